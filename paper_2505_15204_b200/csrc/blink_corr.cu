// CMAC correlator on the 5th-generation tensor cores -- SURVEY 8(f) rank 4 (last item).
// PAPER.md eq. 3 (L98), section 6.2.2 (L172-178): visibilities = voltages of every pair of inputs, conjugate-multiplied
// and accumulated over an integration interval and the averaged fine channels, divided by their number, stored as a
// lower-triangular matrix per (interval, output channel).  DESIGN.md reading R17 / section 5.8.
//
// The paper gives each (baseline, channel, interval) to a warp and reduces across lanes.  Here the operation is what it is
// algebraically -- per (interval t, output channel c) the Hermitian product X X^H of the [A inputs] x [K samples] complex
// int8 matrix -- and runs as int8 tensor-core GEMMs (tcgen05.mma kind::i8, int32 accumulators in TMEM, exact):
//   a row of X in memory is (re0, im0, re1, im1, ...) = the real vector a_i of length 2K,
//   Re S_ij = sum r_i r_j + i_i i_j = a_i . a_j,        Im S_ij = sum i_i r_j - r_i i_j = a_i . b''_j,  b''_j = (-im0, re0, -im1, re1, ...)
// so ONE MMA per K step with A = 128 rows of X and B = [128 rows of X ; their 128 transformed rows] (N = 256) leaves
// Re in TMEM columns 0..127 and Im in columns 128..255 of a 128 x 128 output tile.
//
// One persistent CTA per SM; a unit = (t, c, tile (I, J <= I)) of the lower triangle.  Warp roles:
//   warp 0      TMA producer: [128 rows][128 bytes] boxes of X_J (and X_I when I != J) into a 4-stage ring (128B swizzle);
//               the K tail of an interval and rows beyond A are zero-filled by the tensor map's bounds
//   warps 2-9   build the transformed rows b'' of every stage in shared memory (byte permute + per-byte two's complement; -128 is outside the input contract)
//   warp 1      one lane issues the MMAs (4 K-steps of 32 bytes per stage), tcgen05.commit frees the stage / publishes the tile
//   warps 10-13 epilogue: tcgen05.ld the int32 tile (double-buffered in TMEM: 2 x 256 columns), convert, divide by the number
//               of accumulated samples (one fp32 division, as the oracle), store the triangular matrix
#include "blink_common.cuh"
#include "blink_fft.cuh"
#include "blink_tma.cuh"

namespace blink {

#ifndef BLINK_CORR_XF
#define BLINK_CORR_XF 4
#endif
#ifndef BLINK_CORR_EP
#define BLINK_CORR_EP 4
#endif
#ifndef BLINK_CORR_STAGES
#define BLINK_CORR_STAGES 4
#endif
// measured on the one-second shape (profiles/r2_corr.md): 4 transform warps are as fast as 8; a ring of 3 stages (which is what
// 8 epilogue warps' staging buffers leave room for) costs 12 %, and 8 epilogue warps on top of it give nothing back
constexpr int kCorrXfWarps = BLINK_CORR_XF;                     // warps that build the transformed rows (a multiple of 4)
constexpr int kCorrEpWarps = BLINK_CORR_EP;                     // epilogue warps: 4, or 8 = two per TMEM lane quadrant (column blocks h, h + 2)
constexpr int kCorrThreads = (2 + kCorrXfWarps + kCorrEpWarps) * 32;
constexpr int kCorrStages = BLINK_CORR_STAGES;
static_assert(kCorrXfWarps % 4 == 0 && (kCorrEpWarps == 4 || kCorrEpWarps == 8), "epilogue warp w reads TMEM lane quadrant w % 4");
constexpr int kCorrTile = 128;                                  // rows / columns of an output tile
constexpr int kCorrChunk = 128;                                 // K bytes per stage row (64 complex samples) = swizzle span
constexpr int kCorrRowsBytes = kCorrTile * kCorrChunk;          // 16 KB: 128 rows x 128 bytes
constexpr int kCorrStageBytes = 3 * kCorrRowsBytes;             // X_I | X_J | b''_J
constexpr int kCorrOutBytes = 32 * 33 * 8;                     // per epilogue warp: 32 x 32 complex64, rows padded to 33
constexpr size_t kCorrSmem = (size_t)kCorrStages * kCorrStageBytes + 1024 /* alignment */ + 256 /* barriers */ + kCorrEpWarps * kCorrOutBytes;

struct CorrArgs {
    int A, T, C, n_t, n_avg;
    int n_tiles_side, n_tiles, n_units;
    int nk, last_ksteps;                                        // chunks per (interval, fine channel); K steps of the last one
    int tail_box;                                               // bytes per row staged for the last chunk: 32, 64 or 128
    float norm, rnorm;                                          // n_t * n_avg and its correctly rounded reciprocal
    float2 *vis;
};

__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint64_t *bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// K-major operand tile whose rows are `span` = 128 / 64 / 32 bytes in the swizzle of that width: 8-row groups span x 8 bytes
// apart (SBO), layout type 2 / 4 / 6 (bits 61-63), descriptor version 1 (bit 46); LBO is unused for swizzled K-major tiles
__device__ __forceinline__ uint64_t umma_desc_k(uint32_t saddr, uint32_t span)
{
    const uint64_t type = span == 128u ? 2ull : span == 64u ? 4ull : 6ull;
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | (1ull << 16) | ((uint64_t)(span >> 1) << 32) | (1ull << 46) | (type << 61);
}
__device__ __forceinline__ void umma_i8(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate)
{
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n\t"
        "}\n" ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&r)[32])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
          "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
          "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr)
        : "memory");
}

// unit -> (t, c, I, J): the tiles of one (t, c) are consecutive units, so the CTAs working on them share X through L2;
__device__ __forceinline__ void corr_unit(const CorrArgs &a, int u, int &t, int &c, int &I, int &J)
{
    const int item = u / a.n_tiles;
    int k = u - item * a.n_tiles;
    c = item / a.T;                                             // t fastest: the CTAs running at the same time read
    t = item - c * a.T;                                         // neighbouring intervals of the same rows (DRAM pages)
    I = 0;
    while (k > I) { k -= I + 1; ++I; }                          // row I holds tiles J = 0..I
    J = k;
}

// k-th tile of this CTA: unit blockIdx.x + k gridDim.x
__device__ __forceinline__ bool corr_tile(const CorrArgs &a, int k, int &t, int &c, int &I, int &J)
{
    const long long u = (long long)blockIdx.x + (long long)k * gridDim.x;
    if (u >= a.n_units) return false;
    corr_unit(a, (int)u, t, c, I, J);
    return true;
}

__global__ void __launch_bounds__(kCorrThreads, 1)
corr_kernel(const CorrArgs a, const __grid_constant__ CUtensorMap tmap, const __grid_constant__ CUtensorMap tmap_tail)
{
    extern __shared__ __align__(16) unsigned char corr_smem[];
    const uint32_t base = smem_u32(corr_smem);
    unsigned char *tiles = corr_smem + (((base + 1023u) & ~1023u) - base);         // 1024-byte aligned stage ring
    uint64_t *bars = reinterpret_cast<uint64_t *>(tiles + (size_t)kCorrStages * kCorrStageBytes);
    uint64_t *full_tma = bars, *full_xf = bars + kCorrStages, *empty = bars + 2 * kCorrStages;
    uint64_t *tmem_full = bars + 3 * kCorrStages, *tmem_empty = tmem_full + 2;
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(tmem_empty + 2);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // stage slots (16 KB each): A block X_I | X_J | b''_J
    constexpr uint32_t xj_off = (uint32_t)kCorrRowsBytes;      // X_J, followed by its transformed copy
    // the last chunk of an (interval, fine channel) holds a.tail_box bytes per row (32 / 64: narrower swizzle; 128: like the rest)
    const uint32_t tail_rows_bytes = (uint32_t)kCorrTile * (uint32_t)a.tail_box;

    if (threadIdx.x == 0) {
        for (int s = 0; s < kCorrStages; ++s) {
            mbar_init(&full_tma[s], 1);
            mbar_init(&full_xf[s], kCorrXfWarps * 32);
            mbar_init(&empty[s], 1);
        }
        for (int b = 0; b < 2; ++b) {
            mbar_init(&tmem_full[b], 1);
            mbar_init(&tmem_empty[b], kCorrEpWarps * 32);
        }
        fence_mbar_init();
        tma_prefetch_desc(&tmap);
        tma_prefetch_desc(&tmap_tail);
    }
    if (warp == 1) {                                            // TMEM: all 512 columns (two 128 x 256 int32 accumulators)
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(512) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;
    const int chunks = a.n_avg * a.nk;

    if (warp == 0) {
        if (lane == 0) {
            uint32_t s = 0, ph = 0;                             // ring position as (stage, phase) counters
            int t, c, I, J;
            for (int k = 0; corr_tile(a, k, t, c, I, J); ++k) {
                for (int fi = 0; fi < a.n_avg; ++fi) {          // nested (fine channel, chunk): no divisions in the single-thread loops
                    const int f = c * a.n_avg + fi;
                    for (int kc = 0; kc < a.nk; ++kc) {
                        mbar_wait(&empty[s], ph ^ 1u);
                        unsigned char *st = tiles + (size_t)s * kCorrStageBytes;
                        const bool tail = kc == a.nk - 1;
                        const CUtensorMap *map = tail ? &tmap_tail : &tmap;
                        const uint32_t rows_bytes = tail ? tail_rows_bytes : (uint32_t)kCorrRowsBytes;
                        mbar_expect_tx(&full_tma[s], I == J ? rows_bytes : 2 * rows_bytes);
                        tma_load_4d(st + kCorrRowsBytes, map, &full_tma[s], kc * kCorrChunk, t, J * kCorrTile, f);
                        if (I != J) tma_load_4d(st, map, &full_tma[s], kc * kCorrChunk, t, I * kCorrTile, f);
                        if (++s == kCorrStages) { s = 0; ph ^= 1u; }
                    }
                }
            }
        }
    } else if (warp == 1) {
        if (lane == 0) {
            // instruction descriptor: D = S32 (2 << 4), A = B = signed 8 bit (1 << 7, 1 << 10), both K-major, N = 256, M = 128
            const uint32_t idesc = (2u << 4) | (1u << 7) | (1u << 10) | ((256u >> 3) << 17) | ((128u >> 4) << 24);
            uint32_t s = 0, ph = 0, n = 0;
            int t, c, I, J;
            for (int k = 0; corr_tile(a, k, t, c, I, J); ++k, ++n) {
                const uint32_t b = n & 1u;
                mbar_wait(&tmem_empty[b], ((n >> 1) & 1u) ^ 1u);
                tc_fence_after();
                const uint32_t d = tmem_base + b * 256u;
                uint32_t acc = 0;
                for (int fi = 0; fi < a.n_avg; ++fi) {
                    for (int kc = 0; kc < a.nk; ++kc) {
                        mbar_wait(&full_tma[s], ph);
                        mbar_wait(&full_xf[s], ph);
                        tc_fence_after();
                        const uint32_t st = smem_u32(tiles + (size_t)s * kCorrStageBytes);
                        const bool tail = kc == a.nk - 1;
                        const uint64_t adesc = umma_desc_k(I == J ? st + xj_off : st, tail ? (uint32_t)a.tail_box : 128u);
                        const uint64_t bdesc = umma_desc_k(st + xj_off, tail ? (uint32_t)a.tail_box : 128u);
                        const int ksteps = tail ? a.last_ksteps : 4;
                        for (int ks = 0; ks < ksteps; ++ks) {   // 32 bytes of K per instruction: +2 in units of 16 bytes
                            umma_i8(d, adesc + 2u * ks, bdesc + 2u * ks, idesc, acc);
                            acc = 1u;
                        }
                        tc_commit(&empty[s]);
                        if (++s == kCorrStages) { s = 0; ph ^= 1u; }
                    }
                }
                tc_commit(&tmem_full[b]);
            }
        }
    } else if (warp < 2 + kCorrXfWarps) {
        constexpr int XT = kCorrXfWarps * 32, XV = 1024 / XT;      // threads, 16-byte vectors per thread and full stage
        const int tx = threadIdx.x - 64;
        const int tail_vec = (int)(tail_rows_bytes / 16u);      // 16-byte vectors of a tail block (256 / 512 / 1024)
        auto xf = [](uint32_t w) {                              // bytes (r0, i0, r1, i1) -> (-i0, r0, -i1, r1)
            const uint32_t sw = __byte_perm(w, 0u, 0x2301);                   // (i0, r0, i1, r1)
            // -x = ~x + 1 on bytes 0 and 2: with bytes 1 and 3 cleared first, each +1 carries at most into the
            // cleared byte above it and is masked away
            const uint32_t neg = (~sw & 0x00FF00FFu) + 0x00010001u;
            return (neg & 0x00FF00FFu) | (sw & 0xFF00FF00u);
        };
        uint32_t s = 0, ph = 0;
        int t, c, I, J;
        for (int k = 0; corr_tile(a, k, t, c, I, J); ++k) {
            for (int q = 0, kc = 0; q < chunks; ++q) {
                mbar_wait(&full_tma[s], ph);
                // (re, im) -> (-im, re), same (swizzled) slot of the block that follows X_J: the B operand is 256 rows in a row,
                // so the transformed rows of a narrow tail block start right after its 128 x tail_box bytes
                const int nvec = (kc == a.nk - 1) ? tail_vec : 1024;
                kc = (kc == a.nk - 1) ? 0 : kc + 1;
                const uint4 *src = reinterpret_cast<const uint4 *>(tiles + (size_t)s * kCorrStageBytes + xj_off);
                uint4 *dst = const_cast<uint4 *>(src) + nvec;
                if (nvec == 1024) {
                    uint4 v[XV];
#pragma unroll
                    for (int m = 0; m < XV; ++m) v[m] = src[tx + m * XT];
#pragma unroll
                    for (int m = 0; m < XV; ++m) dst[tx + m * XT] = make_uint4(xf(v[m].x), xf(v[m].y), xf(v[m].z), xf(v[m].w));
                } else {
                    for (int i = tx; i < nvec; i += XT) {
                        const uint4 v = src[i];
                        dst[i] = make_uint4(xf(v.x), xf(v.y), xf(v.z), xf(v.w));
                    }
                }
                fence_proxy_async();                            // generic-proxy writes -> the tensor core's async-proxy reads
                mbar_arrive(&full_xf[s]);
                if (++s == kCorrStages) { s = 0; ph ^= 1u; }
            }
        }
    } else {
        // sum / norm, correctly rounded, without the division subroutine: y = RN(1 / norm) from the host, q = RN(a y), then
        // two residual corrections with exact remainders r = a - norm q (fma) -- the sequence IEEE division itself uses once
        // range checks are out of the way (|a| < 2^31, 1 <= norm <= 66000: no overflow, underflow or subnormals; a = 0 gives +0)
        // on (re, im) pairs with the packed fp32 instructions (mul / fma.f32x2: the same IEEE operations, half the issue slots)
        const float2 nnrm2 = make_float2(-a.norm, -a.norm), rn2 = make_float2(a.rnorm, a.rnorm);
        auto div_norm2 = [nnrm2, rn2](uint32_t vr, uint32_t vi) {
            const float2 x = make_float2((float)(int)vr, (float)(int)vi);
            float2 q = pk_mul(x, rn2);
            q = pk_fma(pk_fma(nnrm2, q, x), rn2, q);
            return pk_fma(pk_fma(nnrm2, q, x), rn2, q);
        };
        const int q4 = warp & 3;                                // TMEM lane quadrant this warp may read
        const int ew = warp - 2 - kCorrXfWarps;                 // epilogue warp; with 8 of them, warps ew and ew + 4 share a quadrant
        const int h = ew >> 2, hstep = kCorrEpWarps / 4;        // and take the 32-column blocks h, h + 2
        float2 *stage = reinterpret_cast<float2 *>(reinterpret_cast<unsigned char *>(tmem_slot + 4) + (size_t)ew * kCorrOutBytes);
        const size_t ntri = (size_t)a.A * (a.A + 1) / 2;
        uint32_t n = 0;
        int t, c, I, J;
        for (int k = 0; corr_tile(a, k, t, c, I, J); ++k, ++n) {
            const uint32_t b = n & 1u;
            mbar_wait(&tmem_full[b], (n >> 1) & 1u);
            tc_fence_after();
            float2 *mat = a.vis + ((size_t)t * a.C + c) * ntri;
            const int nblk = I == J ? q4 + 1 : 4;               // 32-column blocks at or below the diagonal for some row of this warp
            for (int cj = h; cj < nblk; cj += hstep) {
                uint32_t re[32], im[32];
                const uint32_t taddr = tmem_base + ((uint32_t)(q4 * 32) << 16) + b * 256u + (uint32_t)cj * 32u;
                tmem_ld32(taddr, re);
                tmem_ld32(taddr + 128u, im);
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                // a lane holds 32 columns of ONE row; the matrix wants a warp to write 32 consecutive columns of a row
                // (256 contiguous bytes = 8 full sectors per store instead of 32 partial ones): transpose through shared memory
#pragma unroll
                for (int k = 0; k < 32; ++k) stage[lane * 33 + k] = div_norm2(re[k], im[k]);
                __syncwarp();
                const int gj = J * kCorrTile + cj * 32 + lane;
                const int gi0 = I * kCorrTile + q4 * 32;
                float2 *dst = mat + (size_t)gi0 * (gi0 + 1) / 2 + gj;   // row gi starts gi (gi + 1) / 2 entries in: +gi + 1 per row
#pragma unroll 8
                for (int r = 0; r < 32; ++r) {
                    const int gi = gi0 + r;
                    if (gi < a.A && gj <= gi) *dst = stage[r * 33 + lane];
                    dst += gi + 1;
                }
                __syncwarp();
            }
            tc_fence_before();
            mbar_arrive(&tmem_empty[b]);
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512) : "memory");
    }
}


}  // namespace blink

using namespace blink;

extern "C" int blink_correlate(const int8_t *volt, int F, int A, int Ns, int n_t, int n_avg, blink_c64 *vis, void *stream)
{
    if (!volt || !vis || F < 1 || A < 1 || Ns < 1 || n_t < 1 || n_avg < 1) return BLINK_ERR_INVALID_ARG;
    if (Ns % n_t != 0 || F % n_avg != 0) return BLINK_ERR_INVALID_ARG;
    if (!aligned16(volt) || (reinterpret_cast<uintptr_t>(vis) & 7u)) return BLINK_ERR_INVALID_ARG;
    // tensor-map strides are multiples of 16 bytes (n_t % 8), a box row must fit the interval (n_t >= 64), and int32 sums
    // must hold: n_t n_avg 2 127^2 < 2^31
    if (n_t % 8 != 0 || n_t < 64 || A > 4096 || (long long)n_t * n_avg > 66000) return BLINK_ERR_UNSUPPORTED;
    int rc = ensure_device();
    if (rc != BLINK_OK) return rc;
    CorrArgs a{};
    a.A = A; a.T = Ns / n_t; a.C = F / n_avg; a.n_t = n_t; a.n_avg = n_avg;
    a.n_tiles_side = (A + kCorrTile - 1) / kCorrTile;
    a.n_tiles = a.n_tiles_side * (a.n_tiles_side + 1) / 2;
    const long long units = (long long)a.T * a.C * a.n_tiles;
    if (units > 0x7fffffffLL) return BLINK_ERR_UNSUPPORTED;
    a.n_units = (int)units;
    const int kbytes = 2 * n_t;
    a.nk = (kbytes + kCorrChunk - 1) / kCorrChunk;
    a.last_ksteps = (kbytes - (a.nk - 1) * kCorrChunk + 31) / 32;
    a.norm = (float)((long long)n_t * n_avg);
    a.rnorm = (float)(1.0 / (double)((long long)n_t * n_avg));
    a.vis = reinterpret_cast<float2 *>(vis);
    // the K tail of an (interval, fine channel): 2 n_t = (nk - 1) 128 + tail bytes.  A tail of at most 32 / 64 bytes is staged as
    // 32 / 64-byte rows (tensor map and UMMA descriptor in the swizzle of that width): the paper's 20 ms interval is 400 bytes =
    // 3 x 128 + 16, and a fourth full-width chunk would stage and transform 128 bytes per row for 16 valid ones
    const int tail_bytes = kbytes - (a.nk - 1) * kCorrChunk;
    a.tail_box = tail_bytes <= 32 ? 32 : tail_bytes <= 64 ? 64 : 128;
    CUtensorMap tmap, tmap_tail;
    // volt as bytes: [F][A][T][2 n_t], innermost first {2 n_t, T, A, F}; a box = 128 bytes x 1 interval x 128 inputs x 1 channel
    const uint32_t box_rows = (uint32_t)kCorrTile;
    const uint64_t dims[4] = {(uint64_t)kbytes, (uint64_t)a.T, (uint64_t)A, (uint64_t)F};
    const uint64_t strides[3] = {(uint64_t)kbytes, (uint64_t)Ns * 2, (uint64_t)A * Ns * 2};
    const uint32_t box[4] = {(uint32_t)kCorrChunk, 1u, box_rows, 1u};
    const uint32_t box_tail[4] = {(uint32_t)a.tail_box, 1u, box_rows, 1u};
    if (encode_tensor_map_4d_u8(&tmap, volt, dims, strides, box, kCorrChunk) != 0 ||
        encode_tensor_map_4d_u8(&tmap_tail, volt, dims, strides, box_tail, a.tail_box) != 0) {
        set_error_text("cuTensorMapEncodeTiled failed (correlator voltages)");
        return BLINK_ERR_CUDA;
    }
    int ctas = sm_count() > 0 ? sm_count() : 148;
    BLINK_CUDA_TRY(cudaFuncSetAttribute(corr_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kCorrSmem));
    if (ctas > a.n_units) ctas = a.n_units;
    corr_kernel<<<ctas, kCorrThreads, kCorrSmem, static_cast<cudaStream_t>(stream)>>>(a, tmap, tmap_tail);
    BLINK_LAUNCH_CHECK("corr_kernel");
    return BLINK_OK;
}
