// Fused imaging kernel: visibilities -> dirty images, the uv grid is never materialised.
//
// What makes this possible:
//   * the gridded plane is Hermitian, G[-v][-u] = conj(G[v][u]) (every sample is gridded with its conjugate,
//     reading R1), so only the half plane u >= 0 is gridded: N x N/2 cells (column u = N/2 is always empty, R4);
//   * pass 1 transforms that half plane along v, one u-column at a time, in shared memory, and leaves
//     H[u][ky] (N/2 x N complex64) in a per-CTA scratch in global memory (L2-resident at N = 512);
//   * pass 2 turns row pairs (ky, ky+1) into TWO real image rows with ONE N-point complex transform:
//     Z[n] = S1[n] + i S2[n] (n < N/2), Z[N-n] = conj(S1[n]) + i conj(S2[n]);  Re z = row ky, Im z = row ky+1.
//     Its input tiles [KY ky][N/2 u] are TRANSPOSED reads of the scratch, staged by TMA (128B-swizzled),
//     double-buffered behind an mbarrier pipeline; the fftshift (index XOR N/2), the 1/W normalisation and the
//     real-part extraction are part of the store.
// One persistent CTA per SM walks over (t,c) work items; per item it computes the cell indices once (bit-exact
// twin of the oracle), bins the samples by u-tile with a counting sort in shared memory, and reuses the bins
// for all P polarisations.  PAPER.md L190-194 (gridding, batched inverse 2D FFT, shift); L150 (fp32).
#include <algorithm>

#include "blink_common.cuh"
#include "blink_fft.cuh"
#include "blink_tma.cuh"

namespace blink {

constexpr int kFusedThreads = 512;

template <int N>
struct FusedCfg {
    static constexpr int H = N / 2;
    static constexpr int TG = N / kE;                          // threads per transform
    static constexpr int G = kFusedThreads / TG;               // groups per CTA
    static constexpr int KU = 2 * G;                           // u-columns per pass-1 tile (2 per group)
    static constexpr int NT = H / KU;                          // pass-1 tiles in the half plane
    static constexpr int SLOTS = N;                            // column length (XOR-swizzled, no padding)
    static constexpr int KY = (8192 / N) < 16 ? (8192 / N) : 16;   // ky rows per pass-2 stage
    static constexpr int ROWB = KY * 8;                        // stage row bytes (= TMA swizzle span)
    static constexpr int PAIRS = KY / 2;
    static constexpr int BOX_ROWS = H < 256 ? H : 256;
    static constexpr int NBOX = H / BOX_ROWS;
    static constexpr int STAGE_BYTES = H * ROWB;
    static constexpr int NIT = N / KY;                         // pass-2 stages per image
    static constexpr int LOG_TILE = 13;                        // KU * N == 8192 cells per tile
    static_assert(KU * N == 8192, "tile is 8192 cells");
    static_assert(PAIRS <= G, "one pair per group per stage");
};

struct FusedArgs {
    const float2 *vis; const float *uvw_m;
    int T, C, P, B, weighting;
    int tc0, ntc, c_base;
    float *image; float *wsum; int32_t *cell_idx;              // indexed by absolute tc / image
    float2 *scratch;                                           // [gridDim.x][H][N]
    const float *su; const float *sv; const uint32_t *sb;      // per timestep: baselines sorted by |u| (presort_kernel)
    const float2 *tw;
};

struct ExchangePadded2 {
    float2 *c0, *c1;
    __device__ __forceinline__ void put(int w, const float2 (&v)[2]) const
    {
        const int o = xsw(w);
        c0[o] = v[0];
        c1[o] = v[1];
    }
    __device__ __forceinline__ void get(int w, float2 (&v)[2]) const
    {
        const int o = xsw(w);
        v[0] = c0[o];
        v[1] = c1[o];
    }
};

template <int N>
__host__ __device__ constexpr size_t fused_region_bytes(bool uniform)
{
    using Cfg = FusedCfg<N>;
    const size_t p1 = (size_t)Cfg::KU * Cfg::SLOTS * (uniform ? 12 : 8);
    const size_t p2 = 2 * (size_t)Cfg::STAGE_BYTES + (size_t)Cfg::G * Cfg::SLOTS * 8;
    return p1 > p2 ? p1 : p2;
}
// shared memory: vis row [B] float2 | tile offsets [NT+1] | owner ids [KU*SLOTS] u16 | pad to 1024 |
//                union(pass-1 tile (+counts), pass-2 stages + exchange) | mbarriers
template <int N>
__host__ __device__ constexpr size_t fused_front_bytes(int B)
{
    using Cfg = FusedCfg<N>;
    return (size_t)B * 8 + (size_t)(Cfg::NT + 1) * 4 + (size_t)Cfg::KU * Cfg::SLOTS * 2;
}
template <int N>
static size_t fused_smem_bytes(int B, bool uniform)
{
    return align_up(fused_front_bytes<N>(B), 1024) + fused_region_bytes<N>(uniform) + 1024 + 64;
}

// ------------------------------------------------------------------------------------------ presort
// One CTA per timestep: sorts the baselines by |u_m| (bitonic sort of (key, index) pairs in shared memory).
// For every channel the u-tile of a sample, rint(|u_m| * s_c) / KU, is then non-decreasing along the sorted
// order (fp32 multiply by s_c > 0 and rint are monotone), so a tile's samples are ONE contiguous range and no
// per-image binning is needed.  The sample is stored folded into the half plane u >= 0:
//   su = |u_m|, sv = (u_m < 0 ? -v_m : v_m), sb = b | (u_m < 0) << 31   (bit 31: use conj(V) at (-u,-v)).
// rint(-x) = -rint(x) and (-a) * s = -(a * s) exactly, so the folded cell is exactly the mirror cell (R1, R2).
constexpr int kSortThreads = 1024;
constexpr int kSortMaxB = 16384;

__global__ void __launch_bounds__(kSortThreads)
presort_kernel(const float *__restrict__ uvw_m, int B, int np2, float *__restrict__ su, float *__restrict__ sv,
               uint32_t *__restrict__ sb)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float *key = reinterpret_cast<float *>(smem_raw);
    uint32_t *idx = reinterpret_cast<uint32_t *>(smem_raw) + np2;
    const int t = blockIdx.x;
    const float *uvw = uvw_m + (size_t)t * B * 3;
    for (int i = threadIdx.x; i < np2; i += kSortThreads) {
        float k = __int_as_float(0x7f800000);                               // +inf: padding and NaN sort last
        if (i < B) {
            const float a = fabsf(uvw[3 * i]);
            if (a == a) k = a;
        }
        key[i] = k;
        idx[i] = (uint32_t)i;
    }
    __syncthreads();
    for (int k = 2; k <= np2; k <<= 1) {
        for (int j = k >> 1; j > 0; j >>= 1) {
            for (int i = threadIdx.x; i < np2; i += kSortThreads) {
                const int x = i ^ j;
                if (x > i) {
                    const float a = key[i], b = key[x];
                    const uint32_t ia = idx[i], ib = idx[x];
                    const bool gt = (a > b) || (a == b && ia > ib);         // (key, index) order: padding stays last
                    const bool up = (i & k) == 0;
                    if (gt == up) {
                        key[i] = b; key[x] = a;
                        idx[i] = ib; idx[x] = ia;
                    }
                }
            }
            __syncthreads();
        }
    }
    for (int i = threadIdx.x; i < B; i += kSortThreads) {
        const uint32_t b = idx[i];                                          // < B: real samples sort before the padding
        const float u = uvw[3 * b], v = uvw[3 * b + 1];
        const bool neg = u < 0.0f;
        su[(size_t)t * B + i] = fabsf(u);
        sv[(size_t)t * B + i] = neg ? -v : v;
        sb[(size_t)t * B + i] = b | (neg ? 0x80000000u : 0u);
    }
}

// ------------------------------------------------------------------------------------------ fused kernel
template <int N>
__global__ void __launch_bounds__(kFusedThreads, 1)
fused_image_kernel(const FusedArgs a, const __grid_constant__ ScaleBlock sc, const __grid_constant__ CUtensorMap tmap)
{
    using Cfg = FusedCfg<N>;
    constexpr int H = Cfg::H, TG = Cfg::TG, KU = Cfg::KU, NT = Cfg::NT, SLOTS = Cfg::SLOTS;
    constexpr int IT = 2;                                      // samples per thread per accumulation round
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    const bool uniform = a.weighting == BLINK_W_UNIFORM;
    const int B = a.B;

    // ---- shared memory carve-up (pointer arithmetic on the array keeps every access in the shared window) ----
    float2 *visrow = reinterpret_cast<float2 *>(smem_raw);                     // [B]
    uint32_t *toff = reinterpret_cast<uint32_t *>(smem_raw + (size_t)B * 8);   // [NT+1]
    unsigned short *own = reinterpret_cast<unsigned short *>(smem_raw + (size_t)B * 8 + (size_t)(NT + 1) * 4);
    const uint32_t front = (uint32_t)fused_front_bytes<N>(B);
    const uint32_t base_addr = smem_u32(smem_raw);
    unsigned char *region = smem_raw + (((base_addr + front + 1023u) & ~1023u) - base_addr);
    float2 *tile = reinterpret_cast<float2 *>(region);                         // pass 1: [KU][SLOTS]
    uint32_t *cnt = reinterpret_cast<uint32_t *>(region + (size_t)KU * SLOTS * 8);   // pass 1 (uniform)
    unsigned char *stage = region;                                             // pass 2: [2][STAGE_BYTES]
    float2 *xbuf = reinterpret_cast<float2 *>(region + 2 * (size_t)Cfg::STAGE_BYTES);   // pass 2: [G][SLOTS]
    uint64_t *bars = reinterpret_cast<uint64_t *>(region + fused_region_bytes<N>(uniform));   // full[2]
    __shared__ int s_nin, s_occ;

    const int g = threadIdx.x / TG;
    const int tid = threadIdx.x % TG;
    const int lane = threadIdx.x & 31;
    float2 *scratch = a.scratch + (size_t)blockIdx.x * H * N;
    // barrier over ONE transform group (its columns / exchange buffer are private to it)
    auto sync = [g] {
        if constexpr (TG == 32) __syncwarp();
        else if constexpr (Cfg::G <= 15) asm volatile("bar.sync %0, %1;" ::"r"(g + 1), "r"(TG) : "memory");
        else __syncthreads();
    };
    const float lim = (float)(H - 1);

    if (threadIdx.x == 0) {
        mbar_init(&bars[0], 1);
        mbar_init(&bars[1], 1);
        fence_mbar_init();
        tma_prefetch_desc(&tmap);
    }
    uint32_t uses0 = 0, uses1 = 0;                                             // completed phases per barrier
    Twiddles<N> twr;
    twr.init(tid, a.tw);
    __syncthreads();

    for (int tc = a.tc0 + blockIdx.x; tc < a.tc0 + a.ntc; tc += gridDim.x) {
        const int t = tc / a.C, c = tc - t * a.C;
        const float s = sc.s[c - a.c_base];
        const float *su = a.su + (size_t)t * B;
        const float *sv = a.sv + (size_t)t * B;
        const uint32_t *sb = a.sb + (size_t)t * B;

        // u-tile of sorted sample j for this channel (NT = beyond the grid)
        auto tile_of = [&](int j) -> int {
            const float xr = rintf(__fmul_rn(__ldg(su + j), s));
            return (xr <= lim) ? (int)xr / KU : NT;
        };
        // ---- tile boundaries: toff[tl] = first sorted sample whose tile is >= tl -------------------------
        for (int i = threadIdx.x; i <= NT; i += kFusedThreads) toff[i] = (uint32_t)B;
        if (threadIdx.x == 0) { s_nin = 0; s_occ = 0; }
        __syncthreads();
        for (int j = threadIdx.x; j < B; j += kFusedThreads) {
            const int tj = tile_of(j);
            const int tp = j > 0 ? tile_of(j - 1) : -1;
            for (int tl = tp + 1; tl <= tj; ++tl) toff[tl] = (uint32_t)j;
        }
        // ---- optional output: cell index of every baseline, in baseline order (a1) -----------------------
        if (a.cell_idx) {
            const float *uvw = a.uvw_m + (size_t)t * B * 3;
            for (int b = threadIdx.x; b < B; b += kFusedThreads)
                a.cell_idx[(size_t)tc * B + b] = cell_of(uvw[3 * b], uvw[3 * b + 1], s, N, H);
        }
        __syncthreads();
        const int j_end = (int)toff[NT];                                        // samples [0, j_end) have |iu| <= H-1
        const int n_tiles = j_end > 0 ? tile_of(j_end - 1) + 1 : 0;
        const int ulim = n_tiles * KU;                                          // scratch rows written by pass 1
        const int n_box = (ulim + Cfg::BOX_ROWS - 1) / Cfg::BOX_ROWS;
        float wsum_val = 0.f;

        for (int p = 0; p < a.P; ++p) {
            const size_t img_idx = (size_t)tc * a.P + p;
            float *img = a.image + img_idx * N * N;
            // ---- stage this image's visibility row in shared memory (coalesced, 16-byte loads when aligned) ----
            __syncthreads();                                                    // previous readers of visrow are done
            {
                const float2 *vrow = a.vis + img_idx * B;
                if (((img_idx * (size_t)B) & 1) == 0) {
                    const float4 *src = reinterpret_cast<const float4 *>(vrow);
                    float4 *dst = reinterpret_cast<float4 *>(visrow);
                    for (int i = threadIdx.x; i < B / 2; i += kFusedThreads) dst[i] = __ldcs(src + i);
                    if ((B & 1) && threadIdx.x == 0) visrow[B - 1] = vrow[B - 1];
                } else {
                    for (int i = threadIdx.x; i < B; i += kFusedThreads) visrow[i] = vrow[i];
                }
            }
            int my_occ = 0, my_in = 0;
            // ================= pass 1: grid a u-tile in shared memory, transform its columns along v =====
            for (int tl = 0; tl < n_tiles; ++tl) {
                __syncthreads();                                                // previous users of the region are done
                for (int i = threadIdx.x; i < KU * SLOTS / 2; i += kFusedThreads)
                    reinterpret_cast<float4 *>(tile)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
                if (uniform)
                    for (int i = threadIdx.x; i < KU * SLOTS / 4; i += kFusedThreads)
                        reinterpret_cast<uint4 *>(cnt)[i] = make_uint4(0u, 0u, 0u, 0u);
                const int k0 = (int)toff[tl], k1 = (int)toff[tl + 1];
                // accumulate in rounds of IT * 512 samples.  Shared-memory float atomics are CAS loops (~2 cycles per
                // lane), and cells rarely collide, so: (1) every sample writes its id into the owner array, (2) the
                // sample whose id survived adds with plain loads/stores, (3) only the losers (and the rare second
                // half of an iu == 0 sample) use atomics.
                for (int r0 = k0; r0 < k1; r0 += IT * kFusedThreads) {
                    int o[IT], o2[IT];
                    float2 v[IT];
#pragma unroll
                    for (int m = 0; m < IT; ++m) {
                        o[m] = -1; o2[m] = -1;
                        const int j = r0 + m * kFusedThreads + threadIdx.x;
                        if (j < k1) {
                            const float xr = rintf(__fmul_rn(__ldg(su + j), s));
                            const float yr = rintf(__fmul_rn(__ldg(sv + j), s));
                            if (fabsf(yr) <= lim) {                              // NaN fails; |iu| <= H-1 by construction
                                const int iu = (int)xr, iv = (int)yr;
                                const uint32_t bb = __ldg(sb + j);
                                float2 vv = visrow[bb & 0x7fffffffu];
                                if (bb >> 31) vv.y = -vv.y;
                                v[m] = vv;
                                const int ul = iu - tl * KU, row = iv + H;
                                o[m] = ul * SLOTS + xsw(row);
                                if (iu == 0) { const int row2 = H - iv; o2[m] = xsw(row2); }
                                ++my_in;
                            }
                        }
                    }
                    __syncthreads();                                            // tile zeroed / previous round complete
#pragma unroll
                    for (int m = 0; m < IT; ++m)
                        if (o[m] >= 0) own[o[m]] = (unsigned short)(m * kFusedThreads + threadIdx.x);
                    __syncthreads();
                    bool lose[IT];
#pragma unroll
                    for (int m = 0; m < IT; ++m) {
                        lose[m] = false;
                        if (o[m] >= 0) {
                            if (own[o[m]] == (unsigned short)(m * kFusedThreads + threadIdx.x)) {
                                float2 q = tile[o[m]];
                                q.x += v[m].x; q.y += v[m].y;
                                tile[o[m]] = q;
                                if (uniform) cnt[o[m]] += 1u;
                            } else {
                                lose[m] = true;
                            }
                        }
                    }
                    __syncthreads();
#pragma unroll
                    for (int m = 0; m < IT; ++m) {
                        if (lose[m]) {
                            atomicAdd(&tile[o[m]].x, v[m].x);
                            atomicAdd(&tile[o[m]].y, v[m].y);
                            if (uniform) atomicAdd(&cnt[o[m]], 1u);
                        }
                        if (o2[m] >= 0) {                                       // iu == 0: the conjugate lies in column 0 too
                            atomicAdd(&tile[o2[m]].x, v[m].x);
                            atomicAdd(&tile[o2[m]].y, -v[m].y);
                            if (uniform) atomicAdd(&cnt[o2[m]], 1u);
                        }
                    }
                }
                __syncthreads();
                if (uniform) {                                                  // a3: divide by the cell count
                    for (int i = threadIdx.x; i < KU * SLOTS; i += kFusedThreads) {
                        const uint32_t cc = cnt[i];
                        if (cc) {
                            float2 q = tile[i];
                            q.x = __fdiv_rn(q.x, (float)cc); q.y = __fdiv_rn(q.y, (float)cc);
                            tile[i] = q;
                            // occupied cells of the FULL plane: the mirror image of a u > 0 cell is occupied too
                            my_occ += (tl == 0 && i < SLOTS) ? 1 : 2;
                        }
                    }
                    __syncthreads();
                }
                {
                    float2 *c0 = tile + (size_t)(2 * g) * SLOTS, *c1 = c0 + SLOTS;
                    ExchangePadded2 xch{c0, c1};
                    float2 v[2][kE];
#pragma unroll
                    for (int e = 0; e < kE; ++e) {                              // transform index n lives in centred row n ^ H
                        const int r = tid + (e ^ (kE / 2)) * TG;
                        v[0][e] = c0[xsw(r)];
                        v[1][e] = c1[xsw(r)];
                    }
                    fft_inverse<N, 2>(v, tid, xch, twr, sync);
                    float2 *d0 = scratch + (size_t)(tl * KU + 2 * g) * N, *d1 = d0 + N;
#pragma unroll
                    for (int e = 0; e < kE; ++e) {
                        d0[tid + e * TG] = v[0][e];
                        d1[tid + e * TG] = v[1][e];
                    }
                }
            }
            if (p == 0) {                                                       // weight sum (a3), shared by the P planes
#pragma unroll
                for (int d = 16; d > 0; d >>= 1) {
                    my_occ += __shfl_xor_sync(0xffffffffu, my_occ, d);
                    my_in += __shfl_xor_sync(0xffffffffu, my_in, d);
                }
                if (lane == 0) { atomicAdd(&s_occ, my_occ); atomicAdd(&s_nin, my_in); }
            }
            // scratch stores (generic proxy) must be visible to the TMA loads (async proxy) below
            __threadfence();
            asm volatile("fence.proxy.async;" ::: "memory");
            __syncthreads();
            if (p == 0) wsum_val = uniform ? (float)s_occ : (float)(2 * s_nin);
            if (wsum_val == 0.f) {                                              // W = 0: zero image (uniform over the CTA)
                for (int i = threadIdx.x; i < N * N / 4; i += kFusedThreads)
                    reinterpret_cast<float4 *>(img)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
                continue;
            }
            const float inv_w = 1.0f / wsum_val;

            // ================= pass 2: row pairs -> two real image rows per transform ===================
            auto issue = [&](int it) {                                          // thread 0 only
                uint64_t *bar = &bars[it & 1];
                unsigned char *dst = stage + (size_t)(it & 1) * Cfg::STAGE_BYTES;
                mbar_expect_tx(bar, (uint32_t)(n_box * Cfg::BOX_ROWS * Cfg::ROWB));
                for (int bx = 0; bx < n_box; ++bx)
                    tma_load_3d(dst + (size_t)bx * Cfg::BOX_ROWS * Cfg::ROWB, &tmap, bar, 2 * it * Cfg::KY,
                                bx * Cfg::BOX_ROWS, (int)blockIdx.x);
            };
            if (threadIdx.x == 0) { issue(0); issue(1); }
            for (int it = 0; it < Cfg::NIT; ++it) {
                const int sbuf = it & 1;
                mbar_wait(&bars[sbuf], (sbuf ? uses1 : uses0) & 1u);
                if (sbuf) ++uses1; else ++uses0;
                float2 z[1][kE];
                if (g < Cfg::PAIRS) {
                    ExchangeTilePair<Cfg::ROWB> st{stage + (size_t)sbuf * Cfg::STAGE_BYTES, g};
#pragma unroll
                    for (int e = 0; e < kE / 2; ++e) {                          // n = u < H: S1 + i S2
                        const int u = tid + e * TG;
                        float4 q = make_float4(0.f, 0.f, 0.f, 0.f);
                        if (u < ulim) q = *st.at_row(u);
                        z[0][e] = make_float2(q.x - q.w, q.y + q.z);
                    }
#pragma unroll
                    for (int e = kE / 2; e < kE; ++e) {                         // n > H: conj(S1[N-n]) + i conj(S2[N-n])
                        const int u = N - (tid + e * TG);                       // in [1, H]; u == H is the empty Nyquist column
                        float4 q = make_float4(0.f, 0.f, 0.f, 0.f);
                        if (u < ulim && u < H) q = *st.at_row(u);
                        z[0][e] = make_float2(q.x + q.w, q.z - q.y);
                    }
                }
                __syncthreads();                                                // everyone has read this stage buffer
                if (threadIdx.x == 0 && it + 2 < Cfg::NIT) {
                    fence_proxy_async();
                    issue(it + 2);
                }
                if (g < Cfg::PAIRS) {
                    ExchangePadded1 xch{xbuf + (size_t)g * SLOTS};
                    fft_inverse<N, 1>(z, tid, xch, twr, sync);
                    const int ky = it * Cfg::KY + 2 * g;
                    float *r0 = img + (size_t)(ky ^ H) * N, *r1 = img + (size_t)((ky + 1) ^ H) * N;
#pragma unroll
                    for (int e = 0; e < kE; ++e) {
                        const int x = (tid + e * TG) ^ H;
                        __stcs(r0 + x, z[0][e].x * inv_w);
                        __stcs(r1 + x, z[0][e].y * inv_w);
                    }
                }
            }
        }
        if (threadIdx.x == 0) a.wsum[tc] = wsum_val;
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------ counts (optional output)
__global__ void counts_kernel(const float *__restrict__ uvw_m, const ScaleBlock sc, int C, int B, int n, int tc0, int c_base,
                              uint32_t *__restrict__ counts)
{
    const int tc = tc0 + blockIdx.y;
    const int t = tc / C, c = tc - t * C;
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    const float *p = uvw_m + ((size_t)t * B + b) * 3;
    const int cell = cell_of(p[0], p[1], sc.s[c - c_base], n, n / 2);
    if (cell < 0) return;
    uint32_t *dst = counts + (size_t)tc * n * n;
    atomicAdd(&dst[cell], 1u);
    atomicAdd(&dst[mirror_of(cell, n)], 1u);
}

// ------------------------------------------------------------------------------------------ host
bool fused_supported(int P, int B, int n_pix, int weighting)
{
    (void)P;
    if (B > kSortMaxB) return false;
    const bool uni = weighting == BLINK_W_UNIFORM;
    size_t need;
    switch (n_pix) {
        case 256: need = fused_smem_bytes<256>(B, uni); break;
        case 512: need = fused_smem_bytes<512>(B, uni); break;
        case 1024: need = fused_smem_bytes<1024>(B, uni); break;
        case 2048: need = fused_smem_bytes<2048>(B, uni); break;
        case 4096: need = fused_smem_bytes<4096>(B, uni); break;
        default: return false;
    }
    return need <= 227 * 1024;
}

static size_t sort_bytes(int T, int B) { return align_up((size_t)T * B * 4, 256) * 3; }
size_t fused_workspace_bytes(int T, int B, int n_pix, int ctas)
{
    return sort_bytes(T, B) + (size_t)ctas * (n_pix / 2) * n_pix * sizeof(float2);
}
int fused_default_ctas() { return sm_count() > 0 ? sm_count() : 148; }

// sub-ranges of flattened (t,c) that stay inside one block of <= 1024 channels
template <class F>
static int for_channel_blocks(int C, int tc0, int ntc, const double *freqs_hz, int n_pix, double pixscale_rad, F &&f)
{
    int tc = tc0;
    const int tc_end = tc0 + ntc;
    while (tc < tc_end) {
        const int t = tc / C, c = tc - t * C;
        const int c_base = (c / 1024) * 1024;
        const int c_lim = c_base + 1024 < C ? c_base + 1024 : C;
        int end = (C <= 1024) ? tc_end : t * C + c_lim;
        if (end > tc_end) end = tc_end;
        ScaleBlock sc;
        for (int k = 0; k < 1024; ++k) sc.s[k] = (c_base + k < C) ? scale_for(freqs_hz[c_base + k], n_pix, pixscale_rad) : 0.f;
        int rc = f(tc, end - tc, c_base, sc);
        if (rc != BLINK_OK) return rc;
        tc = end;
    }
    return BLINK_OK;
}

template <int N>
static int launch_fused(const FusedArgs &base, const double *freqs_hz, double pixscale_rad, void *workspace,
                        size_t workspace_bytes, cudaStream_t st)
{
    using Cfg = FusedCfg<N>;
    const size_t per_cta = (size_t)Cfg::H * N * sizeof(float2);
    const size_t sortb = sort_bytes(base.T, base.B);
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u) || workspace_bytes < sortb + per_cta)
        return BLINK_ERR_WORKSPACE;
    int ctas = option(BLINK_OPT_FUSED_CTAS);
    if (ctas <= 0) ctas = fused_default_ctas();
    ctas = (int)std::min<size_t>((size_t)ctas, (workspace_bytes - sortb) / per_cta);
    // workspace: su | sv | sb (baselines of every timestep sorted by |u|) | per-CTA scratch
    unsigned char *wsp = static_cast<unsigned char *>(workspace);
    float *su = reinterpret_cast<float *>(wsp);
    float *sv = reinterpret_cast<float *>(wsp + sortb / 3);
    uint32_t *sb = reinterpret_cast<uint32_t *>(wsp + 2 * (sortb / 3));
    void *scratch = wsp + sortb;
    {
        int np2 = 1;
        while (np2 < base.B) np2 <<= 1;
        const size_t ssm = (size_t)np2 * 8;
        BLINK_CUDA_TRY(cudaFuncSetAttribute(presort_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ssm));
        presort_kernel<<<base.T, kSortThreads, ssm, st>>>(base.uvw_m, base.B, np2, su, sv, sb);
        BLINK_LAUNCH_CHECK("presort_kernel");
    }
    const size_t smem = fused_smem_bytes<N>(base.B, base.weighting == BLINK_W_UNIFORM);
    BLINK_CUDA_TRY(cudaFuncSetAttribute(fused_image_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    CUtensorMap tmap;
    // scratch viewed as float32 [ctas][H rows (u)][2N (ky re/im)]; boxes of [BOX_ROWS u][KY ky]
    int rc = encode_tensor_map_3d_f32(&tmap, scratch, 2ull * N, (uint64_t)Cfg::H, (uint64_t)ctas, (uint64_t)N * 8,
                                      (uint64_t)Cfg::H * N * 8, 2 * Cfg::KY, Cfg::BOX_ROWS, 1,
                                      Cfg::ROWB >= 32 ? Cfg::ROWB : 0);
    if (rc != 0) { set_error_text("cuTensorMapEncodeTiled failed (fused scratch)"); return BLINK_ERR_CUDA; }
    return for_channel_blocks(base.C, base.tc0, base.ntc, freqs_hz, N, pixscale_rad,
                              [&](int tc0, int ntc, int c_base, const ScaleBlock &sc) -> int {
                                  FusedArgs a = base;
                                  a.tc0 = tc0; a.ntc = ntc; a.c_base = c_base;
                                  a.scratch = static_cast<float2 *>(scratch);
                                  a.su = su; a.sv = sv; a.sb = sb;
                                  a.tw = twiddle_table();
                                  const int grid = ntc < ctas ? ntc : ctas;
                                  fused_image_kernel<N><<<grid, kFusedThreads, smem, st>>>(a, sc, tmap);
                                  BLINK_LAUNCH_CHECK("fused_image_kernel");
                                  return (int)BLINK_OK;
                              });
}

int fused_image(const float2 *vis, const float *uvw_m, const double *freqs_hz, double pixscale_rad, int T, int C, int P,
                int B, int n_pix, int weighting, int tc0, int ntc, float *image, float *wsum, int32_t *cell_idx,
                void *workspace, size_t workspace_bytes, cudaStream_t st)
{
    FusedArgs a{};
    a.vis = vis; a.uvw_m = uvw_m; a.T = T; a.C = C; a.P = P; a.B = B; a.weighting = weighting;
    a.tc0 = tc0; a.ntc = ntc; a.image = image; a.wsum = wsum; a.cell_idx = cell_idx;
    switch (n_pix) {
        case 256: return launch_fused<256>(a, freqs_hz, pixscale_rad, workspace, workspace_bytes, st);
        case 512: return launch_fused<512>(a, freqs_hz, pixscale_rad, workspace, workspace_bytes, st);
        case 1024: return launch_fused<1024>(a, freqs_hz, pixscale_rad, workspace, workspace_bytes, st);
        case 2048: return launch_fused<2048>(a, freqs_hz, pixscale_rad, workspace, workspace_bytes, st);
        case 4096: return launch_fused<4096>(a, freqs_hz, pixscale_rad, workspace, workspace_bytes, st);
        default: return BLINK_ERR_UNSUPPORTED;
    }
}

int counts_only(const float *uvw_m, const double *freqs_hz, double pixscale_rad, int T, int C, int B, int n_pix, int tc0,
                int ntc, uint32_t *counts, cudaStream_t st)
{
    (void)T;
    const size_t n2 = (size_t)n_pix * n_pix;
    BLINK_CUDA_TRY(cudaMemsetAsync(counts + (size_t)tc0 * n2, 0, (size_t)ntc * n2 * sizeof(uint32_t), st));
    return for_channel_blocks(C, tc0, ntc, freqs_hz, n_pix, pixscale_rad,
                              [&](int s0, int m, int c_base, const ScaleBlock &sc) -> int {
                                  for (int y0 = 0; y0 < m; y0 += 65535) {
                                      const int my = m - y0 < 65535 ? m - y0 : 65535;
                                      dim3 grid((B + 255) / 256, my);
                                      counts_kernel<<<grid, 256, 0, st>>>(uvw_m, sc, C, B, n_pix, s0 + y0, c_base, counts);
                                      BLINK_LAUNCH_CHECK("counts_kernel");
                                  }
                                  return (int)BLINK_OK;
                              });
}

}  // namespace blink
