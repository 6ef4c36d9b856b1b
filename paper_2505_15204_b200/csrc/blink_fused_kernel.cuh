// Fused imaging kernel (template) and its launcher, shared by blink_fused.cu (nearest-cell gridding) and
// blink_fused_conv.cu (convolutional gridding, support radius R > 0).  See blink_fused.cu for the design notes.
#pragma once
#include <algorithm>

#include "blink_common.cuh"
#include "blink_fft.cuh"
#include "blink_tma.cuh"

namespace blink {

constexpr int kFusedThreads = 512;

template <int N>
struct FusedCfg {
    static constexpr int H = N / 2;
    static constexpr int TG = N / kE;                          // threads per transform group
    static constexpr int G = kFusedThreads / TG;               // groups per CTA
    static constexpr int KY = (8192 / N) < 16 ? (8192 / N) : 16;   // ky rows per pass-2 sub-tile
    static constexpr int ROWB = KY * 8;                        // sub-tile row bytes (= TMA swizzle span)
    static constexpr int PPS = KY / 2;                         // row pairs per sub-tile
    static constexpr int NSUB = G / PPS;                       // sub-tiles per stage: every group gets a pair
    static constexpr int KYS = KY * NSUB;                      // ky rows per stage
    static constexpr int NIT = N / KYS;                        // pass-2 stages per image
    static constexpr int BOX_ROWS = H < 256 ? H : 256;
    static constexpr int SUB_BYTES = H * ROWB;
    static constexpr int STAGE_BYTES = NSUB * SUB_BYTES;       // 32 KB for every N
    static constexpr int COL_BYTES = G * 2 * N * 8;            // pass-1 column pairs of all groups (64 KB)
    static_assert(NSUB >= 1 && NSUB * PPS == G, "one row pair per group per stage");
    static_assert(SUB_BYTES % 1024 == 0, "swizzled sub-tiles stay 1024-byte aligned");
};

struct FusedArgs {
    const float2 *vis; const float *uvw_m;
    int T, C, P, B, weighting;
    int tc0, ntc, c_base;
    float *image; float *wsum; int32_t *cell_idx;              // indexed by absolute tc / image
    float2 *scratch;                                           // [gridDim.x][H][N]
    const float *su; const uint2 *svb;                         // per timestep: baselines sorted by |u| (presort_kernel)
    const float2 *tw;
    GainRef cal;                                               // optional per-antenna gains applied at the load
    // teams: `team` consecutive CTAs image one (t,c) together (column pairs and pass-2 tiles dealt round-robin over the ranks;
    // one scratch shared by the team, double-buffered; one global-memory barrier per image).  team == 1: a CTA per image.
    int team;
    unsigned *team_ctr;                                        // [n_teams] arrivals so far (monotonic)
    unsigned *team_w;                                          // [n_teams][2 parities][2] running totals of (occupied cells, samples)
};

constexpr size_t kTeamBytes = 4096;                            // team_ctr + team_w of up to 148 teams, 256-aligned

// Convolutional gridding (reading R16): the NORMALISED tap weight of tap j = -R..R of one axis,
//   w_j(f) = k(j - f) / sum_i k(i - f),  f = x - rint(x) in [-1/2, 1/2],  k = Kaiser-Bessel window of support S = 2R+1,
// is a smooth function of f and is evaluated as a polynomial in f (Horner, fp32).  The coefficients are fitted on the
// host in double (Chebyshev interpolation, conv_fit_taps in blink_fused_conv.cu) and travel as a kernel parameter.
#ifndef BLINK_CONV_TERMS
#define BLINK_CONV_TERMS 12
#endif
constexpr int kConvTerms = BLINK_CONV_TERMS;
constexpr int kConvMaxSupport = 7;
struct ConvPoly { float c[kConvMaxSupport][kConvTerms]; const float *inv_taper; };     // c[j + R][k] multiplies f^k

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
    __device__ __forceinline__ void put2(int wt, int wr, const float2 (&v)[2]) const
    {
        const int o = xsw(wt) ^ xsw(wr);
        c0[o] = v[0];
        c1[o] = v[1];
    }
    template <int TG>
    __device__ __forceinline__ void get_e(int tid, int e, float2 (&v)[2]) const
    {
        const int o = xsw_e<TG>(xsw(tid), e);
        v[0] = c0[o];
        v[1] = c1[o];
    }
};

// shared memory: vis row [B] float2 | column offsets [H+2] | pad to 1024 |
//                union(pass 1: column pairs (+ counts), pass 2: NS stages + exchange arrays) | mbarriers
template <int N>
__host__ __device__ constexpr size_t fused_region_bytes(bool uniform, int ns)
{
    using Cfg = FusedCfg<N>;
    (void)uniform;                                             // columns | counts | staged samples (2 rounds x 8 bytes per thread)
    const size_t p1 = (size_t)Cfg::COL_BYTES + (size_t)Cfg::COL_BYTES / 2 + (size_t)kFusedThreads * 16;
    const size_t p2 = (size_t)ns * Cfg::STAGE_BYTES + (size_t)Cfg::G * N * 8;
    return p1 > p2 ? p1 : p2;
}
template <int N>
__host__ __device__ constexpr size_t fused_front_bytes(int B)
{
    return (((size_t)B * 8 + 15) & ~(size_t)15) + (size_t)(FusedCfg<N>::H + 2) * 4;
}
template <int N>
static size_t fused_smem_bytes(int B, bool uniform, int ns)
{
    return align_up(fused_front_bytes<N>(B), 1024) + fused_region_bytes<N>(uniform, ns) + 1024 + 128;
}
constexpr size_t kSmemLimit = 227 * 1024;
// pipeline depth that fits next to the visibility row: 3 stages, else 2, else 0 (not supported)
template <int N>
static int fused_stages(int B, bool uniform)
{
    if (fused_smem_bytes<N>(B, uniform, 3) <= kSmemLimit) return 3;
    if (fused_smem_bytes<N>(B, uniform, 2) <= kSmemLimit) return 2;
    return 0;
}

// defined in blink_fused.cu
int fused_default_ctas();
int presort_launch(const float *uvw_m, int T, int B, float *su, uint2 *svb, cudaStream_t st);
size_t sort_bytes(int T, int B);

// ------------------------------------------------------------------------------------------ fused kernel
template <int N, int NS, int R = 0, bool TEAM = false>
__global__ void __launch_bounds__(kFusedThreads, 1)
fused_image_kernel(const FusedArgs a, const __grid_constant__ ScaleBlock sc, const __grid_constant__ CUtensorMap tmap,
                   const __grid_constant__ ConvPoly cpoly)
{
    using Cfg = FusedCfg<N>;
    constexpr int H = Cfg::H, TG = Cfg::TG, G = Cfg::G;
    extern __shared__ __align__(16) unsigned char smem_raw[];    // the 1024-byte alignment TMA needs is established below
    const bool uniform = a.weighting == BLINK_W_UNIFORM;
    const int B = a.B;
    const int g = threadIdx.x / TG;
    const int tid = threadIdx.x % TG;
    const int lane = threadIdx.x & 31;

    // ---- shared memory carve-up (pointer arithmetic on the array keeps every access in the shared window) ----
    float2 *visrow = reinterpret_cast<float2 *>(smem_raw);                                        // [B]
    uint32_t *coff = reinterpret_cast<uint32_t *>(smem_raw + (((size_t)B * 8 + 15) & ~(size_t)15));   // [H+2]
    const uint32_t front = (uint32_t)fused_front_bytes<N>(B);
    const uint32_t base_addr = smem_u32(smem_raw);
    unsigned char *region = smem_raw + (((base_addr + front + 1023u) & ~1023u) - base_addr);
    // pass 1: this group's column pair (XOR-swizzled slots) and, for uniform weighting, its cell counts
    float2 *c0 = reinterpret_cast<float2 *>(region) + (size_t)g * 2 * N, *c1 = c0 + N;
    uint32_t *n0 = reinterpret_cast<uint32_t *>(region + Cfg::COL_BYTES) + (size_t)g * 2 * N, *n1 = n0 + N;
    constexpr int kPre = 2;                                    // sample rounds staged ahead per unit
    uint2 *pre = reinterpret_cast<uint2 *>(region + Cfg::COL_BYTES + Cfg::COL_BYTES / 2) + (size_t)g * kPre * TG;
    // pass 2: NS stages of transposed scratch tiles, then one exchange array per group
    unsigned char *stage = region;
    float2 *xbuf = reinterpret_cast<float2 *>(region + (size_t)NS * Cfg::STAGE_BYTES) + (size_t)g * N;
    uint64_t *full = reinterpret_cast<uint64_t *>(region + fused_region_bytes<N>(uniform, NS));   // [NS]
    uint64_t *visbar = full + NS;
    __shared__ int s_nin, s_occ, s_ncol;
    __shared__ unsigned s_done[4];                             // per stage buffer: groups that have released it (running count)

    // TEAM == false compiles to the one-CTA-per-image kernel (K = 1, rank = 0: the compiler folds the team arithmetic away)
    const int K = TEAM ? a.team : 1, team_id = (int)blockIdx.x / K, rank = (int)blockIdx.x - team_id * K, n_teams = (int)gridDim.x / K;
    unsigned tcs = 0;                                          // (t,c) items this team has imaged so far
    __shared__ unsigned s_prev[4];                             // thread 0: team totals (occ, nin) at the last use of each parity
    if (threadIdx.x == 0) s_prev[0] = s_prev[1] = s_prev[2] = s_prev[3] = 0u;
    // barrier over ONE transform group (its columns / exchange array are private to it)
    auto gsync = [g] {
        if constexpr (TG == 32) __syncwarp();
        else if constexpr (G <= 15 && G > 1) asm volatile("bar.sync %0, %1;" ::"r"(g + 1), "r"(TG) : "memory");
        else __syncthreads();
    };
    const float lim = (float)(H - 1 - R);                      // R > 0: the whole support of a sample stays on the grid (R16)

    if (threadIdx.x == 0) {
        for (int k = 0; k < NS; ++k) {
            mbar_init(&full[k], 1);
            s_done[k] = 0u;
        }
        mbar_init(visbar, 1);
        fence_mbar_init();
        tma_prefetch_desc(&tmap);
    }
    // pipeline bookkeeping, identical in every thread: stage and use count of the next tile to consume
    uint32_t cs = 0, ck = 0;
    uint32_t vph = 0;
    Twiddles<N> twr;
    twr.init(tid, a.tw);
    // visibility rows arrive by bulk async copy when every row start is 16-byte aligned (B even)
    const bool bulk = (B & 1) == 0;
    const int tc_end = a.tc0 + a.ntc;
    __syncthreads();
    if (bulk && threadIdx.x == 0 && a.tc0 + team_id < tc_end) {
        mbar_expect_tx(visbar, (uint32_t)B * 8u);
        bulk_load_1d(visrow, a.vis + (size_t)(a.tc0 + team_id) * a.P * B, (uint32_t)B * 8u, visbar);
    }

    for (int tc = a.tc0 + team_id; tc < tc_end; tc += n_teams, ++tcs) {
        const int t = tc / a.C, c = tc - t * a.C;
        const float s = sc.s[c - a.c_base];
        const float *su = a.su + (size_t)t * B;
        const uint2 *svb = a.svb + (size_t)t * B;
        // column of sorted sample value x = |u_m| for this channel (H = beyond the grid, NaN included)
        auto col_of = [&](float x) -> int {
            int i;
            const float xr = rint_rne(__fmul_rn(x, s), i);
            return (xr <= lim) ? i : H;
        };
        int n_cp = 0, ulim = 0, n_box = 0;
        float wsum_val = 0.f;

        for (int p = 0; p < a.P; ++p) {
            const unsigned seq = tcs * (unsigned)a.P + (unsigned)p;   // planes this team has imaged so far
            const size_t img_idx = (size_t)tc * a.P + p;
            float *img = a.image + img_idx * N * N;
            // scratch slot: a CTA's own (team of one), else the team's two slots in turn -- the slot read by pass 2 of plane
            // seq is rewritten by pass 1 of plane seq + 2, after every CTA has passed the barrier of plane seq + 1
            const int slot = K == 1 ? (int)blockIdx.x : 2 * team_id + (int)(seq & 1u);
            float2 *scratch = a.scratch + (size_t)slot * H * N;
            __syncthreads();                                    // (C) every group has finished the previous pass 2
            {                                                   // the region was last used by pass 2: clear the columns
                const int n16 = (Cfg::COL_BYTES + (uniform ? Cfg::COL_BYTES / 2 : 0)) / 16;
                for (int i = threadIdx.x; i < n16; i += kFusedThreads)
                    reinterpret_cast<float4 *>(region)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
            }
            if (p == 0) {
                if (threadIdx.x == 0) { s_nin = 0; s_occ = 0; }
                // ---- column offsets: coff[u] = first sorted sample whose column is >= u, u = 0..H+1 -------
                // (sample j = B is a sentinel of column H+1, so every entry is written exactly once)
                for (int j0 = threadIdx.x; j0 <= B; j0 += 4 * kFusedThreads) {
                    float xs[4], xp[4];
#pragma unroll
                    for (int m = 0; m < 4; ++m) {
                        const int j = j0 + m * kFusedThreads;
                        xs[m] = j < B ? __ldg(su + j) : 0.f;
                        xp[m] = (j > 0 && j <= B) ? __ldg(su + j - 1) : 0.f;
                    }
#pragma unroll
                    for (int m = 0; m < 4; ++m) {
                        const int j = j0 + m * kFusedThreads;
                        if (j <= B) {
                            const int cj = j < B ? col_of(xs[m]) : H + 1;
                            const int cq = j > 0 ? col_of(xp[m]) : -1;
                            for (int u = cq + 1; u <= cj; ++u) coff[u] = (uint32_t)j;
                            if (cj >= H && cq < H) s_ncol = cq + 1 + (cq >= 0 ? R : 0);   // occupied columns are [0, cq + R]
                        }
                    }
                }
                // ---- optional output: cell index of every baseline, in baseline order (a1) ---------------
                if (a.cell_idx && rank == 0) {
                    const float *uvw = a.uvw_m + (size_t)t * B * 3;
                    for (int b = threadIdx.x; b < B; b += kFusedThreads)
                        a.cell_idx[(size_t)tc * B + b] = cell_of(uvw[3 * b], uvw[3 * b + 1], s, N, H, R);
                }
            }
            if (!bulk) {                                        // odd B: rows are only 8-byte aligned
                const float2 *vrow = a.vis + img_idx * B;
                for (int i = threadIdx.x; i < B; i += kFusedThreads) visrow[i] = vrow[i];
            }
            __syncthreads();                                    // (A)
            if (p == 0) {
                n_cp = (s_ncol + 1) / 2;                        // column pairs that hold samples
                ulim = 2 * n_cp;                                // scratch rows written by pass 1
                n_box = (ulim + Cfg::BOX_ROWS - 1) / Cfg::BOX_ROWS;
            }
            if (bulk) { mbar_wait(visbar, vph); vph ^= 1u; }
            if (a.cal.gains) {                                  // corrections fused into the load (R15): one sweep over the staged row
                const float2 *gc = a.cal.gains + ((size_t)c * a.P + p) * a.cal.A;
                for (int i = threadIdx.x; i < B; i += kFusedThreads) {
                    const int2 ap = __ldg(a.cal.ant + i);
                    const float2 g1 = __ldg(gc + ap.x), g2 = __ldg(gc + ap.y);
                    visrow[i] = cmul(visrow[i], cmul(g1, make_float2(g2.x, -g2.y)));
                }
                __syncthreads();
            }

            // ================= pass 1: each group grids and transforms column pairs (2cp, 2cp+1) ==========
            int my_in = 0, my_occ = 0;
            // one sample of this group's column pair: accumulate V (or conj V) into its cell with shared atomics
            auto grid_one = [&](uint2 sq, bool second, bool col0) {
                int iv;
                const float yr = rint_rne(__fmul_rn(__uint_as_float(sq.x), s), iv);
                if (fabsf(yr) <= lim) {                         // NaN fails; |iu| <= H-1 by construction
                    float2 vv = visrow[sq.y & 0x7fffffffu];
                    if (sq.y >> 31) vv.y = -vv.y;
                    float2 *col = second ? c1 : c0;
                    const int o = xsw(iv + H);
#if BLINK_GRID_EXCH
                    cell_add_exch(&col[o], vv);
#else
                    {                                           // odd lanes imaginary part first: even and odd banks per warp atomic
                        const int odd = lane & 1;
                        float *cell = reinterpret_cast<float *>(&col[o]);
                        atomicAdd(cell + odd, odd ? vv.y : vv.x);
                        atomicAdd(cell + (odd ^ 1), odd ? vv.x : vv.y);
                    }
#endif
                    if (uniform) atomicAdd(second ? &n1[o] : &n0[o], 1u);
                    if (col0) {                                 // iu == 0: the conjugate lies in column 0 too
                        const int o2 = xsw(H - iv);
#if BLINK_GRID_EXCH
                        cell_add_exch(&c0[o2], make_float2(vv.x, -vv.y));
#else
                        atomicAdd(&c0[o2].x, vv.x);
                        atomicAdd(&c0[o2].y, -vv.y);
#endif
                        if (uniform) atomicAdd(&n0[o2], 1u);
                    }
                    ++my_in;
                }
            };
            // Convolutional gridding (R > 0): sorted sample j seen from column pair (u0, u0+1).  Its S x S taps sit at
            // columns iu0-R..iu0+R; the taps at columns <= 0 are ALSO the conjugate sample's taps mirrored into u >= 0
            // (k is even, so the Hermitian sample at (-x,-y) has exactly the mirrored weights).
            auto conv_one = [&](int j, int u0) {
                if constexpr (R == 0) return;
                int iu0, iv0;
                const float x = __fmul_rn(__ldg(su + j), s);
                const float xr = rint_rne(x, iu0);              // in range by construction of the sample range
                const uint2 sq = __ldg(svb + j);
                const float y = __fmul_rn(__uint_as_float(sq.x), s);
                const float yr = rint_rne(y, iv0);
                if (!(fabsf(yr) <= lim)) return;                // NaN fails
                const float fx = __fsub_rn(x, xr), fy = __fsub_rn(y, yr);     // exact (|x - rint x| <= 1/2)
                float2 vv = visrow[sq.y & 0x7fffffffu];
                if (sq.y >> 31) vv.y = -vv.y;
                constexpr int S = 2 * R + 1;
                float wy[S];
#pragma unroll
                for (int i = 0; i < S; ++i) {
                    float w = cpoly.c[i][kConvTerms - 1];
#pragma unroll
                    for (int k = kConvTerms - 2; k >= 0; --k) w = fmaf(w, fy, cpoly.c[i][k]);
                    wy[i] = w;
                }
                // S taps of one column.  (Measured: fp32 atomicAdd on shared memory is a load + CAS spin loop per scalar on
                // sm_100, yet an optimistic batch of 64-bit CAS on the (re, im) pairs -- S loads, S CAS in flight, retry only
                // on interference -- was 1.4x (S = 5) to 2.1x (S = 7) SLOWER than the plain per-scalar adds below.)
                // Odd lanes add the imaginary part first: one warp-wide atomic then touches even AND odd banks (the real parts
                // alone live in the 16 even banks), which cuts the expected bank conflicts of 32 unrelated rows.
#ifndef BLINK_CONV_TAKE
#define BLINK_CONV_TAKE 1
#endif
                const int odd = lane & 1;
                auto add_taps = [&](float2 *col, int row0, int dir, float ar, float ai) {
#if BLINK_CONV_TAKE
                    (void)odd;
#pragma unroll
                    for (int i = 0; i < S; ++i) cell_add_take(&col[xsw(row0 + dir * i)], make_float2(wy[i] * ar, wy[i] * ai));
#else
                    const float first = odd ? ai : ar, second = odd ? ar : ai;
#pragma unroll
                    for (int i = 0; i < S; ++i) {
                        float *cell = reinterpret_cast<float *>(&col[xsw(row0 + dir * i)]);
                        atomicAdd(cell + odd, wy[i] * first);
                        atomicAdd(cell + (odd ^ 1), wy[i] * second);
                    }
#endif
                };
                auto wx_of = [&](int jj) {                      // tap jj - R of the u axis (dynamic index: LDC)
                    float w = cpoly.c[jj][kConvTerms - 1];
#pragma unroll
                    for (int k = kConvTerms - 2; k >= 0; --k) w = fmaf(w, fx, cpoly.c[jj][k]);
                    return w;
                };
#pragma unroll
                for (int k = 0; k < 2; ++k) {
                    const int u = u0 + k;
                    float2 *col = k ? c1 : c0;
                    const int jd = u - iu0;                     // direct tap that lands in column u
                    if (jd >= -R && jd <= R) {
                        const float wx = wx_of(jd + R);
                        add_taps(col, iv0 - R + H, 1, wx * vv.x, wx * vv.y);
                        if (jd == 0) ++my_in;                   // the sample's own column: counted once
                    }
                    const int jm = -u - iu0;                    // tap at column -u, mirrored: conj(V) at row -(iv0 + i)
                    if (jm >= -R) {
                        const float wx = wx_of(jm + R);
                        add_taps(col, H - (iv0 - R), -1, wx * vv.x, -wx * vv.y);
                    }
                }
            };
            // the first kPre*TG samples of a unit are staged one unit ahead with cp.async (each thread copies
            // exactly the entries it will consume, so no barrier is needed on the staging array)
            auto prefetch = [&](int cp_) {
                if (cp_ < n_cp) {
                    const int q0 = (int)coff[2 * cp_], q2 = (int)coff[2 * cp_ + 2];
#pragma unroll
                    for (int m = 0; m < kPre; ++m) {
                        const int j = q0 + tid + m * TG;
                        if (j < q2) cp_async_8(&pre[m * TG + tid], svb + j);
                    }
                }
            };
            if constexpr (R == 0) prefetch(g + G * rank);
            for (int cp = g + G * rank; cp < n_cp; cp += G * K) {
                const int u0 = 2 * cp;
                if constexpr (R == 0) {
                    const int k0 = (int)coff[u0], k1 = (int)coff[u0 + 1], k2 = (int)coff[u0 + 2];
                    cp_async_wait_all();
                    gsync();                                    // the columns are zero again (own-slot clearing below)
#pragma unroll
                    for (int m = 0; m < kPre; ++m) {
                        const int j = k0 + tid + m * TG;
                        if (j < k2) grid_one(pre[m * TG + tid], j >= k1, u0 == 0 && j < k1);
                    }
                    for (int j = k0 + tid + kPre * TG; j < k2; j += TG) grid_one(__ldg(svb + j), j >= k1, u0 == 0 && j < k1);
                    prefetch(cp + G * K);                       // lands while this unit is transformed
                } else {
                    // samples whose support reaches columns u0, u0+1: nearest columns [u0-R, u0+1+R]; the mirrored
                    // taps come from nearest columns [0, R-u0], a subset (coff[H] = first sample beyond the range)
                    const int k0 = (int)coff[u0 > R ? u0 - R : 0];
                    const int k2 = (int)coff[u0 + 2 + R < H ? u0 + 2 + R : H];
                    gsync();
                    for (int j = k0 + tid; j < k2; j += TG) conv_one(j, u0);
                }
                gsync();
                float2 v[2][kE];
#pragma unroll
                for (int e = 0; e < kE; ++e) {                  // transform index n lives in centred row n ^ H
                    const int o = xsw_e<TG>(xsw(tid), e ^ (kE / 2));
                    v[0][e] = c0[o];
                    v[1][e] = c1[o];
                    if (uniform) {                              // a3: divide by the cell count
                        const uint32_t q0 = n0[o], q1 = n1[o];
                        if (q0) {
                            n0[o] = 0u;
                            v[0][e].x = __fdiv_rn(v[0][e].x, (float)q0);
                            v[0][e].y = __fdiv_rn(v[0][e].y, (float)q0);
                            my_occ += (u0 == 0) ? 1 : 2;        // the mirror image of a u > 0 cell is occupied too
                        }
                        if (q1) {
                            n1[o] = 0u;
                            v[1][e].x = __fdiv_rn(v[1][e].x, (float)q1);
                            v[1][e].y = __fdiv_rn(v[1][e].y, (float)q1);
                            my_occ += 2;
                        }
                    }
                }
                ExchangePadded2 xch{c0, c1};
                fft_inverse<N, 2>(v, tid, xch, twr, gsync);
                float2 *d0 = scratch + (size_t)u0 * N, *d1 = d0 + N;
#pragma unroll
                for (int e = 0; e < kE; ++e) {
                    const int o = xsw_e<TG>(xsw(tid), e);       // the slots this thread read last: clear them
                    c0[o] = make_float2(0.f, 0.f);
                    c1[o] = make_float2(0.f, 0.f);
                    d0[tid + e * TG] = v[0][e];
                    d1[tid + e * TG] = v[1][e];
                }
            }
            if (p == 0) {                                       // weight sum (a3), shared by the P planes
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
            __syncthreads();                                    // (B)
            if (TEAM && K > 1) {
                // team barrier: every CTA's share of H[u][ky] (and of the weight sum) is in global memory before anyone's pass 2
                if (threadIdx.x == 0) {
                    unsigned *tw = a.team_w + (size_t)team_id * 4 + (tcs & 1u) * 2;
                    if (p == 0) { atomicAdd(tw, (unsigned)s_occ); atomicAdd(tw + 1, (unsigned)s_nin); }
                    __threadfence();
                    atomicAdd(a.team_ctr + team_id, 1u);
                    const unsigned target = (seq + 1u) * (unsigned)K;
                    unsigned seen;
                    do {
                        asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(a.team_ctr + team_id) : "memory");
                    } while ((int)(seen - target) < 0);
                    if (p == 0) {                               // the (t,c)'s totals = running totals minus their value two items ago
                        unsigned occ, nin;
                        asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(occ) : "l"(tw) : "memory");
                        asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(nin) : "l"(tw + 1) : "memory");
                        const unsigned o = (tcs & 1u) * 2u;
                        s_occ = (int)(occ - s_prev[o]);
                        s_nin = (int)(nin - s_prev[o + 1]);
                        s_prev[o] = occ;
                        s_prev[o + 1] = nin;
                    }
                }
                __syncthreads();
                asm volatile("fence.proxy.async;" ::: "memory"); // the other CTAs' scratch stores before this CTA's TMA loads
            }
            if (bulk && threadIdx.x == 0) {                     // prefetch the next image's visibility row
                size_t nxt = img_idx + 1;
                if (p + 1 == a.P) nxt = (tc + n_teams < tc_end) ? (size_t)(tc + n_teams) * a.P : (size_t)-1;
                if (nxt != (size_t)-1) {
                    mbar_expect_tx(visbar, (uint32_t)B * 8u);
                    bulk_load_1d(visrow, a.vis + nxt * B, (uint32_t)B * 8u, visbar);
                }
            }
            if (p == 0) wsum_val = uniform ? (float)s_occ : (float)(2 * s_nin);
            if (wsum_val == 0.f) {                              // W = 0: zero image (uniform over the CTA)
                for (int i = threadIdx.x; i < N * N / 4; i += kFusedThreads)
                    reinterpret_cast<float4 *>(img)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
                continue;
            }
            const float inv_w = 1.0f / wsum_val;

            // ================= pass 2: row pairs -> two real image rows per transform ===================
            // NS stage buffers behind `full` mbarriers.  A buffer is re-requested by whichever group is the LAST to
            // have pulled its inputs out of it (a shared counter bumped by each group's leader right after the
            // group's first barrier inside the transform), so refills start the moment the buffer is free.
            auto request = [&](int it, uint32_t st_) {
                fence_proxy_async();
                uint64_t *bar = &full[st_];
                unsigned char *dst = stage + (size_t)st_ * Cfg::STAGE_BYTES;
                mbar_expect_tx(bar, (uint32_t)(Cfg::NSUB * n_box * Cfg::BOX_ROWS * Cfg::ROWB));
                for (int sb_ = 0; sb_ < Cfg::NSUB; ++sb_)
                    for (int bx = 0; bx < n_box; ++bx)
                        tma_load_3d(dst + (size_t)sb_ * Cfg::SUB_BYTES + (size_t)bx * Cfg::BOX_ROWS * Cfg::ROWB, &tmap, bar,
                                    2 * (it * Cfg::KYS + sb_ * Cfg::KY), bx * Cfg::BOX_ROWS, slot);
            };
            if (threadIdx.x == 0)                               // this CTA's tiles: it = rank, rank + K, ...
                for (int i = 0; i < NS && rank + i * K < Cfg::NIT; ++i) request(rank + i * K, (cs + (uint32_t)i) % (uint32_t)NS);
            const int sub = g / Cfg::PPS, pair = g % Cfg::PPS;
            for (int it = rank; it < Cfg::NIT; it += K) {
                mbar_wait(&full[cs], ck & 1u);
                const uint32_t st_used = cs;
                float2 z[1][kE];
                {
                    // 16 bytes (S1[u], S2[u]) per u out of the swizzled sub-tile.  The swizzle only involves bits of
                    // (u mod 8) and TG is a multiple of 8, so the address is one per-thread base plus a compile-time
                    // multiple of TG rows -- for u = tid + e TG as well as for the mirrored u = N - (tid + e TG).
                    using XT = ExchangeTilePair<Cfg::ROWB>;
                    const unsigned char *tile = stage + (size_t)cs * Cfg::STAGE_BYTES + (size_t)sub * Cfg::SUB_BYTES;
                    const unsigned char *lo = tile + XT::swz((uint32_t)tid * Cfg::ROWB + (uint32_t)pair * 16u);
                    const unsigned char *hi = tile + XT::swz((uint32_t)(TG - tid) * Cfg::ROWB + (uint32_t)pair * 16u);
#pragma unroll
                    for (int e = 0; e < kE / 2; ++e) {          // n = u < H: S1 + i S2
                        float4 q = make_float4(0.f, 0.f, 0.f, 0.f);
                        if (tid < ulim - e * TG) q = *reinterpret_cast<const float4 *>(lo + (size_t)e * TG * Cfg::ROWB);
                        z[0][e] = make_float2(q.x - q.w, q.y + q.z);
                    }
#pragma unroll
                    for (int e = kE / 2; e < kE; ++e) {         // n > H: conj(S1[N-n]) + i conj(S2[N-n])
                        // u = N - (tid + e TG) = (TG - tid) + (kE - 1 - e) TG, in [1, H]; u == H is the empty Nyquist column
                        float4 q = make_float4(0.f, 0.f, 0.f, 0.f);
                        const bool ok = (TG - tid) < ulim - (kE - 1 - e) * TG && (e > kE / 2 || tid > 0);
                        if (ok) q = *reinterpret_cast<const float4 *>(hi + (size_t)(kE - 1 - e) * TG * Cfg::ROWB);
                        z[0][e] = make_float2(q.x + q.w, q.z - q.y);
                    }
                }
                if (++cs == (uint32_t)NS) { cs = 0; ++ck; }
                auto release = [&](int k) {                     // k == 0: right after the group's first barrier, inputs are in registers
                    if (k == 0 && tid == 0) {
                        __threadfence_block();                  // the group's reads (ordered by its barrier) before the count
                        const unsigned old = atomicAdd(&s_done[st_used], 1u);
                        __threadfence_block();
                        if (old % (unsigned)G == (unsigned)(G - 1) && it + NS * K < Cfg::NIT) request(it + NS * K, st_used);
                    }
                };
                ExchangePadded1 xch{xbuf};
                fft_inverse<N, 1>(z, tid, xch, twr, gsync, release);
                const int ky = it * Cfg::KYS + sub * Cfg::KY + 2 * pair;
                float *r0 = img + (size_t)(ky ^ H) * N + tid, *r1 = img + (size_t)((ky + 1) ^ H) * N + tid;
                if constexpr (R == 0) {
#pragma unroll
                    for (int e = 0; e < kE; ++e) {              // x = (tid + e TG) ^ H = tid + (e ^ kE/2) TG: fftshift
                        __stcs(r0 + (e ^ (kE / 2)) * TG, z[0][e].x * inv_w);
                        __stcs(r1 + (e ^ (kE / 2)) * TG, z[0][e].y * inv_w);
                    }
                } else {                                        // grid correction 1 / (c(y) c(x)) rides on the same store
                    const float t0 = inv_w * __ldg(cpoly.inv_taper + (ky ^ H)), t1 = inv_w * __ldg(cpoly.inv_taper + ((ky + 1) ^ H));
#pragma unroll
                    for (int e = 0; e < kE; ++e) {
                        const float tx = __ldg(cpoly.inv_taper + tid + (e ^ (kE / 2)) * TG);
                        __stcs(r0 + (e ^ (kE / 2)) * TG, z[0][e].x * (t0 * tx));
                        __stcs(r1 + (e ^ (kE / 2)) * TG, z[0][e].y * (t1 * tx));
                    }
                }
            }
        }
        if (threadIdx.x == 0 && rank == 0) a.wsum[tc] = wsum_val;
    }
}

// Team size for ntc (t,c) items on `ctas` resident CTAs.  Cost model, in units of one plane imaged by one CTA alone:
//   K = 1: rounds(1);   K > 1: rounds(K) / K * (1 + c + K f),   rounds(K) = ceil(ntc / (ctas / K)),
// c = what team mode costs whatever its size (the barrier per plane, the totals), f = the per-plane work every member repeats
// (column-offset scan, clearing, pipeline fill) as a fraction of a plane's work.  Fitted to a sweep of K = 1 .. 74 over
// BASELINE.json configs 2, 4 (one timestep) and 5 on a B200: N = 1024: c ~ 0, f = 0.025; 2048: c = 0.06,
// f = 0.007; 4096: c = 0.07, f = 0.002.  Sizes that leave a rank less than ~two rounds of column-pair units (K G > N / 16)
// are not considered; a team is taken only when the model saves >= 3 %.
template <int N>
static int choose_team(int ntc, int ctas)
{
    const int forced = option(BLINK_OPT_FUSED_TEAM);
    const int cand[] = {2, 3, 4, 6, 8, 12, 16, 37, 74, 148};
    if (forced > 0) return forced <= ctas && forced <= FusedCfg<N>::NIT ? forced : 1;
    const double c = N >= 4096 ? 0.07 : N >= 2048 ? 0.06 : N >= 1024 ? 0.0 : 0.05;
    const double f = N >= 4096 ? 0.002 : N >= 2048 ? 0.007 : N >= 1024 ? 0.025 : N >= 512 ? 0.04 : 0.08;
    auto cost = [&](int k) {
        const int teams = ctas / k;
        const double r = (double)((ntc + teams - 1) / teams) / k;
        return k == 1 ? r : r * (1.0 + c + k * f);
    };
    int best = 1;
    double best_c = cost(1);
    for (int k : cand) {
        if (k > ctas || k * FusedCfg<N>::G > N / 16 || k > FusedCfg<N>::NIT) continue;
        const double ck = cost(k);
        if (ck < best_c) { best = k; best_c = ck; }
    }
    if (best_c > 0.97 * cost(1)) best = 1;
    return best;
}

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

// extra: bytes between the sort arrays and the scratch that the caller has filled (the conv taper table), 256-aligned
template <int N, int R = 0>
static int launch_fused(const FusedArgs &base, const double *freqs_hz, double pixscale_rad, void *workspace,
                        size_t workspace_bytes, cudaStream_t st, const ConvPoly *poly = nullptr, size_t extra = 0)
{
    using Cfg = FusedCfg<N>;
    const size_t per_cta = (size_t)Cfg::H * N * sizeof(float2);
    const size_t sortb = sort_bytes(base.T, base.B) + extra + kTeamBytes;
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u) || workspace_bytes < sortb + per_cta)
        return BLINK_ERR_WORKSPACE;
    int ctas = option(BLINK_OPT_FUSED_CTAS);
    if (ctas <= 0) ctas = fused_default_ctas();
    const int slots_max = (int)std::min<size_t>((size_t)ctas, (workspace_bytes - sortb) / per_cta);   // scratch slots that fit
    // workspace: su | svb (baselines of every timestep sorted by |u|) | per-CTA scratch
    unsigned char *wsp = static_cast<unsigned char *>(workspace);
    float *su = reinterpret_cast<float *>(wsp);
    uint2 *svb = reinterpret_cast<uint2 *>(wsp + (sortb - extra - kTeamBytes) / 3);
    unsigned *team_mem = reinterpret_cast<unsigned *>(wsp + sortb - kTeamBytes);
    void *scratch = wsp + sortb;
    {
        int rc = presort_launch(base.uvw_m, base.T, base.B, su, svb, st);
        if (rc != BLINK_OK) return rc;
    }
    ConvPoly cpoly{};
    if (poly) cpoly = *poly;
    const bool uni = base.weighting == BLINK_W_UNIFORM;
    const int ns = fused_stages<N>(base.B, uni);
    if (ns == 0) return BLINK_ERR_UNSUPPORTED;
    const size_t smem = fused_smem_bytes<N>(base.B, uni, ns);
    if (ns == 3) {
        BLINK_CUDA_TRY(cudaFuncSetAttribute(fused_image_kernel<N, 3, R>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        BLINK_CUDA_TRY(cudaFuncSetAttribute(fused_image_kernel<N, 3, R, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    } else {
        BLINK_CUDA_TRY(cudaFuncSetAttribute(fused_image_kernel<N, 2, R>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        BLINK_CUDA_TRY(cudaFuncSetAttribute(fused_image_kernel<N, 2, R, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    }
    CUtensorMap tmap;
    // scratch viewed as float32 [slots][H rows (u)][2N (ky re/im)]; boxes of [BOX_ROWS u][KY ky]
    int rc = encode_tensor_map_3d_f32(&tmap, scratch, 2ull * N, (uint64_t)Cfg::H, (uint64_t)slots_max, (uint64_t)N * 8,
                                      (uint64_t)Cfg::H * N * 8, 2 * Cfg::KY, Cfg::BOX_ROWS, 1,
                                      Cfg::ROWB >= 32 ? Cfg::ROWB : 0);
    if (rc != 0) { set_error_text("cuTensorMapEncodeTiled failed (fused scratch)"); return BLINK_ERR_CUDA; }
    return for_channel_blocks(base.C, base.tc0, base.ntc, freqs_hz, N, pixscale_rad,
                              [&](int tc0, int ntc, int c_base, const ScaleBlock &sc) -> int {
                                  FusedArgs a = base;
                                  a.tc0 = tc0; a.ntc = ntc; a.c_base = c_base;
                                  a.scratch = static_cast<float2 *>(scratch);
                                  a.su = su; a.svb = svb;
                                  a.tw = twiddle_table();
                                  // team size for this launch; a team of K needs two scratch slots (K > 1) or one per CTA (K == 1)
                                  int team = choose_team<N>(ntc, ctas);
                                  while (team > 1 && slots_max < 2) team = 1;
                                  int grid;
                                  if (team == 1) {
                                      grid = std::min(ntc, std::min(ctas, slots_max));
                                  } else {
                                      const int teams = std::min(std::min(ctas / team, slots_max / 2), ntc);
                                      grid = teams * team;
                                      if (cudaMemsetAsync(team_mem, 0, kTeamBytes, st) != cudaSuccess) return (int)BLINK_ERR_CUDA;
                                  }
                                  a.team = team;
                                  a.team_ctr = team_mem;
                                  a.team_w = team_mem + 256;
                                  if (team > 1) {
                                      if (ns == 3) fused_image_kernel<N, 3, R, true><<<grid, kFusedThreads, smem, st>>>(a, sc, tmap, cpoly);
                                      else fused_image_kernel<N, 2, R, true><<<grid, kFusedThreads, smem, st>>>(a, sc, tmap, cpoly);
                                  } else {
                                      if (ns == 3) fused_image_kernel<N, 3, R><<<grid, kFusedThreads, smem, st>>>(a, sc, tmap, cpoly);
                                      else fused_image_kernel<N, 2, R><<<grid, kFusedThreads, smem, st>>>(a, sc, tmap, cpoly);
                                  }
                                  BLINK_LAUNCH_CHECK("fused_image_kernel");
                                  return (int)BLINK_OK;
                              });
}

}  // namespace blink
