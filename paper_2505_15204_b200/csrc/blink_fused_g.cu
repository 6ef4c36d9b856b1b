// Fused imaging kernel for the paper's own image side, 1200 x 1200 (Table 6): visibilities ->
// dirty images with the uv grid never materialised, the design of blink_fused.cu carried over to a side that is not a
// power of two (1200 = 15 x 5 x 16).
//
//   * presort (blink_fused.cu): per timestep the baselines sorted by |u_m|, folded into the half plane u >= 0, so that for
//     every channel the samples of a u-column are one contiguous range of the list;
//   * one persistent CTA per SM walks over (t,c); it holds FG_G transform groups of 160 threads that run DECOUPLED behind
//     their own named barriers.  A group owns one shared-memory array of 2 x 1200 complex64 and works on TWO transforms at
//     a time: 80 + 80 radix-15 butterflies, 240 + 240 radix-5 butterflies (three rounds), 75 + 75 radix-16 butterflies --
//     every stage register-resident (blink_fftg.cuh), in place in the array (read -> barrier -> write -> barrier);
//   * pass 1, per column pair (u0, u0+1): grid the pair's samples into the (zeroed) array with native 64-bit exchanges
//     (cell_add_exch), divide by the cell counts for uniform weighting while loading the first stage, transform along v,
//     and store the result TRANSPOSED, HT[ky][u], to the per-CTA scratch straight from the registers of the last stage;
//   * pass 2, per two row pairs (ky, ky+1), (ky+2, ky+3): Z[u] = HT[ky][u] + i HT[ky+1][u], Z[N-u] = conj + i conj (the
//     Hermitian packing of blink_fused.cu); the four rows -- only the columns u < ulim hold anything -- arrive in a
//     per-group staging buffer by bulk async copies issued one unit ahead, are transformed along u, and stored as two real image rows from the
//     registers of the last stage with the shift, 1/W and the real part folded in (centred index = (j + N/2) mod N).
// Steps a0-a5 of include/blinkimg.h; PAPER.md L190-194 (gridding, inverse 2D FFT, shift), L150 (fp32).
#include <algorithm>

#include "blink_fused_kernel.cuh"
#include "blink_fftg.cuh"

namespace blink {

constexpr int FG_N = 1200, FG_H = 600;
#ifndef BLINK_FG_NT
#define BLINK_FG_NT 2
#endif
constexpr int FG_NT = BLINK_FG_NT;                              // transforms a group works on at a time (2: a column / row-pair PAIR)
constexpr int FG_TG = FG_NT == 2 ? 160 : 96;                    // threads per group (5 or 3 warps): 80 radix-15 butterflies per transform
#ifndef BLINK_FG_GROUPS
#define BLINK_FG_GROUPS 4
#endif
constexpr int FG_G = BLINK_FG_GROUPS;                           // groups per CTA
constexpr int FG_THREADS = FG_TG * FG_G;                        // 640
constexpr int FG_LD = 1208;                                     // leading dimension of a group's arrays (complex64)
constexpr int FG_TW = 1 + 15 + 75;                              // compact twiddle runs of the three stages
constexpr int kFgMaxB = 15000;                                 // the staged visibility row must fit next to the arrays

// shared memory: arrays | twiddle runs | column offsets | mbarriers | U = union( pass 1: visibility row + 16-bit cell counts,
//                                                                               pass 2: per-group staging of 4 rows of HT )
struct FgSmem {
    static constexpr size_t ARR = (size_t)FG_G * FG_NT * FG_LD * sizeof(float2);      // 77.3 KB
    static constexpr size_t CNT = (size_t)FG_G * FG_NT * (FG_N / 2) * sizeof(uint32_t);  // 19.2 KB: 16-bit counts, two per word
    static constexpr size_t TW = ((size_t)FG_TW * sizeof(float2) + 15) & ~(size_t)15;
    static constexpr size_t COFF = ((size_t)(FG_H + 2) * 4 + 15) & ~(size_t)15;
    static constexpr size_t BARS = 128;                                                // visbar + 2 staging barriers per group
    static constexpr size_t STG_G = (size_t)2 * FG_NT * FG_H * sizeof(float2);         // 19.2 KB per group: 4 rows x 600 columns
    static constexpr size_t HEAD = ARR + TW + COFF + BARS;
    __host__ __device__ static size_t front(int B) { return ((size_t)B * 8 + 15) & ~(size_t)15; }
    __host__ __device__ static size_t uni(int B) { return front(B) + CNT > FG_G * STG_G ? front(B) + CNT : FG_G * STG_G; }
    static size_t bytes(int B) { return HEAD + uni(B) + 16; }
};

// One in-place Stockham stage of the group's two transforms (radix R, sub-transform length P; see gstage in blink_fftg.cu):
//   input  element n of transform tr:  load(tr, n)           (FIRST)  or  arr[tr * LD + n]
//   output element j of transform tr:  emit(tr, j, value)    (LAST)   or  arr[tr * LD + j]
// Butterfly i reads n = i + r N/R and writes j = (i - k) R + k + r P, k = i mod P.  All of a thread's butterflies (ROUNDS of
// them) are loaded before the barrier that separates the stage's reads from its writes.
struct FgNoHook { __device__ __forceinline__ void operator()() const {} };
template <int R, int P, bool FIRST, bool LAST, class Sync, class Load, class Emit, class Hook = FgNoHook>
__device__ __forceinline__ void fg_stage(float2 *arr, const float2 *__restrict__ tw, int tid, Sync gsync, Load load, Emit emit,
                                         Hook hook = Hook())
{
    constexpr int nb = FG_N / R, total = FG_NT * nb, ROUNDS = (total + FG_TG - 1) / FG_TG;
    float2 x[ROUNDS][R];
#pragma unroll
    for (int q = 0; q < ROUNDS; ++q) {
        const int idx = tid + q * FG_TG;
        if (idx < total) {
            const int tr = idx >= nb, i = idx - tr * nb;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                if constexpr (FIRST) x[q][r] = load(tr, i + r * nb);
                else x[q][r] = arr[tr * FG_LD + i + r * nb];
            }
            if constexpr (P > 1) gtwiddle<R>(x[q], tw[i % P]);
            gbutterfly<R>(x[q]);
        }
    }
    if constexpr (!LAST) {
        gsync();                                               // every read of the array is done (also the previous unit's)
        hook();                                                // FIRST: the stage's inputs are in registers
#pragma unroll
        for (int q = 0; q < ROUNDS; ++q) {
            const int idx = tid + q * FG_TG;
            if (idx < total) {
                const int tr = idx >= nb, i = idx - tr * nb, k = i % P;
                float2 *d = arr + tr * FG_LD + (i - k) * R + k;
#pragma unroll
                for (int r = 0; r < R; ++r) d[r * P] = x[q][r];
            }
        }
        gsync();
    } else {
#pragma unroll
        for (int q = 0; q < ROUNDS; ++q) {
            const int idx = tid + q * FG_TG;
            if (idx < total) {
                const int tr = idx >= nb, i = idx - tr * nb, k = i % P;
#pragma unroll
                for (int r = 0; r < R; ++r) emit(tr, (i - k) * R + k + r * P, x[q][r]);
            }
        }
    }
}

// the three stages of 1200 = 15 x 5 x 16; twiddle runs at tw + 0 (unused), + 1 (P = 15), + 16 (P = 75)
template <class Sync, class Load, class Emit, class Hook = FgNoHook>
__device__ __forceinline__ void fg_transform2(float2 *arr, const float2 *tw, int tid, Sync gsync, Load load, Emit emit, Hook hook = Hook())
{
    auto no_load = [](int, int) { return make_float2(0.f, 0.f); };
    auto no_emit = [](int, int, float2) {};
    fg_stage<15, 1, true, false>(arr, tw, tid, gsync, load, no_emit, hook);
    fg_stage<5, 15, false, false>(arr, tw + 1, tid, gsync, no_load, no_emit);
    fg_stage<16, 75, false, true>(arr, tw + 16, tid, gsync, no_load, emit);
}

// the same with the last stage's outputs left in the arrays (natural order); ends with a group barrier
template <class Sync, class Load>
__device__ __forceinline__ void fg_transform2_inplace(float2 *arr, const float2 *tw, int tid, Sync gsync, Load load)
{
    auto no_load = [](int, int) { return make_float2(0.f, 0.f); };
    auto no_emit = [](int, int, float2) {};
    fg_stage<15, 1, true, false>(arr, tw, tid, gsync, load, no_emit);
    fg_stage<5, 15, false, false>(arr, tw + 1, tid, gsync, no_load, no_emit);
    fg_stage<16, 75, false, false>(arr, tw + 16, tid, gsync, no_load, no_emit);
}

#ifndef BLINK_FG_PAIRED_STORE
#define BLINK_FG_PAIRED_STORE 1
#endif

// R > 0: convolutional gridding of support S = 2R + 1 (reading R16, blink_fused_kernel.cuh conv_one): a column pair
// gathers every sorted sample whose support reaches it, the taps at columns <= 0 come back as the conjugate's mirrored taps, the
// grid correction rides on the image store; natural weighting only
template <int R>
__global__ void __launch_bounds__(FG_THREADS, 1)
fused_g_kernel(const FusedArgs a, const __grid_constant__ ScaleBlock sc, const float2 *__restrict__ tw_full,
               const __grid_constant__ ConvPoly cpoly)
{
    constexpr int N = FG_N, H = FG_H;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const bool uniform = a.weighting == BLINK_W_UNIFORM;
    const int B = a.B;
    const int g = threadIdx.x / FG_TG, tid = threadIdx.x % FG_TG, lane = threadIdx.x & 31;

    unsigned char *q = smem_raw + ((16 - (smem_u32(smem_raw) & 15u)) & 15u);
    float2 *arr_all = reinterpret_cast<float2 *>(q);             q += FgSmem::ARR;
    float2 *stw = reinterpret_cast<float2 *>(q);                 q += FgSmem::TW;
    uint32_t *coff = reinterpret_cast<uint32_t *>(q);            q += FgSmem::COFF;
    uint64_t *visbar = reinterpret_cast<uint64_t *>(q);          q += FgSmem::BARS;
    uint64_t *stbar = visbar + 1 + 2 * g;                        // this group's two staging barriers
    float2 *visrow = reinterpret_cast<float2 *>(q);                                               // U, pass 1: [B]
    uint32_t *cnt_all = reinterpret_cast<uint32_t *>(q + FgSmem::front(B));
    float2 *stg = reinterpret_cast<float2 *>(q + (size_t)g * FgSmem::STG_G);                      // U, pass 2: [4][ulim]
    float2 *arr = arr_all + (size_t)g * FG_NT * FG_LD;
    uint32_t *cnt = cnt_all + (size_t)g * FG_NT * (N / 2);           // cnt[tr * 600 + (n >> 1)], 16 bits per cell
    __shared__ int s_nin, s_occ, s_ncol;

    float2 *HT = a.scratch + (size_t)blockIdx.x * N * H;         // [N ky][H u], transposed pass-1 output
    auto gsync = [g] { asm volatile("bar.sync %0, %1;" ::"r"(g + 1), "n"(FG_TG) : "memory"); };
    const float lim = (float)(H - 1 - R);                        // R > 0: the whole support of a sample stays on the grid (R16)

    // compact per-stage twiddle runs: stage with sub-transform length P reads W_N^(k N / (P R)), k < P
    for (int k = threadIdx.x; k < FG_TW; k += FG_THREADS) {
        int step, kk;
        if (k < 1) { step = 0; kk = 0; }
        else if (k < 16) { step = N / (15 * 5); kk = k - 1; }
        else { step = N / (75 * 16); kk = k - 16; }
        stw[k] = tw_full[kk * step];
    }
    if (threadIdx.x == 0) {
        for (int k = 0; k <= 2 * FG_G; ++k) mbar_init(visbar + k, 1);
        fence_mbar_init();
    }
    uint32_t vph = 0, sph = 0;                                   // sph: phase bits of the two staging barriers
    const bool bulk = (B & 1) == 0;
    const int tc_end = a.tc0 + a.ntc;
    __syncthreads();
    auto clear_group = [&] {                                    // this group's arrays (and counts): zero for the next gridding
        float4 *z = reinterpret_cast<float4 *>(arr);
        for (int i = tid; i < FG_NT * FG_LD / 2; i += FG_TG) z[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (uniform) for (int i = tid; i < FG_NT * (N / 2); i += FG_TG) cnt[i] = 0u;
    };

    for (int tc = a.tc0 + blockIdx.x; tc < tc_end; tc += gridDim.x) {
        const int t = tc / a.C, c = tc - t * a.C;
        const float s = sc.s[c - a.c_base];
        const float *su = a.su + (size_t)t * B;
        const uint2 *svb = a.svb + (size_t)t * B;
        auto col_of = [&](float x) -> int {                     // column of sorted sample value x = |u_m| (H = off the grid, NaN too)
            int i;
            const float xr = rint_rne(__fmul_rn(x, s), i);
            return (xr <= lim) ? i : H;
        };
        int n_cp = 0, ulim = 0;
        float wsum_val = 0.f;

        for (int p = 0; p < a.P; ++p) {
            const size_t img_idx = (size_t)tc * a.P + p;
            float *img = a.image + img_idx * N * N;
            __syncthreads();                                    // (C) every group has finished the previous pass 2: U is free
            if (bulk) {
                if (threadIdx.x == 0) {                         // the image's visibility row, by one bulk async copy
                    fence_proxy_async();
                    mbar_expect_tx(visbar, (uint32_t)B * 8u);
                    bulk_load_1d(visrow, a.vis + img_idx * B, (uint32_t)B * 8u, visbar);
                }
            } else {
                const float2 *vrow = a.vis + img_idx * B;       // odd B: rows are only 8-byte aligned
                for (int i = threadIdx.x; i < B; i += FG_THREADS) visrow[i] = vrow[i];
            }
            clear_group();
            if (p == 0) {
                if (threadIdx.x == 0) { s_nin = 0; s_occ = 0; }
                // column offsets: coff[u] = first sorted sample whose column is >= u, u = 0..H+1 (sample B = sentinel of column H+1)
                for (int j = threadIdx.x; j <= B; j += FG_THREADS) {
                    const int cj = j < B ? col_of(__ldg(su + j)) : H + 1;
                    const int cq = j > 0 ? col_of(__ldg(su + j - 1)) : -1;
                    for (int u = cq + 1; u <= cj; ++u) coff[u] = (uint32_t)j;
                    if (cj >= H && cq < H) s_ncol = cq + 1 + (cq >= 0 ? R : 0);   // occupied columns are [0, cq + R]
                }
                if (a.cell_idx) {
                    const float *uvw = a.uvw_m + (size_t)t * B * 3;
                    for (int b = threadIdx.x; b < B; b += FG_THREADS)
                        a.cell_idx[(size_t)tc * B + b] = cell_of(uvw[3 * b], uvw[3 * b + 1], s, N, H, R);
                }
            }
            __syncthreads();                                    // (A)
            if (p == 0) {
                n_cp = (s_ncol + 1) / 2;
                ulim = 2 * n_cp;
            }
            if (bulk) { mbar_wait(visbar, vph); vph ^= 1u; }
            if (a.cal.gains) {                                  // corrections fused into the load (R15)
                const float2 *gc = a.cal.gains + ((size_t)c * a.P + p) * a.cal.A;
                for (int i = threadIdx.x; i < B; i += FG_THREADS) {
                    const int2 ap = __ldg(a.cal.ant + i);
                    const float2 g1 = __ldg(gc + ap.x), g2 = __ldg(gc + ap.y);
                    visrow[i] = cmul(visrow[i], cmul(g1, make_float2(g2.x, -g2.y)));
                }
                __syncthreads();
            }

            // ================= pass 1: column pairs (2cp, 2cp+1): grid, transform along v, store transposed ==========
            int my_in = 0, my_occ = 0;
            // the first FG_TG samples of a unit are fetched one unit ahead (one register pair per thread), the rest in the loop
            const int n_un = ulim / FG_NT;                      // units of FG_NT columns (the last column may be an empty one)
            auto first_sample = [&](int cp_) -> uint2 {
                if (cp_ < n_un) {
                    const int j = (int)coff[FG_NT * cp_] + tid;
                    if (j < (int)coff[FG_NT * cp_ + FG_NT]) return __ldg(svb + j);
                }
                return make_uint2(0u, 0u);
            };
            uint2 sq_next = first_sample(g);
            for (int cp = g; cp < n_un; cp += FG_G) {
                const int u0 = FG_NT * cp;
                const int k0 = (int)coff[u0], k1 = (int)coff[u0 + 1], k2 = (int)coff[u0 + FG_NT];
                auto grid_one = [&](uint2 sq, int j) {
                    int iv;
                    const float yr = rint_rne(__fmul_rn(__uint_as_float(sq.x), s), iv);
                    if (fabsf(yr) <= lim) {                     // NaN fails; |iu| <= H-1 by construction
                        float2 vv = visrow[sq.y & 0x7fffffffu];
                        if (sq.y >> 31) vv.y = -vv.y;
                        const int tr = FG_NT == 2 && j >= k1;
                        const int n = iv < 0 ? iv + N : iv;     // transform index of centred row iv + H
                        cell_add_exch(&arr[tr * FG_LD + n], vv);
                        if (uniform) atomicAdd(&cnt[tr * (N / 2) + (n >> 1)], 1u << ((n & 1) * 16));
                        if (u0 == 0 && !tr) {                   // iu == 0: the conjugate lies in column 0 too, at row -iv
                            const int n2 = iv > 0 ? N - iv : -iv;
                            cell_add_exch(&arr[n2], make_float2(vv.x, -vv.y));
                            if (uniform) atomicAdd(&cnt[n2 >> 1], 1u << ((n2 & 1) * 16));
                        }
                        ++my_in;
                    }
                };
                // convolutional gridding: sorted sample j seen from the column pair (u0, u0 + 1); transform index of row iv = iv mod N
                auto conv_one = [&](int j) {
                    if constexpr (R > 0) {
                        constexpr int S = 2 * R + 1;
                        int iu0, iv0;
                        const float x = __fmul_rn(__ldg(su + j), s);
                        const float xr = rint_rne(x, iu0);      // in range by construction of the sample range
                        const uint2 sq = __ldg(svb + j);
                        const float y = __fmul_rn(__uint_as_float(sq.x), s);
                        const float yr = rint_rne(y, iv0);
                        if (!(fabsf(yr) <= lim)) return;        // NaN fails
                        const float fx = __fsub_rn(x, xr), fy = __fsub_rn(y, yr);
                        float2 vv = visrow[sq.y & 0x7fffffffu];
                        if (sq.y >> 31) vv.y = -vv.y;
                        float wy[S];
#pragma unroll
                        for (int i = 0; i < S; ++i) {
                            float w = cpoly.c[i][kConvTerms - 1];
#pragma unroll
                            for (int k = kConvTerms - 2; k >= 0; --k) w = fmaf(w, fy, cpoly.c[i][k]);
                            wy[i] = w;
                        }
                        auto add_taps = [&](int tr, int row0, int dir, float ar, float ai) {
#pragma unroll
                            for (int i = 0; i < S; ++i) {
                                const int row = row0 + dir * i;
                                cell_add_take(&arr[tr * FG_LD + (row < 0 ? row + N : row)], make_float2(wy[i] * ar, wy[i] * ai));
                            }
                        };
                        auto wx_of = [&](int jj) {
                            float w = cpoly.c[jj][kConvTerms - 1];
#pragma unroll
                            for (int k = kConvTerms - 2; k >= 0; --k) w = fmaf(w, fx, cpoly.c[jj][k]);
                            return w;
                        };
#pragma unroll
                        for (int k = 0; k < 2; ++k) {
                            const int u = u0 + k;
                            const int jd = u - iu0;             // direct tap that lands in column u
                            if (jd >= -R && jd <= R) {
                                const float wx = wx_of(jd + R);
                                add_taps(k, iv0 - R, 1, wx * vv.x, wx * vv.y);
                                if (jd == 0) ++my_in;           // the sample's own column: counted once
                            }
                            const int jm = -u - iu0;            // tap at column -u, mirrored: conj(V) at row -(iv0 - R + i)
                            if (jm >= -R) {
                                const float wx = wx_of(jm + R);
                                add_taps(k, -(iv0 - R), -1, wx * vv.x, -wx * vv.y);
                            }
                        }
                    }
                };
                gsync();                                        // the arrays are zero (clear_group of the previous unit / image)
                if constexpr (R == 0) {
                    if (k0 + tid < k2) grid_one(sq_next, k0 + tid);
                    for (int j = k0 + tid + FG_TG; j < k2; j += FG_TG) grid_one(__ldg(svb + j), j);
                    sq_next = first_sample(cp + FG_G);          // lands while this unit is transformed
                } else {
                    // samples whose support reaches columns u0, u0 + 1: nearest columns [u0 - R, u0 + 1 + R] (the mirrored taps come
                    // from nearest columns [0, R - u0], a subset); coff[H] = first sample beyond the range
                    const int c0 = (int)coff[u0 > R ? u0 - R : 0], c2 = (int)coff[u0 + 2 + R < H ? u0 + 2 + R : H];
                    for (int j = c0 + tid; j < c2; j += FG_TG) conv_one(j);
                    (void)k0; (void)k1; (void)k2; (void)grid_one; (void)sq_next;
                }
                gsync();
                auto load = [&](int tr, int n) -> float2 {      // a3: divide by the cell count (uniform weighting)
                    float2 v = arr[tr * FG_LD + n];
                    if (uniform) {
                        const uint32_t cn = (cnt[tr * (N / 2) + (n >> 1)] >> ((n & 1) * 16)) & 0xffffu;
                        if (cn) {
                            v.x = __fdiv_rn(v.x, (float)cn);
                            v.y = __fdiv_rn(v.y, (float)cn);
                            my_occ += (u0 + tr == 0) ? 1 : 2;   // the mirror image of a u > 0 cell is occupied too
                        }
                    }
                    return v;
                };
#if BLINK_FG_PAIRED_STORE
                // The last stage leaves a thread with 16 outputs of ONE column; stored straight from the registers they are
                // 8-byte pieces 4800 bytes apart (32 sectors per warp instruction, a quarter of each written).  Through the
                // group's arrays instead: (HT[ky][u0], HT[ky][u0 + 1]) leaves as one 16-byte store, and the slots a thread
                // reads are the slots it zeroes for the next unit (ncu: these stores were the kernel's top lg / mio throttle).
                static_assert(FG_NT == 2, "paired stores want a column pair per group");
                fg_transform2_inplace(arr, stw, tid, gsync, load);      // ends with a group barrier: outputs are in the arrays
                {
                    float4 *dst = reinterpret_cast<float4 *>(HT + u0);  // u0 even, H even: 16-byte aligned
                    for (int ky = tid; ky < N; ky += FG_TG) {
                        const float2 v0 = arr[ky], v1 = arr[FG_LD + ky];
                        arr[ky] = make_float2(0.f, 0.f);
                        arr[FG_LD + ky] = make_float2(0.f, 0.f);
                        dst[(size_t)ky * (H / 2)] = make_float4(v0.x, v0.y, v1.x, v1.y);
                    }
                    if (uniform) for (int i = tid; i < FG_NT * (N / 2); i += FG_TG) cnt[i] = 0u;
                }
#else
                auto emit = [&](int tr, int ky, float2 v) { HT[(size_t)ky * H + u0 + tr] = v; };
                fg_transform2(arr, stw, tid, gsync, load, emit);
                gsync();                                        // the last stage's reads are done: zero for the next unit
                clear_group();
#endif
            }
            if (p == 0) {
#pragma unroll
                for (int d = 16; d > 0; d >>= 1) {
                    my_occ += __shfl_xor_sync(0xffffffffu, my_occ, d);
                    my_in += __shfl_xor_sync(0xffffffffu, my_in, d);
                }
                if (lane == 0) { atomicAdd(&s_occ, my_occ); atomicAdd(&s_nin, my_in); }
            }
            // HT stores (generic proxy) must be visible to the bulk copies (async proxy) of pass 2
            __threadfence();
            asm volatile("fence.proxy.async;" ::: "memory");
            __syncthreads();                                    // (B) pass 1 is over: U turns into the staging buffers
            if (p == 0) wsum_val = uniform ? (float)s_occ : (float)(2 * s_nin);
            if (wsum_val == 0.f) {
                for (int i = threadIdx.x; i < N * N / 4; i += FG_THREADS)
                    reinterpret_cast<float4 *>(img)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
                continue;
            }
            const float inv_w = 1.0f / wsum_val;

            // ================= pass 2: two row pairs per unit -> four real image rows ===================================
            // The four rows HT[ky0 .. ky0+3][0 .. ulim) of a unit are staged by bulk async copies into the group's buffer one
            // unit ahead: the request for unit k+1 goes out right after the barrier that follows unit k's first-stage reads
            // (the only reads of the buffer), so it lands while unit k runs its remaining stages and stores.
            const uint32_t row_bytes = (uint32_t)ulim * 8u;     // ulim is even: a multiple of 16 bytes
            // the buffer holds four rows of up to 600 columns: with ulim <= 300 (the paper's MWA coverage fills ~200) it is
            // split into two halves and the requests run TWO units ahead
            const int nbuf = ulim <= H / 2 ? 2 : 1;
            constexpr int RU = 2 * FG_NT, NU = N / RU;          // rows of HT per unit, units per image
            auto request = [&](int unit, int b) {
                fence_proxy_async();
                mbar_expect_tx(stbar + b, (uint32_t)RU * row_bytes);
#pragma unroll
                for (int r = 0; r < RU; ++r)
                    bulk_load_1d(stg + (size_t)(RU * b + r) * ulim, HT + (size_t)(RU * unit + r) * H, row_bytes, stbar + b);
            };
            if (tid == 0)
                for (int b = 0; b < nbuf; ++b)
                    if (g + b * FG_G < NU) request(g + b * FG_G, b);
            int it = 0;
            for (int unit = g; unit < NU; unit += FG_G, ++it) {
                const int ky0 = RU * unit;
                const int b = nbuf == 2 ? (it & 1) : 0;
                mbar_wait(stbar + b, (sph >> b) & 1u);
                sph ^= 1u << b;
                const float2 *sb = stg + (size_t)(RU * b) * ulim;
                auto load = [&](int tr, int n) -> float2 {
                    const float2 *r0 = sb + (size_t)(2 * tr) * ulim, *r1 = r0 + ulim;
                    if (n < H) {                                // Z[u] = S1 + i S2
                        if (n >= ulim) return make_float2(0.f, 0.f);
                        const float2 s1 = r0[n], s2 = r1[n];
                        return make_float2(s1.x - s2.y, s1.y + s2.x);
                    }
                    const int u = N - n;                        // Z[N - u] = conj(S1) + i conj(S2); u = H is the empty column
                    if (u >= ulim || n == H) return make_float2(0.f, 0.f);
                    const float2 s1 = r0[u], s2 = r1[u];
                    return make_float2(s1.x + s2.y, s2.x - s1.y);
                };
                auto emit = [&](int tr, int j, float2 z) {
                    const int ky = ky0 + 2 * tr;
                    const int y0 = ky < H ? ky + H : ky - H, y1 = ky + 1 < H ? ky + 1 + H : ky + 1 - H;
                    const int x = j < H ? j + H : j - H;        // fftshift of both axes
                    if constexpr (R == 0) {
                        __stcs(img + (size_t)y0 * N + x, z.x * inv_w);
                        __stcs(img + (size_t)y1 * N + x, z.y * inv_w);
                    } else {                                    // grid correction 1 / (c(y) c(x)) rides on the same store
                        const float tx = inv_w * __ldg(cpoly.inv_taper + x);
                        __stcs(img + (size_t)y0 * N + x, z.x * (tx * __ldg(cpoly.inv_taper + y0)));
                        __stcs(img + (size_t)y1 * N + x, z.y * (tx * __ldg(cpoly.inv_taper + y1)));
                    }
                };
                auto after_first_reads = [&] {                  // runs right after the first stage's read -> write barrier
                    if (tid == 0 && unit + nbuf * FG_G < NU) request(unit + nbuf * FG_G, b);
                };
                fg_transform2(arr, stw, tid, gsync, load, emit, after_first_reads);
            }
        }
        if (threadIdx.x == 0) a.wsum[tc] = wsum_val;
    }
}

// ------------------------------------------------------------------------------------------ host
bool fused_g_supported(int B, int n_pix)
{
    return n_pix == FG_N && B <= kFgMaxB && B <= 16384 && FgSmem::bytes(B) <= kSmemLimit;
}
size_t fused_g_workspace_bytes(int T, int B, int ctas)
{
    return sort_bytes(T, B) + align_up((size_t)FG_N * sizeof(float2), 256) + (size_t)ctas * FG_N * FG_H * sizeof(float2);
}
int gfft_fill_twiddles(float2 *dst, int n, cudaStream_t st);      // blink_fftg.cu: dst[m] = exp(2 pi i m / n), evaluated in double

int fused_g_image(const float2 *vis, const float *uvw_m, const double *freqs_hz, double pixscale_rad, int T, int C, int P, int B,
                  int weighting, int tc0, int ntc, float *image, float *wsum, int32_t *cell_idx, void *workspace,
                  size_t workspace_bytes, cudaStream_t st, GainRef cal, const ConvPoly *poly, int R, size_t extra)
{
    // extra: bytes between the sort arrays and the twiddle table that the caller has filled (the conv taper table), 256-aligned
    const size_t per_cta = (size_t)FG_N * FG_H * sizeof(float2);
    const size_t twb = align_up((size_t)FG_N * sizeof(float2), 256);
    const size_t sortb = sort_bytes(T, B) + extra;
    if (R < 0 || R > 3 || (R > 0 && (!poly || weighting != BLINK_W_NATURAL))) return BLINK_ERR_INVALID_ARG;
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u) || workspace_bytes < sortb + twb + per_cta) return BLINK_ERR_WORKSPACE;
    int ctas = option(BLINK_OPT_FUSED_CTAS);
    if (ctas <= 0) ctas = fused_default_ctas();
    ctas = (int)std::min<size_t>((size_t)ctas, (workspace_bytes - sortb - twb) / per_cta);
    unsigned char *wsp = static_cast<unsigned char *>(workspace);
    float *su = reinterpret_cast<float *>(wsp);
    uint2 *svb = reinterpret_cast<uint2 *>(wsp + (sortb - extra) / 3);
    float2 *tw = reinterpret_cast<float2 *>(wsp + sortb);
    float2 *scratch = reinterpret_cast<float2 *>(wsp + sortb + twb);
    int rc = presort_launch(uvw_m, T, B, su, svb, st);
    if (rc != BLINK_OK) return rc;
    rc = gfft_fill_twiddles(tw, FG_N, st);
    if (rc != BLINK_OK) return rc;
    const size_t smem = FgSmem::bytes(B);
    BLINK_CUDA_TRY(cudaFuncSetAttribute(fused_g_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    BLINK_CUDA_TRY(cudaFuncSetAttribute(fused_g_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    BLINK_CUDA_TRY(cudaFuncSetAttribute(fused_g_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    BLINK_CUDA_TRY(cudaFuncSetAttribute(fused_g_kernel<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    ConvPoly cpoly{};
    if (poly) cpoly = *poly;
    FusedArgs base{};
    base.cal = cal;
    base.vis = vis; base.uvw_m = uvw_m; base.T = T; base.C = C; base.P = P; base.B = B; base.weighting = weighting;
    base.image = image; base.wsum = wsum; base.cell_idx = cell_idx;
    return for_channel_blocks(C, tc0, ntc, freqs_hz, FG_N, pixscale_rad,
                              [&](int s0, int m, int c_base, const ScaleBlock &sc) -> int {
                                  FusedArgs a = base;
                                  a.tc0 = s0; a.ntc = m; a.c_base = c_base;
                                  a.scratch = scratch; a.su = su; a.svb = svb;
                                  const int grid = m < ctas ? m : ctas;
                                  if (R == 0) fused_g_kernel<0><<<grid, FG_THREADS, smem, st>>>(a, sc, tw, cpoly);
                                  else if (R == 1) fused_g_kernel<1><<<grid, FG_THREADS, smem, st>>>(a, sc, tw, cpoly);
                                  else if (R == 2) fused_g_kernel<2><<<grid, FG_THREADS, smem, st>>>(a, sc, tw, cpoly);
                                  else fused_g_kernel<3><<<grid, FG_THREADS, smem, st>>>(a, sc, tw, cpoly);
                                  BLINK_LAUNCH_CHECK("fused_g_kernel");
                                  return (int)BLINK_OK;
                              });
}

}  // namespace blink
