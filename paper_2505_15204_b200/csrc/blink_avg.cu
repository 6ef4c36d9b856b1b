// blink_image_avg: dirty images averaged over fine channels (and optionally timesteps).
//
// PAPER.md L284 "Images belonging to the same time bin are averaged together", L251 "averaged in time over
// the entire processed time frame and frequency over the 30.72 MHz bandwidth".  The mean of the normalised
// images, A = (1/n) sum_{t,c} Re F[G_tc] / W_tc, is by linearity of the transform ONE transform of the combined
// grid sum_{t,c} G_tc / (n W_tc) (every channel is gridded in its own cell units, which is exactly what makes
// all images share one pixel grid, R3/R14).  So instead of 38400 transforms and a 40 GB image stream
// per second of data the path is: one pass over the visibilities that scatters each sample (and its conjugate),
// pre-multiplied by its weight, into T*P (or P) L2-resident combined grids with vector atomics
// (red.global.add.v2.f32), then the unfused batched transform (blink_fft2d.cu) of those few grids.
#include <algorithm>

#include "blink_common.cuh"
#include "blink_sort.cuh"

namespace blink {

int presort_launch(const float *uvw_m, int T, int B, float *su, uint2 *svb, cudaStream_t st);      // blink_fused.cu
size_t sort_bytes(int T, int B);

constexpr int kAvgThreads = 256;
// avg_grid_kernel: an item is a chain of returning L2 atomics per thread (ncu: 3 % issue-active, 133 us per (t,c) with 256 threads
// at 10296 baselines = 40 samples per thread): 1024 threads keep four times as many of them in flight
constexpr int kAvgGridThreads = 1024;

struct AvgArgs {
    const float2 *vis; const float *uvw_m;
    int T, C, P, B, n, weighting, avg_time;
    int tc0, ntc, c_base;
    float2 *grid;                 // [n_out][n][n] combined grids, centred, zeroed by the caller
    float *wsum;                  // [T*C]
    uint32_t *cnt;                // uniform weighting: [gridDim.x][n*n] count planes, all zero between items
    float inv_navg;               // 1 / (number of images per output)
    float *wq;                    // uniform, fast route: [T*C][B] weight of every sample, 1 / (n W count) or 0 (else NULL)
};

// One persistent CTA per (t,c) item.  Sweep 1 finds the weight sum W of the item (natural: samples placed;
// uniform: occupied cells, counted exactly as "first arrival" on a per-CTA count plane); sweep 2 adds every
// sample times 1 / (n W) (uniform: also / count of its cell) to the combined grid of its output image.
__global__ void __launch_bounds__(kAvgGridThreads)
avg_grid_kernel(const AvgArgs a, const __grid_constant__ ScaleBlock sc)
{
    __shared__ int s_in[kAvgGridThreads / 32], s_first[kAvgGridThreads / 32];
    const bool uniform = a.weighting == BLINK_W_UNIFORM;
    const int n = a.n, h = n / 2, B = a.B;
    const size_t n2 = (size_t)n * n;
    uint32_t *cnt = uniform ? a.cnt + (size_t)blockIdx.x * n2 : nullptr;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int tc = a.tc0 + blockIdx.x; tc < a.tc0 + a.ntc; tc += gridDim.x) {
        const int t = tc / a.C, c = tc - t * a.C;
        const float s = sc.s[c - a.c_base];
        const float *uvw = a.uvw_m + (size_t)t * B * 3;
        // ---- sweep 1: weight sum ---------------------------------------------------------------------
        int n_in = 0, n_first = 0;
        for (int b = threadIdx.x; b < B; b += kAvgGridThreads) {
            const int cell = cell_of(uvw[3 * b], uvw[3 * b + 1], s, n, h);
            if (cell >= 0) {
                ++n_in;
                if (uniform) {
                    n_first += atomicAdd(&cnt[cell], 1u) == 0u;
                    n_first += atomicAdd(&cnt[mirror_of(cell, n)], 1u) == 0u;
                }
            }
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            n_in += __shfl_xor_sync(0xffffffffu, n_in, d);
            n_first += __shfl_xor_sync(0xffffffffu, n_first, d);
        }
        if (lane == 0) { s_in[warp] = n_in; s_first[warp] = n_first; }
        __syncthreads();
        n_in = 0; n_first = 0;
#pragma unroll
        for (int k = 0; k < kAvgGridThreads / 32; ++k) { n_in += s_in[k]; n_first += s_first[k]; }
        const float W = uniform ? (float)n_first : (float)(2 * n_in);
        if (threadIdx.x == 0) a.wsum[tc] = W;
        // ---- sweep 2 ------------------------------------------------------------------------------------
        if (a.wq) {                                                     // fast route: only the per-sample weights; the
            const float wbase = W > 0.f ? a.inv_navg / W : 0.f;         // run-length scatter kernel does the adding
            for (int b = threadIdx.x; b < B; b += kAvgGridThreads) {
                const int cell = cell_of(uvw[3 * b], uvw[3 * b + 1], s, n, h);
                a.wq[(size_t)tc * B + b] = cell >= 0 ? wbase / (float)__ldcg(&cnt[cell]) : 0.f;
            }
        } else if (W > 0.f) {                                           // weighted scatter into the combined grids
            const float wbase = a.inv_navg / W;
            for (int b = threadIdx.x; b < B; b += kAvgGridThreads) {
                const int cell = cell_of(uvw[3 * b], uvw[3 * b + 1], s, n, h);
                if (cell < 0) continue;
                const int mir = mirror_of(cell, n);
                float w1 = wbase, w2 = wbase;
                if (uniform) {                                          // the counts live in L2 (atomics): bypass L1
                    w1 = wbase / (float)__ldcg(&cnt[cell]);
                    w2 = wbase / (float)__ldcg(&cnt[mir]);
                }
                for (int p = 0; p < a.P; ++p) {
                    const float2 v = a.vis[((size_t)tc * a.P + p) * B + b];
                    float2 *g = a.grid + (size_t)(a.avg_time ? p : t * a.P + p) * n2;
                    atomicAdd(&g[cell], make_float2(v.x * w1, v.y * w1));
                    atomicAdd(&g[mir], make_float2(v.x * w2, -v.y * w2));
                }
            }
        }
        if (uniform) {                                                  // leave the count plane clean for the next item
            __syncthreads();
            for (int b = threadIdx.x; b < B; b += kAvgGridThreads) {
                const int cell = cell_of(uvw[3 * b], uvw[3 * b + 1], s, n, h);
                if (cell >= 0) {
                    __stcg(&cnt[cell], 0u);
                    __stcg(&cnt[mirror_of(cell, n)], 0u);
                }
            }
            __threadfence();
        }
        __syncthreads();
    }
}

// ---- uniform weighting, column route: per-sample weights WITHOUT count planes or global atomics ----------------------
// avg_grid_kernel counts on a 4 N^2-byte plane per CTA with returning L2 atomics, a chain of round trips per thread (ncu: 3-6 %
// issue-active, 0.54-0.80 of the 1.13-1.40 ms of a config-4 timestep).  With the baselines of a timestep sorted by |u| and folded
// into the half plane u >= 0 (the fused kernels' presort: su = |u|, svb = {sign(u) v, b | conj << 31}), the samples of one grid
// COLUMN are a contiguous range for every channel, so a warp counts a column in an N-entry shared-memory array, reads the counts
// back for its samples and zeroes what it touched.  A half-plane cell's count is the full plane's count of that cell (a sample with
// u < 0 sits on its conjugate's cell), column 0 takes the sample and its conjugate, and newly occupied cells count twice off the
// axis (cell + mirror): W and every weight are exactly those of avg_grid_kernel.
constexpr int kAvgColThreads = 256, kAvgColWarps = kAvgColThreads / 32;
static size_t avg_col_smem(int n) { return ((size_t)(n / 2 + 2 + 3) / 4 * 4 + (size_t)kAvgColWarps * n) * sizeof(uint32_t); }
__global__ void __launch_bounds__(kAvgColThreads)
avg_uniform_cols_kernel(const AvgArgs a, const __grid_constant__ ScaleBlock sc, const float *__restrict__ su_all,
                        const uint2 *__restrict__ svb_all)
{
    extern __shared__ uint32_t col_sm[];
    __shared__ int s_first[kAvgColWarps];
    __shared__ int s_ncol;                                              // occupied columns are [0, s_ncol)
    const int n = a.n, H = n / 2, B = a.B;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t *coff = col_sm;                                            // [H + 2]: first sorted sample of column u
    uint32_t *cw = col_sm + (H + 2 + 3) / 4 * 4 + (size_t)warp * n;    // this warp's count column
    const float lim = (float)(H - 1);
    for (int i = threadIdx.x; i < kAvgColWarps * n; i += kAvgColThreads) col_sm[(H + 2 + 3) / 4 * 4 + i] = 0u;
    for (int tc = a.tc0 + blockIdx.x; tc < a.tc0 + a.ntc; tc += gridDim.x) {
        const int t = tc / a.C, c = tc - t * a.C;
        const float s = sc.s[c - a.c_base];
        const float *su = su_all + (size_t)t * B;
        const uint2 *svb = svb_all + (size_t)t * B;
        float *wq = a.wq + (size_t)tc * B;
        auto col_of = [&](float x) -> int {
            int i;
            const float xr = rint_rne(__fmul_rn(x, s), i);
            return (xr <= lim) ? i : H;                                 // NaN: H
        };
        __syncthreads();                                                // the previous item's readers of coff are done
        for (int j = threadIdx.x; j <= B; j += kAvgColThreads) {
            const int cj = j < B ? col_of(__ldg(su + j)) : H + 1;
            const int cq = j > 0 ? col_of(__ldg(su + j - 1)) : -1;
            for (int u = cq + 1; u <= cj; ++u) coff[u] = (uint32_t)j;
            if (cj >= H && cq < H) s_ncol = cq + 1;                     // exactly one j sees the step off the grid
        }
        __syncthreads();
        const int ncol = s_ncol;
        int n_first = 0;
        // a column holds a handful of samples (10296 baselines over ~700 occupied columns): the common case is ONE sample per lane,
        // fetched once -- and one column ahead -- and kept in registers through the three steps (count, read back, clear); the first
        // version re-read svb from L2 in each step and spent 0.18 ms per config-4 timestep waiting for those loads
        auto fetch = [&](int u_, int &k0_, int &k1_) -> uint2 {
            k0_ = k1_ = 0;
            if (u_ < ncol) { k0_ = (int)coff[u_]; k1_ = (int)coff[u_ + 1]; }
            return (k0_ + lane < k1_) ? __ldg(svb + k0_ + lane) : make_uint2(0u, 0u);
        };
        int k0n, k1n;
        uint2 sqn = fetch(warp, k0n, k1n);
        for (int u = warp; u < ncol; u += kAvgColWarps) {
            const int k0 = k0n, k1 = k1n;
            const uint2 sq0 = sqn;
            sqn = fetch(u + kAvgColWarps, k0n, k1n);
            if (k0 == k1) continue;
            if (k1 - k0 <= 32) {
                int iv = 0;
                bool ok = false;
                if (k0 + lane < k1) {
                    const float yr = rint_rne(__fmul_rn(__uint_as_float(sq0.x), s), iv);
                    ok = fabsf(yr) <= lim;
                }
                if (ok) {
                    n_first += (atomicAdd(&cw[iv + H], 1u) == 0u) ? (u == 0 ? 1 : 2) : 0;
                    if (u == 0) n_first += atomicAdd(&cw[H - iv], 1u) == 0u;
                }
                __syncwarp();
                if (k0 + lane < k1) wq[sq0.y & 0x7fffffffu] = ok ? (float)cw[iv + H] : 0.f;
                __syncwarp();
                if (ok) {
                    cw[iv + H] = 0u;
                    if (u == 0) cw[H - iv] = 0u;
                }
                __syncwarp();
                continue;
            }
            for (int j = k0 + lane; j < k1; j += 32) {                  // count
                int iv;
                const float yr = rint_rne(__fmul_rn(__uint_as_float(__ldg(&svb[j].x)), s), iv);
                if (fabsf(yr) <= lim) {
                    n_first += (atomicAdd(&cw[iv + H], 1u) == 0u) ? (u == 0 ? 1 : 2) : 0;
                    if (u == 0) n_first += atomicAdd(&cw[H - iv], 1u) == 0u;
                }
            }
            __syncwarp();
            for (int j = k0 + lane; j < k1; j += 32) {                  // read back: the count of every sample's cell, as a float
                int iv;
                const uint2 sq = __ldg(svb + j);
                const float yr = rint_rne(__fmul_rn(__uint_as_float(sq.x), s), iv);
                wq[sq.y & 0x7fffffffu] = fabsf(yr) <= lim ? (float)cw[iv + H] : 0.f;
            }
            __syncwarp();
            for (int j = k0 + lane; j < k1; j += 32) {                  // leave the column clean
                int iv;
                const float yr = rint_rne(__fmul_rn(__uint_as_float(__ldg(&svb[j].x)), s), iv);
                if (fabsf(yr) <= lim) {
                    cw[iv + H] = 0u;
                    if (u == 0) cw[H - iv] = 0u;
                }
            }
            __syncwarp();
        }
        for (int j = (int)coff[H] + threadIdx.x; j < B; j += kAvgColThreads) wq[__ldg(&svb[j].y) & 0x7fffffffu] = 0.f;   // off the grid in u
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) n_first += __shfl_xor_sync(0xffffffffu, n_first, d);
        if (lane == 0) s_first[warp] = n_first;
        __syncthreads();                                                // also: every count of this item is in wq
        n_first = 0;
#pragma unroll
        for (int k = 0; k < kAvgColWarps; ++k) n_first += s_first[k];
        const float W = (float)n_first;
        if (threadIdx.x == 0) a.wsum[tc] = W;
        const float wbase = W > 0.f ? a.inv_navg / W : 0.f;
        for (int b = threadIdx.x; b < B; b += kAvgColThreads) {
            const float cnt = __ldcg(wq + b);                           // written by other warps of this CTA: read it from L2
            wq[b] = cnt > 0.f ? wbase / cnt : 0.f;
        }
    }
}

// ---- natural weighting: run-length scatter --------------------------------------------------------------
// W of every (t,c) first (cells only, no visibilities).  Same thread layout as the scatter below: one thread per
// (baseline, timestep, chunk of channels) keeps (u, v) in registers and walks the channels; a warp's 32 baselines
// are counted with one ballot per channel into shared counters, flushed with one global atomic per channel.
constexpr int kAvgChunk = 128;
// |x| against the grid edge h - 1/2 with round-to-nearest-even at the tie: rint(h - 1/2) is h (off the grid) for even h
// and h-1 (on the grid) for odd h
__device__ __forceinline__ bool on_grid_edge(float x, float edge, int h) { return (h & 1) ? (x <= edge) : (x < edge); }
__global__ void __launch_bounds__(kAvgThreads)
avg_count_kernel(const AvgArgs a, const __grid_constant__ ScaleBlock sc, unsigned *__restrict__ n_in, int t_lo, int c_lo, int nc,
                 int nchunk, int bblocks)
{
    __shared__ unsigned s_cnt[kAvgChunk];
    const int bx = (int)(blockIdx.x % (unsigned)bblocks);
    int y = (int)(blockIdx.x / (unsigned)bblocks);
    const int k = y % nchunk;
    const int t = t_lo + y / nchunk;
    const int b = bx * kAvgThreads + threadIdx.x;
    for (int i = threadIdx.x; i < kAvgChunk; i += kAvgThreads) s_cnt[i] = 0u;
    __syncthreads();
    const int n = a.n, h = n / 2;
    // A sample is on the grid iff |rint(u s)| <= h-1 and |rint(v s)| <= h-1.  For even h, h-1 is odd and the tie
    // |x| = h-1/2 rounds away to h: the test is |u s| < h - 1/2 on the fp32 products; for odd h (N = 2 mod 4) the tie
    // rounds to the even h-1 and stays on the grid: |u s| <= h - 1/2 (on_grid_edge).  Because fp32 multiplication by
    // s > 0 is monotone it is ONE product: max(|u|, |v|) * s against h - 1/2 (NaN in either coordinate fails).
    float m_uv = __int_as_float(0x7fc00000);                            // NaN: never on the grid
    if (b < a.B) {
        const float u = a.uvw_m[((size_t)t * a.B + b) * 3], v = a.uvw_m[((size_t)t * a.B + b) * 3 + 1];
        m_uv = (u == u && v == v) ? fmaxf(fabsf(u), fabsf(v)) : m_uv;
    }
    (void)n;
    const float edge = (float)h - 0.5f;
    const int c0 = c_lo + k * kAvgChunk, c1 = min(c0 + kAvgChunk, c_lo + nc);
    for (int c = c0; c < c1; ++c) {
        const unsigned m = __ballot_sync(0xffffffffu, on_grid_edge(__fmul_rn(m_uv, sc.s[c - a.c_base]), edge, h));
        if ((threadIdx.x & 31) == 0 && m) atomicAdd(&s_cnt[c - c0], (unsigned)__popc(m));
    }
    __syncthreads();
    for (int i = threadIdx.x; i < c1 - c0; i += kAvgThreads)
        if (s_cnt[i]) atomicAdd(&n_in[(size_t)t * a.C + c0 + i], s_cnt[i]);
}
// Faster route to the same counts when a timestep's baselines fit in shared memory: the predicate
// max(|u|,|v|) * s < h - 1/2 is monotone in max(|u|,|v|), so sort that key once per timestep (bitonic, keys only)
// and the count of every channel is ONE binary search with the exact predicate.
constexpr int kAvgSortMaxB = 16384;
__global__ void __launch_bounds__(1024) avg_sortm_kernel(const float *__restrict__ uvw_m, int B, int np2, float *__restrict__ sorted_m)
{
    extern __shared__ float key[];
    const float *uvw = uvw_m + (size_t)blockIdx.x * B * 3;
    for (int i = threadIdx.x; i < np2; i += 1024) {
        float k = __int_as_float(0x7f800000);                            // +inf: padding, NaN coordinates
        if (i < B) {
            const float u = uvw[3 * i], v = uvw[3 * i + 1];
            if (u == u && v == v) k = fmaxf(fabsf(u), fabsf(v));
        }
        key[i] = k;
    }
    __syncthreads();
    for (int k = 2; k <= np2; k <<= 1)
        for (int j = k >> 1; j > 0; j >>= 1) {
            for (int i = threadIdx.x; i < np2; i += 1024) {
                const int x = i ^ j;
                if (x > i) {
                    const float p = key[i], q = key[x];
                    if ((p > q) == ((i & k) == 0)) { key[i] = q; key[x] = p; }
                }
            }
            __syncthreads();
        }
    for (int i = threadIdx.x; i < B; i += 1024) sorted_m[(size_t)blockIdx.x * B + i] = key[i];
}
// the same with the keys in registers (blink_sort.cuh) for EPT * 512 < B <= EPT * 1024
template <int EPT>
__global__ void __launch_bounds__(1024) avg_sortm_regs_kernel(const float *__restrict__ uvw_m, int B, float *__restrict__ sorted_m)
{
    extern __shared__ float key_s[];
    const float *uvw = uvw_m + (size_t)blockIdx.x * B * 3;
    float key[EPT];
    uint32_t val[EPT];
#pragma unroll
    for (int r = 0; r < EPT; ++r) {
        const int i = r * 1024 + (int)threadIdx.x;
        float k = __int_as_float(0x7f800000);                            // +inf: padding, NaN coordinates
        if (i < B) {
            const float u = uvw[3 * i], v = uvw[3 * i + 1];
            if (u == u && v == v) k = fmaxf(fabsf(u), fabsf(v));
        }
        key[r] = k;
        val[r] = 0u;
    }
    block_bitonic_sort<EPT, false>(key, val, key_s, nullptr);
#pragma unroll
    for (int r = 0; r < EPT; ++r) key_s[threadIdx.x * EPT + r] = key[r];
    __syncthreads();
    for (int i = threadIdx.x; i < B; i += 1024) sorted_m[(size_t)blockIdx.x * B + i] = key_s[i];
}
__global__ void avg_wsearch_kernel(const AvgArgs a, const __grid_constant__ ScaleBlock sc, const float *__restrict__ sorted_m,
                                   float *__restrict__ winv)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.ntc) return;
    const int tc = a.tc0 + i;
    const int t = tc / a.C, c = tc - t * a.C;
    const int h = a.n / 2;
    const float s = sc.s[c - a.c_base], edge = (float)h - 0.5f;
    const float *m = sorted_m + (size_t)t * a.B;
    int lo = 0, hi = a.B;                                               // first index whose sample is off the grid
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (on_grid_edge(__fmul_rn(__ldg(m + mid), s), edge, h)) lo = mid + 1; else hi = mid;
    }
    const float W = (float)(2 * lo);
    a.wsum[tc] = W;
    winv[tc] = lo > 0 ? a.inv_navg / W : 0.f;
}
// wsum[tc] = 2 * samples placed, winv[tc] = 1 / (n W) or 0 (in place over the counters)
__global__ void avg_winv_kernel(const AvgArgs a, float *__restrict__ winv)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.ntc) return;
    const int tc = a.tc0 + i;
    const unsigned n_in = reinterpret_cast<const unsigned *>(winv)[tc];
    const float W = (float)(2u * n_in);
    a.wsum[tc] = W;
    winv[tc] = n_in > 0u ? a.inv_navg / W : 0.f;
}

// One thread per (baseline, timestep, polarisation, chunk of kAvgChunk channels).  Along the channel axis a
// baseline's cell moves slowly (the scale changes by 2.6e-4 per 40 kHz channel), so the thread keeps the
// weighted sum of the current cell in registers and only touches the grid when the cell changes: ~20-60x fewer
// atomics than one per sample.  Visibility reads stay coalesced (baseline is the fastest axis of vis).
// WQ: per-sample weights wq [T*C][B] (uniform weighting) instead of one weight per (t,c) (natural: winv [T*C])
template <bool WQ>
__global__ void __launch_bounds__(kAvgThreads)
avg_scatter_runs_kernel(const AvgArgs a, const __grid_constant__ ScaleBlock sc, const float *__restrict__ winv,
                        const float *__restrict__ wq, int t_lo,
                        int c_lo, int nc, int nchunk, int bblocks)
{
    const int bx = (int)(blockIdx.x % (unsigned)bblocks);
    int y = (int)(blockIdx.x / (unsigned)bblocks);
    const int k = y % nchunk; y /= nchunk;
    const int p = y % a.P;
    const int t = t_lo + y / a.P;
    const int b = bx * kAvgThreads + threadIdx.x;
    if (b >= a.B) return;
    const int n = a.n, h = n / 2;
    const size_t n2 = (size_t)n * n;
    const float u = a.uvw_m[((size_t)t * a.B + b) * 3], v = a.uvw_m[((size_t)t * a.B + b) * 3 + 1];
    float2 *g = a.grid + (size_t)(a.avg_time ? p : t * a.P + p) * n2;
    const int c0 = c_lo + k * kAvgChunk, c1 = min(c0 + kAvgChunk, c_lo + nc);
    int cur = -1;
    float2 acc = make_float2(0.f, 0.f);
    auto flush = [&] {
        if (cur >= 0) {
            atomicAdd(&g[cur], acc);
            atomicAdd(&g[mirror_of(cur, n)], make_float2(acc.x, -acc.y));
        }
    };
    // ncu: this kernel is bound by instruction issue (83 % issue-active, 75 thread instructions per sample at first, most of
    // them 64-bit address arithmetic), not by its loads or atomics.  So: running pointers with 32-bit strides, and the cell is
    // re-derived only when the rounded coordinates change -- the integer part of x + 1.5 * 2^23 sits in the mantissa of the sum
    // (rint_rne), cell_of() is a function of these two sums alone, so equal bits = same cell, same range decision.
    constexpr int kAvgAhead = 8;
    const unsigned vs = (unsigned)a.P * (unsigned)a.B;          // elements between consecutive channels of one (t, p, b)
    const float2 *vp = a.vis + ((size_t)(t * a.C + c0) * a.P + p) * a.B + b;
    const float *wp = WQ ? wq + ((size_t)t * a.C + c0) * a.B + b : winv + (size_t)t * a.C + c0;
    const unsigned ws = WQ ? (unsigned)a.B : 1u;
    const float *sp = sc.s + (c0 - a.c_base);
    int kx = 0x7fc00001, ky = 0x7fc00001;                       // bit patterns no valid sum has
    auto step = [&](float s, float2 x, float w) {
        const int bx = __float_as_int(__fadd_rn(__fmul_rn(u, s), 12582912.0f));
        const int by = __float_as_int(__fadd_rn(__fmul_rn(v, s), 12582912.0f));
        if (bx != kx || by != ky) {
            kx = bx;
            ky = by;
            const int cell = cell_of(u, v, s, n, h);
            if (cell != cur) {
                flush();
                cur = cell;
                acc = make_float2(0.f, 0.f);
            }
        }
        if (cur >= 0) {
            acc.x = fmaf(x.x, w, acc.x);
            acc.y = fmaf(x.y, w, acc.y);
        }
    };
    int c = c0;
    for (; c + kAvgAhead <= c1; c += kAvgAhead) {
        float2 x[kAvgAhead];
        float w[kAvgAhead];
#pragma unroll
        for (int j = 0; j < kAvgAhead; ++j) {
            x[j] = __ldcs(vp + (size_t)((unsigned)j * vs));
            if constexpr (WQ) w[j] = __ldcs(wp + (size_t)((unsigned)j * ws));
            else w[j] = __ldg(wp + j);
        }
#pragma unroll
        for (int j = 0; j < kAvgAhead; ++j) step(sp[j], x[j], w[j]);
        vp += (size_t)(kAvgAhead * vs);
        wp += (size_t)(kAvgAhead * ws);
        sp += kAvgAhead;
    }
    for (; c < c1; ++c) {
        step(*sp, __ldcs(vp), WQ ? __ldcs(wp) : __ldg(wp));
        vp += vs;
        wp += ws;
        ++sp;
    }
    flush();
}

static size_t avg_grid_bytes(int T, int P, int n_pix, int avg_time)
{
    // the combined grids, then (sides that are not a power of two) the transform's twiddle table
    return align_up((size_t)(avg_time ? 1 : T) * P * n_pix * n_pix * sizeof(float2), 256) + gfft_workspace_bytes(n_pix);
}
static int avg_max_planes() { return 2 * (sm_count() > 0 ? sm_count() : 148); }
// workspace: combined grids | natural: winv [T*C] float | uniform: count planes
size_t avg_workspace_bytes(int T, int C, int P, int B, int n_pix, int weighting, bool minimum)
{
    size_t b = avg_grid_bytes(T, P, n_pix, 0);
    if (weighting == BLINK_W_NATURAL) b += align_up((size_t)T * C * sizeof(float), 256) + (minimum ? 0 : align_up((size_t)T * B * sizeof(float), 256));
    if (weighting == BLINK_W_UNIFORM) {
        const size_t plane = (size_t)n_pix * n_pix * sizeof(uint32_t);
        size_t planes = minimum ? 1 : (size_t)avg_max_planes();
        if (!minimum) planes = std::max<size_t>(1, std::min<size_t>(planes, ((size_t)2 << 30) / plane));
        b += planes * plane;
        if (!minimum) b += align_up((size_t)T * C * B * sizeof(float), 256);   // per-sample weights: the run-length scatter route
        if (!minimum && B <= 16384) b += sort_bytes(T, B);                      // baselines sorted by |u|: the column route
    }
    return b;
}

}  // namespace blink

using namespace blink;

extern "C" int blink_image_avg(const blink_c64 *vis, const float *uvw_m, const double *freqs_hz, int T, int C, int P, int B,
                               int n_pix, double pixscale_rad, int weighting, int avg_time, float *image_avg, float *wsum,
                               void *workspace, size_t workspace_bytes, void *stream)
{
    if (!vis || !uvw_m || !freqs_hz || !image_avg || !wsum) return BLINK_ERR_INVALID_ARG;
    if (T < 1 || C < 1 || P < 1 || B < 1 || !(pixscale_rad > 0.0)) return BLINK_ERR_INVALID_ARG;
    if (weighting != BLINK_W_NATURAL && weighting != BLINK_W_UNIFORM) return BLINK_ERR_INVALID_ARG;
    if (!size_supported(n_pix) || B > kMaxBaselines) return BLINK_ERR_UNSUPPORTED;
    if ((long long)T * C * P > 0x3fffffffLL) return BLINK_ERR_UNSUPPORTED;
    if (!aligned16(vis) || !aligned16(image_avg)) return BLINK_ERR_INVALID_ARG;
    int rc = ensure_device();
    if (rc != BLINK_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const bool uni = weighting == BLINK_W_UNIFORM;
    const size_t n2 = (size_t)n_pix * n_pix;
    const size_t gbytes = avg_grid_bytes(T, P, n_pix, avg_time ? 1 : 0);
    const size_t plane = n2 * sizeof(uint32_t);
    const size_t winv_bytes = align_up((size_t)T * C * sizeof(float), 256);
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u) || workspace_bytes < gbytes + (uni ? plane : winv_bytes))
        return BLINK_ERR_WORKSPACE;
    float *winv = reinterpret_cast<float *>(static_cast<unsigned char *>(workspace) + gbytes);   // natural only
    // sorted max(|u|,|v|) per timestep, when it fits in shared memory and in the workspace (else: ballot counting)
    float *sorted_m = nullptr;
    const size_t sm_bytes = align_up((size_t)T * B * sizeof(float), 256);
    // (the sort costs ~0.1 ms whatever the batch: only worth it for large batches)
    const int wopt = option(BLINK_OPT_AVG_WSUM);
    const bool want_sort = wopt == 1 || (wopt == 0 && (long long)T * C * B >= (32LL << 20));
    if (!uni && want_sort && B <= kAvgSortMaxB && workspace_bytes >= gbytes + winv_bytes + sm_bytes) {
        sorted_m = reinterpret_cast<float *>(static_cast<unsigned char *>(workspace) + gbytes + winv_bytes);
        int np2 = 1;
        while (np2 < B) np2 <<= 1;
        if (np2 == 8192) {
            BLINK_CUDA_TRY(cudaFuncSetAttribute(avg_sortm_regs_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, np2 * 4));
            avg_sortm_regs_kernel<8><<<T, 1024, (size_t)np2 * 4, st>>>(uvw_m, B, sorted_m);
        } else if (np2 == 16384) {
            BLINK_CUDA_TRY(cudaFuncSetAttribute(avg_sortm_regs_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, np2 * 4));
            avg_sortm_regs_kernel<16><<<T, 1024, (size_t)np2 * 4, st>>>(uvw_m, B, sorted_m);
        } else {
            BLINK_CUDA_TRY(cudaFuncSetAttribute(avg_sortm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, np2 * 4));
            avg_sortm_kernel<<<T, 1024, (size_t)np2 * 4, st>>>(uvw_m, B, np2, sorted_m);
        }
        BLINK_LAUNCH_CHECK("avg_sortm_kernel");
    }
    float2 *grid = static_cast<float2 *>(workspace);
    uint32_t *cnt = uni ? reinterpret_cast<uint32_t *>(static_cast<unsigned char *>(workspace) + gbytes) : nullptr;
    int ctas = 8 * (sm_count() > 0 ? sm_count() : 148);
    // uniform, fast route: per-sample weights [T*C][B] behind the count planes, when the workspace has room for them
    float *wq = nullptr;
    const size_t wq_bytes = align_up((size_t)T * C * B * sizeof(float), 256);
    if (uni) {
        size_t avail = workspace_bytes - gbytes;
        if (avail >= plane + wq_bytes) {
            ctas = (int)std::min<size_t>((size_t)avg_max_planes(), (avail - wq_bytes) / plane);
            wq = reinterpret_cast<float *>(static_cast<unsigned char *>(workspace) + gbytes + (size_t)ctas * plane);
        } else {
            ctas = (int)std::min<size_t>((size_t)avg_max_planes(), avail / plane);
        }
    }
    // uniform, column route: grid | per-sample weights | sorted baselines; no count planes
    const float *col_su = nullptr;
    const uint2 *col_svb = nullptr;
    int col_ctas = 0;
    if (uni && B <= 16384 && n_pix <= 4096 && option(BLINK_OPT_AVG_WSUM) != 2 &&
        workspace_bytes >= gbytes + wq_bytes + sort_bytes(T, B)) {
        unsigned char *wsp = static_cast<unsigned char *>(workspace) + gbytes;
        wq = reinterpret_cast<float *>(wsp);
        float *su = reinterpret_cast<float *>(wsp + wq_bytes);
        uint2 *svb = reinterpret_cast<uint2 *>(wsp + wq_bytes + sort_bytes(T, B) / 3);
        int rc2 = presort_launch(uvw_m, T, B, su, svb, st);
        if (rc2 != BLINK_OK) return rc2;
        col_su = su; col_svb = svb;
        const size_t csm = avg_col_smem(n_pix);
        BLINK_CUDA_TRY(cudaFuncSetAttribute(avg_uniform_cols_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)csm));
        const int per_sm = (int)std::max<size_t>(1, std::min<size_t>(8, ((size_t)227 * 1024) / (csm + 1024)));
        col_ctas = per_sm * (sm_count() > 0 ? sm_count() : 148);
    }
    BLINK_CUDA_TRY(cudaMemsetAsync(grid, 0, gbytes, st));
    if (uni && !col_su) BLINK_CUDA_TRY(cudaMemsetAsync(cnt, 0, (size_t)ctas * plane, st));
    const int n_out = (avg_time ? 1 : T) * P;
    int tc = 0;
    const int tc_end = T * C;
    while (tc < tc_end) {                                       // blocks of <= 1024 channels (scales travel as a kernel parameter)
        const int t = tc / C, c = tc - t * C;
        const int c_base = (c / 1024) * 1024;
        const int c_lim = c_base + 1024 < C ? c_base + 1024 : C;
        const int end = (C <= 1024) ? tc_end : t * C + c_lim;
        ScaleBlock sc;
        for (int k = 0; k < 1024; ++k) sc.s[k] = (c_base + k < C) ? scale_for(freqs_hz[c_base + k], n_pix, pixscale_rad) : 0.f;
        AvgArgs a{};
        a.vis = reinterpret_cast<const float2 *>(vis); a.uvw_m = uvw_m;
        a.T = T; a.C = C; a.P = P; a.B = B; a.n = n_pix; a.weighting = weighting; a.avg_time = avg_time ? 1 : 0;
        a.tc0 = tc; a.ntc = end - tc; a.c_base = c_base;
        a.grid = grid; a.wsum = wsum; a.cnt = cnt;
        a.inv_navg = (float)(1.0 / (avg_time ? (double)T * C : (double)C));
        a.wq = wq;
        if (uni) {
            if (col_su) {
                const int gridx = a.ntc < col_ctas ? a.ntc : col_ctas;
                avg_uniform_cols_kernel<<<gridx, kAvgColThreads, avg_col_smem(n_pix), st>>>(a, sc, col_su, col_svb);
                BLINK_LAUNCH_CHECK("avg_uniform_cols_kernel");
            } else {
                const int gridx = a.ntc < ctas ? a.ntc : ctas;
                avg_grid_kernel<<<gridx, kAvgGridThreads, 0, st>>>(a, sc);
                BLINK_LAUNCH_CHECK("avg_grid_kernel");
            }
            if (wq) {
                const int nt = (C <= 1024) ? T : 1, nc = (C <= 1024) ? C : a.ntc;
                const int nchunk = (nc + kAvgChunk - 1) / kAvgChunk, bblocks = (B + kAvgThreads - 1) / kAvgThreads;
                const long long blocks = (long long)bblocks * nchunk * P * nt;
                if (blocks > 0x7fffffffLL) return BLINK_ERR_UNSUPPORTED;
                avg_scatter_runs_kernel<true><<<(unsigned)blocks, kAvgThreads, 0, st>>>(a, sc, nullptr, wq, t, c, nc, nchunk, bblocks);
                BLINK_LAUNCH_CHECK("avg_scatter_runs_kernel");
            }
        } else {
            // this segment: all timesteps x all channels (C <= 1024) or one timestep x one block of channels
            const int nt = (C <= 1024) ? T : 1, nc = (C <= 1024) ? C : a.ntc;
            const int nchunk = (nc + kAvgChunk - 1) / kAvgChunk, bblocks = (B + kAvgThreads - 1) / kAvgThreads;
            if ((long long)bblocks * nchunk * nt > 0x7fffffffLL) return BLINK_ERR_UNSUPPORTED;
            if (sorted_m) {
                avg_wsearch_kernel<<<(a.ntc + 255) / 256, 256, 0, st>>>(a, sc, sorted_m, winv);
                BLINK_LAUNCH_CHECK("avg_wsearch_kernel");
            } else {
                BLINK_CUDA_TRY(cudaMemsetAsync(winv + tc, 0, (size_t)a.ntc * sizeof(float), st));
                avg_count_kernel<<<(unsigned)(bblocks * nchunk * nt), kAvgThreads, 0, st>>>(a, sc, reinterpret_cast<unsigned *>(winv), t,
                                                                                           c, nc, nchunk, bblocks);
                BLINK_LAUNCH_CHECK("avg_count_kernel");
                avg_winv_kernel<<<(a.ntc + 255) / 256, 256, 0, st>>>(a, winv);
                BLINK_LAUNCH_CHECK("avg_winv_kernel");
            }
            const long long blocks = (long long)bblocks * nchunk * P * nt;
            if (blocks > 0x7fffffffLL) return BLINK_ERR_UNSUPPORTED;
            avg_scatter_runs_kernel<false><<<(unsigned)blocks, kAvgThreads, 0, st>>>(a, sc, winv, nullptr, t, c, nc, nchunk, bblocks);
            BLINK_LAUNCH_CHECK("avg_scatter_runs_kernel");
        }
        tc = end;
    }
    // steps a4-a5 on the combined grids: already normalised, so no scale
    float2 *tw_generic = is_pow2(n_pix) ? nullptr
                                        : reinterpret_cast<float2 *>(static_cast<unsigned char *>(workspace) + gbytes - gfft_workspace_bytes(n_pix));
    return fft2d_range(grid, n_pix, n_out, nullptr, 1, 0, image_avg, nullptr, st, tw_generic, true);
}
