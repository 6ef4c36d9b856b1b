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

namespace blink {

constexpr int kAvgThreads = 256;

struct AvgArgs {
    const float2 *vis; const float *uvw_m;
    int T, C, P, B, n, weighting, avg_time;
    int tc0, ntc, c_base;
    float2 *grid;                 // [n_out][n][n] combined grids, centred, zeroed by the caller
    float *wsum;                  // [T*C]
    uint32_t *cnt;                // uniform weighting: [gridDim.x][n*n] count planes, all zero between items
    float inv_navg;               // 1 / (number of images per output)
};

// One persistent CTA per (t,c) item.  Sweep 1 finds the weight sum W of the item (natural: samples placed;
// uniform: occupied cells, counted exactly as "first arrival" on a per-CTA count plane); sweep 2 adds every
// sample times 1 / (n W) (uniform: also / count of its cell) to the combined grid of its output image.
__global__ void __launch_bounds__(kAvgThreads)
avg_grid_kernel(const AvgArgs a, const __grid_constant__ ScaleBlock sc)
{
    __shared__ int s_in[kAvgThreads / 32], s_first[kAvgThreads / 32];
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
        for (int b = threadIdx.x; b < B; b += kAvgThreads) {
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
        for (int k = 0; k < kAvgThreads / 32; ++k) { n_in += s_in[k]; n_first += s_first[k]; }
        const float W = uniform ? (float)n_first : (float)(2 * n_in);
        if (threadIdx.x == 0) a.wsum[tc] = W;
        // ---- sweep 2: weighted scatter into the combined grids ---------------------------------------
        if (W > 0.f) {
            const float wbase = a.inv_navg / W;
            for (int b = threadIdx.x; b < B; b += kAvgThreads) {
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
            for (int b = threadIdx.x; b < B; b += kAvgThreads) {
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

static size_t avg_grid_bytes(int T, int P, int n_pix, int avg_time)
{
    return align_up((size_t)(avg_time ? 1 : T) * P * n_pix * n_pix * sizeof(float2), 256);
}
static int avg_max_planes() { return 2 * (sm_count() > 0 ? sm_count() : 148); }
size_t avg_workspace_bytes(int T, int P, int n_pix, int weighting, bool minimum)
{
    size_t b = avg_grid_bytes(T, P, n_pix, 0);
    if (weighting == BLINK_W_UNIFORM) {
        const size_t plane = (size_t)n_pix * n_pix * sizeof(uint32_t);
        size_t planes = minimum ? 1 : (size_t)avg_max_planes();
        if (!minimum) planes = std::max<size_t>(1, std::min<size_t>(planes, ((size_t)2 << 30) / plane));
        b += planes * plane;
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
    if (!is_pow2(n_pix) || n_pix < 32 || n_pix > 4096 || B > kMaxBaselines) return BLINK_ERR_UNSUPPORTED;
    if ((long long)T * C * P > 0x3fffffffLL) return BLINK_ERR_UNSUPPORTED;
    if (!aligned16(vis) || !aligned16(image_avg)) return BLINK_ERR_INVALID_ARG;
    int rc = ensure_device();
    if (rc != BLINK_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const bool uni = weighting == BLINK_W_UNIFORM;
    const size_t n2 = (size_t)n_pix * n_pix;
    const size_t gbytes = avg_grid_bytes(T, P, n_pix, avg_time ? 1 : 0);
    const size_t plane = n2 * sizeof(uint32_t);
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u) || workspace_bytes < gbytes + (uni ? plane : 0))
        return BLINK_ERR_WORKSPACE;
    float2 *grid = static_cast<float2 *>(workspace);
    uint32_t *cnt = uni ? reinterpret_cast<uint32_t *>(static_cast<unsigned char *>(workspace) + gbytes) : nullptr;
    int ctas = 8 * (sm_count() > 0 ? sm_count() : 148);
    if (uni) ctas = (int)std::min<size_t>((size_t)avg_max_planes(), (workspace_bytes - gbytes) / plane);
    BLINK_CUDA_TRY(cudaMemsetAsync(grid, 0, gbytes, st));
    if (uni) BLINK_CUDA_TRY(cudaMemsetAsync(cnt, 0, (size_t)ctas * plane, st));
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
        const int gridx = a.ntc < ctas ? a.ntc : ctas;
        avg_grid_kernel<<<gridx, kAvgThreads, 0, st>>>(a, sc);
        BLINK_LAUNCH_CHECK("avg_grid_kernel");
        tc = end;
    }
    // steps a4-a5 on the combined grids: already normalised, so no scale
    return fft2d_range(grid, n_pix, n_out, nullptr, 1, 0, image_avg, nullptr, st);
}
