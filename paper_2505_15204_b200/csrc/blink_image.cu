// blink_image: steps a0-a5, visibilities in -> dirty images out, and its host-buffer twin.
// Path selection (BLINK_OPT_IMAGE_PATH): fused kernel (blink_fused.cu) when the size is supported,
// else the unfused chain grid -> row pass -> column pass over chunks of (t,c) that fit the workspace.
#include <algorithm>

#include "blink_common.cuh"

namespace blink {

// fused path (blink_fused.cu)
bool fused_supported(int P, int B, int n_pix, int weighting);
size_t fused_workspace_bytes(int T, int B, int n_pix, int ctas);
int fused_default_ctas();
int fused_image(const float2 *vis, const float *uvw_m, const double *freqs_hz, double pixscale_rad, int T, int C,
                int P, int B, int n_pix, int weighting, int tc0, int ntc, float *image, float *wsum,
                int32_t *cell_idx, void *workspace, size_t workspace_bytes, cudaStream_t st, GainRef cal);
size_t avg_workspace_bytes(int T, int C, int P, int B, int n_pix, int weighting, bool minimum);   // blink_avg.cu
size_t fused_conv_workspace_bytes(int T, int B, int n_pix, int ctas);                               // blink_fused_conv.cu
size_t conv_unfused_workspace_bytes(int T, int C, int P, int n_pix, bool minimum);
int counts_only(const float *uvw_m, const double *freqs_hz, double pixscale_rad, int T, int C, int B, int n_pix,
                int tc0, int ntc, uint32_t *counts, cudaStream_t st);

// sides that are not a power of two keep one row extent per (t,c) behind the grids (see image_device)
static size_t ext_bytes(int n_pix) { return is_pow2(n_pix) ? 0 : 16; }
static size_t unfused_bytes_per_tc(int P, int B, int n_pix, int weighting, bool have_counts)
{
    const size_t n2 = (size_t)n_pix * n_pix;
    size_t b = (size_t)P * n2 * sizeof(float2);
    if (!have_counts && grid_needs_global_counts(B, n_pix, weighting)) b += n2 * sizeof(uint32_t);
    return b + ext_bytes(n_pix);                               // + the (t,c)'s row extent (an int; 16 keeps the arrays aligned)
}

static bool use_fused(int P, int B, int n_pix, int weighting)
{
    const int path = option(BLINK_OPT_IMAGE_PATH);
    if (path == 1) return false;
    return fused_supported(P, B, n_pix, weighting);
}

// auto path only: batches of at most 4 Mi pixels (64 images of 256^2, 16 of 512^2, 4 of 1024^2, 1 of 2048^2: the measured
// cross-over of the two paths on a B200 -- e.g. 32 x 512^2: unfused 113 us, fused 91 us; 8 x 512^2: 44 / 89 us) go through
// the unfused chain
static bool small_batch(int ntc, int P, int n_pix)
{
    return option(BLINK_OPT_IMAGE_PATH) == 0 && (size_t)ntc * P * n_pix * n_pix <= ((size_t)4 << 20);
}

static int image_device(const float2 *vis, const float *uvw_m, const double *freqs_hz, int T, int C, int P, int B,
                        int n_pix, double pixscale_rad, int weighting, int tc0, int ntc, float *image, float *wsum,
                        int32_t *cell_idx, uint32_t *counts, void *workspace, size_t workspace_bytes, cudaStream_t st,
                        GainRef cal = GainRef())
{
    // image / wsum / cell_idx / counts are indexed by ABSOLUTE tc; the range [tc0, tc0+ntc) is processed
    const size_t n2 = (size_t)n_pix * n_pix;
    if (cal.gains && !use_fused(P, B, n_pix, weighting)) return BLINK_ERR_UNSUPPORTED;   // callers apply the gains first there (blink_image_cal)
    bool fused = use_fused(P, B, n_pix, weighting);
    // A handful of images leaves most SMs idle under the fused kernel (one CTA per image: 144 us for ONE 256 x 256 image,
    // config 1); the unfused chain spreads the rows and columns of an image over many CTAs (56 us).  Taken when the whole
    // range fits the workspace as one chunk; otherwise the fused kernel runs as before.
    if (fused && !cal.gains && small_batch(ntc, P, n_pix) &&
        workspace_bytes >= gfft_workspace_bytes(n_pix) + (size_t)ntc * unfused_bytes_per_tc(P, B, n_pix, weighting, counts != nullptr))
        fused = false;
    if (fused) {
        int rc = fused_image(vis, uvw_m, freqs_hz, pixscale_rad, T, C, P, B, n_pix, weighting, tc0, ntc, image, wsum,
                             cell_idx, workspace, workspace_bytes, st, cal);
        if (rc != BLINK_OK) return rc;
        if (counts) return counts_only(uvw_m, freqs_hz, pixscale_rad, T, C, B, n_pix, tc0, ntc, counts, st);
        return BLINK_OK;
    }
    const size_t per_tc = unfused_bytes_per_tc(P, B, n_pix, weighting, counts != nullptr);
    const size_t twb = gfft_workspace_bytes(n_pix);            // sides that are not a power of two: twiddle table first
    if (!workspace || workspace_bytes < twb + per_tc || !aligned16(workspace)) return BLINK_ERR_WORKSPACE;
    float2 *tw_generic = twb ? static_cast<float2 *>(workspace) : nullptr;
    workspace = static_cast<unsigned char *>(workspace) + twb;
    workspace_bytes -= twb;
    const int chunk = (int)std::min<size_t>((size_t)ntc, workspace_bytes / per_tc);
    float2 *wgrid = static_cast<float2 *>(workspace);
    const bool ws_counts = per_tc - ext_bytes(n_pix) > (size_t)P * n2 * sizeof(float2);
    uint32_t *wcounts = ws_counts ? reinterpret_cast<uint32_t *>(wgrid + (size_t)chunk * P * n2) : nullptr;
    // sides that are not a power of two: the gridder reports how many rows v >= 0 of each (t,c) hold data, and the
    // Hermitian transform neither reads nor transforms the rest (MWA-like uv coverage fills ~1/3 of a 1200 grid's rows)
    int *vrows = is_pow2(n_pix) ? nullptr
                                : reinterpret_cast<int *>(static_cast<unsigned char *>(workspace) + (size_t)chunk * (per_tc - ext_bytes(n_pix)));
    for (int s = tc0; s < tc0 + ntc; s += chunk) {
        const int m = std::min(chunk, tc0 + ntc - s);
        // counts: caller's array (absolute index) or the workspace copy (chunk-relative)
        uint32_t *cptr = counts ? counts + (size_t)s * n2 : wcounts;
        int rc = grid_range(vis, uvw_m, freqs_hz, pixscale_rad, T, C, P, B, n_pix, weighting, s, m, s, wgrid, wsum,
                            cell_idx, cptr, st, /*half_only=*/!is_pow2(n_pix), vrows);
        if (rc != BLINK_OK) return rc;
        rc = fft2d_range(wgrid, n_pix, m * P, wsum, P, s * P, image + (size_t)s * P * n2, nullptr, st, tw_generic, true, vrows, P);
        if (rc != BLINK_OK) return rc;
    }
    return BLINK_OK;
}

// One thread per visibility (pair), in place: the paper's own form of the corrections.
// A thread keeps its baselines' antenna pairs and walks the (t,c,p) rows; even B moves two visibilities per 16-byte access.
__device__ __forceinline__ float2 gain_factor(const float2 *gc, int2 ap)
{
    const float2 g1 = __ldg(gc + ap.x), g2 = __ldg(gc + ap.y);
    return make_float2(g1.x * g2.x + g1.y * g2.y, g1.y * g2.x - g1.x * g2.y);                 // g1 conj(g2)
}
template <int VEC>
__global__ void __launch_bounds__(256)
apply_gains_kernel(float2 *vis, const float2 *src, const float2 *__restrict__ gains, const int2 *__restrict__ ant, long long n_rows,
                   int C, int P, int B, int A)
{
    const int b = (blockIdx.x * blockDim.x + threadIdx.x) * VEC;
    if (b >= B) return;
    int2 ap[VEC];
#pragma unroll
    for (int k = 0; k < VEC; ++k) ap[k] = ant[b + k];                                         // VEC == 2 only when B is even
    for (long long row = blockIdx.y; row < n_rows; row += gridDim.y) {                        // row = (t*C + c)*P + p
        const int p = (int)(row % P), c = (int)((row / P) % C);
        const float2 *gc = gains + ((size_t)c * P + p) * A;
        float2 *dst = vis + row * B + b;
        const float2 *in = src + row * B + b;                                                  // src == vis: in place
        if constexpr (VEC == 2) {
            const float2 f0 = gain_factor(gc, ap[0]), f1 = gain_factor(gc, ap[1]);
            float4 v = *reinterpret_cast<const float4 *>(in);
            v = make_float4(f0.x * v.x - f0.y * v.y, f0.x * v.y + f0.y * v.x, f1.x * v.z - f1.y * v.w, f1.x * v.w + f1.y * v.z);
            *reinterpret_cast<float4 *>(dst) = v;
        } else {
            const float2 f = gain_factor(gc, ap[0]);
            const float2 v = *in;
            *dst = make_float2(f.x * v.x - f.y * v.y, f.x * v.y + f.y * v.x);
        }
    }
}

// Stokes I (reading R18): gridding, weighting (W and the cell counts are shared by the planes of a (t,c)) and the
// transform are linear in V, so (I_XX + I_YY) / 2 is ONE image of the visibilities (V_XX + V_YY) / 2: half the work of
// imaging both planes.  One thread per visibility pair of the output row, 16-byte accesses when B is even.
template <int VEC>
__global__ void __launch_bounds__(256)
stokes_combine_kernel(const float2 *__restrict__ vis, float2 *__restrict__ out, long long n_tc, int P, int B)
{
    const int b = (blockIdx.x * blockDim.x + threadIdx.x) * VEC;
    if (b >= B) return;
    for (long long tc = blockIdx.y; tc < n_tc; tc += gridDim.y) {
        const float2 *xx = vis + (tc * P) * B + b, *yy = vis + (tc * P + (P - 1)) * B + b;
        float2 *dst = out + tc * B + b;
        if constexpr (VEC == 2) {
            const float4 a = __ldcs(reinterpret_cast<const float4 *>(xx)), c = __ldcs(reinterpret_cast<const float4 *>(yy));
            *reinterpret_cast<float4 *>(dst) = make_float4(0.5f * (a.x + c.x), 0.5f * (a.y + c.y), 0.5f * (a.z + c.z), 0.5f * (a.w + c.w));
        } else {
            const float2 a = __ldcs(xx), c = __ldcs(yy);
            *dst = make_float2(0.5f * (a.x + c.x), 0.5f * (a.y + c.y));
        }
    }
}

// samples outside blink_correlate's input contract (int8 -128): grid-stride count, one atomic per CTA
__global__ void __launch_bounds__(256) volt_range_kernel(const int4 *__restrict__ v16, size_t n16, const int8_t *__restrict__ tail,
                                                         int n_tail, unsigned long long *__restrict__ count)
{
    unsigned c = 0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += (size_t)gridDim.x * blockDim.x) {
        const int4 q = __ldcs(v16 + i);
        const unsigned w[4] = {(unsigned)q.x, (unsigned)q.y, (unsigned)q.z, (unsigned)q.w};
#pragma unroll
        for (int k = 0; k < 4; ++k) c += __popc(__vcmpeq4(w[k], 0x80808080u) & 0x01010101u);
    }
    if (blockIdx.x == 0 && (int)threadIdx.x < n_tail && tail[threadIdx.x] == (int8_t)-128) ++c;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) c += __shfl_xor_sync(0xffffffffu, c, d);
    __shared__ unsigned s;
    if (threadIdx.x == 0) s = 0;
    __syncthreads();
    if ((threadIdx.x & 31) == 0 && c) atomicAdd(&s, c);
    __syncthreads();
    if (threadIdx.x == 0 && s) atomicAdd(count, (unsigned long long)s);
}

}  // namespace blink

using namespace blink;

static int check_common(const void *vis, const void *uvw_m, const double *freqs_hz, int T, int C, int P, int B, int n_pix,
                        double pixscale_rad, int weighting)
{
    if (!vis || !uvw_m || !freqs_hz) return BLINK_ERR_INVALID_ARG;
    if (T < 1 || C < 1 || P < 1 || B < 1 || !(pixscale_rad > 0.0)) return BLINK_ERR_INVALID_ARG;
    if (weighting != BLINK_W_NATURAL && weighting != BLINK_W_UNIFORM) return BLINK_ERR_INVALID_ARG;
    if (!size_supported(n_pix) || B > kMaxBaselines) return BLINK_ERR_UNSUPPORTED;
    if ((long long)T * C * P > 0x3fffffffLL) return BLINK_ERR_UNSUPPORTED;
    return BLINK_OK;
}

extern "C" int blink_workspace_bytes(int op, int T, int C, int P, int B, int n_pix, int weighting, size_t *bytes,
                                     size_t *min_bytes)
{
    if (!bytes) return BLINK_ERR_INVALID_ARG;
    if (!size_supported(n_pix)) return BLINK_ERR_UNSUPPORTED;
    if (T < 1 || C < 1 || P < 1 || B < 0) return BLINK_ERR_INVALID_ARG;
    const size_t n2 = (size_t)n_pix * n_pix;
    size_t rec = 0, mn = 0;
    switch (op) {
        case BLINK_OP_GRID:
            rec = mn = grid_needs_global_counts(B, n_pix, weighting) ? (size_t)T * C * n2 * sizeof(uint32_t) : 0;
            break;
        case BLINK_OP_FFT2D:
            rec = mn = gfft_workspace_bytes(n_pix);
            break;
        case BLINK_OP_IMAGE_CAL: {                              // fused sizes: as blink_image; else + the corrected copy
            size_t r1 = 0, m1 = 0;
            int rc1 = blink_workspace_bytes(BLINK_OP_IMAGE, T, C, P, B, n_pix, weighting, &r1, &m1);
            if (rc1 != BLINK_OK) return rc1;
            const size_t corr = use_fused(P, B, n_pix, weighting) ? 0 : align_up((size_t)T * C * P * B * sizeof(float2), 256);
            rec = corr + r1;
            mn = corr + m1;
            break;
        }
        case BLINK_OP_IMAGE_STOKES_I: {                         // combined visibilities + a one-plane blink_image
            if (P != 2 && P != 4) return BLINK_ERR_INVALID_ARG;
            size_t r1 = 0, m1 = 0;
            int rc1 = blink_workspace_bytes(BLINK_OP_IMAGE, T, C, 1, B, n_pix, weighting, &r1, &m1);
            if (rc1 != BLINK_OK) return rc1;
            const size_t comb = align_up((size_t)T * C * B * sizeof(float2), 256);
            rec = comb + r1;
            mn = comb + m1;
            break;
        }
        case BLINK_OP_IMAGE:
        case BLINK_OP_IMAGE_HOST: {
            if (use_fused(P, B, n_pix, weighting)) {
                int ctas = option(BLINK_OPT_FUSED_CTAS);
                if (ctas <= 0) ctas = fused_default_ctas();
                rec = fused_workspace_bytes(T, B, n_pix, ctas);
                mn = fused_workspace_bytes(T, B, n_pix, 1);
                const int ntc = op == BLINK_OP_IMAGE_HOST ? C : T * C;        // (t,c) per image_device call
                if (small_batch(ntc, P, n_pix))                              // room for the small-batch route (see image_device)
                    rec = std::max(rec, gfft_workspace_bytes(n_pix) + (size_t)ntc * unfused_bytes_per_tc(P, B, n_pix, weighting, false));
            } else {
                const size_t per_tc = unfused_bytes_per_tc(P, B, n_pix, weighting, false);
                mn = gfft_workspace_bytes(n_pix) + per_tc;
                rec = gfft_workspace_bytes(n_pix) + per_tc * std::min<size_t>((size_t)T * C, 256);
            }
            if (op == BLINK_OP_IMAGE_HOST) {
                // device staging: uvw for all timesteps, wsum, and two slots of one timestep of vis + images
                size_t stage = align_up((size_t)T * B * 3 * sizeof(float), 256) + align_up((size_t)T * C * sizeof(float), 256) +
                               2 * (align_up((size_t)C * P * B * sizeof(float2), 256) + align_up((size_t)C * P * n2 * sizeof(float), 256));
                rec = 2 * align_up(rec, 256) + stage;             // one compute workspace per pipeline slot
                mn = 2 * align_up(mn, 256) + stage;
            }
            break;
        }
        case BLINK_OP_IMAGE_AVG:
            rec = avg_workspace_bytes(T, C, P, B, n_pix, weighting, false);
            mn = avg_workspace_bytes(T, C, P, B, n_pix, weighting, true);
            break;
        case BLINK_OP_IMAGE_CONV: {
            if (!(is_pow2(n_pix) || n_pix == 1200) || !fused_supported(P, B, n_pix, BLINK_W_NATURAL)) {
                rec = conv_unfused_workspace_bytes(T, C, P, n_pix, false);
                mn = conv_unfused_workspace_bytes(T, C, P, n_pix, true);
                break;
            }
            int ctas = option(BLINK_OPT_FUSED_CTAS);
            if (ctas <= 0) ctas = fused_default_ctas();
            rec = fused_conv_workspace_bytes(T, B, n_pix, ctas);
            mn = fused_conv_workspace_bytes(T, B, n_pix, 1);
            break;
        }
        default:
            return BLINK_ERR_INVALID_ARG;
    }
    *bytes = rec;
    if (min_bytes) *min_bytes = mn;
    return BLINK_OK;
}

extern "C" int blink_image(const blink_c64 *vis, const float *uvw_m, const double *freqs_hz, int T, int C, int P, int B,
                           int n_pix, double pixscale_rad, int weighting, float *image, float *wsum, int32_t *cell_idx,
                           uint32_t *counts, void *workspace, size_t workspace_bytes, void *stream)
{
    int rc = check_common(vis, uvw_m, freqs_hz, T, C, P, B, n_pix, pixscale_rad, weighting);
    if (rc != BLINK_OK) return rc;
    if (!image || !wsum) return BLINK_ERR_INVALID_ARG;
    if (!aligned16(vis) || !aligned16(image) || (counts && !aligned16(counts))) return BLINK_ERR_INVALID_ARG;
    rc = ensure_device();
    if (rc != BLINK_OK) return rc;
    return image_device(reinterpret_cast<const float2 *>(vis), uvw_m, freqs_hz, T, C, P, B, n_pix, pixscale_rad, weighting,
                        0, T * C, image, wsum, cell_idx, counts, workspace, workspace_bytes,
                        static_cast<cudaStream_t>(stream));
}

extern "C" int blink_image_host(const blink_c64 *vis_host, const float *uvw_m_host, const double *freqs_hz, int T, int C,
                                int P, int B, int n_pix, double pixscale_rad, int weighting, float *image_host,
                                float *wsum_host, void *workspace, size_t workspace_bytes)
{
    int rc = check_common(vis_host, uvw_m_host, freqs_hz, T, C, P, B, n_pix, pixscale_rad, weighting);
    if (rc != BLINK_OK) return rc;
    if (!image_host || !wsum_host || !workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u)) return BLINK_ERR_INVALID_ARG;   // the fused path needs 256
    rc = ensure_device();
    if (rc != BLINK_OK) return rc;
    size_t need = 0, need_min = 0;
    rc = blink_workspace_bytes(BLINK_OP_IMAGE_HOST, T, C, P, B, n_pix, weighting, &need, &need_min);
    if (rc != BLINK_OK) return rc;
    if (workspace_bytes < need_min) return BLINK_ERR_WORKSPACE;

    const size_t n2 = (size_t)n_pix * n_pix;
    const size_t uvw_b = align_up((size_t)T * B * 3 * sizeof(float), 256);
    const size_t wsum_b = align_up((size_t)T * C * sizeof(float), 256);
    const size_t vis_b = align_up((size_t)C * P * B * sizeof(float2), 256);
    const size_t img_b = align_up((size_t)C * P * n2 * sizeof(float), 256);
    const size_t stage = uvw_b + wsum_b + 2 * (vis_b + img_b);
    unsigned char *w = static_cast<unsigned char *>(workspace);
    float *d_uvw = reinterpret_cast<float *>(w);
    float *d_wsum = reinterpret_cast<float *>(w + uvw_b);
    unsigned char *slots = w + uvw_b + wsum_b;
    unsigned char *compute_ws = w + stage;
    const size_t compute_bytes = (workspace_bytes - stage) / 2 / 256 * 256;       // one half per slot

    // two pipelines (slots): H2D vis(t) -> image(t) -> D2H images(t), each on its own stream.  Streams and the event are
    // created per call on the CURRENT device and destroyed on every exit path (after draining both streams).
    cudaStream_t streams[2] = {nullptr, nullptr};
    cudaEvent_t uvw_ready = nullptr;
    int result = BLINK_OK;
    auto fail = [&](cudaError_t e, const char *where) {
        if (e != cudaSuccess && result == BLINK_OK) { set_cuda_error(e, where); result = BLINK_ERR_CUDA; }
        return e != cudaSuccess;
    };
    for (int k = 0; k < 2 && result == BLINK_OK; ++k)
        fail(cudaStreamCreateWithFlags(&streams[k], cudaStreamNonBlocking), "cudaStreamCreateWithFlags");
    if (result == BLINK_OK) fail(cudaEventCreateWithFlags(&uvw_ready, cudaEventDisableTiming), "cudaEventCreateWithFlags");
    if (result == BLINK_OK) {
        fail(cudaMemcpyAsync(d_uvw, uvw_m_host, (size_t)T * B * 3 * sizeof(float), cudaMemcpyHostToDevice, streams[0]), "cudaMemcpyAsync(uvw)") ||
            fail(cudaEventRecord(uvw_ready, streams[0]), "cudaEventRecord") ||
            fail(cudaStreamWaitEvent(streams[1], uvw_ready, 0), "cudaStreamWaitEvent");
    }
    for (int t = 0; t < T && result == BLINK_OK; ++t) {
        const int k = t & 1;
        cudaStream_t st = streams[k];
        float2 *d_vis = reinterpret_cast<float2 *>(slots + (size_t)k * (vis_b + img_b));
        float *d_img = reinterpret_cast<float *>(slots + (size_t)k * (vis_b + img_b) + vis_b);
        const size_t vis_elems = (size_t)C * P * B;
        if (fail(cudaMemcpyAsync(d_vis, reinterpret_cast<const float2 *>(vis_host) + (size_t)t * vis_elems,
                                 vis_elems * sizeof(float2), cudaMemcpyHostToDevice, st), "cudaMemcpyAsync(vis)"))
            break;
        // one timestep as a T=1 problem: uvw of timestep t, outputs of timestep t
        result = image_device(d_vis, d_uvw + (size_t)t * B * 3, freqs_hz, 1, C, P, B, n_pix, pixscale_rad, weighting, 0, C,
                              d_img, d_wsum + (size_t)t * C, nullptr, nullptr, compute_ws + (size_t)k * compute_bytes,
                              compute_bytes, st);
        if (result != BLINK_OK) break;
        fail(cudaMemcpyAsync(image_host + (size_t)t * C * P * n2, d_img, (size_t)C * P * n2 * sizeof(float),
                             cudaMemcpyDeviceToHost, st), "cudaMemcpyAsync(images)");
    }
    for (int k = 0; k < 2; ++k)                                 // drain on every path: nothing may still be in flight on return
        if (streams[k]) fail(cudaStreamSynchronize(streams[k]), "cudaStreamSynchronize");
    if (result == BLINK_OK)
        fail(cudaMemcpy(wsum_host, d_wsum, (size_t)T * C * sizeof(float), cudaMemcpyDeviceToHost), "cudaMemcpy(wsum)");
    if (uvw_ready) cudaEventDestroy(uvw_ready);
    for (int k = 0; k < 2; ++k)
        if (streams[k]) cudaStreamDestroy(streams[k]);
    return result;
}


static int check_gains(const void *gains, const void *ant_pairs, int A)
{
    if (!gains || !ant_pairs || A < 1) return BLINK_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(gains) & 7u) || (reinterpret_cast<uintptr_t>(ant_pairs) & 7u)) return BLINK_ERR_INVALID_ARG;
    return BLINK_OK;
}

static int launch_gains(float2 *dst, const float2 *src, const float2 *g, const int2 *ap, int T, int C, int P, int B, int A, cudaStream_t st)
{
    const long long n_rows = (long long)T * C * P;
    const unsigned rows_y = (unsigned)std::min<long long>(n_rows, 2048);
    if ((B & 1) == 0 && aligned16(dst) && aligned16(src))
        apply_gains_kernel<2><<<dim3((B / 2 + 255) / 256, rows_y), 256, 0, st>>>(dst, src, g, ap, n_rows, C, P, B, A);
    else
        apply_gains_kernel<1><<<dim3((B + 255) / 256, rows_y), 256, 0, st>>>(dst, src, g, ap, n_rows, C, P, B, A);
    BLINK_LAUNCH_CHECK("apply_gains_kernel");
    return BLINK_OK;
}

extern "C" int blink_apply_gains(blink_c64 *vis, const blink_c64 *gains, const int32_t *ant_pairs, int T, int C, int P, int B,
                                 int A, void *stream)
{
    if (!vis || T < 1 || C < 1 || P < 1 || B < 1) return BLINK_ERR_INVALID_ARG;
    int rc = check_gains(gains, ant_pairs, A);
    if (rc != BLINK_OK) return rc;
    rc = ensure_device();
    if (rc != BLINK_OK) return rc;
    float2 *v = reinterpret_cast<float2 *>(vis);
    return launch_gains(v, v, reinterpret_cast<const float2 *>(gains), reinterpret_cast<const int2 *>(ant_pairs), T, C, P, B, A,
                        static_cast<cudaStream_t>(stream));
}

extern "C" int blink_image_cal(const blink_c64 *vis, const float *uvw_m, const double *freqs_hz, const blink_c64 *gains,
                               const int32_t *ant_pairs, int A, int T, int C, int P, int B, int n_pix, double pixscale_rad,
                               int weighting, float *image, float *wsum, void *workspace, size_t workspace_bytes, void *stream)
{
    int rc = check_common(vis, uvw_m, freqs_hz, T, C, P, B, n_pix, pixscale_rad, weighting);
    if (rc != BLINK_OK) return rc;
    if (!image || !wsum || !aligned16(vis) || !aligned16(image)) return BLINK_ERR_INVALID_ARG;
    rc = check_gains(gains, ant_pairs, A);
    if (rc != BLINK_OK) return rc;
    rc = ensure_device();
    if (rc != BLINK_OK) return rc;
    GainRef cal;
    cal.gains = reinterpret_cast<const float2 *>(gains);
    cal.ant = reinterpret_cast<const int2 *>(ant_pairs);
    cal.A = A;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const float2 *v = reinterpret_cast<const float2 *>(vis);
    if (!use_fused(P, B, n_pix, weighting)) {
        // sizes the fused kernel does not cover (the paper's 1200 and 8192 among them): the corrected visibilities go to the
        // head of the workspace (out of place: `vis` stays untouched here too) and the unfused chain images them
        const size_t corr = align_up((size_t)T * C * P * B * sizeof(float2), 256);
        if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u) || workspace_bytes < corr) return BLINK_ERR_WORKSPACE;
        float2 *vc = static_cast<float2 *>(workspace);
        rc = launch_gains(vc, v, cal.gains, cal.ant, T, C, P, B, A, st);
        if (rc != BLINK_OK) return rc;
        return image_device(vc, uvw_m, freqs_hz, T, C, P, B, n_pix, pixscale_rad, weighting, 0, T * C, image, wsum, nullptr, nullptr,
                            static_cast<unsigned char *>(workspace) + corr, workspace_bytes - corr, st);
    }
    return image_device(v, uvw_m, freqs_hz, T, C, P, B, n_pix, pixscale_rad, weighting, 0, T * C, image, wsum, nullptr, nullptr,
                        workspace, workspace_bytes, st, cal);
}

extern "C" int blink_image_stokes_i(const blink_c64 *vis, const float *uvw_m, const double *freqs_hz, int T, int C, int P, int B,
                                    int n_pix, double pixscale_rad, int weighting, float *image, float *wsum,
                                    void *workspace, size_t workspace_bytes, void *stream)
{
    int rc = check_common(vis, uvw_m, freqs_hz, T, C, P, B, n_pix, pixscale_rad, weighting);
    if (rc != BLINK_OK) return rc;
    if (P != 2 && P != 4) return BLINK_ERR_INVALID_ARG;
    if (!image || !wsum || !aligned16(vis) || !aligned16(image)) return BLINK_ERR_INVALID_ARG;
    rc = ensure_device();
    if (rc != BLINK_OK) return rc;
    // workspace: the combined visibilities [T][C][B] | the workspace of the one-plane blink_image that follows
    const size_t comb = align_up((size_t)T * C * B * sizeof(float2), 256);
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u) || workspace_bytes < comb) return BLINK_ERR_WORKSPACE;
    float2 *vm = static_cast<float2 *>(workspace);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const long long n_tc = (long long)T * C;
    const unsigned rows_y = (unsigned)std::min<long long>(n_tc, 4096);
    const float2 *v = reinterpret_cast<const float2 *>(vis);
    if ((B & 1) == 0)
        stokes_combine_kernel<2><<<dim3((B / 2 + 255) / 256, rows_y), 256, 0, st>>>(v, vm, n_tc, P, B);
    else
        stokes_combine_kernel<1><<<dim3((B + 255) / 256, rows_y), 256, 0, st>>>(v, vm, n_tc, P, B);
    BLINK_LAUNCH_CHECK("stokes_combine_kernel");
    return image_device(vm, uvw_m, freqs_hz, T, C, 1, B, n_pix, pixscale_rad, weighting, 0, T * C, image, wsum, nullptr, nullptr,
                        static_cast<unsigned char *>(workspace) + comb, workspace_bytes - comb, st);
}

extern "C" int blink_volt_out_of_range(const int8_t *volt, size_t n_bytes, unsigned long long *count, void *stream)
{
    if (!volt || !count || !aligned16(volt)) return BLINK_ERR_INVALID_ARG;
    int rc = ensure_device();
    if (rc != BLINK_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    BLINK_CUDA_TRY(cudaMemsetAsync(count, 0, sizeof(unsigned long long), st));
    const size_t n16 = n_bytes / 16;
    const int blocks = (int)std::min<size_t>((n16 + 255) / 256 + 1, (size_t)(sm_count() > 0 ? sm_count() : 148) * 8);
    volt_range_kernel<<<blocks, 256, 0, st>>>(reinterpret_cast<const int4 *>(volt), n16, volt + n16 * 16, (int)(n_bytes - n16 * 16), count);
    BLINK_LAUNCH_CHECK("volt_range_kernel");
    return BLINK_OK;
}
