// Convolutional (anti-aliasing) gridding in the fused imaging kernel -- SURVEY 8(f) rank 2.
// PAPER.md L192 ("Visibilities are not convolved with any kernel at this stage, a feature to be introduced in the near
// future to alleviate the effects of source aliasing"), L351 ("The implementation of a gridding kernel to minimise
// aliasing is in progress").  The paper defines no kernel; reading R16 fixes a separable Kaiser-Bessel window
// of odd support S = 3, 5, 7 with per-sample normalised taps and the matching grid correction in the image plane.
//
// Device side: fused_image_kernel<N, NS, R> (blink_fused_kernel.cuh) with R = (S-1)/2 > 0 -- a column pair gathers the
// samples whose support reaches it (one contiguous range of the |u|-sorted list), the taps that fall at u <= 0 are
// mirrored into the gridded half plane as the conjugate sample's taps, and 1 / (c(y) c(x)) rides on the image store.
// Host side (this file): the polynomial form of the normalised tap weights, the taper table kernel, the C ABI.
#include <math.h>
#include <algorithm>

#include "blink_fused_kernel.cuh"

namespace blink {

int fused_g_image(const float2 *vis, const float *uvw_m, const double *freqs_hz, double pixscale_rad, int T, int C, int P, int B,
                  int weighting, int tc0, int ntc, float *image, float *wsum, int32_t *cell_idx, void *workspace,
                  size_t workspace_bytes, cudaStream_t st, GainRef cal, const ConvPoly *poly, int R, size_t extra);      // blink_fused_g.cu

bool fused_supported(int P, int B, int n_pix, int weighting);          // blink_fused.cu
size_t fused_workspace_bytes(int T, int B, int n_pix, int ctas);
int fused_default_ctas();

// ---- Kaiser-Bessel window on the host (double) -----------------------------------------------------------------
// I0 by the ascending series up to |x| = 12, by the large-argument asymptotic expansion beyond.
static double host_i0(double x)
{
    x = fabs(x);
    if (x < 12.0) {
        const double y = x * x * 0.25;
        double t = 1.0, acc = 1.0;
        for (int m = 1; m < 200; ++m) {
            t *= y / ((double)m * m);
            acc += t;
            if (t < acc * 1e-18) break;
        }
        return acc;
    }
    // I0(x) ~ e^x / sqrt(2 pi x) * sum_m ((2m-1)!!)^2 / (m! (8x)^m)
    double t = 1.0, acc = 1.0;
    for (int m = 1; m < 60; ++m) {
        const double f = (2.0 * m - 1.0);
        const double nt = t * f * f / ((double)m * 8.0 * x);
        if (nt >= t || nt < 1e-18 * acc) { if (nt < t) acc += nt; break; }
        t = nt;
        acc += t;
    }
    return exp(x) / sqrt(2.0 * 3.14159265358979323846 * x) * acc;
}
static double host_kb(double d, int S, double beta)
{
    const double a = 2.0 * d / S;
    double z = 1.0 - a * a;
    if (z < 0.0) z = 0.0;                                              // |d| = S/2 within rounding
    return host_i0(beta * sqrt(z));                                    // the common factor 1 / I0(beta) cancels in the taps
}
static void host_taps(double f, int S, double beta, double *w)
{
    const int r = (S - 1) / 2;
    double sum = 0.0;
    for (int j = -r; j <= r; ++j) sum += (w[j + r] = host_kb((double)j - f, S, beta));
    for (int j = 0; j < S; ++j) w[j] /= sum;
}

// Fits w_j(f), f in [-1/2, 1/2], for every tap: Chebyshev interpolation at kConvTerms nodes in t = 2f, converted to
// monomial coefficients of f.  Returns the largest |fit - direct| over a dense check grid (double evaluation).
double conv_fit_taps(int S, double beta, ConvPoly *out)
{
    constexpr int M = kConvTerms;
    const double pi = 3.14159265358979323846;
    double node[M], val[kConvMaxSupport][M];
    for (int m = 0; m < M; ++m) {
        node[m] = cos(pi * (m + 0.5) / M);
        double w[kConvMaxSupport];
        host_taps(0.5 * node[m], S, beta, w);
        for (int j = 0; j < S; ++j) val[j][m] = w[j];
    }
    double mono[kConvMaxSupport][M];
    for (int j = 0; j < S; ++j) {
        double cheb[M];
        for (int k = 0; k < M; ++k) {
            double acc = 0.0;
            for (int m = 0; m < M; ++m) acc += val[j][m] * cos(pi * k * (m + 0.5) / M);
            cheb[k] = acc * (k == 0 ? 1.0 : 2.0) / M;
        }
        // T_0 = 1, T_1 = t, T_{k+1} = 2 t T_k - T_{k-1}  ->  coefficients of t^q
        double tkm[M] = {0}, tk[M] = {0}, acc[M] = {0};
        tkm[0] = 1.0;
        tk[1] = 1.0;
        for (int q = 0; q < M; ++q) acc[q] = cheb[0] * tkm[q] + (M > 1 ? cheb[1] * tk[q] : 0.0);
        for (int k = 2; k < M; ++k) {
            double tn[M] = {0};
            for (int q = 0; q < M; ++q) tn[q] = (q > 0 ? 2.0 * tk[q - 1] : 0.0) - tkm[q];
            for (int q = 0; q < M; ++q) { acc[q] += cheb[k] * tn[q]; tkm[q] = tk[q]; tk[q] = tn[q]; }
        }
        double p2 = 1.0;
        for (int q = 0; q < M; ++q) { mono[j][q] = acc[q] * p2; p2 *= 2.0; }       // t = 2 f
    }
    for (int j = 0; j < kConvMaxSupport; ++j)
        for (int q = 0; q < M; ++q) out->c[j][q] = j < S ? (float)mono[j][q] : 0.f;
    double worst = 0.0;
    for (int i = 0; i <= 400; ++i) {
        const double f = -0.5 + i / 400.0;
        double w[kConvMaxSupport];
        host_taps(f, S, beta, w);
        for (int j = 0; j < S; ++j) {
            double v = mono[j][M - 1];
            for (int q = M - 2; q >= 0; --q) v = v * f + mono[j][q];
            worst = fmax(worst, fabs(v - w[j]));
        }
    }
    return worst;
}

// ---- grid correction table: inv_c[x] = 1 / c((x - h)/N), c = window transform normalised to c(0) = 1 ------------
//   int_{-S/2}^{S/2} k(d) cos(2 pi d xi) dd  ~  sinh(q)/q,  q = sqrt(beta^2 - (pi S xi)^2)   (sin(q')/q' beyond the null)
__global__ void conv_taper_kernel(float *__restrict__ inv_c, int n, int S, double beta)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= n) return;
    const double xi = (double)(x - n / 2) / (double)n;
    const double a = 3.14159265358979323846 * (double)S * xi;
    const double z = beta * beta - a * a;
    const double q = sqrt(fabs(z));
    double ft;
    if (q < 1e-8) ft = 1.0;
    else ft = z > 0.0 ? sinh(q) / q : sin(q) / q;
    const double c = ft / (sinh(beta) / beta);
    inv_c[x] = (float)(1.0 / c);
}

static size_t taper_bytes(int n_pix) { return align_up((size_t)n_pix * sizeof(float), 256); }
size_t fused_conv_workspace_bytes(int T, int B, int n_pix, int ctas) { return fused_workspace_bytes(T, B, n_pix, ctas) + taper_bytes(n_pix); }

template <int N>
static int launch_conv(const FusedArgs &a, int R, const double *freqs_hz, double pixscale_rad, void *ws, size_t wsb,
                       cudaStream_t st, const ConvPoly *poly, size_t extra)
{
    switch (R) {
        case 1: return launch_fused<N, 1>(a, freqs_hz, pixscale_rad, ws, wsb, st, poly, extra);
        case 2: return launch_fused<N, 2>(a, freqs_hz, pixscale_rad, ws, wsb, st, poly, extra);
        case 3: return launch_fused<N, 3>(a, freqs_hz, pixscale_rad, ws, wsb, st, poly, extra);
        default: return BLINK_ERR_UNSUPPORTED;
    }
}

// ---- every other supported size (the paper's 1200 and 8192 among them): the plain form --------------------------------
// One thread per (baseline, (t,c)) evaluates the sample's taps once and adds them, and the mirrored conjugate taps, to the
// full complex grids of the P planes with global vector atomics (red.global.add.v2.f32); the unfused transform
// (blink_fft2d.cu / blink_fftg.cu) follows and one elementwise pass applies the grid correction.  A fallback, not a tuned
// path: it exists so that the convolutional gridder covers every side blink_image covers.
template <int R>
__global__ void __launch_bounds__(256)
conv_scatter_kernel(const float2 *__restrict__ vis, const float *__restrict__ uvw_m, const __grid_constant__ ScaleBlock sc,
                    const __grid_constant__ ConvPoly poly, int C, int P, int B, int n, int tc0, int c_base, float2 *__restrict__ grid,
                    unsigned *__restrict__ n_in, int32_t *__restrict__ cell_idx)
{
    constexpr int S = 2 * R + 1;
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    const int tc = tc0 + blockIdx.y, t = tc / C, c = tc - t * C, h = n / 2;
    const float s = sc.s[c - c_base];
    const float *q = uvw_m + ((size_t)t * B + b) * 3;
    int iu0, iv0;
    const float x = __fmul_rn(q[0], s), y = __fmul_rn(q[1], s);
    const float xr = rint_rne(x, iu0), yr = rint_rne(y, iv0);
    const float lim = (float)(h - 1 - R);
    const bool ok = fabsf(xr) <= lim && fabsf(yr) <= lim;       // NaN fails: the whole support stays on the grid (R16)
    if (cell_idx) cell_idx[(size_t)tc * B + b] = ok ? (iv0 + h) * n + (iu0 + h) : -1;
    if (!ok) return;
    const float fx = __fsub_rn(x, xr), fy = __fsub_rn(y, yr);
    float wx[S], wy[S];
#pragma unroll
    for (int i = 0; i < S; ++i) {
        float a = poly.c[i][kConvTerms - 1], d = a;
#pragma unroll
        for (int k = kConvTerms - 2; k >= 0; --k) { a = fmaf(a, fx, poly.c[i][k]); d = fmaf(d, fy, poly.c[i][k]); }
        wx[i] = a;
        wy[i] = d;
    }
    atomicAdd(&n_in[tc], 1u);
    for (int p = 0; p < P; ++p) {
        const float2 v = __ldg(vis + ((size_t)tc * P + p) * B + b);
        float2 *g = grid + ((size_t)blockIdx.y * P + p) * n * n;
#pragma unroll
        for (int i = 0; i < S; ++i) {
            const int r0 = iv0 - R + i;
#pragma unroll
            for (int j = 0; j < S; ++j) {
                const int q0 = iu0 - R + j;
                const float w = wy[i] * wx[j];
                atomicAdd(g + (size_t)(r0 + h) * n + (q0 + h), make_float2(w * v.x, w * v.y));
                atomicAdd(g + (size_t)(h - r0) * n + (h - q0), make_float2(w * v.x, -w * v.y));     // conjugate sample: mirrored taps
            }
        }
    }
}
__global__ void conv_wsum_kernel(const unsigned *__restrict__ n_in, float *__restrict__ wsum, int tc0, int m)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < m) wsum[tc0 + i] = (float)(2u * n_in[tc0 + i]);
}
// image[i][y][x] *= inv_c[y] inv_c[x]  (n is even: float2 accesses)
__global__ void __launch_bounds__(256) conv_correct_kernel(float *__restrict__ image, const float *__restrict__ inv_c, int n, size_t n_rows)
{
    const int half = n / 2;
    for (size_t row = blockIdx.x; row < n_rows; row += gridDim.x) {
        const float cy = inv_c[row % n];
        float2 *r = reinterpret_cast<float2 *>(image + row * n);
        for (int k = threadIdx.x; k < half; k += blockDim.x) {
            float2 v = r[k];
            v.x *= cy * inv_c[2 * k];
            v.y *= cy * inv_c[2 * k + 1];
            r[k] = v;
        }
    }
}

static size_t conv_unfused_fixed(int T, int C, int n_pix)
{
    return gfft_workspace_bytes(n_pix) + taper_bytes(n_pix) + align_up((size_t)T * C * sizeof(unsigned), 256);
}
size_t conv_unfused_workspace_bytes(int T, int C, int P, int n_pix, bool minimum)
{
    const size_t per_tc = (size_t)P * n_pix * n_pix * sizeof(float2);
    return conv_unfused_fixed(T, C, n_pix) + per_tc * (minimum ? 1 : std::min<size_t>((size_t)T * C, 256));
}

static int conv_unfused(const float2 *vis, const float *uvw_m, const double *freqs_hz, int T, int C, int P, int B, int n_pix,
                        double pixscale_rad, int support, double beta, const ConvPoly &poly_in, float *image, float *wsum,
                        int32_t *cell_idx, void *workspace, size_t workspace_bytes, cudaStream_t st)
{
    const size_t n2 = (size_t)n_pix * n_pix, per_tc = (size_t)P * n2 * sizeof(float2);
    const size_t fixed = conv_unfused_fixed(T, C, n_pix);
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u) || workspace_bytes < fixed + per_tc) return BLINK_ERR_WORKSPACE;
    unsigned char *w = static_cast<unsigned char *>(workspace);
    float2 *tw_generic = gfft_workspace_bytes(n_pix) ? reinterpret_cast<float2 *>(w) : nullptr;
    float *inv_c = reinterpret_cast<float *>(w + gfft_workspace_bytes(n_pix));
    unsigned *n_in = reinterpret_cast<unsigned *>(w + gfft_workspace_bytes(n_pix) + taper_bytes(n_pix));
    float2 *wgrid = reinterpret_cast<float2 *>(w + fixed);
    const int chunk = (int)std::min<size_t>((size_t)T * C, std::min<size_t>((workspace_bytes - fixed) / per_tc, 65535));
    conv_taper_kernel<<<(n_pix + 255) / 256, 256, 0, st>>>(inv_c, n_pix, support, beta);
    BLINK_LAUNCH_CHECK("conv_taper_kernel");
    BLINK_CUDA_TRY(cudaMemsetAsync(n_in, 0, (size_t)T * C * sizeof(unsigned), st));
    ConvPoly poly = poly_in;
    poly.inv_taper = inv_c;
    const int R = (support - 1) / 2;
    return for_channel_blocks(C, 0, T * C, freqs_hz, n_pix, pixscale_rad, [&](int s0, int m, int c_base, const ScaleBlock &sc) -> int {
        for (int s = s0; s < s0 + m; s += chunk) {
            const int mm = std::min(chunk, s0 + m - s);
            BLINK_CUDA_TRY(cudaMemsetAsync(wgrid, 0, (size_t)mm * per_tc, st));
            const dim3 g((B + 255) / 256, mm);
            if (R == 1) conv_scatter_kernel<1><<<g, 256, 0, st>>>(vis, uvw_m, sc, poly, C, P, B, n_pix, s, c_base, wgrid, n_in, cell_idx);
            else if (R == 2) conv_scatter_kernel<2><<<g, 256, 0, st>>>(vis, uvw_m, sc, poly, C, P, B, n_pix, s, c_base, wgrid, n_in, cell_idx);
            else conv_scatter_kernel<3><<<g, 256, 0, st>>>(vis, uvw_m, sc, poly, C, P, B, n_pix, s, c_base, wgrid, n_in, cell_idx);
            BLINK_LAUNCH_CHECK("conv_scatter_kernel");
            conv_wsum_kernel<<<(mm + 255) / 256, 256, 0, st>>>(n_in, wsum, s, mm);
            BLINK_LAUNCH_CHECK("conv_wsum_kernel");
            float *img = image + (size_t)s * P * n2;
            int rc = fft2d_range(wgrid, n_pix, mm * P, wsum, P, s * P, img, nullptr, st, tw_generic, /*hermitian=*/true);
            if (rc != BLINK_OK) return rc;
            const size_t n_rows = (size_t)mm * P * n_pix;
            conv_correct_kernel<<<(unsigned)std::min<size_t>(n_rows, (size_t)148 * 16), 256, 0, st>>>(img, inv_c, n_pix, n_rows);
            BLINK_LAUNCH_CHECK("conv_correct_kernel");
        }
        return (int)BLINK_OK;
    });
}

}  // namespace blink

using namespace blink;

static double conv_beta(int support, double beta) { return beta > 0.0 ? beta : 2.34 * support; }
static int conv_check(int support, double beta)
{
    if (support != 3 && support != 5 && support != 7) return BLINK_ERR_UNSUPPORTED;
    // the correction must stay positive over the whole image: first null of the window transform beyond |xi| = 1/2
    if (!(beta >= 1.7 * support) || !(beta <= 60.0)) return BLINK_ERR_INVALID_ARG;
    return BLINK_OK;
}

extern "C" int blink_conv_taps_host(double f, int support, double beta, float *w, double *fit_error)
{
    if (!w || !(f >= -0.5 && f <= 0.5)) return BLINK_ERR_INVALID_ARG;
    beta = conv_beta(support, beta);
    int rc = conv_check(support, beta);
    if (rc != BLINK_OK) return rc;
    ConvPoly poly;
    const double err = conv_fit_taps(support, beta, &poly);
    if (fit_error) *fit_error = err;
    const float ff = (float)f;
    for (int j = 0; j < support; ++j) {                                // the kernel's evaluation: fp32 Horner
        float v = poly.c[j][kConvTerms - 1];
        for (int k = kConvTerms - 2; k >= 0; --k) v = fmaf(v, ff, poly.c[j][k]);
        w[j] = v;
    }
    return BLINK_OK;
}

extern "C" int blink_image_conv(const blink_c64 *vis, const float *uvw_m, const double *freqs_hz, int T, int C, int P, int B,
                                int n_pix, double pixscale_rad, int support, double beta, float *image, float *wsum,
                                int32_t *cell_idx, void *workspace, size_t workspace_bytes, void *stream)
{
    if (!vis || !uvw_m || !freqs_hz || !image || !wsum) return BLINK_ERR_INVALID_ARG;
    if (T < 1 || C < 1 || P < 1 || B < 1 || !(pixscale_rad > 0.0)) return BLINK_ERR_INVALID_ARG;
    if (!aligned16(vis) || !aligned16(image)) return BLINK_ERR_INVALID_ARG;
    beta = conv_beta(support, beta);
    int rc = conv_check(support, beta);
    if (rc != BLINK_OK) return rc;
    if ((long long)T * C * P > 0x3fffffffLL) return BLINK_ERR_UNSUPPORTED;
    if (!size_supported(n_pix) || B > kMaxBaselines) return BLINK_ERR_UNSUPPORTED;
    rc = ensure_device();
    if (rc != BLINK_OK) return rc;
    if (!(is_pow2(n_pix) || n_pix == 1200) || !fused_supported(P, B, n_pix, BLINK_W_NATURAL)) {   // outside the fused kernels: the plain form
        ConvPoly poly_u;
        conv_fit_taps(support, beta, &poly_u);
        return conv_unfused(reinterpret_cast<const float2 *>(vis), uvw_m, freqs_hz, T, C, P, B, n_pix, pixscale_rad, support, beta,
                            poly_u, image, wsum, cell_idx, workspace, workspace_bytes, static_cast<cudaStream_t>(stream));
    }
    const size_t extra = taper_bytes(n_pix);
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u) ||
        workspace_bytes < fused_conv_workspace_bytes(T, B, n_pix, 1))
        return BLINK_ERR_WORKSPACE;
    ConvPoly poly;
    conv_fit_taps(support, beta, &poly);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    float *inv_c = reinterpret_cast<float *>(static_cast<unsigned char *>(workspace) + sort_bytes(T, B));
    conv_taper_kernel<<<(n_pix + 255) / 256, 256, 0, st>>>(inv_c, n_pix, support, beta);
    BLINK_LAUNCH_CHECK("conv_taper_kernel");
    FusedArgs a{};
    a.vis = reinterpret_cast<const float2 *>(vis); a.uvw_m = uvw_m; a.T = T; a.C = C; a.P = P; a.B = B;
    a.weighting = BLINK_W_NATURAL; a.tc0 = 0; a.ntc = T * C; a.image = image; a.wsum = wsum; a.cell_idx = cell_idx;
    poly.inv_taper = inv_c;                          // [N] 1 / c((x - h)/N), read by the image store
    const int R = (support - 1) / 2;
    switch (n_pix) {
        case 256: return launch_conv<256>(a, R, freqs_hz, pixscale_rad, workspace, workspace_bytes, st, &poly, extra);
        case 512: return launch_conv<512>(a, R, freqs_hz, pixscale_rad, workspace, workspace_bytes, st, &poly, extra);
        case 1024: return launch_conv<1024>(a, R, freqs_hz, pixscale_rad, workspace, workspace_bytes, st, &poly, extra);
        case 2048: return launch_conv<2048>(a, R, freqs_hz, pixscale_rad, workspace, workspace_bytes, st, &poly, extra);
        case 4096: return launch_conv<4096>(a, R, freqs_hz, pixscale_rad, workspace, workspace_bytes, st, &poly, extra);
        case 1200: return fused_g_image(a.vis, uvw_m, freqs_hz, pixscale_rad, T, C, P, B, BLINK_W_NATURAL, 0, T * C, image, wsum, cell_idx,
                                        workspace, workspace_bytes, st, GainRef(), &poly, R, extra);
        default: return BLINK_ERR_UNSUPPORTED;
    }
}
