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

#include "blink_fused_kernel.cuh"

namespace blink {

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
    if (!is_pow2(n_pix) || !fused_supported(P, B, n_pix, BLINK_W_NATURAL)) return BLINK_ERR_UNSUPPORTED;
    rc = ensure_device();
    if (rc != BLINK_OK) return rc;
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
        default: return BLINK_ERR_UNSUPPORTED;
    }
}
