/*
 * blinkimg.h -- C ABI of libblinkimg: batched dirty imaging on one NVIDIA B200 (sm_100a).
 *
 * The hot path of the BLINK high-time-resolution imager (arXiv 2505.15204; PAPER.md in the
 * reference folder): for every (timestep t, fine channel c, polarisation p)
 *   a0  cells per metre  s_c = float(f_c * N * pixscale / c0)          (u in wavelengths;
 *                                                                       DESIGN.md reading R3)
 *   a1  nearest uv cell  iu = rint(u_m * s_c), iv = rint(v_m * s_c)     ("placed ... based on
 *                                                                       the (u,v) coordinates"; R2, R4)
 *   a2  accumulate       G[cell] += V, G[cell'] += conj(V)              (no gridding
 *                                                                       kernel; conjugate at (-u,-v): R1)
 *   a3  weighting        natural (default) or uniform (BASELINE.json; R9), weight sum W
 *   a4  inverse FFT along u (rows)      \  PAPER.md L108-110 eq. 5: "2D inverse FFT",
 *   a5  inverse FFT along v (columns)   /  batched over all grids; sign +, unnormalised (R5)
 *       + fftshift (L194), * 1/W (R6), real part  ->  float32 dirty image (L150: fp32 throughout)
 *
 * Image index i = (t*C + c)*P + p, n_img = T*C*P.  N = n_pix (even, 32..8192, no prime factor above 5), h = N/2.  All arrays are dense,
 * row-major, last index fastest.  "centred" means the DC cell / phase-centre pixel is [h][h];
 * column index = u / l axis, row index = v / m axis (R7, R8).
 *
 * Pointers are DEVICE pointers owned by the caller unless marked HOST.  Complex numbers are
 * interleaved float pairs (re, im) = CUDA float2 = torch.complex64.  Every call is asynchronous
 * on `stream` (a cudaStream_t passed as void*; NULL = the legacy default stream), allocates and
 * frees nothing, never writes to its inputs (one documented exception: blink_fft2d_inverse may
 * clobber `grid`), fully overwrites its outputs, and returns BLINK_OK or a negative error code.
 * No exceptions, no stderr output, no exit().  Concurrent calls on different streams with
 * disjoint workspaces and outputs are allowed.  There is no CPU fallback: on a machine without
 * an sm_100 device every compute call returns BLINK_ERR_CUDA.
 */
#ifndef BLINKIMG_H
#define BLINKIMG_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct blink_c64 { float re, im; } blink_c64;       /* == float2 == complex64 */

enum { BLINK_W_NATURAL = 0, BLINK_W_UNIFORM = 1 };
enum { BLINK_OP_GRID = 0, BLINK_OP_FFT2D = 1, BLINK_OP_IMAGE = 2, BLINK_OP_IMAGE_HOST = 3, BLINK_OP_IMAGE_AVG = 4,
       BLINK_OP_IMAGE_CONV = 5, BLINK_OP_IMAGE_STOKES_I = 6, BLINK_OP_IMAGE_CAL = 7 };
enum {
    BLINK_OK = 0,
    BLINK_ERR_INVALID_ARG = -1,   /* NULL / misaligned pointer, non-positive size, bad enum          */
    BLINK_ERR_UNSUPPORTED = -2,   /* n_pix odd, outside [32, 8192] or with a prime factor > 5; B > 2^18-1 */
    BLINK_ERR_WORKSPACE   = -3,   /* workspace smaller than blink_workspace_bytes() reports           */
    BLINK_ERR_CUDA        = -4    /* a CUDA runtime/driver call failed: see blink_last_cuda_error()   */
};

/* Options for blink_set_option: tuning / test switches of the CALLING THREAD (thread-local; defaults in brackets).
 * A call reads the options of the thread that issues it, so a switch set by one thread never changes the route of a
 * call made by another; there is no process-wide mutable state besides the launch counter. */
enum {
    BLINK_OPT_IMAGE_PATH = 0,     /* [0] 0 = auto (fused where supported; batches of <= 4 Mi pixels take the unfused chain when the
                                         workspace holds them), 1 = force unfused (grid -> rows -> columns), 2 = force fused */
    BLINK_OPT_FUSED_CTAS = 1,     /* [0] 0 = auto (one persistent CTA per SM), else CTAs for the fused kernel  */
    BLINK_OPT_GRID_CHUNK_B = 2,   /* [0] 0 = auto, else baselines per gridder chunk (tests the spill path)     */
    BLINK_OPT_AVG_WSUM = 3,       /* [0] blink_image_avg weight sums: 0 = auto, 1 = sort + binary search, 2 = ballot counting */
    BLINK_OPT_CORR_PATH = 4,      /* [0] blink_correlate: 0 = auto, 1 = one CTA per tile; 2 is reserved (the 3-CTA multicast and the cta_group::2 pair kernels were measured slower and are gone: profiles/r2_corr.md) */
    BLINK_OPT_FUSED_TEAM = 5      /* [0] fused kernel: CTAs that image one (t,c) together: 0 = auto (1 for large batches; more when the batch
                                         leaves the last round of one-CTA-per-image half empty), else the team size */
};

const char *blink_strerror(int code);
const char *blink_last_cuda_error(void);          /* text of the last CUDA failure on this thread, or "" */
int blink_set_option(int key, int value);
int blink_get_option(int key, int *value);
/* Number of kernels this library has launched in this process so far (all threads). */
unsigned long long blink_kernel_launches(void);

/*
 * Workspace a call needs for the given problem (bytes; may be 0).  For BLINK_OP_IMAGE this is the
 * RECOMMENDED size; blink_image accepts anything >= the minimum it reports via *min_bytes (may be
 * NULL) and chunks the batch to fit.  For BLINK_OP_FFT2D pass the batch as T (C = P = 1, B = 0).
 */
int blink_workspace_bytes(int op, int T, int C, int P, int B, int n_pix, int weighting,
                          size_t *bytes, size_t *min_bytes);

/*
 * Steps a0-a3: grid every image of the batch.
 *   vis       in  [T][C][P][B] complex64, baseline fastest, cross-correlations only (R10)
 *   uvw_m     in  [T][B][3] float32 metres (u, v, w); w is read-compatible but unused
 *   freqs_hz  in  HOST [C] double
 *   grid      out [T*C*P][N][N] complex64, centred
 *   wsum      out [T*C] float32: natural = 2*B_in (samples placed incl. conjugates); uniform = number
 *                 of occupied cells.  Shared by the P polarisations of a (t,c).
 *   cell_idx  out OPTIONAL (NULL ok) [T][C][B] int32: centred linear cell (iv+h)*N + (iu+h), -1 if dropped
 *   counts    out OPTIONAL (NULL ok) [T*C][N][N] uint32 samples per cell (vis + conjugates)
 * Samples with |iu| > h-1 or |iv| > h-1 (or non-finite uvw) are dropped with their conjugate (R4).
 * Uniform weighting divides each occupied cell by its count.  A (t,c) with W = 0 gives a zero grid.
 * Visibilities are binned by uv row-band tile and accumulated in shared memory; when the binned
 * list of a (t,c) does not fit on chip the baselines are processed in chunks and every chunk after
 * the first is added to the grid with global atomics (the spill path).
 */
int blink_grid(const blink_c64 *vis, const float *uvw_m, const double *freqs_hz,
               int T, int C, int P, int B, int n_pix, double pixscale_rad, int weighting,
               blink_c64 *grid, float *wsum, int32_t *cell_idx, uint32_t *counts,
               void *workspace, size_t workspace_bytes, void *stream);

/*
 * Steps a4-a5 on arbitrary complex grids (Hermitian or not):
 *   image[i][y][x] = (1/scale) * Re sum_{r,q} grid[i][r][q] * exp(+2 pi i ((q-h)(x-h) + (r-h)(y-h)) / N)
 *   grid        in  [batch][N][N] complex64, centred.  CLOBBERED (used as the row-pass output).
 *   scale       in  OPTIONAL [ceil(batch / scale_stride_div)] float32; image i is multiplied by
 *                   1/scale[i / scale_stride_div]; an entry of 0 gives a zero image; NULL = unscaled
 *   image       out [batch][N][N] float32, centred
 *   image_imag  out OPTIONAL [batch][N][N] float32: the imaginary part, same scaling (debug / tests)
 * Row pass in shared memory, then a column pass whose tiles are staged by TMA with the fftshift,
 * the 1/W normalisation and the real-part extraction fused into its store.
 * Sides that are not a power of two run a mixed-radix transform instead and need `workspace` >=
 * blink_workspace_bytes(BLINK_OP_FFT2D) (an N-entry twiddle table); powers of two need none.
 */
int blink_fft2d_inverse(blink_c64 *grid, int n_pix, int batch,
                        const float *scale, int scale_stride_div,
                        float *image, float *image_imag,
                        void *workspace, size_t workspace_bytes, void *stream);

/*
 * Steps a0-a5 fused: visibilities in, dirty images out; the uv grids are never materialised in
 * full.  Arguments as blink_grid, plus
 *   image     out [T*C*P][N][N] float32, centred, = Re(...) / W ; W = 0 gives a zero image
 * The batch is processed in chunks that fit `workspace`.
 */
int blink_image(const blink_c64 *vis, const float *uvw_m, const double *freqs_hz,
                int T, int C, int P, int B, int n_pix, double pixscale_rad, int weighting,
                float *image, float *wsum, int32_t *cell_idx, uint32_t *counts,
                void *workspace, size_t workspace_bytes, void *stream);

/*
 * blink_image with HOST buffers (vis, uvw_m, image, wsum are HOST pointers, ideally pinned):
 * copies inputs to the device, images, copies the images back, pipelined per timestep on internal
 * streams.  `workspace` is a DEVICE buffer of at least blink_workspace_bytes(BLINK_OP_IMAGE_HOST)
 * that also holds the device staging copies.  Synchronous: returns when `image` is complete.
 */
int blink_image_host(const blink_c64 *vis_host, const float *uvw_m_host, const double *freqs_hz,
                     int T, int C, int P, int B, int n_pix, double pixscale_rad, int weighting,
                     float *image_host, float *wsum_host,
                     void *workspace, size_t workspace_bytes);

/*
 * Dirty images averaged over fine channels, or over fine channels and timesteps ("Images
 * belonging to the same time bin are averaged together"; L251 "averaged in time ... and frequency over the
 * 30.72 MHz bandwidth"; reading R14):
 *   avg_time == 0:  image_avg[t*P + p] = (1/C)     sum_c     image[(t*C + c)*P + p]        out [T*P][N][N]
 *   avg_time != 0:  image_avg[p]       = (1/(T*C)) sum_{t,c} image[(t*C + c)*P + p]        out [P][N][N]
 * with image[] exactly what blink_image produces (each image normalised by its own W; a (t,c) with W = 0
 * contributes a zero image and still counts in the mean).  The individual images are never formed: by linearity
 * the samples are scattered, pre-multiplied by 1/(n W_tc) (uniform: also by 1/count of their cell), into one
 * combined uv grid per output image with global vector atomics, and only those grids are transformed.
 * Inputs as blink_grid; wsum out [T*C] as blink_image.  `workspace` >= blink_workspace_bytes(BLINK_OP_IMAGE_AVG)
 * (minimum via *min_bytes): the combined grids and, for uniform weighting, per-CTA count planes.  With the recommended
 * size the per-sample weights [T*C][B] and the baselines sorted by |u| (12 bytes per (timestep, baseline)) fit as well, and
 * uniform weighting takes the faster column route (counts per grid column in shared memory, no count planes) for
 * n_pix <= 4096 and B <= 16384; results do not depend on the route.
 */
int blink_image_avg(const blink_c64 *vis, const float *uvw_m, const double *freqs_hz,
                    int T, int C, int P, int B, int n_pix, double pixscale_rad, int weighting,
                    int avg_time, float *image_avg, float *wsum,
                    void *workspace, size_t workspace_bytes, void *stream);

/*
 * Visibility corrections as per-antenna complex gains ("precomputed calibration solutions are
 * applied to visibilities, followed by geometric and cable length corrections"; reading R15):
 *   V'[t][c][p][b] = g[c][p][a1(b)] * conj(g[c][p][a2(b)]) * V[t][c][p][b]
 *   gains      in  [C][P][A] complex64 (a per-antenna phase carries the cable-length and geometric delays)
 *   ant_pairs  in  [B][2] int32, (a1, a2) of every baseline, 0 <= a < A; 8-byte aligned
 * blink_apply_gains corrects `vis` IN PLACE, one thread per visibility (the paper's own form).
 * blink_image_cal is blink_image of the corrected visibilities; `vis` is not modified and never written.  Where the fused
 * kernel runs (n_pix a power of two in [256, 4096], B <= 16384) the correction is fused into the gridder's load; for every
 * other supported size (the paper's 1200 and 8192 among them) the corrected visibilities are written to the head of the
 * workspace and imaged by the unfused chain.  `workspace` >= blink_workspace_bytes(BLINK_OP_IMAGE_CAL) minimum, 256-byte
 * aligned.  Other arguments as blink_image.
 */
int blink_apply_gains(blink_c64 *vis, const blink_c64 *gains, const int32_t *ant_pairs,
                      int T, int C, int P, int B, int A, void *stream);
int blink_image_cal(const blink_c64 *vis, const float *uvw_m, const double *freqs_hz,
                    const blink_c64 *gains, const int32_t *ant_pairs, int A,
                    int T, int C, int P, int B, int n_pix, double pixscale_rad, int weighting,
                    float *image, float *wsum, void *workspace, size_t workspace_bytes, void *stream);

/*
 * blink_image with a convolutional (anti-aliasing) gridding kernel -- the step the paper names as its next one
 * ("Visibilities are not convolved with any kernel at this stage, a feature to be introduced in the
 * near future to alleviate the effects of source aliasing"; L351).  The paper defines no kernel; DESIGN.md reading
 * R16 fixes the one used here:
 *   k(d)   = I0(beta sqrt(1 - (2d/S)^2)) / I0(beta), |d| <= S/2   (Kaiser-Bessel window, S = support = 3, 5 or 7 cells)
 *   x      = u_m * s_c (one fp32 multiply, as step a1), iu0 = rint(x), fx = x - iu0; the same along v
 *   taps   cell (iv0+i, iu0+j), i,j = -r..r, r = (S-1)/2, += wy_i wx_j V with wx_j = k(j - fx) / sum_j' k(j' - fx)
 *          (the S taps of an axis sum to 1), and the mirror cell += wy_i wx_j conj(V)
 *   range  a sample (and its conjugate) is dropped when |iu0| or |iv0| > h-1-r: the whole support stays on the grid
 *   W      natural weighting: 2 * (samples placed); uniform weighting is not offered with a kernel
 *   image  = Re IDFT(G) / W / (c((y-h)/N) c((x-h)/N)), c(xi) = (sinh(q)/q) / (sinh(beta)/beta),
 *            q = sqrt(beta^2 - (pi S xi)^2): the transform of the window, normalised to c(0) = 1 (grid correction)
 *   support   3, 5 or 7, else BLINK_ERR_UNSUPPORTED
 *   beta      <= 0 selects 2.34 * support; otherwise 1.7 * support <= beta <= 60 (the correction must stay positive
 *             over the whole image), else BLINK_ERR_INVALID_ARG
 *   cell_idx  out OPTIONAL [T][C][B]: the NEAREST cell (iv0+h)*N + (iu0+h) of every baseline, -1 if dropped
 * Runs in the fused kernels for n_pix a power of two in [256, 4096] (B <= 16384) and for the paper's 1200 (B <= 15000); every
 * other supported side (32 .. 8192, prime factors 2, 3, 5: 8192 among them) takes the plain form -- taps scattered into full grids with
 * global vector atomics, the unfused transform, one elementwise correction pass -- in chunks that fit the workspace.
 * `workspace` >= blink_workspace_bytes(BLINK_OP_IMAGE_CONV) minimum, 256-byte aligned.  Other arguments as blink_image.
 * The tap weights are evaluated as degree-11 polynomials in the offset, fitted on the host at every call;
 * blink_conv_taps_host (HOST pointers, no GPU needed) returns the weights exactly as the kernel evaluates them for
 * one offset f in [-1/2, 1/2], plus the largest deviation of the fit from the window's definition (tests).
 */
int blink_image_conv(const blink_c64 *vis, const float *uvw_m, const double *freqs_hz,
                     int T, int C, int P, int B, int n_pix, double pixscale_rad, int support, double beta,
                     float *image, float *wsum, int32_t *cell_idx,
                     void *workspace, size_t workspace_bytes, void *stream);
int blink_conv_taps_host(double f, int support, double beta, float *w /* HOST [support] */, double *fit_error /* HOST, opt */);

/*
 * CMAC correlator (eq. 3; section 6.2.2: "only the Conjugate Multiply Accumulate (CMAC) operation
 * was developed ... the result is divided by the integration time and number of averaged frequency channels.
 * Visibilities are stored in a lower triangular matrix form for each integration interval and output frequency
 * channel"; reading R17 for the sample format and array order the paper leaves open):
 *   volt  in  [F][A][Ns][2] int8: fine channel, input (tile x polarisation), time sample, (re, im); values in
 *             [-127, 127] (MWA Phase I VCS samples are 4 + 4 bit: [-8, 7]); 16-byte aligned
 *   n_t       samples per integration interval: T = Ns / n_t intervals (Ns % n_t == 0; n_t a multiple of 8, >= 64)
 *   n_avg     contiguous fine channels averaged into one output channel: C = F / n_avg (F % n_avg == 0)
 *   vis   out [T][C][A(A+1)/2] complex64: entry i(i+1)/2 + j (j <= i, autocorrelations included) =
 *             (float)(sum_{f,s} x_i conj(x_j)) / (float)(n_t n_avg); the integer sum is exact (int32 accumulators:
 *             n_t * n_avg <= 66000), the division is one correctly rounded fp32 operation
 * Runs on the int8 tensor cores (tcgen05.mma kind::i8, accumulators in TMEM), one persistent CTA per SM; needs no
 * workspace.  BLINK_ERR_UNSUPPORTED for n_t not a multiple of 8 or below 64, A > 4096, n_t * n_avg > 66000.
 */
int blink_correlate(const int8_t *volt, int F, int A, int Ns, int n_t, int n_avg, blink_c64 *vis, void *stream);
/*
 * Input-contract check for blink_correlate: *count (DEVICE, 8 bytes, written asynchronously on `stream`) = number of the
 * n_bytes int8 samples at `volt` (16-byte aligned) that equal -128.  The correlator negates imaginary parts bytewise and
 * -(-128) does not exist in int8, so such a sample silently corrupts the imaginary parts of its products; callers that
 * cannot guarantee [-127, 127] run this first (one read of the voltages).
 */
int blink_volt_out_of_range(const int8_t *volt, size_t n_bytes, unsigned long long *count, void *stream);

/*
 * Stokes I dirty images (the paper images XX only and "does not form Stokes I"; L351 future work;
 * DESIGN.md reading R18):  image[t*C + c] = (I_XX + I_YY) / 2  with I_XX, I_YY exactly blink_image's images of the planes
 * p = 0 and p = P-1 of vis [T][C][P][B] (P = 2: XX, YY;  P = 4: XX, XY, YX, YY; other P: BLINK_ERR_INVALID_ARG).
 * W and the uniform-weighting cell counts are shared by the planes of a (t,c), so the result is one image of the mean
 * visibilities (V_XX + V_YY) / 2, which is how it is computed: half the work of imaging both planes.
 *   image  out [T*C][N][N] float32;  wsum out [T*C];  other arguments as blink_image.
 * `workspace` >= blink_workspace_bytes(BLINK_OP_IMAGE_STOKES_I) minimum, 256-byte aligned (holds the combined visibilities).
 */
int blink_image_stokes_i(const blink_c64 *vis, const float *uvw_m, const double *freqs_hz,
                         int T, int C, int P, int B, int n_pix, double pixscale_rad, int weighting,
                         float *image, float *wsum, void *workspace, size_t workspace_bytes, void *stream);

/*
 * blink_image without a workspace argument, for callers that cannot allocate device memory (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc).  The scratch blink_image needs lives in one built-in device array of
 * blink_static_scratch_bytes() = 32 MiB that every GPU which loads the library holds until the process exits.  The call
 * allocates and frees nothing (no cudaMalloc / cudaFree / allocating library routine) and runs blink_image's own kernels with
 * that array as the workspace (fewer persistent CTAs / smaller chunks than a recommended-size workspace would give).
 *   - A problem whose MINIMUM blink_image workspace (blink_workspace_bytes(BLINK_OP_IMAGE), *min_bytes) exceeds the array is
 *     refused with BLINK_ERR_WORKSPACE before anything is launched; blink_last_cuda_error() names both sizes.  The fused
 *     kernels need 12 T B bytes + one half plane (n_pix^2 * 4 bytes: 16 MiB at 2048, so 4096 does not fit); the unfused chain
 *     needs P * n_pix^2 * 8 bytes + an n_pix-entry table.
 *   - All calls on a device share the array and it keeps the last call's contents; what must start at zero is cleared
 *     in-stream by the call itself.  Calls on one stream are ordered and safe; calls that OVERLAP on the GPU (different
 *     streams, unordered threads) race on the array and must not be made.
 * Arguments as blink_image (no cell_idx / counts outputs).  Results are blink_image's.
 */
size_t blink_static_scratch_bytes(void);
int blink_image_static(const blink_c64 *vis, const float *uvw_m, const double *freqs_hz,
                       int T, int C, int P, int B, int n_pix, double pixscale_rad, int weighting,
                       float *image, float *wsum, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* BLINKIMG_H */
