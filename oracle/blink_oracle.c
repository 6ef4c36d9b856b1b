/*
 * blink_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU statement of what libblinkimg computes: nearest-cell
 * gridding of visibilities (+ Hermitian conjugates) and the centred inverse 2D DFT that turns a
 * grid into a dirty image (eq. 5, L190-194 section 6.2.4).  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 * It shares no code, header, table or constant generator with paper_2505_15204_b200/csrc.
 *
 * Precision: visibilities and uvw arrive as float32 ("32 bit floating point");
 * the CELL INDEX is decided in float32 exactly as DESIGN.md reading R2 states (one fp32 multiply,
 * round-to-nearest-even) because floating point decides an integer there; everything else
 * (accumulation, DFT) is float64.
 *
 * Pins (tests/test_oracle_pins.py, all run without a GPU):
 *   oracle_scale / oracle_cell    : exact on-grid inputs, mirror invariant r+r'=N, brute-force
 *                                   float64 evaluation away from half-cell boundaries
 *   oracle_grid_one               : W = 2*B_in = sum(cnt); sum(G) = sum 2 Re V; Hermitian grid;
 *                                   3-antenna hand case
 *   oracle_idft2_direct           : single-cell closed form cos(2 pi (ku x + kv y)/N + arg V)
 *   oracle_ifft2_radix2           : == oracle_idft2_direct on 32x32 (north_star check 4),
 *                                   == numpy.fft.ifft2 with shifts, Parseval, linearity; sizes that are not a
 *                                   power of two (direct 1D sums): == oracle_idft2_direct at 12 and 20,
 *                                   == numpy.fft.ifft2 at 30, 48, 150, single-cell closed form at 1200
 *   oracle_sparse_image           : == radix-2 image on a full-size image
 *   oracle_image_one              : unit source at phase centre -> 1.0 at [h][h]; on-grid offset
 *                                   source peaks at its pixel with value 1.0; |Im| < 1e-6 peak
 *   oracle_image_avg              : unit sources -> 1.0 at the centre of the mean; == one numpy.fft transform
 *                                   of the 1/W-weighted sum of independently re-gridded channels; centre-pixel
 *                                   closed form with an empty channel counted in the mean
 *   oracle_apply_gains            : identity for unit gains; pure phases rotate by phi_a1 - phi_a2; independent
 *                                   numpy evaluation; undoing a simulated corruption restores the image
 *   oracle_image_stokes_i         : unit sources -> 1.0; YY = -XX -> 0; XX-only -> half the XX image; single-baseline
 *                                   closed form; == the image of the averaged visibilities (linearity)
 * Nothing here is "parity unpinned".
 *
 * Build: gcc -O2 -ffp-contract=off -fPIC -shared -pthread -o liboracle.so blink_oracle.c -lm
 */
#include <math.h>
#include <fenv.h>
#include <pthread.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_C0 299792458.0
#define ORACLE_PI 3.14159265358979323846264338327950288

/* ------------------------------------------------------------------------------------------
 * a0. cells per metre for channel frequency f (reading R3):
 *     u in wavelengths is u_m f / c, the uv cell is 1/(N pixscale) wavelengths,
 *     so cells = u_m * f * N * pixscale / c.  Evaluated left to right in double, rounded ONCE
 *     to float.
 * ---------------------------------------------------------------------------------------- */
float oracle_scale(double f_hz, int n_pix, double pixscale_rad)
{
    double s = f_hz * (double)n_pix;
    s = s * pixscale_rad;
    s = s / ORACLE_C0;
    return (float)s;
}

/* ------------------------------------------------------------------------------------------
 * a1. nearest cell of one baseline ("placed ... based on the (u, v) coordinates";
 *     readings R2 (round half to even), R4 (drop when |iu| or |iv| > h-1), w ignored (L114)).
 *     Returns the centred linear cell (iv+h)*N + (iu+h), or -1 when dropped.
 * ---------------------------------------------------------------------------------------- */
int32_t oracle_cell(float u_m, float v_m, float s, int n_pix)
{
    const int h = n_pix / 2;
    volatile float x = u_m * s;            /* one IEEE fp32 multiply, no contraction */
    volatile float y = v_m * s;
    float xr = nearbyintf(x);              /* FE_TONEAREST: ties to even */
    float yr = nearbyintf(y);
    const float lim = (float)(h - 1);
    if (!(fabsf(xr) <= lim && fabsf(yr) <= lim)) return -1;    /* NaN fails -> dropped */
    int iu = (int)xr, iv = (int)yr;
    return (int32_t)((iv + h) * n_pix + (iu + h));
}

/* cell of the Hermitian conjugate sample at (-u,-v): (h-iv)*N + (h-iu)  (reading R1) */
static int32_t mirror_cell(int32_t cell, int n_pix)
{
    const int h = n_pix / 2;
    int r = cell / n_pix, q = cell % n_pix;
    int iv = r - h, iu = q - h;
    return (int32_t)((h - iv) * n_pix + (h - iu));
}
int32_t oracle_mirror_cell(int32_t cell, int n_pix) { return mirror_cell(cell, n_pix); }

/* all (t, c, b) indices of a batch: cell_idx[T][C][B] */
void oracle_cells(const float *uvw_m, const double *freqs_hz, int T, int C, int B,
                  int n_pix, double pixscale_rad, int32_t *cell_idx)
{
    fesetround(FE_TONEAREST);
    for (int t = 0; t < T; ++t)
        for (int c = 0; c < C; ++c) {
            float s = oracle_scale(freqs_hz[c], n_pix, pixscale_rad);
            for (int b = 0; b < B; ++b) {
                const float *p = uvw_m + ((size_t)t * B + b) * 3;
                cell_idx[((size_t)t * C + c) * B + b] = oracle_cell(p[0], p[1], s, n_pix);
            }
        }
}

/* ------------------------------------------------------------------------------------------
 * a2 + a3. grid ONE image (natural weighting is the paper's default,
 *     uniform weighting is BASELINE.json's, reading R9).
 *   vis      [B] complex64 as float pairs, uvw_t [B][3] metres
 *   grid     [N][N] complex128 as double pairs, centred (DC at [h][h]); zeroed here
 *   cnt      [N][N] samples per cell (vis + conjugates); zeroed here
 *   cell_idx [B] (may be NULL)
 *   returns W: natural = sum(cnt) = 2 B_in ; uniform = number of occupied cells
 * ---------------------------------------------------------------------------------------- */
double oracle_grid_one(const float *vis, const float *uvw_t, double f_hz, int B, int n_pix,
                       double pixscale_rad, int weighting, double *grid, uint32_t *cnt,
                       int32_t *cell_idx)
{
    const size_t n2 = (size_t)n_pix * n_pix;
    fesetround(FE_TONEAREST);
    memset(grid, 0, n2 * 2 * sizeof(double));
    memset(cnt, 0, n2 * sizeof(uint32_t));
    float s = oracle_scale(f_hz, n_pix, pixscale_rad);
    for (int b = 0; b < B; ++b) {                                  /* baseline order */
        int32_t cell = oracle_cell(uvw_t[3 * b], uvw_t[3 * b + 1], s, n_pix);
        if (cell_idx) cell_idx[b] = cell;
        if (cell < 0) continue;
        int32_t cellc = mirror_cell(cell, n_pix);
        double re = (double)vis[2 * b], im = (double)vis[2 * b + 1];
        grid[2 * (size_t)cell] += re;   grid[2 * (size_t)cell + 1] += im;      /* G[cell]  += V       */
        grid[2 * (size_t)cellc] += re;  grid[2 * (size_t)cellc + 1] -= im;     /* G[cell'] += conj(V) */
        cnt[cell] += 1;  cnt[cellc] += 1;
    }
    double W = 0.0;
    if (weighting == 0) {
        for (size_t k = 0; k < n2; ++k) W += (double)cnt[k];
    } else {
        for (size_t k = 0; k < n2; ++k)
            if (cnt[k] > 0) {
                grid[2 * k] /= (double)cnt[k];
                grid[2 * k + 1] /= (double)cnt[k];
                W += 1.0;
            }
    }
    return W;
}

/* ------------------------------------------------------------------------------------------
 * a4 + a5, THE DEFINITION (sign + because eq. 4 L104 has e^{-i2pi(ul+vm)} in V;
 * unnormalised; centred on both sides, reading R7: DC cell [h][h] <-> phase-centre pixel [h][h]):
 *     out[y][x] = sum_{r,q} G[r][q] exp(+2 pi i ((q-h)(x-h) + (r-h)(y-h)) / N)
 * O(N^4): for N <= 64 only.  out is complex [N][N] as double pairs.
 * ---------------------------------------------------------------------------------------- */
void oracle_idft2_direct(const double *grid, int n, double *out)
{
    const int h = n / 2;
    for (int y = 0; y < n; ++y)
        for (int x = 0; x < n; ++x) {
            double sr = 0.0, si = 0.0;
            for (int r = 0; r < n; ++r)
                for (int q = 0; q < n; ++q) {
                    double gr = grid[2 * ((size_t)r * n + q)], gi = grid[2 * ((size_t)r * n + q) + 1];
                    if (gr == 0.0 && gi == 0.0) continue;
                    /* reduce the integer phase mod N before the trig call: exact */
                    long long k = (long long)(q - h) * (x - h) + (long long)(r - h) * (y - h);
                    k %= n; if (k < 0) k += n;
                    double a = 2.0 * ORACLE_PI * (double)k / (double)n;
                    double cr = cos(a), ci = sin(a);
                    sr += gr * cr - gi * ci;
                    si += gr * ci + gi * cr;
                }
            out[2 * ((size_t)y * n + x)] = sr;
            out[2 * ((size_t)y * n + x) + 1] = si;
        }
}

/* same definition, looping over OCCUPIED cells only and over all pixels: O(nnz N^2).
 * img[y][x] = (1/W) Re(...), imag part optionally to img_im. */
void oracle_sparse_image(const double *grid, int n, double W, double *img, double *img_im)
{
    const int h = n / 2;
    const size_t n2 = (size_t)n * n;
    /* table of the N distinct phases, exact argument reduction by integer arithmetic */
    double *ct = (double *)malloc(sizeof(double) * n), *st = (double *)malloc(sizeof(double) * n);
    for (int k = 0; k < n; ++k) { ct[k] = cos(2.0 * ORACLE_PI * k / n); st[k] = sin(2.0 * ORACLE_PI * k / n); }
    for (size_t p = 0; p < n2; ++p) { img[p] = 0.0; if (img_im) img_im[p] = 0.0; }
    for (int r = 0; r < n; ++r)
        for (int q = 0; q < n; ++q) {
            double gr = grid[2 * ((size_t)r * n + q)], gi = grid[2 * ((size_t)r * n + q) + 1];
            if (gr == 0.0 && gi == 0.0) continue;
            for (int y = 0; y < n; ++y)
                for (int x = 0; x < n; ++x) {
                    long long k = (long long)(q - h) * (x - h) + (long long)(r - h) * (y - h);
                    k %= n; if (k < 0) k += n;
                    img[(size_t)y * n + x] += gr * ct[k] - gi * st[k];
                    if (img_im) img_im[(size_t)y * n + x] += gr * st[k] + gi * ct[k];
                }
        }
    double inv = (W > 0.0) ? 1.0 / W : 0.0;
    for (size_t p = 0; p < n2; ++p) { img[p] *= inv; if (img_im) img_im[p] *= inv; }
    free(ct); free(st);
}

/* ------------------------------------------------------------------------------------------
 * The FAST route to the same numbers: textbook iterative radix-2 decimation-in-time FFT
 * (bit reversal, log2 n butterfly levels), sign +, unnormalised, in double; applied to rows
 * then columns.  The centring is done by index arithmetic exactly as the definition reads:
 * frequency index k = (q - h) mod N on input, pixel x = (j + h) mod N on output, where the
 * plain transform is X[j] = sum_k x[k] e^{+2 pi i j k / N}.
 * ---------------------------------------------------------------------------------------- */
static void fft1d_radix2_inverse(double *re, double *im, int n)
{
    /* bit-reversal permutation */
    for (int i = 1, j = 0; i < n; ++i) {
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) { double t = re[i]; re[i] = re[j]; re[j] = t; t = im[i]; im[i] = im[j]; im[j] = t; }
    }
    for (int len = 2; len <= n; len <<= 1) {
        int half = len >> 1;
        for (int i = 0; i < n; i += len)
            for (int k = 0; k < half; ++k) {
                double a = 2.0 * ORACLE_PI * (double)k / (double)len;     /* + sign: inverse */
                double wr = cos(a), wi = sin(a);
                double xr = re[i + k + half] * wr - im[i + k + half] * wi;
                double xi = re[i + k + half] * wi + im[i + k + half] * wr;
                re[i + k + half] = re[i + k] - xr;  im[i + k + half] = im[i + k] - xi;
                re[i + k] += xr;                    im[i + k] += xi;
            }
    }
}

/* Sizes that are not a power of two (the paper images at 1200 x 1200): the 1D transform is the
 * plain sum X[j] = sum_k x[k] e^{+2 pi i j k / n}, O(n^2), with the n roots of unity tabulated once and indexed
 * by (j k) mod n (exact periodicity, no large arguments).  Same sign and normalisation as the radix-2 routine. */
static void dft1d_direct_inverse(double *re, double *im, int n)
{
    double *wr = (double *)malloc(sizeof(double) * n), *wi = (double *)malloc(sizeof(double) * n);
    double *xr = (double *)malloc(sizeof(double) * n), *xi = (double *)malloc(sizeof(double) * n);
    for (int m = 0; m < n; ++m) {
        double a = 2.0 * ORACLE_PI * (double)m / (double)n;
        wr[m] = cos(a); wi[m] = sin(a);
        xr[m] = re[m]; xi[m] = im[m];
    }
    for (int j = 0; j < n; ++j) {
        double sr = 0.0, si = 0.0;
        int m = 0;                                        /* (j*k) mod n, advanced by j per term */
        for (int k = 0; k < n; ++k) {
            sr += xr[k] * wr[m] - xi[k] * wi[m];
            si += xr[k] * wi[m] + xi[k] * wr[m];
            m += j; if (m >= n) m -= n;
        }
        re[j] = sr; im[j] = si;
    }
    free(wr); free(wi); free(xr); free(xi);
}
static void fft1d_inverse_any(double *re, double *im, int n)
{
    if ((n & (n - 1)) == 0) fft1d_radix2_inverse(re, im, n);
    else dft1d_direct_inverse(re, im, n);
}

/* out[y][x] (complex, double pairs) = centred unnormalised inverse 2D DFT of grid[r][q]
 * (radix-2 rows and columns when n is a power of two, direct 1D sums otherwise) */
void oracle_ifft2_radix2(const double *grid, int n, double *out)
{
    const int h = n / 2;
    double *re = (double *)malloc(sizeof(double) * n), *im = (double *)malloc(sizeof(double) * n);
    double *tmp = (double *)malloc(sizeof(double) * 2 * (size_t)n * n);
    /* rows: u -> x */
    for (int r = 0; r < n; ++r) {
        for (int q = 0; q < n; ++q) {
            int k = ((q - h) % n + n) % n;
            re[k] = grid[2 * ((size_t)r * n + q)];
            im[k] = grid[2 * ((size_t)r * n + q) + 1];
        }
        fft1d_inverse_any(re, im, n);
        for (int j = 0; j < n; ++j) {
            int x = (j + h) % n;
            tmp[2 * ((size_t)r * n + x)] = re[j];
            tmp[2 * ((size_t)r * n + x) + 1] = im[j];
        }
    }
    /* columns: v -> y */
    for (int x = 0; x < n; ++x) {
        for (int r = 0; r < n; ++r) {
            int k = ((r - h) % n + n) % n;
            re[k] = tmp[2 * ((size_t)r * n + x)];
            im[k] = tmp[2 * ((size_t)r * n + x) + 1];
        }
        fft1d_inverse_any(re, im, n);
        for (int j = 0; j < n; ++j) {
            int y = (j + h) % n;
            out[2 * ((size_t)y * n + x)] = re[j];
            out[2 * ((size_t)y * n + x) + 1] = im[j];
        }
    }
    free(re); free(im); free(tmp);
}

/* ------------------------------------------------------------------------------------------
 * One dirty image, start to end (a0..a5): grid, weight, transform, divide by W, real part.
 *   image [N][N] double; image_im (may be NULL) the imaginary part, also / W
 *   grid_out (may be NULL) [N][N] complex128; cnt_out (may be NULL); cell_idx (may be NULL)
 *   returns W.  W == 0 -> all-zero image.
 * ---------------------------------------------------------------------------------------- */
double oracle_image_one(const float *vis, const float *uvw_t, double f_hz, int B, int n_pix,
                        double pixscale_rad, int weighting, double *image, double *image_im,
                        double *grid_out, uint32_t *cnt_out, int32_t *cell_idx)
{
    const size_t n2 = (size_t)n_pix * n_pix;
    double *grid = grid_out ? grid_out : (double *)malloc(sizeof(double) * 2 * n2);
    uint32_t *cnt = cnt_out ? cnt_out : (uint32_t *)malloc(sizeof(uint32_t) * n2);
    double *cimg = (double *)malloc(sizeof(double) * 2 * n2);
    double W = oracle_grid_one(vis, uvw_t, f_hz, B, n_pix, pixscale_rad, weighting, grid, cnt, cell_idx);
    oracle_ifft2_radix2(grid, n_pix, cimg);
    double inv = (W > 0.0) ? 1.0 / W : 0.0;
    for (size_t p = 0; p < n2; ++p) {
        image[p] = cimg[2 * p] * inv;
        if (image_im) image_im[p] = cimg[2 * p + 1] * inv;
    }
    free(cimg);
    if (!grid_out) free(grid);
    if (!cnt_out) free(cnt);
    return W;
}

/* ------------------------------------------------------------------------------------------
 * Batch driver: images img_ids[0..n_ids) of a [T][C][P][B] visibility set, one image per task,
 * nthreads POSIX threads.  images [n_ids][N][N] double, wsum [n_ids] double.
 * Image index i = (t*C + c)*P + p.
 * ---------------------------------------------------------------------------------------- */
typedef struct {
    const float *vis, *uvw_m; const double *freqs_hz;
    int T, C, P, B, n_pix, weighting; double pixscale_rad;
    const int64_t *img_ids; int n_ids; double *images; double *wsum;
    int tid, nthreads;
} batch_job_t;

static void *batch_worker(void *arg)
{
    batch_job_t *j = (batch_job_t *)arg;
    const size_t n2 = (size_t)j->n_pix * j->n_pix;
    for (int k = j->tid; k < j->n_ids; k += j->nthreads) {
        int64_t i = j->img_ids[k];
        int p = (int)(i % j->P);
        int c = (int)((i / j->P) % j->C);
        int t = (int)(i / ((int64_t)j->P * j->C));
        const float *v = j->vis + 2 * ((((size_t)t * j->C + c) * j->P + p) * (size_t)j->B);
        const float *uvw = j->uvw_m + (size_t)t * j->B * 3;
        j->wsum[k] = oracle_image_one(v, uvw, j->freqs_hz[c], j->B, j->n_pix, j->pixscale_rad,
                                      j->weighting, j->images + (size_t)k * n2, NULL, NULL, NULL, NULL);
    }
    return NULL;
}

int oracle_image_batch(const float *vis, const float *uvw_m, const double *freqs_hz,
                       int T, int C, int P, int B, int n_pix, double pixscale_rad, int weighting,
                       const int64_t *img_ids, int n_ids, double *images, double *wsum, int nthreads)
{
    if (nthreads < 1) nthreads = 1;
    if (nthreads > 256) nthreads = 256;
    pthread_t th[256];
    batch_job_t jobs[256];
    for (int k = 0; k < nthreads; ++k) {
        batch_job_t jb = { vis, uvw_m, freqs_hz, T, C, P, B, n_pix, weighting, pixscale_rad,
                           img_ids, n_ids, images, wsum, k, nthreads };
        jobs[k] = jb;
        if (pthread_create(&th[k], NULL, batch_worker, &jobs[k]) != 0) return -1;
    }
    for (int k = 0; k < nthreads; ++k) pthread_join(th[k], NULL);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Averaged images ("Images belonging to the same time bin are averaged together";
 * L251 "averaged in time over the entire processed time frame and frequency over the 30.72 MHz
 * bandwidth"; reading R14): the plain definition -- image every (t, c, p) with
 * oracle_image_one, then take the arithmetic mean over c (avg_time == 0: out [T][P][N][N]) or over
 * (t, c) (avg_time != 0: out [P][N][N]).  Images with W == 0 are zero and still count in the mean.
 * Pins (tests/test_oracle_pins.py): mean of unit-source images has 1.0 at the centre; linearity
 * (equals the transform of the W-weighted sum of the grids, evaluated independently with numpy);
 * centre pixel closed form mean_c(sum 2 Re V / W_c).
 * ---------------------------------------------------------------------------------------- */
int oracle_image_avg(const float *vis, const float *uvw_m, const double *freqs_hz,
                     int T, int C, int P, int B, int n_pix, double pixscale_rad, int weighting,
                     int avg_time, double *out)
{
    const size_t n2 = (size_t)n_pix * n_pix;
    const size_t n_out = avg_time ? (size_t)P : (size_t)T * P;
    double *img = (double *)malloc(sizeof(double) * n2);
    if (!img) return -1;
    for (size_t k = 0; k < n_out * n2; ++k) out[k] = 0.0;
    for (int t = 0; t < T; ++t)
        for (int c = 0; c < C; ++c)
            for (int p = 0; p < P; ++p) {
                const float *v = vis + 2 * ((((size_t)t * C + c) * P + p) * (size_t)B);
                oracle_image_one(v, uvw_m + (size_t)t * B * 3, freqs_hz[c], B, n_pix, pixscale_rad,
                                 weighting, img, NULL, NULL, NULL, NULL);
                double *dst = out + (avg_time ? (size_t)p : (size_t)t * P + p) * n2;
                for (size_t k = 0; k < n2; ++k) dst[k] += img[k];
            }
    const double inv = 1.0 / (avg_time ? (double)T * C : (double)C);
    for (size_t k = 0; k < n_out * n2; ++k) out[k] *= inv;
    free(img);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Stokes I images ("BLINK currently images only the XX polarisation ... does not form Stokes I";
 * L351 lists it as future work, reading R18): the plain definition --
 * image the XX plane (p = 0) and the YY plane (p = P-1; P = 2: XX, YY; P = 4: XX, XY, YX, YY) of every (t, c) with
 * oracle_image_one and take I = (I_XX + I_YY) / 2 pixel by pixel.  out [n_ids][N][N], wsum [n_ids] (the W the two
 * planes share); tc_ids index (t, c) pairs, tc = t*C + c.
 * Pins (tests/test_oracle_pins.py): unit sources in XX and YY -> 1.0 at the centre; YY = -XX -> zero image;
 * XX-only signal -> half the XX image; a single baseline against the closed-form cosine of the mean visibility;
 * equals one image of the averaged visibilities (linearity, evaluated through oracle_image_one independently).
 * ---------------------------------------------------------------------------------------- */
int oracle_image_stokes_i(const float *vis, const float *uvw_m, const double *freqs_hz,
                          int T, int C, int P, int B, int n_pix, double pixscale_rad, int weighting,
                          const int64_t *tc_ids, int n_ids, double *out, double *wsum)
{
    const size_t n2 = (size_t)n_pix * n_pix;
    if (P != 2 && P != 4) return -1;
    double *xx = (double *)malloc(sizeof(double) * n2), *yy = (double *)malloc(sizeof(double) * n2);
    if (!xx || !yy) { free(xx); free(yy); return -1; }
    for (int k = 0; k < n_ids; ++k) {
        const int64_t tc = tc_ids[k];
        const int t = (int)(tc / C), c = (int)(tc % C);
        if (t < 0 || t >= T) { free(xx); free(yy); return -1; }
        const float *vxx = vis + 2 * ((((size_t)t * C + c) * P + 0) * (size_t)B);
        const float *vyy = vis + 2 * ((((size_t)t * C + c) * P + (P - 1)) * (size_t)B);
        const float *uvw = uvw_m + (size_t)t * B * 3;
        const double W = oracle_image_one(vxx, uvw, freqs_hz[c], B, n_pix, pixscale_rad, weighting, xx, NULL, NULL, NULL, NULL);
        oracle_image_one(vyy, uvw, freqs_hz[c], B, n_pix, pixscale_rad, weighting, yy, NULL, NULL, NULL, NULL);
        for (size_t q = 0; q < n2; ++q) out[(size_t)k * n2 + q] = 0.5 * (xx[q] + yy[q]);
        wsum[k] = W;
    }
    free(xx); free(yy);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Calibration / cable / geometric corrections as per-antenna complex gains (PAPER.md L182-184:
 * "precomputed calibration solutions are applied to visibilities, followed by geometric and cable
 * length corrections ... Visibilities are one-to-one mapped to GPU threads"; reading R15):
 *   V'[t][c][p][b] = g[c][p][a1(b)] * conj(g[c][p][a2(b)]) * V[t][c][p][b]
 * evaluated in double, stored back as complex64 (the paper corrects its fp32 visibilities in place).
 * A per-antenna phase exp(i phi_a) covers cable length and geometric delay (both are differences of
 * per-antenna delays).  Pins (tests/test_oracle_pins.py): unit gains are the identity; pure phases
 * rotate by phi_a1 - phi_a2 and keep |V|; an independent numpy evaluation; applying the gains that undo
 * a simulated corruption restores the uncorrupted image.
 * ---------------------------------------------------------------------------------------- */
void oracle_apply_gains(const float *vis, const float *gains, const int32_t *ant_pairs,
                        int T, int C, int P, int B, int A, float *vis_out)
{
    for (int t = 0; t < T; ++t)
        for (int c = 0; c < C; ++c)
            for (int p = 0; p < P; ++p) {
                const float *g = gains + 2 * (((size_t)c * P + p) * (size_t)A);
                const size_t row = (((size_t)t * C + c) * P + p) * (size_t)B;
                for (int b = 0; b < B; ++b) {
                    const int a1 = ant_pairs[2 * b], a2 = ant_pairs[2 * b + 1];
                    const double g1r = g[2 * a1], g1i = g[2 * a1 + 1], g2r = g[2 * a2], g2i = g[2 * a2 + 1];
                    const double fr = g1r * g2r + g1i * g2i, fi = g1i * g2r - g1r * g2i;      /* g1 * conj(g2) */
                    const double vr = vis[2 * (row + b)], vi = vis[2 * (row + b) + 1];
                    vis_out[2 * (row + b)] = (float)(fr * vr - fi * vi);
                    vis_out[2 * (row + b) + 1] = (float)(fr * vi + fi * vr);
                }
            }
}

/* ------------------------------------------------------------------------------------------
 * Convolutional (anti-aliasing) gridding -- SURVEY 8(f) rank 2.  PAPER.md L192: "Visibilities are not
 * convolved with any kernel at this stage, a feature to be introduced in the near future to alleviate the
 * effects of source aliasing"; L351 "The implementation of a gridding kernel to minimise aliasing is in
 * progress".  The paper defines no kernel, so DESIGN.md reading R16 fixes one (the separable Kaiser-Bessel
 * window that WSClean, the paper's comparison imager, uses by default):
 *
 *   k(d)   = I0(beta sqrt(1 - (2 d / S)^2)) / I0(beta)   for |d| <= S/2, else 0      (S odd: 1, 3, 5, 7)
 *   x      = u_m * s_c (ONE fp32 multiply, as in a1), iu0 = rint(x), fx = x - iu0 in [-1/2, 1/2]  (exact)
 *   taps   j = -r..r (r = (S-1)/2) at column iu0 + j, distance d = j - fx from the sample,
 *          weight wx_j = k(j - fx) / sum_i k(i - fx)       (normalised: the S taps of an axis sum to 1)
 *   the same along v; cell (iv0 + i, iu0 + j) += wy_i wx_j V, mirror cell (-(iv0+i), -(iu0+j)) += wy_i wx_j conj(V)
 *          (the Hermitian sample at (-x,-y) has offsets -fx, -fy and k is even: exactly the mirrored taps)
 *   range  a sample is dropped (with its conjugate) when |iu0| or |iv0| > h - 1 - r, so that the whole
 *          support stays inside |iu|, |iv| <= h - 1 (reading R4 extended)
 *   W      natural weighting only: W = 2 B_in (every sample carries total weight 1)
 *   image  I[y][x] = (1/W) Re IDFT(G)[y][x] / (c((y-h)/N) c((x-h)/N)),   the grid correction
 *          c(xi) = int_{-S/2}^{S/2} k(d) cos(2 pi d xi) dd / int_{-S/2}^{S/2} k(d) dd      (c(0) = 1)
 * S = 1 is nearest-cell gridding (the only tap has normalised weight 1): the S = 1 GRID equals
 * oracle_grid_one's; the library itself offers S = 3, 5, 7.
 * Pins (tests/test_oracle_pins.py): I0 series vs scipy.special.i0 / numpy.i0; taps sum to 1, are symmetric
 * at fx = 0 and mirror under fx -> -fx; S = 1 grid == oracle_grid_one; sum(G) = sum 2 Re V; Hermitian;
 * independent numpy re-gridding (np.add.at over an outer product); quadrature taper vs the closed form
 * sinh(sqrt(beta^2 - (pi S xi)^2)) / sqrt(...) normalised; unit source -> exactly 1.0 at the centre;
 * single off-grid baseline: the corrected image is closer to the exact (ungridded) cosine than nearest-cell
 * gridding is, inside the central half of the field.
 * ---------------------------------------------------------------------------------------- */
static double bessel_i0_series(double x)
{
    /* I0(x) = sum_k ((x/2)^2)^k / (k!)^2 ; terms decay once k > x/2 ; |x| <= ~60 here */
    const double q = 0.25 * x * x;
    double term = 1.0, sum = 1.0;
    for (int k = 1; k < 500; ++k) {
        term *= q / ((double)k * (double)k);
        sum += term;
        if (term < 1e-17 * sum) break;
    }
    return sum;
}
double oracle_bessel_i0(double x) { return bessel_i0_series(x); }

double oracle_kb(double d, int S, double beta)
{
    const double a = 2.0 * d / (double)S;
    const double z = 1.0 - a * a;
    if (z < 0.0) return (z > -1e-14) ? 1.0 / bessel_i0_series(beta) : 0.0;   /* |d| = S/2 up to rounding */
    return bessel_i0_series(beta * sqrt(z)) / bessel_i0_series(beta);
}

/* w[0..S) : normalised tap weights of one axis for fractional offset f = x - rint(x) */
void oracle_conv_taps(double f, int S, double beta, double *w)
{
    const int r = (S - 1) / 2;
    double sum = 0.0;
    for (int j = -r; j <= r; ++j) { w[j + r] = oracle_kb((double)j - f, S, beta); sum += w[j + r]; }
    for (int j = 0; j < S; ++j) w[j] /= sum;
}

/* grid correction c(xi), xi = (pixel - h)/N in [-1/2, 1/2): composite Simpson over the support */
double oracle_conv_taper(double xi, int S, double beta)
{
    const int M = 8192;                             /* even number of intervals */
    const double lo = -0.5 * (double)S, hstep = (double)S / (double)M;
    double num = 0.0, den = 0.0;
    for (int m = 0; m <= M; ++m) {
        const double d = lo + hstep * (double)m;
        const double wq = (m == 0 || m == M) ? 1.0 : ((m & 1) ? 4.0 : 2.0);
        const double kd = oracle_kb(d, S, beta);
        num += wq * kd * cos(2.0 * ORACLE_PI * d * xi);
        den += wq * kd;
    }
    return num / den;
}

/* nearest cell of the convolutional gridder: oracle_cell with the tighter range h-1-r; -1 when dropped.
 * fx, fy (may be NULL) receive the exact offsets x - iu0, y - iv0. */
int32_t oracle_cell_conv(float u_m, float v_m, float s, int n_pix, int S, double *fx, double *fy)
{
    const int h = n_pix / 2, r = (S - 1) / 2;
    volatile float x = u_m * s;
    volatile float y = v_m * s;
    float xr = nearbyintf(x);
    float yr = nearbyintf(y);
    const float lim = (float)(h - 1 - r);
    if (!(fabsf(xr) <= lim && fabsf(yr) <= lim)) return -1;
    if (fx) *fx = (double)x - (double)xr;
    if (fy) *fy = (double)y - (double)yr;
    return (int32_t)(((int)yr + h) * n_pix + ((int)xr + h));
}

double oracle_grid_conv_one(const float *vis, const float *uvw_t, double f_hz, int B, int n_pix,
                            double pixscale_rad, int S, double beta, double *grid, int32_t *cell_idx)
{
    const size_t n2 = (size_t)n_pix * n_pix;
    const int h = n_pix / 2, r = (S - 1) / 2;
    fesetround(FE_TONEAREST);
    memset(grid, 0, n2 * 2 * sizeof(double));
    float s = oracle_scale(f_hz, n_pix, pixscale_rad);
    double W = 0.0, wx[16], wy[16];
    for (int b = 0; b < B; ++b) {
        double fx, fy;
        int32_t cell = oracle_cell_conv(uvw_t[3 * b], uvw_t[3 * b + 1], s, n_pix, S, &fx, &fy);
        if (cell_idx) cell_idx[b] = cell;
        if (cell < 0) continue;
        const int iv0 = cell / n_pix - h, iu0 = cell % n_pix - h;
        oracle_conv_taps(fx, S, beta, wx);
        oracle_conv_taps(fy, S, beta, wy);
        const double re = (double)vis[2 * b], im = (double)vis[2 * b + 1];
        for (int i = -r; i <= r; ++i)
            for (int j = -r; j <= r; ++j) {
                const double w = wy[i + r] * wx[j + r];
                const size_t k = (size_t)(iv0 + i + h) * n_pix + (size_t)(iu0 + j + h);
                const size_t km = (size_t)(h - (iv0 + i)) * n_pix + (size_t)(h - (iu0 + j));
                grid[2 * k] += w * re;   grid[2 * k + 1] += w * im;
                grid[2 * km] += w * re;  grid[2 * km + 1] -= w * im;
            }
        W += 2.0;
    }
    return W;
}

double oracle_image_conv_one(const float *vis, const float *uvw_t, double f_hz, int B, int n_pix,
                             double pixscale_rad, int S, double beta, double *image, double *image_im,
                             double *grid_out, int32_t *cell_idx)
{
    const size_t n2 = (size_t)n_pix * n_pix;
    const int h = n_pix / 2;
    double *grid = grid_out ? grid_out : (double *)malloc(sizeof(double) * 2 * n2);
    double *cimg = (double *)malloc(sizeof(double) * 2 * n2);
    double *c = (double *)malloc(sizeof(double) * n_pix);
    double W = oracle_grid_conv_one(vis, uvw_t, f_hz, B, n_pix, pixscale_rad, S, beta, grid, cell_idx);
    oracle_ifft2_radix2(grid, n_pix, cimg);
    for (int x = 0; x < n_pix; ++x) c[x] = oracle_conv_taper((double)(x - h) / (double)n_pix, S, beta);
    double inv = (W > 0.0) ? 1.0 / W : 0.0;
    for (int y = 0; y < n_pix; ++y)
        for (int x = 0; x < n_pix; ++x) {
            const size_t p = (size_t)y * n_pix + x;
            const double corr = inv / (c[y] * c[x]);
            image[p] = cimg[2 * p] * corr;
            if (image_im) image_im[p] = cimg[2 * p + 1] * corr;
        }
    free(cimg); free(c);
    if (!grid_out) free(grid);
    return W;
}

/* batch driver, as oracle_image_batch */
typedef struct {
    const float *vis, *uvw_m; const double *freqs_hz;
    int T, C, P, B, n_pix, S; double pixscale_rad, beta;
    const int64_t *img_ids; int n_ids; double *images; double *wsum;
    int tid, nthreads;
} conv_job_t;

static void *conv_worker(void *arg)
{
    conv_job_t *j = (conv_job_t *)arg;
    const size_t n2 = (size_t)j->n_pix * j->n_pix;
    for (int k = j->tid; k < j->n_ids; k += j->nthreads) {
        int64_t i = j->img_ids[k];
        int p = (int)(i % j->P);
        int c = (int)((i / j->P) % j->C);
        int t = (int)(i / ((int64_t)j->P * j->C));
        const float *v = j->vis + 2 * ((((size_t)t * j->C + c) * j->P + p) * (size_t)j->B);
        const float *uvw = j->uvw_m + (size_t)t * j->B * 3;
        j->wsum[k] = oracle_image_conv_one(v, uvw, j->freqs_hz[c], j->B, j->n_pix, j->pixscale_rad, j->S, j->beta,
                                           j->images + (size_t)k * n2, NULL, NULL, NULL);
    }
    return NULL;
}

int oracle_image_conv_batch(const float *vis, const float *uvw_m, const double *freqs_hz,
                            int T, int C, int P, int B, int n_pix, double pixscale_rad, int S, double beta,
                            const int64_t *img_ids, int n_ids, double *images, double *wsum, int nthreads)
{
    if (nthreads < 1) nthreads = 1;
    if (nthreads > 256) nthreads = 256;
    if (S < 1 || S > 15 || !(S & 1)) return -2;
    pthread_t th[256];
    conv_job_t jobs[256];
    for (int k = 0; k < nthreads; ++k) {
        conv_job_t jb = { vis, uvw_m, freqs_hz, T, C, P, B, n_pix, S, pixscale_rad, beta,
                          img_ids, n_ids, images, wsum, k, nthreads };
        jobs[k] = jb;
        if (pthread_create(&th[k], NULL, conv_worker, &jobs[k]) != 0) return -1;
    }
    for (int k = 0; k < nthreads; ++k) pthread_join(th[k], NULL);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * CMAC correlator -- SURVEY 8(f) rank 4 (last item).  PAPER.md eq. 3 (L98) and section 6.2.2
 * (L172-178): "voltage data from every pair of antennas are combined to produce visibilities ...
 * only the Conjugate Multiply Accumulate (CMAC) operation was developed ... partial results are
 * summed together ... and the result is divided by the integration time and number of averaged
 * frequency channels.  Visibilities are stored in a lower triangular matrix form for each
 * integration interval and output frequency channel."  DESIGN.md reading R17 fixes what the paper
 * leaves open (sample format and array order):
 *   volt [F][A][Ns][2] int8: fine channel f, input a (tile x polarisation), time sample, (re, im);
 *        MWA Phase I VCS samples are 4 + 4 bit, i.e. values in [-8, 7]; any value in [-127, 127] is allowed
 *   interval t = samples [t n_t, (t+1) n_t), T = Ns / n_t;  output channel c = fine channels [c n_avg, (c+1) n_avg)
 *   S[t][c][i][j] = sum_{f in c} sum_{s in t} x_i(f,s) conj(x_j(f,s))      for j <= i   (exact, 64-bit integers)
 *   vis [T][C][A(A+1)/2] complex64, entry i(i+1)/2 + j = (float)S / (float)(n_t n_avg): ONE fp32 division of two
 *        exactly representable integers (|S| < 2^24 whenever n_t n_avg max|x|^2 2 < 2^24; larger sums are first
 *        rounded to fp32 by the int -> float conversion, on both sides)
 * Pins (tests/test_oracle_corr_pins.py): hand-worked two-input case (tests/golden/cmac_two_inputs.txt);
 * constant inputs -> c_i conj(c_j); autos real and = mean |x|^2; conjugate symmetry under swapping inputs;
 * independent numpy einsum; averaging n_avg channels = mean of the single-channel results (exact sums);
 * a common signal with per-input phase steps -> the phase differences; independent noise -> cross terms
 * within 6 sigma of zero.
 * ---------------------------------------------------------------------------------------- */
int oracle_correlate(const int8_t *volt, int F, int A, int Ns, int n_t, int n_avg, float *vis)
{
    if (n_t < 1 || n_avg < 1 || Ns % n_t != 0 || F % n_avg != 0) return -1;
    const int T = Ns / n_t, C = F / n_avg;
    const size_t ntri = (size_t)A * (A + 1) / 2;
    const float norm = (float)((long long)n_t * n_avg);
    for (int t = 0; t < T; ++t)
        for (int c = 0; c < C; ++c)
            for (int i = 0; i < A; ++i)
                for (int j = 0; j <= i; ++j) {
                    long long sr = 0, si = 0;
                    for (int f = c * n_avg; f < (c + 1) * n_avg; ++f) {
                        const int8_t *xi = volt + 2 * (((size_t)f * A + i) * Ns + (size_t)t * n_t);
                        const int8_t *xj = volt + 2 * (((size_t)f * A + j) * Ns + (size_t)t * n_t);
                        for (int s = 0; s < n_t; ++s) {
                            const long long ar = xi[2 * s], ai = xi[2 * s + 1], br = xj[2 * s], bi = xj[2 * s + 1];
                            sr += ar * br + ai * bi;           /* (ar + i ai)(br - i bi) */
                            si += ai * br - ar * bi;
                        }
                    }
                    float *o = vis + 2 * (((size_t)t * C + c) * ntri + (size_t)i * (i + 1) / 2 + j);
                    o[0] = (float)sr / norm;
                    o[1] = (float)si / norm;
                }
    return 0;
}
