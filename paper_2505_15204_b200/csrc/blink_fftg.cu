// Centred inverse 2D transform for image sides that are NOT a power of two (N even, N = 2^a 3^b 5^c; the paper
// images at 1200 x 1200).  Same definition as blink_fft2d.cu (sign +, unnormalised, fftshift,
// 1/scale, real part; readings R5-R7), different machinery: a mixed-radix Stockham transform whose every stage
// goes through shared memory (two ping-pong arrays), radices 15, 16 (register-resident 3 x 5 / 4 x 4 butterflies), 5, 3, 4, 2,
// twiddles from an N-entry table
// exp(+2 pi i m / N) that an init kernel writes (in double) into the caller's workspace.
//   pass 1 (gfft_rows_kernel): rows, in place, input taken at the centred column (n + h) mod N, output in natural x;
//   pass 2 (gfft_cols_kernel): KC columns per CTA, output row / column moved by h again, scaled, real part stored.
// This is the fallback for the paper's own sizes, not a tuned path.
#include <algorithm>

#include "blink_common.cuh"
#include "blink_fft.cuh"
#include "blink_fftg.cuh"

namespace blink {

// Threads per CTA.  The paper's side 1200 runs as 15 x 5 x 16 (register-resident radix-15 and radix-16 butterflies: three
// stages and three CTA barriers per transform instead of the five of 5 x 5 x 3 x 4 x 4 -- the barriers between stages were
// the measured bound of round 1's column pass: 3.3 warps waiting at one per issuing warp).  Four transforms per CTA are then
// 320 + 960 + 300 butterflies: with 320 threads that is 1 + 3 + 1 rounds with (almost) every thread busy.
constexpr int kGRowThreads = 512, kGColThreads = 480, kGThreads1200 = 320;
template <int NN> __host__ __device__ constexpr int grow_threads() { return NN == 1200 ? kGThreads1200 : kGRowThreads; }
template <int NN> __host__ __device__ constexpr int gcol_threads() { return NN == 1200 ? kGThreads1200 : kGColThreads; }
constexpr int kGRowsMax = 4;                       // rows per round of a row-pass CTA
struct GPlan {
    int n, nst;
    int radix[16];
    int toff[16];                                  // stage s reads its twiddles W_n^(k n / (P_s R_s)), k < P_s, at table[toff[s] + k]
};

// The N-entry table exp(2 pi i m / N) of the workspace is re-packed per CTA into one COMPACT run per stage (stage s: P_s
// consecutive entries), because a warp of a stage reads the entries k * step for consecutive k: out of the full table that is
// a stride of `step` complex numbers -- 16 at the radix-3 stage of 1200, i.e. every lane in the same bank (measured: 32
// wavefronts per load, 19 % of the column kernel's shared-memory traffic); out of the compact run it is unit stride.
__device__ __forceinline__ void stage_twiddles(float2 *__restrict__ stw, const float2 *__restrict__ tw, const GPlan &pl)
{
    int P = 1;
    for (int s = 0; s < pl.nst; ++s) {
        const int step = pl.n / (P * pl.radix[s]);
        for (int k = threadIdx.x; k < P; k += blockDim.x) stw[pl.toff[s] + k] = tw[k * step];
        P *= pl.radix[s];
    }
}

__global__ void gfft_twiddle_kernel(float2 *tw, int n)
{
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= n) return;
    double s, c;
    sincospi(2.0 * (double)m / (double)n, &s, &c);
    tw[m] = make_float2((float)c, (float)s);
}

int gfft_fill_twiddles(float2 *dst, int n, cudaStream_t st)
{
    gfft_twiddle_kernel<<<(n + 255) / 256, 256, 0, st>>>(dst, n);
    BLINK_LAUNCH_CHECK("gfft_twiddle_kernel");
    return BLINK_OK;
}

// exact i / d for 0 <= i < 2^16 by a float reciprocal ((i + 1/2) / d is at least 1/(2d) away from an integer, far
// more than the rounding error of the product)
__device__ __forceinline__ int fdiv_small(int i, int d, float inv_d) { (void)d; return (int)(((float)i + 0.5f) * inv_d); }

// One Stockham stage (radix R, sub-transform length P) of `nt` independent transforms of length n stored with
// leading dimension ld: src[tr][i + r*(n/R)] -> dst[tr][(i - k)*R + k + r*P], k = i mod P, inputs r >= 1
// twiddled by W_n^(r k n/(P R)).  Reads are unit-stride in i; writes are runs of P consecutive elements, which is
// why the plan puts the odd radices first (P grows past a warp before the radix-4 stages: no bank conflicts there).
// NN / PP: n and P when they are known at compile time (the paper's side 1200 has its own instantiation: every
// division and remainder below becomes a multiply-shift and the stage loop is specialised), else 0 = run-time values.
template <int R, int NN = 0, int PP = 0>
__device__ __forceinline__ void gstage(const float2 *__restrict__ src, float2 *__restrict__ dst, int nt, int n_rt, int ld, int p_rt,
                                       const float2 *__restrict__ tw)
{
    const int n = NN ? NN : n_rt, P = PP ? PP : p_rt;
    if constexpr (NN != 0 && PP != 0) {
        constexpr int nb = NN / R;
        for (int idx = threadIdx.x; idx < nt * nb; idx += blockDim.x) {
            const int tr = idx / nb, i = idx - tr * nb;
            const int k = i % PP;
            const float2 *s = src + (size_t)tr * ld + i;
            float2 x[R];
#pragma unroll
            for (int r = 0; r < R; ++r) x[r] = s[r * nb];
            if constexpr (PP > 1) gtwiddle<R>(x, tw[k]);      // compact per-stage run (stage_twiddles)
            gbutterfly<R>(x);
            float2 *d = dst + (size_t)tr * ld + (i - k) * R + k;
#pragma unroll
            for (int r = 0; r < R; ++r) d[r * PP] = x[r];
        }
        return;
    }
    const int nb = n / R;
    const float inv_nb = 1.0f / (float)nb, inv_p = 1.0f / (float)P;
    for (int idx = threadIdx.x; idx < nt * nb; idx += blockDim.x) {
        const int tr = fdiv_small(idx, nb, inv_nb), i = idx - tr * nb;
        const int k = i - P * fdiv_small(i, P, inv_p);
        const float2 *s = src + (size_t)tr * ld + i;
        float2 x[R];
#pragma unroll
        for (int r = 0; r < R; ++r) x[r] = s[r * nb];
        if (P > 1) gtwiddle<R>(x, tw[k]);                      // one table read per butterfly; w^2.. are products
        gbutterfly<R>(x);
        float2 *d = dst + (size_t)tr * ld + (i - k) * R + k;
#pragma unroll
        for (int r = 0; r < R; ++r) d[r * P] = x[r];
    }
}

// all stages; returns the array that holds the result (natural order)
template <int NN>
__device__ __forceinline__ float2 *gfft_run(float2 *a, float2 *b, int nt, int ld, const GPlan &pl, const float2 *tw)
{
    if constexpr (NN == 1200) {                                // 15 * 5 * 16, the plan gfft2d_range builds for 1200
        gstage<15, 1200, 1>(a, b, nt, 1200, ld, 1, tw);       __syncthreads();          // toff = 0, 1, 16 (gfft2d_range)
        gstage<5, 1200, 15>(b, a, nt, 1200, ld, 15, tw + 1);  __syncthreads();
        gstage<16, 1200, 75>(a, b, nt, 1200, ld, 75, tw + 16); __syncthreads();
        return b;
    }
    int P = 1;
    for (int s = 0; s < pl.nst; ++s) {
        const int R = pl.radix[s];
        const float2 *tws = tw + pl.toff[s];
        if (R == 16) gstage<16>(a, b, nt, pl.n, ld, P, tws);
        else if (R == 15) gstage<15>(a, b, nt, pl.n, ld, P, tws);
        else if (R == 4) gstage<4>(a, b, nt, pl.n, ld, P, tws);
        else if (R == 2) gstage<2>(a, b, nt, pl.n, ld, P, tws);
        else if (R == 3) gstage<3>(a, b, nt, pl.n, ld, P, tws);
        else gstage<5>(a, b, nt, pl.n, ld, P, tws);
        __syncthreads();
        float2 *t = a; a = b; b = t;
        P *= R;
    }
    return a;
}

// ------------------------------------------------------------------------------------------ rows
template <int NN>
__global__ void __launch_bounds__(grow_threads<NN>())
gfft_rows_kernel(float2 *__restrict__ grid, long long n_rows, const GPlan pl, const float2 *__restrict__ tw, int nr, int rows_per_img,
                 int row_off, const int *__restrict__ ext, int ext_div)
{
    // logical row L -> image L / rows_per_img, row row_off + L % rows_per_img (Hermitian grids: only the rows v >= 0)
    // ext (optional): image i holds data only in its first ext[i / ext_div] logical rows; the others are all zero, so is
    // their transform, and nobody reads them: they are skipped (not read, not written)
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int n = NN ? NN : pl.n, h = n / 2;
    float2 *a = reinterpret_cast<float2 *>(smem_raw), *b = a + (size_t)nr * n;
    float2 *stw = b + (size_t)nr * n;                          // the twiddle table, staged once per CTA
    stage_twiddles(stw, tw, pl);
    __syncthreads();
    for (long long base = (long long)blockIdx.x * nr; base < n_rows; base += (long long)gridDim.x * nr) {
        const int cnt = (int)(n_rows - base < nr ? n_rows - base : nr);
        // per row of this round (nr <= kGRowsMax): where it lives in the grid and whether it has to be transformed (bit tr of
        // `live`, the same value in every thread).  The 64-bit divisions happen here, once per row -- inside the element loops
        // below they were most of the kernel's instructions (ncu: 350 k thread instructions per 1200-point row).
        float2 *grow[kGRowsMax];
        unsigned live = 0u;
#pragma unroll
        for (int tr = 0; tr < kGRowsMax; ++tr) {
            grow[tr] = grid;
            if (tr < cnt) {
                const long long L = base + tr, im = L / rows_per_img;
                const int r = (int)(L - im * rows_per_img);
                grow[tr] = grid + (im * n + row_off + r) * n;
                if (ext == nullptr || r < __ldg(ext + im / ext_div)) live |= 1u << tr;
            }
        }
        if (live == 0u) continue;
#pragma unroll
        for (int tr = 0; tr < kGRowsMax; ++tr) {
            if (tr >= cnt) break;
            const bool lv = (live >> tr) & 1u;
            for (int j = threadIdx.x; j < n; j += blockDim.x) {
                int q = j + h;                                 // transform index j lives in centred column (j + h) mod n
                if (q >= n) q -= n;
                a[(size_t)tr * n + j] = lv ? grow[tr][q] : make_float2(0.f, 0.f);
            }
        }
        __syncthreads();
        const float2 *res = gfft_run<NN>(a, b, cnt, n, pl, stw);
#pragma unroll
        for (int tr = 0; tr < kGRowsMax; ++tr) {
            if (tr >= cnt || !((live >> tr) & 1u)) continue;
            for (int j = threadIdx.x; j < n; j += blockDim.x) grow[tr][j] = res[(size_t)tr * n + j];   // natural (unshifted) x order
        }
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------ columns + epilogue
template <int NN>
__global__ void __launch_bounds__(gcol_threads<NN>())
gfft_cols_kernel(const float2 *__restrict__ grid, const GPlan pl, const float2 *__restrict__ tw, int kc, const float *__restrict__ scale,
                 int scale_div, int img_base, float *__restrict__ image, float *__restrict__ image_imag)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int n = NN ? NN : pl.n, h = n / 2;
    const int ld = n + 1;                                      // odd leading dimension: the kc columns of a row fall in different banks
    float2 *a = reinterpret_cast<float2 *>(smem_raw), *b = a + (size_t)kc * ld;
    float2 *stw = b + (size_t)kc * ld;
    stage_twiddles(stw, tw, pl);
    const int x0 = blockIdx.x * kc, img = blockIdx.y;
    const size_t img_off = (size_t)img * n * n;
    const int lg = 31 - __clz(kc);                             // kc is a power of two (gfft2d_range): shifts, not divisions
    for (int idx = threadIdx.x; idx < n * kc; idx += blockDim.x) {
        const int j = idx >> lg, c = idx & (kc - 1);           // c fastest: kc consecutive columns of one row
        int r = j + h;                                         // transform index j lives in centred row (j + h) mod n
        if (r >= n) r -= n;
        a[(size_t)c * ld + j] = grid[img_off + (size_t)r * n + x0 + c];
    }
    __syncthreads();
    const float2 *res = gfft_run<NN>(a, b, kc, ld, pl, stw);
    float s = 1.0f;
    if (scale != nullptr) {
        const float w = scale[(img_base + img) / scale_div];
        s = (w != 0.0f) ? 1.0f / w : 0.0f;
    }
    for (int idx = threadIdx.x; idx < n * kc; idx += blockDim.x) {
        const int j = idx >> lg, c = idx & (kc - 1);
        int y = j + h, x = x0 + c + h;                         // fftshift of both axes
        if (y >= n) y -= n;
        if (x >= n) x -= n;
        const float2 v = res[(size_t)c * ld + j];
        image[img_off + (size_t)y * n + x] = v.x * s;
        if (image_imag != nullptr) image_imag[img_off + (size_t)y * n + x] = v.y * s;
    }
}

// Hermitian grids (everything the library's own gridders produce: G[-v][-u] = conj G[v][u], row and column -N/2
// empty): after the row pass R[-v][x] = conj R[v][x], so only the rows v >= 0 were transformed, and two columns
// x1, x2 become ONE complex transform Z[v] = R[v][x1] + i R[v][x2], Z[-v] = conj R[v][x1] + i conj R[v][x2] whose
// real part is image column x1 and imaginary part image column x2.  Half the reads, half the transforms.
template <int NN>
__global__ void __launch_bounds__(gcol_threads<NN>())
gfft_cols_herm_kernel(const float2 *__restrict__ grid, const GPlan pl, const float2 *__restrict__ tw, int kc, const float *__restrict__ scale,
                      int scale_div, int img_base, float *__restrict__ image, const int *__restrict__ ext, int ext_div, int ext_base, int ld)
{
    // ld (herm_ld): the leading dimension that makes the transposing accesses below -- lane -> (row v + lane / np, pair lane % np),
    // address pair * ld + row -- fall into every bank exactly twice (the minimum for 8-byte words)
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int n = NN ? NN : pl.n, h = n / 2, np = kc / 2;                // np column pairs = transforms per CTA
    float2 *a = reinterpret_cast<float2 *>(smem_raw), *b = a + (size_t)np * ld;
    float2 *stw = b + (size_t)np * ld;
    stage_twiddles(stw, tw, pl);
    const int x0 = blockIdx.x * kc, img = blockIdx.y;
    const size_t img_off = (size_t)img * n * n;
    const int vu = ext != nullptr ? __ldg(ext + (ext_base + img) / ext_div) : h;      // rows v >= vu are zero and are not read
    const int lg = 31 - __clz(np);                             // np is a power of two (gfft2d_range): shifts, not divisions
    for (int idx = threadIdx.x; idx < h * np; idx += blockDim.x) {
        const int v = idx >> lg, p = idx & (np - 1);           // p fastest: consecutive 16-byte column pairs of one row
        float4 q = make_float4(0.f, 0.f, 0.f, 0.f);
        if (v < vu) q = *reinterpret_cast<const float4 *>(grid + img_off + (size_t)(h + v) * n + x0 + 2 * p);
        a[(size_t)p * ld + v] = make_float2(q.x - q.w, q.y + q.z);                   // S1 + i S2
        if (v > 0) a[(size_t)p * ld + n - v] = make_float2(q.x + q.w, q.z - q.y);    // conj S1 + i conj S2
    }
    for (int p = threadIdx.x; p < np; p += blockDim.x) a[(size_t)p * ld + h] = make_float2(0.f, 0.f);   // the empty row -N/2
    __syncthreads();
    const float2 *res = gfft_run<NN>(a, b, np, ld, pl, stw);
    float s = 1.0f;
    if (scale != nullptr) {
        const float w = scale[(img_base + img) / scale_div];
        s = (w != 0.0f) ? 1.0f / w : 0.0f;
    }
    for (int idx = threadIdx.x; idx < n * np; idx += blockDim.x) {
        const int j = idx >> lg, p = idx & (np - 1);
        int y = j + h, x = x0 + 2 * p + h, x1 = x0 + 2 * p + 1 + h;      // fftshift of both axes
        if (y >= n) y -= n;
        if (x >= n) x -= n;
        if (x1 >= n) x1 -= n;
        const float2 z = res[(size_t)p * ld + j];
        if ((h & 1) == 0) {                                    // x is even, x1 = x + 1 < n: one aligned 8-byte store
            *reinterpret_cast<float2 *>(image + img_off + (size_t)y * n + x) = make_float2(z.x * s, z.y * s);
        } else {
            image[img_off + (size_t)y * n + x] = z.x * s;
            image[img_off + (size_t)y * n + x1] = z.y * s;
        }
    }
}

// ------------------------------------------------------------------------------------------ host
bool size_supported(int n)
{
    if (n < 32 || n > kMaxPix || (n & 1)) return false;
    while (n % 2 == 0) n /= 2;
    while (n % 3 == 0) n /= 3;
    while (n % 5 == 0) n /= 5;
    return n == 1;
}
// leading dimension of the Hermitian column kernel's arrays for np transforms per CTA: np * (ld mod 16) = 32 (mod 16 banks of
// 8 bytes) spreads the np x (32 / np) lanes of a transposing access over all banks; np <= 2 needs nothing but keeps the odd pad
static int herm_ld(int n, int np)
{
    const int want = np == 4 ? 8 : np == 8 ? 4 : 1;
    return n + (want - n % 16 + 16) % 16;
}
size_t gfft_workspace_bytes(int n) { return is_pow2(n) ? 0 : align_up((size_t)n * sizeof(float2), 256); }

int gfft2d_range(float2 *grid, int n, int batch, const float *scale, int scale_div, int img_base, float *image,
                 float *image_imag, float2 *tw, cudaStream_t st, bool hermitian, const int *row_extent, int ext_div)
{
    if (image_imag) hermitian = false;                          // the imaginary part is only defined for the general transform
    if (batch == 0) return BLINK_OK;
    if (!tw) return BLINK_ERR_WORKSPACE;
    GPlan pl{};
    pl.n = n;
    int m = n;
    while (m % 15 == 0) { pl.radix[pl.nst++] = 15; m /= 15; }  // odd radices first (see gstage); 15 and 16 in registers
    while (m % 5 == 0) { pl.radix[pl.nst++] = 5; m /= 5; }
    while (m % 3 == 0) { pl.radix[pl.nst++] = 3; m /= 3; }
    while (m % 16 == 0) { pl.radix[pl.nst++] = 16; m /= 16; }
    while (m % 4 == 0) { pl.radix[pl.nst++] = 4; m /= 4; }
    while (m % 2 == 0) { pl.radix[pl.nst++] = 2; m /= 2; }
    if (m != 1) return BLINK_ERR_UNSUPPORTED;
    for (int s = 0, P = 1, off = 0; s < pl.nst; ++s) { pl.toff[s] = off; off += P; P *= pl.radix[s]; }   // sum of P_s < n: fits the n-entry array
    gfft_twiddle_kernel<<<(n + 255) / 256, 256, 0, st>>>(tw, n);
    BLINK_LAUNCH_CHECK("gfft_twiddle_kernel");
    const size_t per = 2 * (size_t)(n + 16) * sizeof(float2);   // ping + pong of one transform (padded leading dimension: n + 1, or herm_ld)
    const size_t twb = (size_t)n * sizeof(float2);              // + the twiddle table staged in shared memory
    const size_t budget = 200 * 1024 - twb;
    // rows per round: the paper's side takes 4 (two CTAs of 320 threads per SM), the others 2 as before
    int nr = (int)std::min<size_t>(n == 1200 ? 4 : 2, n == 1200 ? (100 * 1024 - twb) / per : budget / per);
    int kc = 1;
    for (int c = 8; c >= 1; c >>= 1)
        if ((n / 2) % c == 0 && (size_t)c * per <= budget) { kc = c; break; }
    if (nr < 1) return BLINK_ERR_UNSUPPORTED;
    // the paper's side has compile-time instantiations (same algorithm, constant index arithmetic)
    auto rows_k = n == 1200 ? gfft_rows_kernel<1200> : gfft_rows_kernel<0>;
    auto cols_k = n == 1200 ? gfft_cols_kernel<1200> : gfft_cols_kernel<0>;
    auto herm_k = n == 1200 ? gfft_cols_herm_kernel<1200> : gfft_cols_herm_kernel<0>;
    BLINK_CUDA_TRY(cudaFuncSetAttribute(rows_k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(nr * per + twb)));
    BLINK_CUDA_TRY(cudaFuncSetAttribute(cols_k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(kc * per + twb)));
    const int rows_per_img = hermitian ? n / 2 : n, row_off = hermitian ? n / 2 : 0;
    const long long n_rows = (long long)batch * rows_per_img;
    const long long want = (n_rows + nr - 1) / nr, cap = (long long)sm_count() * 8;
    const int row_threads = n == 1200 ? grow_threads<1200>() : grow_threads<0>();
    const int col_threads = n == 1200 ? gcol_threads<1200>() : gcol_threads<0>();
    rows_k<<<(unsigned)(want < cap ? want : cap), row_threads, nr * per + twb, st>>>(grid, n_rows, pl, tw, nr, rows_per_img, row_off,
                                                                                           hermitian ? row_extent : nullptr, ext_div);
    BLINK_LAUNCH_CHECK("gfft_rows_kernel");
    // Hermitian: kc columns are kc/2 transforms; keep two CTAs per SM when the arrays allow it
    int kch = 2;
    for (int c = 16; c >= 2; c >>= 1)
        if (n % c == 0 && (size_t)(c / 2) * per + twb <= 100 * 1024) { kch = c; break; }
    if (hermitian && (size_t)(kch / 2) * per > budget) hermitian = false;
    if (!hermitian && row_extent) return BLINK_ERR_UNSUPPORTED;   // skipped rows are only defined for the Hermitian consumer (cannot happen: kch = 2 always fits)
    if (hermitian)
        BLINK_CUDA_TRY(cudaFuncSetAttribute(herm_k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)((kch / 2) * per + twb)));
    for (int b0 = 0; b0 < batch; b0 += 65535) {
        const int nb = batch - b0 < 65535 ? batch - b0 : 65535;
        if (hermitian)
            herm_k<<<dim3(n / kch, nb), col_threads, (kch / 2) * per + twb, st>>>(grid + (size_t)b0 * n * n, pl, tw, kch, scale,
                                                                                          scale_div, img_base + b0,
                                                                                          image + (size_t)b0 * n * n, row_extent, ext_div, b0,
                                                                                          herm_ld(n, kch / 2));
        else
            cols_k<<<dim3(n / kc, nb), col_threads, kc * per + twb, st>>>(grid + (size_t)b0 * n * n, pl, tw, kc, scale, scale_div,
                                                                           img_base + b0, image + (size_t)b0 * n * n,
                                                                           image_imag ? image_imag + (size_t)b0 * n * n : nullptr);
        BLINK_LAUNCH_CHECK("gfft_cols_kernel");
    }
    return BLINK_OK;
}

}  // namespace blink
