// Internal helpers shared by the libblinkimg translation units (not part of the C ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/blinkimg.h"

namespace blink {

// --- error plumbing ---------------------------------------------------------------------------
void set_cuda_error(cudaError_t e, const char *where);          // records text for blink_last_cuda_error()
void set_error_text(const char *text);
void count_launch(unsigned n = 1);

#define BLINK_CUDA_TRY(expr)                                                     \
    do {                                                                         \
        cudaError_t _e = (expr);                                                 \
        if (_e != cudaSuccess) { ::blink::set_cuda_error(_e, #expr); return BLINK_ERR_CUDA; } \
    } while (0)

#define BLINK_LAUNCH_CHECK(name)                                                 \
    do {                                                                         \
        cudaError_t _e = cudaGetLastError();                                     \
        if (_e != cudaSuccess) { ::blink::set_cuda_error(_e, name); return BLINK_ERR_CUDA; } \
        ::blink::count_launch();                                                 \
    } while (0)

int  option(int key);
int  ensure_device();             // checks for an sm_100 device, uploads the twiddle table once per device
int  sm_count();

static inline bool is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }
constexpr int kMaxPix = 8192;           // largest image side (the fused kernel stops at 4096: blink_image falls back to the unfused chain)
static inline bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// step a0 (R3): cells per metre, double left to right, rounded once to float
static inline float scale_for(double f_hz, int n_pix, double pixscale_rad)
{
    double s = f_hz * (double)n_pix;
    s = s * pixscale_rad;
    s = s / 299792458.0;
    return (float)s;
}

constexpr int kMaxChannels = 4096;      // per-channel scales are passed to kernels through a device array
constexpr int kMaxBaselines = (1 << 18) - 1;

// device twiddle table W[m] = exp(+2 pi i m / 8192), m in [0, 8192), built in double on the host
constexpr int kTwiddleN = 8192;
const float2 *twiddle_table();          // device pointer (after ensure_device())

// per-antenna gain corrections fused into the gridder's load (R15): V' = g[c][p][a1] conj(g[c][p][a2]) V
struct GainRef {
    const float2 *gains = nullptr;      // [C][P][A] complex64 (device) or NULL
    const int2 *ant = nullptr;          // [B] antenna pair (a1, a2) of every baseline (device)
    int A = 0;
};

// per-channel scales travel as a kernel parameter (<= 1024 channels per launch)
struct ScaleBlock { float s[1024]; };

#ifdef __CUDACC__
#ifndef BLINK_GRID_EXCH
#define BLINK_GRID_EXCH 1
#endif
// Round to nearest, ties to even, WITHOUT the quarter-rate conversion unit (FRND / F2I): adding and subtracting
// 1.5 * 2^23 with two correctly rounded fp32 adds (never contracted into an fma) gives exactly rint(x) for
// |x| < 2^22, and the integer sits in the mantissa of the intermediate sum.  For larger |x| (and inf / NaN) the
// result keeps its huge magnitude (or stays NaN), so the range test that follows still rejects it; `i` is only
// meaningful once that test has passed.  Measured: the averaging path was bound by 4 FRND/F2I per sample.
__device__ __forceinline__ float rint_rne(float x, int &i)
{
    const float t = __fadd_rn(x, 12582912.0f);
    i = __float_as_int(t) - 0x4B400000;
    return __fadd_rn(t, -12582912.0f);
}
// step a1 (R2, R4): nearest cell of one baseline, bit-exact twin of the oracle's fp32 recipe
__device__ __forceinline__ bool cell_coords(float u_m, float v_m, float s, int h, int &iu, int &iv, int r = 0)
{
    const float x = __fmul_rn(u_m, s);            // one IEEE fp32 multiply, never contracted
    const float y = __fmul_rn(v_m, s);
    const float xr = rint_rne(x, iu), yr = rint_rne(y, iv);     // round to nearest, ties to even
    const float lim = (float)(h - 1 - r);                       // r: support radius of the convolutional gridder (R16)
    return fabsf(xr) <= lim && fabsf(yr) <= lim;                // NaN fails
}
__device__ __forceinline__ int cell_of(float u_m, float v_m, float s, int n, int h, int r = 0)
{
    int iu, iv;
    if (!cell_coords(u_m, v_m, s, h, iu, iv, r)) return -1;
    return (iv + h) * n + (iu + h);
}
// Accumulate one complex sample into a shared-memory cell WITHOUT floating-point atomics.  fp32 atomicAdd on shared memory
// is a load + compare-and-swap spin loop per scalar on sm_100 (ATOMS.CAST.SPIN; profiles/r1_fused_v2.md: 17 wavefronts per
// warp instruction), but the 64-bit exchange ATOMS.EXCH.64 is native.  Cells start at zero and almost every cell of a
// nearest-cell grid receives ONE sample (1.04-1.22 per occupied cell), so: put the sample and look at what
// came out.  Zero bits: the cell was empty, done -- one instruction.  Otherwise the value that came out is now this
// thread's to re-add: take whatever is in the cell (exchange with zero), add, put the sum back; repeat while a put
// displaces a non-zero value.  Invariant: cell + values in flight = sum of the samples; a value is in flight in exactly one
// thread; every exit leaves nothing in flight.  Bit-identical samples are handled like any other (no tags, no compares of
// values).  A displaced -0.0 merely costs one more round.
__device__ __forceinline__ void cell_add_exch(float2 *cell, float2 v)
{
    unsigned long long *p = reinterpret_cast<unsigned long long *>(cell);
    unsigned long long out = atomicExch(p, *reinterpret_cast<unsigned long long *>(&v));
    while (out != 0ull) {
        const unsigned long long cur = atomicExch(p, 0ull);
        const float2 a = *reinterpret_cast<float2 *>(&out), b = *reinterpret_cast<const float2 *>(&cur);
        float2 sum = make_float2(a.x + b.x, a.y + b.y);
        out = atomicExch(p, *reinterpret_cast<unsigned long long *>(&sum));
    }
}

// The same without the optimistic first put, for cells that usually hold a value already (convolutional gridding: a cell is
// hit ~S^2 times): take what is there (exchange with zero), add, put the sum back; a non-zero value coming out of the put
// arrived in between and is re-added the same way.  Two native atomics per complex tap instead of two load + CAS spin loops.
__device__ __forceinline__ void cell_add_take(float2 *cell, float2 v)
{
    unsigned long long *p = reinterpret_cast<unsigned long long *>(cell);
    for (;;) {
        const unsigned long long cur = atomicExch(p, 0ull);
        const float2 c = *reinterpret_cast<const float2 *>(&cur);
        float2 sum = make_float2(v.x + c.x, v.y + c.y);
        const unsigned long long out = atomicExch(p, *reinterpret_cast<unsigned long long *>(&sum));
        if (out == 0ull) break;
        v = *reinterpret_cast<const float2 *>(&out);
    }
}
__device__ __forceinline__ int mirror_of(int cell, int n)
{
    const int r = cell / n, q = cell - r * n;
    return (n - r) * n + (n - q);                 // (h - iv)*N + (h - iu)
}
#endif

// --- internal entry points used across translation units ---------------------------------------
// gridder over the flattened (t,c) range [tc0, tc0+ntc).  wsum / cell_idx are indexed by the absolute tc,
// grid / counts by (tc - out_tc0) so that a chunk can land at the start of a workspace buffer.
int grid_range(const float2 *vis, const float *uvw_m, const double *freqs_hz, double pixscale_rad, int T, int C,
               int P, int B, int n_pix, int weighting, int tc0, int ntc, int out_tc0, float2 *grid, float *wsum,
               int32_t *cell_idx, uint32_t *counts, cudaStream_t st, bool half_only = false, int *row_extent = nullptr);
bool grid_needs_global_counts(int B, int n_pix, int weighting);
// hermitian: the grids come from the library's own gridders (G[-v][-u] = conj G[v][u], row / column -N/2 empty)
// tw_generic: device array of n_pix complex64 (gfft_workspace_bytes) for sides that are not a power of two, else unused
// row_extent (hermitian, generic sides only; written by grid_range): image i only has data in its rows v = 0 ..
// row_extent[i / ext_div] - 1; the rows above are neither read nor transformed (they need not even be initialised)
int fft2d_range(float2 *grid, int n_pix, int batch, const float *scale, int scale_div, int scale_img_base,
                float *image, float *image_imag, cudaStream_t st, float2 *tw_generic = nullptr, bool hermitian = false,
                const int *row_extent = nullptr, int ext_div = 1);
// image sides: even, 32..kMaxPix, only prime factors 2, 3, 5 (powers of two run the tuned kernels)
bool size_supported(int n_pix);
size_t gfft_workspace_bytes(int n_pix);
int gfft2d_range(float2 *grid, int n, int batch, const float *scale, int scale_div, int img_base, float *image,
                 float *image_imag, float2 *tw, cudaStream_t st, bool hermitian, const int *row_extent = nullptr, int ext_div = 1);

}  // namespace blink
