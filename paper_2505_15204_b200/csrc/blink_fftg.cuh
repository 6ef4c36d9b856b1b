// Register-resident small inverse DFTs (sign +, natural order in and out) and twiddle helpers shared by the mixed-radix
// transforms for image sides that are not a power of two: blink_fftg.cu (unfused chain) and blink_fused_g.cu (fused kernel
// at the paper's side 1200).  Radices 2, 3, 4, 5 directly; 15 = 3 x 5 and 16 = 4 x 4 by decimation in time.
#pragma once
#include "blink_fft.cuh"

namespace blink {

// The butterflies below use the packed fp32 pair instructions of sm_100 (blink_fft.cuh: add / mul / fma.f32x2 on a 64-bit
// register pair = one complex number), half the issue slots of the scalar forms.
__device__ __forceinline__ float2 bcast(float c) { return make_float2(c, c); }
__device__ __forceinline__ void gdft3(float2 &x0, float2 &x1, float2 &x2)
{
    const float c = 0.86602540378443864676f;                   // sin(2 pi / 3)
    const float2 t = cadd(x1, x2), d = csub(x1, x2);
    const float2 m = pk_fma(t, bcast(-0.5f), x0);              // x0 - t / 2
    x0 = cadd(x0, t);
    x1 = pk_fma(make_float2(d.y, d.x), make_float2(-c, c), m); // m + i c d
    x2 = pk_fma(make_float2(d.y, d.x), make_float2(c, -c), m); // m - i c d
}
__device__ __forceinline__ void gdft5(float2 &x0, float2 &x1, float2 &x2, float2 &x3, float2 &x4)
{
    const float c1 = 0.30901699437494742410f, c2 = -0.80901699437494742410f;      // cos(2 pi / 5), cos(4 pi / 5)
    const float s1 = 0.95105651629515357212f, s2 = 0.58778525229247312917f;       // sin(2 pi / 5), sin(4 pi / 5)
    const float2 a1 = cadd(x1, x4), a2 = cadd(x2, x3), b1 = csub(x1, x4), b2 = csub(x2, x3);
    const float2 p1 = pk_fma(a2, bcast(c2), pk_fma(a1, bcast(c1), x0));
    const float2 p2 = pk_fma(a2, bcast(c1), pk_fma(a1, bcast(c2), x0));
    const float2 q1 = pk_fma(b2, bcast(s2), pk_mul(b1, bcast(s1)));
    const float2 q2 = pk_fma(b2, bcast(-s1), pk_mul(b1, bcast(s2)));
    x0 = cadd(x0, cadd(a1, a2));
    x1 = add_i(p1, q1);                                        // p1 + i q1
    x4 = sub_i(p1, q1);
    x2 = add_i(p2, q2);                                        // p2 + i q2
    x3 = sub_i(p2, q2);
}

// x * exp(+2 pi i m / n) for compile-time constants (c, s) = (cos, sin)(2 pi m / n)
__device__ __forceinline__ float2 cmulc(float2 x, float c, float s) { return cmul(x, make_float2(c, s)); }

// 16-point inverse DFT in registers, natural order in and out: 4 x 4 decimation in time.
//   A[k1][n2] = sum_n1 x[n2 + 4 n1] W4^(n1 k1);  X[k1 + 4 k2] = sum_n2 (W16^(n2 k1) A[k1][n2]) W4^(n2 k2)
__device__ __forceinline__ void gdft16(float2 (&x)[16])
{
#pragma unroll
    for (int j = 0; j < 4; ++j) dft4(x[j], x[j + 4], x[j + 8], x[j + 12]);          // x[n2 + 4 k1] = A[k1][n2]
    const float c1 = 0.92387953251128674f, s1 = 0.38268343236508978f, r2 = 0.70710678118654752f;
    x[5] = cmulc(x[5], c1, s1);    x[6] = cmulc(x[6], r2, r2);    x[7] = cmulc(x[7], s1, c1);        // W16^1, ^2, ^3
    x[9] = cmulc(x[9], r2, r2);    x[10] = make_float2(-x[10].y, x[10].x);                             // W16^2, ^4 = i
    x[11] = cmulc(x[11], -r2, r2);                                                                     // W16^6
    x[13] = cmulc(x[13], s1, c1);  x[14] = cmulc(x[14], -r2, r2); x[15] = cmulc(x[15], -c1, -s1);     // W16^3, ^6, ^9
#pragma unroll
    for (int k = 0; k < 4; ++k) dft4(x[4 * k], x[4 * k + 1], x[4 * k + 2], x[4 * k + 3]);             // x[4 k1 + k2] = X[k1 + 4 k2]
    float2 y[16];
#pragma unroll
    for (int k1 = 0; k1 < 4; ++k1)
#pragma unroll
        for (int k2 = 0; k2 < 4; ++k2) y[k1 + 4 * k2] = x[4 * k1 + k2];
#pragma unroll
    for (int k = 0; k < 16; ++k) x[k] = y[k];
}
// 15-point inverse DFT in registers, natural order in and out: 3 x 5 decimation in time.
//   A[k1][n2] = sum_n1 x[n2 + 5 n1] W3^(n1 k1);  X[k1 + 3 k2] = sum_n2 (W15^(n2 k1) A[k1][n2]) W5^(n2 k2)
__device__ __forceinline__ void gdft15(float2 (&x)[15])
{
#pragma unroll
    for (int j = 0; j < 5; ++j) gdft3(x[j], x[j + 5], x[j + 10]);                    // x[n2 + 5 k1] = A[k1][n2]
    x[6] = cmulc(x[6], 0.91354545764260087f, 0.40673664307580015f);                   // W15^1
    x[7] = cmulc(x[7], 0.66913060635885824f, 0.74314482547739413f);                   // W15^2
    x[8] = cmulc(x[8], 0.30901699437494745f, 0.95105651629515353f);                   // W15^3
    x[9] = cmulc(x[9], -0.10452846326765333f, 0.9945218953682734f);                   // W15^4
    x[11] = cmulc(x[11], 0.66913060635885824f, 0.74314482547739413f);                 // W15^2
    x[12] = cmulc(x[12], -0.10452846326765333f, 0.9945218953682734f);                 // W15^4
    x[13] = cmulc(x[13], -0.80901699437494734f, 0.58778525229247325f);                // W15^6
    x[14] = cmulc(x[14], -0.97814760073380569f, -0.20791169081775907f);               // W15^8
#pragma unroll
    for (int k = 0; k < 3; ++k) gdft5(x[5 * k], x[5 * k + 1], x[5 * k + 2], x[5 * k + 3], x[5 * k + 4]);   // x[5 k1 + k2] = X[k1 + 3 k2]
    float2 y[15];
#pragma unroll
    for (int k1 = 0; k1 < 3; ++k1)
#pragma unroll
        for (int k2 = 0; k2 < 5; ++k2) y[k1 + 3 * k2] = x[5 * k1 + k2];
#pragma unroll
    for (int k = 0; k < 15; ++k) x[k] = y[k];
}
template <int R>
__device__ __forceinline__ void gbutterfly(float2 (&x)[R])
{
    if constexpr (R == 2) dft2(x[0], x[1]);
    if constexpr (R == 3) gdft3(x[0], x[1], x[2]);
    if constexpr (R == 4) dft4(x[0], x[1], x[2], x[3]);
    if constexpr (R == 5) gdft5(x[0], x[1], x[2], x[3], x[4]);
    if constexpr (R == 15) gdft15(x);
    if constexpr (R == 16) gdft16(x);
}
// inputs r >= 1 times w1^r: the powers are products of at most four factors (w^(2^j) by squaring, the others as
// w^(highest power of two below r) * w^(rest)), so a power carries a handful of roundings, not r of them
template <int R>
__device__ __forceinline__ void gtwiddle(float2 (&x)[R], float2 w1)
{
    float2 w[R > 1 ? R : 2];
    w[1] = w1;
    x[1] = cmul(x[1], w1);
#pragma unroll
    for (int r = 2; r < R; ++r) {
        int hb = 1;
        while (hb * 2 <= r) hb *= 2;
        w[r] = (hb == r) ? cmul(w[r / 2], w[r / 2]) : cmul(w[hb], w[r - hb]);
        x[r] = cmul(x[r], w[r]);
    }
}

}  // namespace blink
