// Cooperative register-resident inverse FFT building blocks (sm_100a).
//
// A group of TG = N/8 threads transforms NV vectors of N complex64 values at once.  Thread `tid`
// of the group holds element n = tid + e*TG in register slot e (e = 0..7) before AND after the
// transform (Stockham auto-sort, decimation in time, radices 8/4 chosen by plan_radix()).  Between
// stages the values cross threads through a shared-memory exchange array addressed by an
// Exchange policy; inside a stage everything is register arithmetic.
//
// Sign +, unnormalised: X[j] = sum_n x[n] exp(+2 pi i j n / N)   (eq. 5, reading R5).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace blink {

constexpr int kE = 8;                                   // elements per thread per vector
__host__ __device__ constexpr int kTwiddleNConst() { return 8192; }   // length of the W table

__host__ __device__ constexpr int ilog2(int n) { return n <= 1 ? 0 : 1 + ilog2(n >> 1); }
// number of radix-4 stages: log2 N = 3 a + 2 b with b in {0,1,2}
__host__ __device__ constexpr int plan_n4(int n) { return (ilog2(n) % 3 == 0) ? 0 : (ilog2(n) % 3 == 2 ? 1 : 2); }
__host__ __device__ constexpr int plan_n8(int n) { return (ilog2(n) - 2 * plan_n4(n)) / 3; }
__host__ __device__ constexpr int plan_stages(int n) { return plan_n8(n) + plan_n4(n); }
__host__ __device__ constexpr int plan_radix(int n, int s) { return s < plan_n8(n) ? 8 : 4; }

// Packed fp32 pairs: sm_100 has FADD2 / FMUL2 / FFMA2 (PTX add/sub/mul/fma .f32x2) that operate on a 64-bit
// register pair -- one issue slot per COMPLEX add instead of two.  ptxas folds the half swap (LO_HI), the
// scalar broadcast (.F32) and per-half signs into operand modifiers, so a + i b, a * w and the 8th-root
// rotations below cost no extra moves (checked with cuobjdump -sass).  Same flop rate as the scalar
// instructions (measured: FADD 1 / clk / SMSP, FADD2 1 / 2 clk), half the issue slots.
__device__ __forceinline__ unsigned long long pk_bits(float2 a) { return *reinterpret_cast<unsigned long long *>(&a); }
__device__ __forceinline__ float2 pk_f2(unsigned long long a) { return *reinterpret_cast<float2 *>(&a); }
__device__ __forceinline__ float2 pk_add(float2 a, float2 b)
{
    unsigned long long c;
    asm("add.f32x2 %0, %1, %2;" : "=l"(c) : "l"(pk_bits(a)), "l"(pk_bits(b)));
    return pk_f2(c);
}
__device__ __forceinline__ float2 pk_sub(float2 a, float2 b)
{
    unsigned long long c;
    asm("sub.f32x2 %0, %1, %2;" : "=l"(c) : "l"(pk_bits(a)), "l"(pk_bits(b)));
    return pk_f2(c);
}
__device__ __forceinline__ float2 pk_mul(float2 a, float2 b)
{
    unsigned long long c;
    asm("mul.f32x2 %0, %1, %2;" : "=l"(c) : "l"(pk_bits(a)), "l"(pk_bits(b)));
    return pk_f2(c);
}
__device__ __forceinline__ float2 pk_fma(float2 a, float2 b, float2 c)
{
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(pk_bits(a)), "l"(pk_bits(b)), "l"(pk_bits(c)));
    return pk_f2(d);
}

__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return pk_add(a, b); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return pk_sub(a, b); }
// a * w = a.x * (w.x, w.y) + a.y * (-w.y, w.x)
__device__ __forceinline__ float2 cmul(float2 a, float2 w)
{
    return pk_fma(make_float2(a.x, a.x), w, pk_mul(make_float2(a.y, a.y), make_float2(-w.y, w.x)));
}
__device__ __forceinline__ float2 add_i(float2 a, float2 b)       // a + i b = (a.x - b.y, a.y + b.x)
{
    return pk_fma(make_float2(b.y, b.x), make_float2(-1.f, 1.f), a);
}
__device__ __forceinline__ float2 sub_i(float2 a, float2 b)       // a - i b = (a.x + b.y, a.y - b.x)
{
    return pk_fma(make_float2(b.y, b.x), make_float2(1.f, -1.f), a);
}

// In-register inverse DFTs of length 2, 4, 8 (natural order in and out).
__device__ __forceinline__ void dft2(float2 &a, float2 &b)
{
    float2 t = a;
    a = cadd(t, b);
    b = csub(t, b);
}
__device__ __forceinline__ void dft4(float2 &x0, float2 &x1, float2 &x2, float2 &x3)
{
    float2 t0 = cadd(x0, x2), t1 = csub(x0, x2), t2 = cadd(x1, x3), d = csub(x1, x3);
    x0 = cadd(t0, t2);
    x2 = csub(t0, t2);
    x1 = add_i(t1, d);
    x3 = sub_i(t1, d);
}
__device__ __forceinline__ void dft8(float2 (&x)[8])
{
    // even / odd halves, then combine with w8^k = exp(+2 pi i k / 8); the 1/sqrt2 of the odd rotations is
    // folded into the final packed fma
    dft4(x[0], x[2], x[4], x[6]);
    dft4(x[1], x[3], x[5], x[7]);
    const float r = 0.70710678118654752440f;
    const float2 pr = make_float2(r, r), nr = make_float2(-r, -r);
    const float2 e0 = x[0], e1 = x[2], e2 = x[4], e3 = x[6];
    const float2 o0 = x[1];
    const float2 t1 = add_i(x[3], x[3]);          // (1 + i) x3     -> o1 = r t1
    const float2 o2 = x[5];                       // o2 = i x5
    const float2 t3 = sub_i(x[7], x[7]);          // (1 - i) x7     -> o3 = (-1 + i) r x7 = -r t3
    x[0] = cadd(e0, o0);          x[4] = csub(e0, o0);
    x[1] = pk_fma(t1, pr, e1);    x[5] = pk_fma(t1, nr, e1);
    x[2] = add_i(e2, o2);         x[6] = sub_i(e2, o2);
    x[3] = pk_fma(t3, nr, e3);    x[7] = pk_fma(t3, pr, e3);
}

// ---------------------------------------------------------------------------------------------
// Exchange policies: where position w (0..N-1) of the group's vector(s) lives in shared memory.
// ---------------------------------------------------------------------------------------------
// XOR swizzle for arrays of 8-byte elements (16 per 128-byte bank row; a 64-bit access is served per
// half warp).  Position w lives in slot xsw(w): bits 4..6 of w are folded into bits 0..2 and bit 6 also
// into bit 3, so the 16 lanes of a half warp hit 16 different bank pairs for the unit-stride loads AND for
// the stride-8 / stride-64 Stockham stores (padding w + w/8 cost a second wavefront on every load:
// profiles/r1_fused.md capture b).  No padding: an N-element vector takes N slots.
__device__ __forceinline__ int xsw(int w) { return w ^ ((w >> 4) & 7) ^ (((w >> 6) & 1) << 3); }

// Slot of position w = tid + e*TG (tid < TG, TG a power of two >= 32) in factored form: the swizzle only touches
// bits 0..3, which belong to tid, and the bits of e*TG it depends on are compile-time, so
//   xsw(tid + e*TG) = e*TG + (xsw(tid) ^ me(e)),  me(e) = swizzle mask of (e*TG mod 128).
// With e known at compile time the unit-stride reads of a transform become one or two per-thread bases plus
// immediate offsets instead of four integer instructions per access.
template <int TG>
__device__ __forceinline__ int xsw_e(int xsw_tid, int e)
{
    const int lowe = (e * TG) & 127;
    return e * TG + (xsw_tid ^ ((lowe >> 4) ^ ((lowe >> 6) << 3)));
}

// One vector, float2 elements.
struct ExchangePadded1 {
    float2 *base;
    __device__ __forceinline__ void put(int w, const float2 (&v)[1]) const { base[xsw(w)] = v[0]; }
    __device__ __forceinline__ void get(int w, float2 (&v)[1]) const { v[0] = base[xsw(w)]; }
    template <int TG>
    __device__ __forceinline__ void get_e(int tid, int e, float2 (&v)[1]) const { v[0] = base[xsw_e<TG>(xsw(tid), e)]; }
    // position wt + wr with disjoint bit fields (wt per thread, wr compile-time): xsw is XOR-linear
    __device__ __forceinline__ void put2(int wt, int wr, const float2 (&v)[1]) const { base[xsw(wt) ^ xsw(wr)] = v[0]; }
};

// Two vectors (a column pair), float4 elements living INSIDE a TMA-written tile whose rows are
// ROWB bytes wide and swizzled by the hardware (CU_TENSOR_MAP_SWIZZLE_{32,64,128}B for ROWB =
// 32/64/128).  Position w is kept in tile row rho(w), 16-byte chunk `pair`; rho permutes the rows
// so that the 8 lanes of a quarter warp always touch 8 different bank groups.
template <int ROWB>
struct ExchangeTilePair {
    unsigned char *tile;            // 1024-byte aligned shared memory
    int pair;                       // which 16-byte chunk of the row (= column pair)
    __device__ __forceinline__ static int rho(int w) { return w ^ (((w >> 3) ^ (w >> 6)) & 7); }
    __device__ __forceinline__ static uint32_t swz(uint32_t off)
    {
        constexpr uint32_t mask = ROWB == 128 ? 7u : (ROWB == 64 ? 3u : (ROWB == 32 ? 1u : 0u));
        return off ^ (((off >> 7) & mask) << 4);
    }
    __device__ __forceinline__ float4 *at_row(int row) const
    {
        return reinterpret_cast<float4 *>(tile + swz((uint32_t)row * ROWB + (uint32_t)pair * 16u));
    }
    __device__ __forceinline__ void put(int w, const float2 (&v)[2]) const
    {
        *at_row(rho(w)) = make_float4(v[0].x, v[0].y, v[1].x, v[1].y);
    }
    __device__ __forceinline__ void get(int w, float2 (&v)[2]) const
    {
        float4 t = *at_row(rho(w));
        v[0] = make_float2(t.x, t.y);
        v[1] = make_float2(t.z, t.w);
    }
    template <int TG>
    __device__ __forceinline__ void get_e(int tid, int e, float2 (&v)[2]) const { get(tid + e * TG, v); }
    __device__ __forceinline__ void put2(int wt, int wr, const float2 (&v)[2]) const { put(wt + wr, v); }
};

// Two vectors, float4 elements in a private dense array (8 elements per 128-byte line), same rho.
struct ExchangeDense2 {
    float4 *base;
    __device__ __forceinline__ static int rho(int w) { return w ^ (((w >> 3) ^ (w >> 6)) & 7); }
    __device__ __forceinline__ void put(int w, const float2 (&v)[2]) const
    {
        base[rho(w)] = make_float4(v[0].x, v[0].y, v[1].x, v[1].y);
    }
    __device__ __forceinline__ void get(int w, float2 (&v)[2]) const
    {
        float4 t = base[rho(w)];
        v[0] = make_float2(t.x, t.y);
        v[1] = make_float2(t.z, t.w);
    }
    template <int TG>
    __device__ __forceinline__ void get_e(int tid, int e, float2 (&v)[2]) const { get(tid + e * TG, v); }
    __device__ __forceinline__ void put2(int wt, int wr, const float2 (&v)[2]) const { put(wt + wr, v); }
};

// ---------------------------------------------------------------------------------------------
// Per-thread twiddle registers.  Which twiddles a thread needs depends only on (tid, stage, butterfly),
// never on the data, so they are read ONCE per kernel from the W_8192 table (built in double on the
// host) and kept in registers: per stage > 0 and butterfly q the powers w^1, w^2 (and w^4 for radix 8)
// of w = exp(+2 pi i k / (P R)); the remaining powers are products of those (<= 2 extra roundings).
// N = 8192 runs with N/8 = 1024 threads per transform (64 registers each): there the three base twiddles are
// fetched from the (L1-resident) table at every use instead.
// ---------------------------------------------------------------------------------------------
template <int N, int E = kE>
struct Twiddles {
    static constexpr int S = plan_stages(N);
    static constexpr bool kInRegs = N <= 4096;
    float2 w[kInRegs ? (S > 1 ? S - 1 : 1) : 1][kInRegs ? E / 4 : 1][3];   // [stage-1][butterfly q][w1, w2, w4]
    const float2 *table;
    int tid_;

    // base twiddle `idx` (0, 1, 2 -> w^1, w^2, w^4) of butterfly q in stage ST (radix R, sub-transform length P)
    template <int ST, int R, int P>
    __device__ __forceinline__ float2 base(int q, int idx) const
    {
        if constexpr (kInRegs) {
            return w[ST - 1][q][idx];
        } else {
            constexpr int step = kTwiddleNConst() / (P * R);
            const int k = (tid_ + q * (N / E)) & (P - 1);
            return __ldg(table + (k * step << idx));
        }
    }

    template <int ST, int P>
    __device__ __forceinline__ void init_stage(int tid, const float2 *__restrict__ tw)
    {
        if constexpr (ST < S) {
            constexpr int R = plan_radix(N, ST);
            constexpr int TG = N / E;
            constexpr int NB = E / R;
            if constexpr (ST > 0) {
                constexpr int step = kTwiddleNConst() / (P * R);
#pragma unroll
                for (int q = 0; q < NB; ++q) {
                    const int k = (tid + q * TG) & (P - 1);
                    w[ST - 1][q][0] = __ldg(tw + k * step);
                    w[ST - 1][q][1] = __ldg(tw + 2 * k * step);
                    if constexpr (R == 8) w[ST - 1][q][2] = __ldg(tw + 4 * k * step);
                }
            }
            init_stage<ST + 1, P * R>(tid, tw);
        }
    }
    __device__ __forceinline__ void init(int tid, const float2 *__restrict__ tw)
    {
        table = tw;
        tid_ = tid;
        if constexpr (kInRegs) init_stage<0, 1>(tid, tw);
    }
};

// One stage: twiddle (skipped when P == 1), radix-R butterflies in registers.
//   v[nv][e] holds x[tid + e*TG].  Butterfly q (q = 0..8/R-1) is i = tid + q*TG and uses slots
//   e = q + r*(8/R), r = 0..R-1.  Twiddle of input r: w^r, w = exp(+2 pi i k / (P R)), k = i mod P.
template <int N, int NV, int R, int P, int ST, int E>
__device__ __forceinline__ void stage_compute(float2 (&v)[NV][E], const Twiddles<N, E> &twr)
{
    constexpr int NB = E / R;                         // butterflies per thread
#pragma unroll
    for (int q = 0; q < NB; ++q) {
        if constexpr (P > 1) {
            float2 wp[R];
            wp[1] = twr.template base<ST, R, P>(q, 0);
            wp[2] = twr.template base<ST, R, P>(q, 1);
            wp[3] = cmul(wp[1], wp[2]);
            if constexpr (R == 8) {
                wp[4] = twr.template base<ST, R, P>(q, 2);
                wp[5] = cmul(wp[1], wp[4]);
                wp[6] = cmul(wp[2], wp[4]);
                wp[7] = cmul(wp[3], wp[4]);
            }
#pragma unroll
            for (int r = 1; r < R; ++r) {
#pragma unroll
                for (int nv = 0; nv < NV; ++nv) v[nv][q + r * NB] = cmul(v[nv][q + r * NB], wp[r]);
            }
        }
#pragma unroll
        for (int nv = 0; nv < NV; ++nv) {
            if constexpr (R == 8) {
                float2 x[8];
#pragma unroll
                for (int r = 0; r < 8; ++r) x[r] = v[nv][q + r * NB];
                dft8(x);
#pragma unroll
                for (int r = 0; r < 8; ++r) v[nv][q + r * NB] = x[r];
            } else {
                dft4(v[nv][q], v[nv][q + NB], v[nv][q + 2 * NB], v[nv][q + 3 * NB]);
            }
        }
    }
}

// scatter the stage outputs to their Stockham positions: y[j + r*P], j = (i - k)*R + k
template <int N, int NV, int R, int P, class X, int E>
__device__ __forceinline__ void stage_put(const float2 (&v)[NV][E], int tid, const X &xch)
{
    constexpr int TG = N / E;
    constexpr int NB = E / R;
#pragma unroll
    for (int q = 0; q < NB; ++q) {
        const int i = tid + q * TG;
        const int k = i & (P - 1);
        const int j = (i - k) * R + k;                  // bits of j and of r*P never overlap (k < P, (i-k)*R multiple of P*R)
#pragma unroll
        for (int r = 0; r < R; ++r) {
            float2 t[NV];
#pragma unroll
            for (int nv = 0; nv < NV; ++nv) t[nv] = v[nv][q + r * NB];
            xch.put2(j, r * P, t);
        }
    }
}

template <int N, int NV, class X, int E>
__device__ __forceinline__ void stage_get(float2 (&v)[NV][E], int tid, const X &xch)
{
    constexpr int TG = N / E;
#pragma unroll
    for (int e = 0; e < E; ++e) {
        float2 t[NV];
        xch.template get_e<TG>(tid, e, t);
#pragma unroll
        for (int nv = 0; nv < NV; ++nv) v[nv][e] = t[nv];
    }
}

// Optional hook: called by every thread right after the k-th group barrier of a transform (k = 0, 1, ...).
struct NoHook {
    __device__ __forceinline__ void operator()(int) const {}
};

template <int N, int NV, int E, int S, int P, class X, class Sync, class Hook>
struct FftStages {
    __device__ __forceinline__ static void run(float2 (&v)[NV][E], int tid, const X &xch, const Twiddles<N, E> &twr,
                                               Sync sync, Hook hook)
    {
        constexpr int R = plan_radix(N, S);
        stage_compute<N, NV, R, P, S, E>(v, twr);
        if constexpr (S + 1 < plan_stages(N)) {
            sync();                                      // everyone has finished reading the array
            hook(2 * S);
            stage_put<N, NV, R, P, X, E>(v, tid, xch);
            sync();                                      // all writes visible
            hook(2 * S + 1);
            stage_get<N, NV, X, E>(v, tid, xch);
            FftStages<N, NV, E, S + 1, P * R, X, Sync, Hook>::run(v, tid, xch, twr, sync, hook);
        }
        // last stage: output j + r*P with P = N/R is again slot layout tid + e*TG -- nothing to move
    }
};

// Full transform.  `sync` must synchronise (at least) all threads of the group and must be called
// by every thread the same number of times (use __syncthreads() when groups share a CTA).
// NOTE: the first sync() also orders the caller's last reads of the exchange array (e.g. the
// initial load out of a TMA tile that doubles as the exchange array) before the first put; `hook(k)`
// runs in every thread right after the k-th sync (callers use it to overlap their own loads with the transform).
template <int N, int NV, int E, class X, class Sync, class Hook = NoHook>
__device__ __forceinline__ void fft_inverse(float2 (&v)[NV][E], int tid, const X &xch, const Twiddles<N, E> &twr,
                                            Sync sync, Hook hook = Hook())
{
    FftStages<N, NV, E, 0, 1, X, Sync, Hook>::run(v, tid, xch, twr, sync, hook);
}

}  // namespace blink
