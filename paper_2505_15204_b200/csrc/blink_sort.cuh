// Block-wide bitonic sort of EPT * 1024 (key, value) pairs held in REGISTERS by a CTA of 1024 threads (the per-timestep
// presorts of the fused imaging kernels and of blink_image_avg: baselines by |u| resp. by max(|u|, |v|)).
// Element i = tid * EPT + r lives in register r of thread tid, so of the 91 (EPT = 8) compare-exchange steps of the network
//   j <  EPT        stay inside a thread (compile-time register pairs),
//   j <  32 EPT     exchange between lanes of a warp (shuffles),
//   j >= 32 EPT     cross warps through shared memory (15 steps of 91 at 8192 elements; slot r * 1024 + tid: conflict-free).
// The first version kept every element in shared memory and paid a CTA barrier for each of the 91 steps (0.108 ms per 8128
// baselines, 4.5 % of config 2's step and 11 % of the averaged-image step; this one: 0.049 ms, bound by the ~6 M thread
// instructions of the network itself).
// Order: ascending in (key, value) -- a total order when the values are distinct indices, so padding (+inf, index >= B) stays last.
#pragma once
#include <stdint.h>

namespace blink {

constexpr int kSortThreads = 1024;

template <bool KV>
__device__ __forceinline__ bool sort_gt(float a, uint32_t ia, float b, uint32_t ib)
{
    if constexpr (KV) return (a > b) || (a == b && ia > ib);
    else return a > b;
}

// key / val: this thread's EPT elements (i = tid * EPT + r); skey / sval: EPT * 1024 words of shared memory each (sval unused
// when !KV).  All 1024 threads must call.  On return the registers hold the sorted sequence in the same layout.
template <int EPT, bool KV>
__device__ __forceinline__ void block_bitonic_sort(float (&key)[EPT], uint32_t (&val)[EPT], float *skey, uint32_t *sval)
{
    constexpr int NP2 = EPT * kSortThreads;
    const int tid = threadIdx.x;
    for (int k = 2; k <= NP2; k <<= 1) {
        int j = k >> 1;
        // ---- partners in other warps: through shared memory ----
        for (; j >= 32 * EPT; j >>= 1) {
#pragma unroll
            for (int r = 0; r < EPT; ++r) {
                skey[r * kSortThreads + tid] = key[r];
                if constexpr (KV) sval[r * kSortThreads + tid] = val[r];
            }
            __syncthreads();
            const int pt = tid ^ (j / EPT);
            const bool lower = (tid & (j / EPT)) == 0, up = ((tid * EPT) & k) == 0;     // k > j >= EPT: bit k lies in the tid part
#pragma unroll
            for (int r = 0; r < EPT; ++r) {
                const float b = skey[r * kSortThreads + pt];
                const uint32_t ib = KV ? sval[r * kSortThreads + pt] : 0u;
                if (sort_gt<KV>(key[r], val[r], b, ib) == (lower == up)) { key[r] = b; val[r] = ib; }
            }
            __syncthreads();
        }
        // ---- partners in the same warp: shuffles ----
        for (; j >= EPT; j >>= 1) {
            const int lj = j / EPT;
            const bool lower = (tid & lj) == 0;
            const bool up = k >= EPT * 2 ? (((tid * EPT) & k) == 0) : true;             // j >= EPT implies k >= 2 EPT
#pragma unroll
            for (int r = 0; r < EPT; ++r) {
                const float b = __shfl_xor_sync(0xffffffffu, key[r], lj);
                const uint32_t ib = KV ? __shfl_xor_sync(0xffffffffu, val[r], lj) : 0u;
                if (sort_gt<KV>(key[r], val[r], b, ib) == (lower == up)) { key[r] = b; val[r] = ib; }
            }
        }
        // ---- partners in the same thread: compile-time register pairs ----
#pragma unroll
        for (int J = EPT / 2; J > 0; J >>= 1) {
            if (J <= j) {                                       // j = min(k / 2, EPT / 2) here; steps J = j, j / 2, ..., 1
#pragma unroll
                for (int r = 0; r < EPT; ++r) {
                    if ((r & J) == 0) {
                        const int r2 = r | J;
                        const bool up = k < EPT ? ((r & k) == 0) : (((tid * EPT + r) & k) == 0);
                        if (sort_gt<KV>(key[r], val[r], key[r2], val[r2]) == up) {
                            const float tk = key[r]; key[r] = key[r2]; key[r2] = tk;
                            const uint32_t tv = val[r]; val[r] = val[r2]; val[r2] = tv;
                        }
                    }
                }
            }
        }
    }
}

}  // namespace blink
