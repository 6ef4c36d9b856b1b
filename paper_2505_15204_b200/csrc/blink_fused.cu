// Fused imaging kernel: visibilities -> dirty images, the uv grid is never materialised.
//
// What makes this possible:
//   * the gridded plane is Hermitian, G[-v][-u] = conj(G[v][u]) (every sample is gridded with its conjugate,
//     reading R1), so only the half plane u >= 0 is gridded: N x N/2 cells (column u = N/2 is always empty, R4);
//   * pass 1 grids and transforms that half plane along v, one u-column PAIR per transform group, in shared
//     memory, and leaves H[u][ky] (N/2 x N complex64) in a per-CTA scratch in global memory (L2-resident);
//   * pass 2 turns row pairs (ky, ky+1) into TWO real image rows with ONE N-point complex transform:
//     Z[n] = S1[n] + i S2[n] (n < N/2), Z[N-n] = conj(S1[n]) + i conj(S2[n]);  Re z = row ky, Im z = row ky+1.
//     Its input tiles [KY ky][N/2 u] are TRANSPOSED reads of the scratch, staged by TMA (128B-swizzled) through a
//     3-stage full/empty mbarrier pipeline; the fftshift (index XOR N/2), the 1/W normalisation and the
//     real-part extraction are part of the store.
// One persistent CTA per SM walks over (t,c) work items.  Inside a pass the transform groups (N/8 threads each)
// run DECOUPLED: a group grids its own two columns with shared-memory atomics (the samples of a column are one
// contiguous range of the per-timestep |u|-sorted baseline list), transforms them and moves on; only three
// CTA-wide barriers per image remain.  The next image's visibility row is prefetched with a bulk async copy
// while pass 2 runs.  PAPER.md L190-194 (gridding, batched inverse 2D FFT, shift); L150 (fp32).
#include "blink_fused_kernel.cuh"
#include "blink_sort.cuh"

namespace blink {

// ------------------------------------------------------------------------------------------ presort
// One CTA per timestep: sorts the baselines by |u_m| (bitonic sort of (key, index) pairs in shared memory).
// For every channel the u-tile of a sample, rint(|u_m| * s_c) / KU, is then non-decreasing along the sorted
// order (fp32 multiply by s_c > 0 and rint are monotone), so a tile's samples are ONE contiguous range and no
// per-image binning is needed.  The sample is stored folded into the half plane u >= 0:
//   su = |u_m|, svb = { bits of sv = (u_m < 0 ? -v_m : v_m), b | (u_m < 0) << 31 }   (bit 31: use conj(V) at (-u,-v)).
// rint(-x) = -rint(x) and (-a) * s = -(a * s) exactly, so the folded cell is exactly the mirror cell (R1, R2).
constexpr int kSortMaxB = 16384;

__global__ void __launch_bounds__(kSortThreads)
presort_kernel(const float *__restrict__ uvw_m, int B, int np2, float *__restrict__ su, uint2 *__restrict__ svb)
{
    extern __shared__ __align__(16) unsigned char sort_raw[];
    float *key = reinterpret_cast<float *>(sort_raw);
    uint32_t *idx = reinterpret_cast<uint32_t *>(sort_raw) + np2;
    const int t = blockIdx.x;
    const float *uvw = uvw_m + (size_t)t * B * 3;
    for (int i = threadIdx.x; i < np2; i += kSortThreads) {
        float k = __int_as_float(0x7f800000);                               // +inf: padding and NaN sort last
        if (i < B) {
            const float a = fabsf(uvw[3 * i]);
            if (a == a) k = a;
        }
        key[i] = k;
        idx[i] = (uint32_t)i;
    }
    __syncthreads();
    for (int k = 2; k <= np2; k <<= 1) {
        for (int j = k >> 1; j > 0; j >>= 1) {
            for (int i = threadIdx.x; i < np2; i += kSortThreads) {
                const int x = i ^ j;
                if (x > i) {
                    const float a = key[i], b = key[x];
                    const uint32_t ia = idx[i], ib = idx[x];
                    const bool gt = (a > b) || (a == b && ia > ib);         // (key, index) order: padding stays last
                    const bool up = (i & k) == 0;
                    if (gt == up) {
                        key[i] = b; key[x] = a;
                        idx[i] = ib; idx[x] = ia;
                    }
                }
            }
            __syncthreads();
        }
    }
    for (int i = threadIdx.x; i < B; i += kSortThreads) {
        const uint32_t b = idx[i];                                          // < B: real samples sort before the padding
        const float u = uvw[3 * b], v = uvw[3 * b + 1];
        const bool neg = u < 0.0f;
        su[(size_t)t * B + i] = fabsf(u);
        svb[(size_t)t * B + i] = make_uint2(__float_as_uint(neg ? -v : v), b | (neg ? 0x80000000u : 0u));
    }
}

// The same for EPT * 1024 >= B > EPT * 512 baselines with the elements in registers (blink_sort.cuh): 8128 baselines in 1 / 10 of
// the time of the shared-memory loop above, which stays for the other sizes.
template <int EPT>
__global__ void __launch_bounds__(kSortThreads)
presort_regs_kernel(const float *__restrict__ uvw_m, int B, float *__restrict__ su, uint2 *__restrict__ svb)
{
    extern __shared__ __align__(16) unsigned char sort_raw[];
    constexpr int NP2 = EPT * kSortThreads;
    float *skey = reinterpret_cast<float *>(sort_raw);
    uint32_t *sval = reinterpret_cast<uint32_t *>(sort_raw) + NP2;
    const int t = blockIdx.x;
    const float *uvw = uvw_m + (size_t)t * B * 3;
    float key[EPT];
    uint32_t val[EPT];
#pragma unroll
    for (int r = 0; r < EPT; ++r) {
        const int i = r * kSortThreads + threadIdx.x;          // coalesced read; any assignment of inputs to slots will do
        float k = __int_as_float(0x7f800000);                  // +inf: padding and NaN sort last
        if (i < B) {
            const float a = fabsf(uvw[3 * i]);
            if (a == a) k = a;
        }
        key[r] = k;
        val[r] = (uint32_t)i;
    }
    block_bitonic_sort<EPT, true>(key, val, skey, sval);
#pragma unroll
    for (int r = 0; r < EPT; ++r) sval[threadIdx.x * EPT + r] = val[r];       // sorted position i = tid * EPT + r
    __syncthreads();
    for (int i = threadIdx.x; i < B; i += kSortThreads) {
        const uint32_t b = sval[i];                            // < B: real samples sort before the padding
        const float u = uvw[3 * b], v = uvw[3 * b + 1];
        const bool neg = u < 0.0f;
        su[(size_t)t * B + i] = fabsf(u);
        svb[(size_t)t * B + i] = make_uint2(__float_as_uint(neg ? -v : v), b | (neg ? 0x80000000u : 0u));
    }
}

// ------------------------------------------------------------------------------------------ counts (optional output)
__global__ void counts_kernel(const float *__restrict__ uvw_m, const ScaleBlock sc, int C, int B, int n, int tc0, int c_base,
                              uint32_t *__restrict__ counts)
{
    const int tc = tc0 + blockIdx.y;
    const int t = tc / C, c = tc - t * C;
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    const float *p = uvw_m + ((size_t)t * B + b) * 3;
    const int cell = cell_of(p[0], p[1], sc.s[c - c_base], n, n / 2);
    if (cell < 0) return;
    uint32_t *dst = counts + (size_t)tc * n * n;
    atomicAdd(&dst[cell], 1u);
    atomicAdd(&dst[mirror_of(cell, n)], 1u);
}

// the fused kernel of the paper's own side, 1200 x 1200 (blink_fused_g.cu)
bool fused_g_supported(int B, int n_pix);
size_t fused_g_workspace_bytes(int T, int B, int ctas);
int fused_g_image(const float2 *vis, const float *uvw_m, const double *freqs_hz, double pixscale_rad, int T, int C, int P, int B,
                  int weighting, int tc0, int ntc, float *image, float *wsum, int32_t *cell_idx, void *workspace,
                  size_t workspace_bytes, cudaStream_t st, GainRef cal, const ConvPoly *poly = nullptr, int R = 0, size_t extra = 0);

// ------------------------------------------------------------------------------------------ host
bool fused_supported(int P, int B, int n_pix, int weighting)
{
    (void)P;
    if (B > kSortMaxB) return false;
    if (n_pix == 1200) return fused_g_supported(B, n_pix);
    const bool uni = weighting == BLINK_W_UNIFORM;
    switch (n_pix) {
        case 256: return fused_stages<256>(B, uni) > 0;
        case 512: return fused_stages<512>(B, uni) > 0;
        case 1024: return fused_stages<1024>(B, uni) > 0;
        case 2048: return fused_stages<2048>(B, uni) > 0;
        case 4096: return fused_stages<4096>(B, uni) > 0;
        default: return false;
    }
}

size_t sort_bytes(int T, int B) { return align_up((size_t)T * B * 4, 256) * 3; }
int presort_launch(const float *uvw_m, int T, int B, float *su, uint2 *svb, cudaStream_t st)
{
    int np2 = 1;
    while (np2 < B) np2 <<= 1;
    const size_t ssm = (size_t)np2 * 8;
    if (np2 == 8 * kSortThreads) {
        BLINK_CUDA_TRY(cudaFuncSetAttribute(presort_regs_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ssm));
        presort_regs_kernel<8><<<T, kSortThreads, ssm, st>>>(uvw_m, B, su, svb);
    } else if (np2 == 16 * kSortThreads) {
        BLINK_CUDA_TRY(cudaFuncSetAttribute(presort_regs_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ssm));
        presort_regs_kernel<16><<<T, kSortThreads, ssm, st>>>(uvw_m, B, su, svb);
    } else {
        BLINK_CUDA_TRY(cudaFuncSetAttribute(presort_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ssm));
        presort_kernel<<<T, kSortThreads, ssm, st>>>(uvw_m, B, np2, su, svb);
    }
    BLINK_LAUNCH_CHECK("presort_kernel");
    return BLINK_OK;
}
size_t fused_workspace_bytes(int T, int B, int n_pix, int ctas)
{
    if (n_pix == 1200) return fused_g_workspace_bytes(T, B, ctas);
    // at least two scratch slots so that a team (two slots in turn) can run when the caller grants the recommended size
    return sort_bytes(T, B) + kTeamBytes + (size_t)ctas * (n_pix / 2) * n_pix * sizeof(float2);
}
int fused_default_ctas() { return sm_count() > 0 ? sm_count() : 148; }

int fused_image(const float2 *vis, const float *uvw_m, const double *freqs_hz, double pixscale_rad, int T, int C, int P,
                int B, int n_pix, int weighting, int tc0, int ntc, float *image, float *wsum, int32_t *cell_idx,
                void *workspace, size_t workspace_bytes, cudaStream_t st, GainRef cal)
{
    FusedArgs a{};
    a.cal = cal;
    a.vis = vis; a.uvw_m = uvw_m; a.T = T; a.C = C; a.P = P; a.B = B; a.weighting = weighting;
    a.tc0 = tc0; a.ntc = ntc; a.image = image; a.wsum = wsum; a.cell_idx = cell_idx;
    switch (n_pix) {
        case 256: return launch_fused<256>(a, freqs_hz, pixscale_rad, workspace, workspace_bytes, st);
        case 512: return launch_fused<512>(a, freqs_hz, pixscale_rad, workspace, workspace_bytes, st);
        case 1024: return launch_fused<1024>(a, freqs_hz, pixscale_rad, workspace, workspace_bytes, st);
        case 2048: return launch_fused<2048>(a, freqs_hz, pixscale_rad, workspace, workspace_bytes, st);
        case 4096: return launch_fused<4096>(a, freqs_hz, pixscale_rad, workspace, workspace_bytes, st);
        case 1200: return fused_g_image(vis, uvw_m, freqs_hz, pixscale_rad, T, C, P, B, weighting, tc0, ntc, image, wsum, cell_idx,
                                        workspace, workspace_bytes, st, cal);
        default: return BLINK_ERR_UNSUPPORTED;
    }
}

int counts_only(const float *uvw_m, const double *freqs_hz, double pixscale_rad, int T, int C, int B, int n_pix, int tc0,
                int ntc, uint32_t *counts, cudaStream_t st)
{
    (void)T;
    const size_t n2 = (size_t)n_pix * n_pix;
    BLINK_CUDA_TRY(cudaMemsetAsync(counts + (size_t)tc0 * n2, 0, (size_t)ntc * n2 * sizeof(uint32_t), st));
    return for_channel_blocks(C, tc0, ntc, freqs_hz, n_pix, pixscale_rad,
                              [&](int s0, int m, int c_base, const ScaleBlock &sc) -> int {
                                  for (int y0 = 0; y0 < m; y0 += 65535) {
                                      const int my = m - y0 < 65535 ? m - y0 : 65535;
                                      dim3 grid((B + 255) / 256, my);
                                      counts_kernel<<<grid, 256, 0, st>>>(uvw_m, sc, C, B, n_pix, s0 + y0, c_base, counts);
                                      BLINK_LAUNCH_CHECK("counts_kernel");
                                  }
                                  return (int)BLINK_OK;
                              });
}

}  // namespace blink
