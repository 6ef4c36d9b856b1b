// Fused imaging kernel: visibilities -> dirty images, the uv grid is never materialised.
//
// What makes this possible:
//   * the gridded plane is Hermitian, G[-v][-u] = conj(G[v][u]) (every sample is gridded with its conjugate,
//     reading R1), so only the half plane u >= 0 is gridded: N x N/2 cells (column u = N/2 is always empty, R4);
//   * pass 1 transforms that half plane along v, one u-column at a time, in shared memory, and leaves
//     H[u][ky] (N/2 x N complex64) in a per-CTA scratch in global memory (L2-resident at N = 512);
//   * pass 2 turns row pairs (ky, ky+1) into TWO real image rows with ONE N-point complex transform:
//     Z[n] = S1[n] + i S2[n] (n < N/2), Z[N-n] = conj(S1[n]) + i conj(S2[n]);  Re z = row ky, Im z = row ky+1.
//     Its input tiles [KY ky][N/2 u] are TRANSPOSED reads of the scratch, staged by TMA (128B-swizzled),
//     double-buffered behind an mbarrier pipeline; the fftshift (index XOR N/2), the 1/W normalisation and the
//     real-part extraction are part of the store.
// One persistent CTA per SM walks over (t,c) work items; per item it computes the cell indices once (bit-exact
// twin of the oracle), bins the samples by u-tile with a counting sort in shared memory, and reuses the bins
// for all P polarisations.  PAPER.md L190-194 (gridding, batched inverse 2D FFT, shift); L150 (fp32).
#include <algorithm>

#include "blink_common.cuh"
#include "blink_fft.cuh"
#include "blink_tma.cuh"

namespace blink {

constexpr int kFusedThreads = 512;

template <int N>
struct FusedCfg {
    static constexpr int H = N / 2;
    static constexpr int TG = N / kE;                          // threads per transform
    static constexpr int G = kFusedThreads / TG;               // groups per CTA
    static constexpr int KU = 2 * G;                           // u-columns per pass-1 tile (2 per group)
    static constexpr int NT = H / KU;                          // pass-1 tiles in the half plane
    static constexpr int SLOTS = N + (N >> 3);                 // padded column length
    static constexpr int KY = (8192 / N) < 16 ? (8192 / N) : 16;   // ky rows per pass-2 stage
    static constexpr int ROWB = KY * 8;                        // stage row bytes (= TMA swizzle span)
    static constexpr int PAIRS = KY / 2;
    static constexpr int BOX_ROWS = H < 256 ? H : 256;
    static constexpr int NBOX = H / BOX_ROWS;
    static constexpr int STAGE_BYTES = H * ROWB;
    static constexpr int NIT = N / KY;                         // pass-2 stages per image
    static constexpr int LOG_TILE = 13;                        // KU * N == 8192 cells per tile
    static_assert(KU * N == 8192, "tile is 8192 cells");
    static_assert(PAIRS <= G, "one pair per group per stage");
};

struct FusedArgs {
    const float2 *vis; const float *uvw_m;
    int T, C, P, B, weighting;
    int tc0, ntc, c_base;
    float *image; float *wsum; int32_t *cell_idx;              // indexed by absolute tc / image
    float2 *scratch;                                           // [gridDim.x][H][N]
    const float2 *tw;
};

struct ExchangePadded2 {
    float2 *c0, *c1;
    __device__ __forceinline__ void put(int w, const float2 (&v)[2]) const
    {
        const int o = w + (w >> 3);
        c0[o] = v[0];
        c1[o] = v[1];
    }
    __device__ __forceinline__ void get(int w, float2 (&v)[2]) const
    {
        const int o = w + (w >> 3);
        v[0] = c0[o];
        v[1] = c1[o];
    }
};

template <int N>
__host__ __device__ constexpr size_t fused_region_bytes(bool uniform)
{
    using Cfg = FusedCfg<N>;
    const size_t p1 = (size_t)Cfg::KU * Cfg::SLOTS * (uniform ? 12 : 8);
    const size_t p2 = 2 * (size_t)Cfg::STAGE_BYTES + (size_t)Cfg::G * Cfg::SLOTS * 8;
    return p1 > p2 ? p1 : p2;
}
template <int N>
static size_t fused_smem_bytes(int B, bool uniform)
{
    using Cfg = FusedCfg<N>;
    // items [2B] + tile offsets/cursors + union(pass-1 tile, pass-2 stages+exchange) + alignment + barriers
    return align_up((size_t)2 * B * 4 + (size_t)(2 * Cfg::NT + 1) * 4, 1024) + fused_region_bytes<N>(uniform) + 1024 + 64;
}

template <int N>
__global__ void __launch_bounds__(kFusedThreads, 1)
fused_image_kernel(const FusedArgs a, const __grid_constant__ ScaleBlock sc, const __grid_constant__ CUtensorMap tmap)
{
    using Cfg = FusedCfg<N>;
    constexpr int H = Cfg::H, TG = Cfg::TG, KU = Cfg::KU, NT = Cfg::NT, SLOTS = Cfg::SLOTS;
    extern __shared__ unsigned char smem_raw[];
    const bool uniform = a.weighting == BLINK_W_UNIFORM;
    const int B = a.B;

    // ---- shared memory carve-up -----------------------------------------------------------------
    uint32_t *items = reinterpret_cast<uint32_t *>(smem_raw);                  // [2B]
    uint32_t *toff = items + 2 * (size_t)B;                                    // [NT+1]
    uint32_t *tcur = toff + NT + 1;                                            // [NT]
    unsigned char *region = reinterpret_cast<unsigned char *>(
        (reinterpret_cast<uintptr_t>(tcur + NT) + 1023) & ~(uintptr_t)1023);
    float2 *tile = reinterpret_cast<float2 *>(region);                         // pass 1: [KU][SLOTS]
    uint32_t *cnt = reinterpret_cast<uint32_t *>(tile + (size_t)KU * SLOTS);   // pass 1 (uniform): [KU][SLOTS]
    unsigned char *stage = region;                                             // pass 2: [2][STAGE_BYTES]
    float2 *xbuf = reinterpret_cast<float2 *>(region + 2 * (size_t)Cfg::STAGE_BYTES);   // pass 2: [G][SLOTS]
    uint64_t *bars = reinterpret_cast<uint64_t *>(region + fused_region_bytes<N>(uniform));   // full[2]
    __shared__ int s_nin, s_umax, s_occ;

    const int g = threadIdx.x / TG;
    const int tid = threadIdx.x % TG;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float2 *scratch = a.scratch + (size_t)blockIdx.x * H * N;
    auto sync = [] { __syncthreads(); };

    if (threadIdx.x == 0) {
        mbar_init(&bars[0], 1);
        mbar_init(&bars[1], 1);
        fence_mbar_init();
        tma_prefetch_desc(&tmap);
    }
    uint32_t uses0 = 0, uses1 = 0;                                             // completed phases per barrier
    __syncthreads();

    for (int tc = a.tc0 + blockIdx.x; tc < a.tc0 + a.ntc; tc += gridDim.x) {
        const int t = tc / a.C, c = tc - t * a.C;
        const float s = sc.s[c - a.c_base];
        const float *uvw = a.uvw_m + (size_t)t * B * 3;

        // ---- index (a1) + histogram of the half-plane samples by u-tile --------------------------
        for (int i = threadIdx.x; i <= NT; i += kFusedThreads) toff[i] = 0;
        if (threadIdx.x == 0) { s_nin = 0; s_umax = 0; s_occ = 0; }
        __syncthreads();
        int my_in = 0, my_umax = 0;
        for (int b = threadIdx.x; b < B; b += kFusedThreads) {
            int iu, iv;
            const bool ok = cell_coords(uvw[3 * b], uvw[3 * b + 1], s, H, iu, iv);
            if (a.cell_idx) a.cell_idx[(size_t)tc * B + b] = ok ? (iv + H) * N + (iu + H) : -1;
            if (ok) {
                ++my_in;
                const int au = iu < 0 ? -iu : iu;
                my_umax = max(my_umax, au);
                atomicAdd(&toff[au / KU], iu == 0 ? 2u : 1u);
            }
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            my_in += __shfl_xor_sync(0xffffffffu, my_in, d);
            my_umax = max(my_umax, __shfl_xor_sync(0xffffffffu, my_umax, d));
        }
        if (lane == 0) { atomicAdd(&s_nin, my_in); atomicMax(&s_umax, my_umax); }
        __syncthreads();
        if (warp == 0) {                                                        // exclusive scan over the u-tiles
            uint32_t carry = 0;
            for (int base = 0; base < NT; base += 32) {
                const uint32_t v = (base + lane < NT) ? toff[base + lane] : 0u;
                uint32_t inc = v;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) {
                    const uint32_t y = __shfl_up_sync(0xffffffffu, inc, d);
                    if (lane >= d) inc += y;
                }
                if (base + lane < NT) { toff[base + lane] = carry + inc - v; tcur[base + lane] = carry + inc - v; }
                carry += __shfl_sync(0xffffffffu, inc, 31);
            }
            if (lane == 0) toff[NT] = carry;
        }
        __syncthreads();
        // ---- counting sort: item = [b:18][conj:1][u_local * N + row : 13] ---------------------------
        for (int b = threadIdx.x; b < B; b += kFusedThreads) {
            int iu, iv;
            if (cell_coords(uvw[3 * b], uvw[3 * b + 1], s, H, iu, iv)) {
                const uint32_t bl = (uint32_t)b << 14;
                if (iu >= 0) {                                                  // the sample itself lies in u >= 0
                    const uint32_t pos = atomicAdd(&tcur[iu / KU], 1u);
                    items[pos] = bl | (uint32_t)((iu % KU) * N + (iv + H));
                }
                if (iu <= 0) {                                                  // its conjugate lies in u >= 0
                    const int u = -iu;
                    const uint32_t pos = atomicAdd(&tcur[u / KU], 1u);
                    items[pos] = bl | (1u << 13) | (uint32_t)((u % KU) * N + (H - iv));
                }
            }
        }
        __syncthreads();
        const int n_in = s_nin;
        const int n_tiles = s_umax / KU + 1;                                    // tiles that can hold samples
        const int ulim = n_tiles * KU;                                          // scratch rows written by pass 1
        const int n_box = (ulim + Cfg::BOX_ROWS - 1) / Cfg::BOX_ROWS;
        float wsum_val = (float)(2 * n_in);

        for (int p = 0; p < a.P; ++p) {
            const size_t img_idx = (size_t)tc * a.P + p;
            float *img = a.image + img_idx * N * N;
            if (n_in == 0) {                                                    // W = 0: zero image
                for (int i = threadIdx.x; i < N * N / 4; i += kFusedThreads)
                    reinterpret_cast<float4 *>(img)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
                continue;
            }
            const float2 *vrow = a.vis + img_idx * B;
            int my_occ = 0;
            // ================= pass 1: grid a u-tile in shared memory, transform its columns along v =====
            for (int tl = 0; tl < n_tiles; ++tl) {
                __syncthreads();                                                // previous users of the region are done
                for (int i = threadIdx.x; i < KU * SLOTS / 2; i += kFusedThreads)
                    reinterpret_cast<float4 *>(tile)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
                if (uniform)
                    for (int i = threadIdx.x; i < KU * SLOTS / 4; i += kFusedThreads)
                        reinterpret_cast<uint4 *>(cnt)[i] = make_uint4(0u, 0u, 0u, 0u);
                __syncthreads();
                const uint32_t k0 = toff[tl], k1 = toff[tl + 1];
                for (uint32_t k = k0 + threadIdx.x; k < k1; k += kFusedThreads) {
                    const uint32_t it = items[k];
                    const int cl = it & 8191u;
                    const int ul = cl / N, r = cl % N;
                    const int o = ul * SLOTS + r + (r >> 3);
                    float2 v = __ldg(vrow + (it >> 14));
                    if (it & (1u << 13)) v.y = -v.y;
                    atomicAdd(&tile[o].x, v.x);
                    atomicAdd(&tile[o].y, v.y);
                    if (uniform) atomicAdd(&cnt[o], 1u);
                }
                __syncthreads();
                if (uniform) {                                                  // a3: divide by the cell count
                    for (int i = threadIdx.x; i < KU * SLOTS; i += kFusedThreads) {
                        const uint32_t cc = cnt[i];
                        if (cc) {
                            float2 v = tile[i];
                            v.x = __fdiv_rn(v.x, (float)cc); v.y = __fdiv_rn(v.y, (float)cc);
                            tile[i] = v;
                            // occupied cells of the FULL plane: the mirror image of a u > 0 cell is occupied too
                            my_occ += (tl == 0 && i < SLOTS) ? 1 : 2;
                        }
                    }
                    __syncthreads();
                }
                {
                    float2 *c0 = tile + (size_t)(2 * g) * SLOTS, *c1 = c0 + SLOTS;
                    ExchangePadded2 xch{c0, c1};
                    float2 v[2][kE];
#pragma unroll
                    for (int e = 0; e < kE; ++e) {                              // transform index n lives in centred row n ^ H
                        const int r = tid + (e ^ (kE / 2)) * TG;
                        v[0][e] = c0[r + (r >> 3)];
                        v[1][e] = c1[r + (r >> 3)];
                    }
                    fft_inverse<N, 2>(v, tid, xch, a.tw, sync);
                    float2 *d0 = scratch + (size_t)(tl * KU + 2 * g) * N, *d1 = d0 + N;
#pragma unroll
                    for (int e = 0; e < kE; ++e) {
                        d0[tid + e * TG] = v[0][e];
                        d1[tid + e * TG] = v[1][e];
                    }
                }
            }
            if (uniform && p == 0) {
#pragma unroll
                for (int d = 16; d > 0; d >>= 1) my_occ += __shfl_xor_sync(0xffffffffu, my_occ, d);
                if (lane == 0) atomicAdd(&s_occ, my_occ);
            }
            // scratch stores (generic proxy) must be visible to the TMA loads (async proxy) below
            __threadfence();
            asm volatile("fence.proxy.async;" ::: "memory");
            __syncthreads();
            if (uniform) wsum_val = (float)s_occ;
            const float inv_w = 1.0f / wsum_val;

            // ================= pass 2: row pairs -> two real image rows per transform ===================
            auto issue = [&](int it) {                                          // thread 0 only
                uint64_t *bar = &bars[it & 1];
                unsigned char *dst = stage + (size_t)(it & 1) * Cfg::STAGE_BYTES;
                mbar_expect_tx(bar, (uint32_t)(n_box * Cfg::BOX_ROWS * Cfg::ROWB));
                for (int bx = 0; bx < n_box; ++bx)
                    tma_load_3d(dst + (size_t)bx * Cfg::BOX_ROWS * Cfg::ROWB, &tmap, bar, 2 * it * Cfg::KY,
                                bx * Cfg::BOX_ROWS, (int)blockIdx.x);
            };
            if (threadIdx.x == 0) { issue(0); issue(1); }
            for (int it = 0; it < Cfg::NIT; ++it) {
                const int sb = it & 1;
                mbar_wait(&bars[sb], (sb ? uses1 : uses0) & 1u);
                if (sb) ++uses1; else ++uses0;
                float2 z[1][kE];
                if (g < Cfg::PAIRS) {
                    ExchangeTilePair<Cfg::ROWB> st{stage + (size_t)sb * Cfg::STAGE_BYTES, g};
#pragma unroll
                    for (int e = 0; e < kE / 2; ++e) {                          // n = u < H: S1 + i S2
                        const int u = tid + e * TG;
                        float4 q = make_float4(0.f, 0.f, 0.f, 0.f);
                        if (u < ulim) q = *st.at_row(u);
                        z[0][e] = make_float2(q.x - q.w, q.y + q.z);
                    }
#pragma unroll
                    for (int e = kE / 2; e < kE; ++e) {                         // n > H: conj(S1[N-n]) + i conj(S2[N-n])
                        const int u = N - (tid + e * TG);                       // in [1, H]; u == H is the empty Nyquist column
                        float4 q = make_float4(0.f, 0.f, 0.f, 0.f);
                        if (u < ulim && u < H) q = *st.at_row(u);
                        z[0][e] = make_float2(q.x + q.w, q.z - q.y);
                    }
                } else {
#pragma unroll
                    for (int e = 0; e < kE; ++e) z[0][e] = make_float2(0.f, 0.f);
                }
                __syncthreads();                                                // everyone has read this stage buffer
                if (threadIdx.x == 0 && it + 2 < Cfg::NIT) {
                    fence_proxy_async();
                    issue(it + 2);
                }
                ExchangePadded1 xch{xbuf + (size_t)g * SLOTS};
                fft_inverse<N, 1>(z, tid, xch, a.tw, sync);
                if (g < Cfg::PAIRS) {
                    const int ky = it * Cfg::KY + 2 * g;
                    float *r0 = img + (size_t)(ky ^ H) * N, *r1 = img + (size_t)((ky + 1) ^ H) * N;
#pragma unroll
                    for (int e = 0; e < kE; ++e) {
                        const int x = (tid + e * TG) ^ H;
                        __stcs(r0 + x, z[0][e].x * inv_w);
                        __stcs(r1 + x, z[0][e].y * inv_w);
                    }
                }
            }
        }
        if (threadIdx.x == 0) a.wsum[tc] = (n_in == 0) ? 0.f : wsum_val;
        __syncthreads();
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

// ------------------------------------------------------------------------------------------ host
bool fused_supported(int P, int B, int n_pix, int weighting)
{
    (void)P;
    const bool uni = weighting == BLINK_W_UNIFORM;
    size_t need;
    switch (n_pix) {
        case 256: need = fused_smem_bytes<256>(B, uni); break;
        case 512: need = fused_smem_bytes<512>(B, uni); break;
        case 1024: need = fused_smem_bytes<1024>(B, uni); break;
        case 2048: need = fused_smem_bytes<2048>(B, uni); break;
        case 4096: need = fused_smem_bytes<4096>(B, uni); break;
        default: return false;
    }
    return need <= 227 * 1024;
}

size_t fused_workspace_bytes(int n_pix, int ctas) { return (size_t)ctas * (n_pix / 2) * n_pix * sizeof(float2); }
int fused_default_ctas() { return sm_count() > 0 ? sm_count() : 148; }

// sub-ranges of flattened (t,c) that stay inside one block of <= 1024 channels
template <class F>
static int for_channel_blocks(int C, int tc0, int ntc, const double *freqs_hz, int n_pix, double pixscale_rad, F &&f)
{
    int tc = tc0;
    const int tc_end = tc0 + ntc;
    while (tc < tc_end) {
        const int t = tc / C, c = tc - t * C;
        const int c_base = (c / 1024) * 1024;
        const int c_lim = c_base + 1024 < C ? c_base + 1024 : C;
        int end = (C <= 1024) ? tc_end : t * C + c_lim;
        if (end > tc_end) end = tc_end;
        ScaleBlock sc;
        for (int k = 0; k < 1024; ++k) sc.s[k] = (c_base + k < C) ? scale_for(freqs_hz[c_base + k], n_pix, pixscale_rad) : 0.f;
        int rc = f(tc, end - tc, c_base, sc);
        if (rc != BLINK_OK) return rc;
        tc = end;
    }
    return BLINK_OK;
}

template <int N>
static int launch_fused(const FusedArgs &base, const double *freqs_hz, double pixscale_rad, void *workspace,
                        size_t workspace_bytes, cudaStream_t st)
{
    using Cfg = FusedCfg<N>;
    const size_t per_cta = (size_t)Cfg::H * N * sizeof(float2);
    if (!workspace || !aligned16(workspace) || workspace_bytes < per_cta) return BLINK_ERR_WORKSPACE;
    int ctas = option(BLINK_OPT_FUSED_CTAS);
    if (ctas <= 0) ctas = fused_default_ctas();
    ctas = (int)std::min<size_t>((size_t)ctas, workspace_bytes / per_cta);
    const size_t smem = fused_smem_bytes<N>(base.B, base.weighting == BLINK_W_UNIFORM);
    BLINK_CUDA_TRY(cudaFuncSetAttribute(fused_image_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    CUtensorMap tmap;
    // scratch viewed as float32 [ctas][H rows (u)][2N (ky re/im)]; boxes of [BOX_ROWS u][KY ky]
    int rc = encode_tensor_map_3d_f32(&tmap, workspace, 2ull * N, (uint64_t)Cfg::H, (uint64_t)ctas, (uint64_t)N * 8,
                                      (uint64_t)Cfg::H * N * 8, 2 * Cfg::KY, Cfg::BOX_ROWS, 1,
                                      Cfg::ROWB >= 32 ? Cfg::ROWB : 0);
    if (rc != 0) { set_error_text("cuTensorMapEncodeTiled failed (fused scratch)"); return BLINK_ERR_CUDA; }
    return for_channel_blocks(base.C, base.tc0, base.ntc, freqs_hz, N, pixscale_rad,
                              [&](int tc0, int ntc, int c_base, const ScaleBlock &sc) -> int {
                                  FusedArgs a = base;
                                  a.tc0 = tc0; a.ntc = ntc; a.c_base = c_base;
                                  a.scratch = static_cast<float2 *>(workspace);
                                  a.tw = twiddle_table();
                                  const int grid = ntc < ctas ? ntc : ctas;
                                  fused_image_kernel<N><<<grid, kFusedThreads, smem, st>>>(a, sc, tmap);
                                  BLINK_LAUNCH_CHECK("fused_image_kernel");
                                  return (int)BLINK_OK;
                              });
}

int fused_image(const float2 *vis, const float *uvw_m, const double *freqs_hz, double pixscale_rad, int T, int C, int P,
                int B, int n_pix, int weighting, int tc0, int ntc, float *image, float *wsum, int32_t *cell_idx,
                void *workspace, size_t workspace_bytes, cudaStream_t st)
{
    FusedArgs a{};
    a.vis = vis; a.uvw_m = uvw_m; a.T = T; a.C = C; a.P = P; a.B = B; a.weighting = weighting;
    a.tc0 = tc0; a.ntc = ntc; a.image = image; a.wsum = wsum; a.cell_idx = cell_idx;
    switch (n_pix) {
        case 256: return launch_fused<256>(a, freqs_hz, pixscale_rad, workspace, workspace_bytes, st);
        case 512: return launch_fused<512>(a, freqs_hz, pixscale_rad, workspace, workspace_bytes, st);
        case 1024: return launch_fused<1024>(a, freqs_hz, pixscale_rad, workspace, workspace_bytes, st);
        case 2048: return launch_fused<2048>(a, freqs_hz, pixscale_rad, workspace, workspace_bytes, st);
        case 4096: return launch_fused<4096>(a, freqs_hz, pixscale_rad, workspace, workspace_bytes, st);
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
