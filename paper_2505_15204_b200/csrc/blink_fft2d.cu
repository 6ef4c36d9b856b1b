// blink_fft2d_inverse: batched centred inverse 2D FFT, complex64 grids -> float32 images.
//   pass 1 (fft_rows_kernel): N-point transforms along u (rows), in place, output in natural
//           (unshifted) x order; register-resident radix-8/4 stages, shared-memory exchanges.
//   pass 2 (fft_cols_kernel): a tile of KC columns x N rows is staged into shared memory by TMA
//           (hardware-swizzled), every thread group transforms a column PAIR with 16-byte shared
//           accesses, and the fftshift, the 1/W scale and the real-part extraction are fused into the
//           store (shift after the FFT; readings R5-R7).
// Centring is index arithmetic only: centred index r <-> transform index r ^ (N/2).
#include "blink_common.cuh"
#include "blink_fft.cuh"
#include "blink_tma.cuh"

namespace blink {

// ------------------------------------------------------------------------------------------ rows
template <int N>
struct RowCfg {
    static constexpr int TG = N / kE;                                  // threads per row
    static constexpr int THREADS = TG > 256 ? TG : 256;
    static constexpr int G = THREADS / TG;                             // rows in flight per CTA
    static constexpr int SLOTS = N;
    static constexpr size_t SMEM = (size_t)G * SLOTS * sizeof(float2);
};

template <int N>
__global__ void __launch_bounds__(RowCfg<N>::THREADS)
fft_rows_kernel(float2 *__restrict__ grid, long long n_rows, const float2 *__restrict__ tw)
{
    using Cfg = RowCfg<N>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *xbuf = reinterpret_cast<float2 *>(smem_raw);
    const int g = threadIdx.x / Cfg::TG;
    const int tid = threadIdx.x % Cfg::TG;
    ExchangePadded1 xch{xbuf + (size_t)g * Cfg::SLOTS};
    auto sync = [] { __syncthreads(); };
    Twiddles<N> twr;
    twr.init(tid, tw);
    for (long long base = (long long)blockIdx.x * Cfg::G; base < n_rows; base += (long long)gridDim.x * Cfg::G) {
        const long long row = base + g;
        const bool valid = row < n_rows;
        float2 *p = grid + row * N;
        float2 v[1][kE];
#pragma unroll
        for (int e = 0; e < kE; ++e)                                   // transform index n = tid + e*TG lives in column n ^ h
            v[0][e] = valid ? p[tid + (e ^ (kE / 2)) * Cfg::TG] : make_float2(0.f, 0.f);
        fft_inverse<N, 1>(v, tid, xch, twr, sync);
        if (valid) {
#pragma unroll
            for (int e = 0; e < kE; ++e) p[tid + e * Cfg::TG] = v[0][e];
        }
    }
}

// --------------------------------------------------------------------------------------- columns
template <int N>
struct ColCfg {
    static constexpr int KC = N <= 512 ? 16 : (N == 1024 ? 8 : (N == 2048 ? 4 : 2));   // columns per tile
    static constexpr int ROWB = KC * 8;                                // tile row bytes = TMA swizzle span
    static constexpr int PAIRS = KC / 2;
    static constexpr int TG = N / kE;
    static constexpr int THREADS = PAIRS * TG;
    static constexpr int BOX_ROWS = N < 256 ? N : 256;
    static constexpr int NBOX = N / BOX_ROWS;
    static constexpr size_t TILE_BYTES = (size_t)N * ROWB;
    static constexpr size_t SMEM = TILE_BYTES + 1024 /*alignment slack*/ + 16 /*mbarrier*/;
};

// staging address of (row y, pair) for the transposed store: rows of KC floats, pairs XOR-permuted so
// that 16 consecutive rows hit 16 different 8-byte bank pairs
template <int KC>
__device__ __forceinline__ int stage_off(int y, int pair)
{
    constexpr int RPL = 32 / KC;                                       // rows per 128-byte line
    constexpr int PPR = KC / 2;                                        // pairs per row
    return y * KC + (((pair ^ (y / RPL)) & (PPR - 1)) << 1);           // in floats
}

template <int N>
__global__ void __launch_bounds__(ColCfg<N>::THREADS)
fft_cols_kernel(const __grid_constant__ CUtensorMap tmap, const float *__restrict__ scale, int scale_div,
                int img_base, float *__restrict__ image, float *__restrict__ image_imag, const float2 *__restrict__ tw)
{
    using Cfg = ColCfg<N>;
    constexpr int h = N / 2;
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    // keep the pointer in the shared window (pointer arithmetic on the array, no integer round trip)
    unsigned char *tile = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint64_t *bar = reinterpret_cast<uint64_t *>(tile + Cfg::TILE_BYTES);

    const int col0 = blockIdx.x * Cfg::KC;                             // first (natural-order) column of the tile
    const int img = blockIdx.y;

    if (threadIdx.x == 0) {
        mbar_init(bar, 1);
        fence_mbar_init();
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        mbar_expect_tx(bar, (uint32_t)Cfg::TILE_BYTES);
#pragma unroll
        for (int b = 0; b < Cfg::NBOX; ++b)
            tma_load_3d(tile + (size_t)b * Cfg::BOX_ROWS * Cfg::ROWB, &tmap, bar, 2 * col0, b * Cfg::BOX_ROWS, img);
    }
    const int pair = threadIdx.x / Cfg::TG;
    const int tid = threadIdx.x % Cfg::TG;
    ExchangeTilePair<Cfg::ROWB> xch{tile, pair};
    mbar_wait(bar, 0);

    // transform index n = tid + e*TG is stored in centred row n ^ h
    float2 v[2][kE];
#pragma unroll
    for (int e = 0; e < kE; ++e) {
        const float4 t = *xch.at_row(tid + (e ^ (kE / 2)) * Cfg::TG);
        v[0][e] = make_float2(t.x, t.y);
        v[1][e] = make_float2(t.z, t.w);
    }
    auto sync = [] { __syncthreads(); };
    Twiddles<N> twr;
    twr.init(tid, tw);
    fft_inverse<N, 2>(v, tid, xch, twr, sync);

    // epilogue: scale, real part, fftshift (y = ky ^ h, x = kx ^ h), transposed through shared memory
    float s = 1.0f;
    if (scale != nullptr) {
        const float w = scale[(img_base + img) / scale_div];
        s = (w != 0.0f) ? 1.0f / w : 0.0f;
    }
    float *st_re = reinterpret_cast<float *>(tile);
    float *st_im = st_re + (size_t)N * Cfg::KC;
    __syncthreads();                                                   // all exchange reads done before reuse
#pragma unroll
    for (int e = 0; e < kE; ++e) {
        const int y = (tid + e * Cfg::TG) ^ h;
        const int o = stage_off<Cfg::KC>(y, pair);
        *reinterpret_cast<float2 *>(st_re + o) = make_float2(v[0][e].x * s, v[1][e].x * s);
        if (image_imag != nullptr) *reinterpret_cast<float2 *>(st_im + o) = make_float2(v[0][e].y * s, v[1][e].y * s);
    }
    __syncthreads();
    const int x0 = col0 ^ h;                                           // KC-aligned, so the tile stays contiguous in x
    const size_t img_off = (size_t)img * N * N;
    for (int idx = threadIdx.x; idx < N * Cfg::PAIRS; idx += Cfg::THREADS) {
        const int y = idx / Cfg::PAIRS, pr = idx % Cfg::PAIRS;
        const int o = stage_off<Cfg::KC>(y, pr);
        const size_t go = img_off + (size_t)y * N + x0 + 2 * pr;
        *reinterpret_cast<float2 *>(image + go) = *reinterpret_cast<const float2 *>(st_re + o);
        if (image_imag != nullptr)
            *reinterpret_cast<float2 *>(image_imag + go) = *reinterpret_cast<const float2 *>(st_im + o);
    }
}

// ------------------------------------------------------------------------------------------ host
template <int N>
static int launch_fft2d(float2 *grid, int batch, const float *scale, int scale_div, int img_base, float *image,
                        float *image_imag, cudaStream_t st)
{
    using RC = RowCfg<N>;
    using CC = ColCfg<N>;
    const float2 *tw = twiddle_table();
    // the attribute belongs to the current device's context: set it on every launch (cheap, idempotent)
    BLINK_CUDA_TRY(cudaFuncSetAttribute(fft_rows_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RC::SMEM));
    BLINK_CUDA_TRY(cudaFuncSetAttribute(fft_cols_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)CC::SMEM));
    // grid.y is limited to 65535: process the batch in slabs
    const long long n_rows = (long long)batch * N;
    long long want = (n_rows + RC::G - 1) / RC::G;
    const long long cap = (long long)sm_count() * 16;
    const int rgrid = (int)(want < cap ? want : cap);
    fft_rows_kernel<N><<<rgrid, RC::THREADS, RC::SMEM, st>>>(grid, n_rows, tw);
    BLINK_LAUNCH_CHECK("fft_rows_kernel");

    for (int b0 = 0; b0 < batch; b0 += 65535) {
        const int nb = batch - b0 < 65535 ? batch - b0 : 65535;
        CUtensorMap tmap;
        int rc = encode_tensor_map_3d_f32(&tmap, grid + (size_t)b0 * N * N, 2ull * N, (uint64_t)N, (uint64_t)nb,
                                          (uint64_t)N * 8, (uint64_t)N * N * 8, 2 * CC::KC, CC::BOX_ROWS, 1,
                                          CC::ROWB >= 32 ? CC::ROWB : 0);
        if (rc != 0) { set_error_text("cuTensorMapEncodeTiled failed"); return BLINK_ERR_CUDA; }
        dim3 g(N / CC::KC, nb);
        fft_cols_kernel<N><<<g, CC::THREADS, CC::SMEM, st>>>(
            tmap, scale, scale_div, img_base + b0, image + (size_t)b0 * N * N,
            image_imag ? image_imag + (size_t)b0 * N * N : nullptr, tw);
        BLINK_LAUNCH_CHECK("fft_cols_kernel");
    }
    return BLINK_OK;
}

int fft2d_range(float2 *grid, int n_pix, int batch, const float *scale, int scale_div, int img_base, float *image,
                float *image_imag, cudaStream_t st, float2 *tw_generic, bool hermitian, const int *row_extent, int ext_div)
{
    if (batch == 0) return BLINK_OK;
    if (!is_pow2(n_pix))
        return size_supported(n_pix) ? gfft2d_range(grid, n_pix, batch, scale, scale_div, img_base, image, image_imag, tw_generic, st, hermitian,
                                                    row_extent, ext_div)
                                     : (int)BLINK_ERR_UNSUPPORTED;
    switch (n_pix) {
        case 32: return launch_fft2d<32>(grid, batch, scale, scale_div, img_base, image, image_imag, st);
        case 64: return launch_fft2d<64>(grid, batch, scale, scale_div, img_base, image, image_imag, st);
        case 128: return launch_fft2d<128>(grid, batch, scale, scale_div, img_base, image, image_imag, st);
        case 256: return launch_fft2d<256>(grid, batch, scale, scale_div, img_base, image, image_imag, st);
        case 512: return launch_fft2d<512>(grid, batch, scale, scale_div, img_base, image, image_imag, st);
        case 1024: return launch_fft2d<1024>(grid, batch, scale, scale_div, img_base, image, image_imag, st);
        case 2048: return launch_fft2d<2048>(grid, batch, scale, scale_div, img_base, image, image_imag, st);
        case 4096: return launch_fft2d<4096>(grid, batch, scale, scale_div, img_base, image, image_imag, st);
        case 8192: return launch_fft2d<8192>(grid, batch, scale, scale_div, img_base, image, image_imag, st);
        default: return BLINK_ERR_UNSUPPORTED;
    }
}

}  // namespace blink

extern "C" int blink_fft2d_inverse(blink_c64 *grid, int n_pix, int batch, const float *scale, int scale_stride_div,
                                   float *image, float *image_imag, void *workspace, size_t workspace_bytes,
                                   void *stream)
{
    using namespace blink;
    if (grid == nullptr || image == nullptr || batch < 0) return BLINK_ERR_INVALID_ARG;
    if (!aligned16(grid) || !aligned16(image) || (image_imag && !aligned16(image_imag))) return BLINK_ERR_INVALID_ARG;
    if (!size_supported(n_pix)) return BLINK_ERR_UNSUPPORTED;
    if (scale != nullptr && scale_stride_div < 1) return BLINK_ERR_INVALID_ARG;
    if (scale == nullptr) scale_stride_div = 1;
    int rc = ensure_device();
    if (rc != BLINK_OK) return rc;
    float2 *tw_generic = nullptr;                              // sides that are not a power of two: twiddle table in the workspace
    if (!is_pow2(n_pix)) {
        if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 15u) || workspace_bytes < gfft_workspace_bytes(n_pix))
            return BLINK_ERR_WORKSPACE;
        tw_generic = static_cast<float2 *>(workspace);
    }
    return fft2d_range(reinterpret_cast<float2 *>(grid), n_pix, batch, scale, scale_stride_div, 0, image, image_imag,
                       static_cast<cudaStream_t>(stream), tw_generic);
}
