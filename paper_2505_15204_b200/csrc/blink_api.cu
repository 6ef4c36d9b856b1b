// libblinkimg: process-wide state (options, error text, launch counter, twiddle table), the TMA
// tensor-map encoder and the workspace query.
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <vector>

#include "blink_common.cuh"
#include "blink_tma.cuh"

namespace blink {

static thread_local char g_err[512] = "";
static std::atomic<unsigned long long> g_launches{0};
static thread_local int g_opts[8];                             // route / test switches of the CALLING thread
static std::mutex g_init_mu;
constexpr int kMaxDevices = 64;
static bool g_dev_ready[kMaxDevices];                           // per device: twiddle table uploaded (guarded by g_init_mu)
static std::atomic<int> g_dev_sms[kMaxDevices];
__device__ float2 g_twiddle[kTwiddleN];

void set_cuda_error(cudaError_t e, const char *where)
{
    snprintf(g_err, sizeof(g_err), "%s: %s (%s)", where, cudaGetErrorName(e), cudaGetErrorString(e));
    (void)cudaGetLastError();                                   // clear the sticky-less error state
}
void set_error_text(const char *text) { snprintf(g_err, sizeof(g_err), "%s", text); }
void count_launch(unsigned n) { g_launches.fetch_add(n, std::memory_order_relaxed); }
int option(int key) { return (key >= 0 && key < 8) ? g_opts[key] : 0; }
int sm_count()
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return 0;
    return g_dev_sms[dev].load(std::memory_order_relaxed);
}

const float2 *twiddle_table()
{
    void *p = nullptr;
    cudaGetSymbolAddress(&p, g_twiddle);
    return static_cast<const float2 *>(p);
}

int ensure_device()
{
    int dev = -1;
    BLINK_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) { set_error_text("device ordinal out of range"); return BLINK_ERR_CUDA; }
    std::lock_guard<std::mutex> lk(g_init_mu);
    if (g_dev_ready[dev]) return BLINK_OK;
    cudaDeviceProp prop;
    BLINK_CUDA_TRY(cudaGetDeviceProperties(&prop, dev));
    if (prop.major != 10) {
        set_error_text("libblinkimg is built for sm_100a only: no compute-capability-10.x device is current");
        return BLINK_ERR_CUDA;
    }
    std::vector<float2> tw(kTwiddleN);
    const double two_pi = 6.283185307179586476925286766559;
    for (int m = 0; m < kTwiddleN; ++m) {
        const double a = two_pi * (double)m / (double)kTwiddleN;
        tw[m] = make_float2((float)std::cos(a), (float)std::sin(a));
    }
    // exact values on the axes and diagonals (cos/sin of multiples of pi/4 rounded from double are already exact
    // for 0 and +-1; force the zeros)
    tw[0] = make_float2(1.f, 0.f);
    tw[kTwiddleN / 4] = make_float2(0.f, 1.f);
    tw[kTwiddleN / 2] = make_float2(-1.f, 0.f);
    tw[3 * kTwiddleN / 4] = make_float2(0.f, -1.f);
    BLINK_CUDA_TRY(cudaMemcpyToSymbol(g_twiddle, tw.data(), sizeof(float2) * kTwiddleN));   // this device's copy of the symbol
    g_dev_sms[dev].store(prop.multiProcessorCount, std::memory_order_relaxed);
    g_dev_ready[dev] = true;
    return BLINK_OK;
}

// ---- tensor map encoder through the runtime's driver entry point (no -lcuda) -------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn()
{
    static EncodeTiledFn fn = nullptr;
    static std::once_flag once;
    std::call_once(once, [] {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    });
    return fn;
}

int encode_tensor_map_3d_f32(CUtensorMap *out, const void *base, uint64_t d0, uint64_t d1, uint64_t d2,
                             uint64_t stride1_bytes, uint64_t stride2_bytes, uint32_t b0, uint32_t b1, uint32_t b2,
                             int swizzle_bytes)
{
    EncodeTiledFn fn = encode_fn();
    if (!fn) return -1;
    cuuint64_t dims[3] = {d0, d1, d2};
    cuuint64_t strides[2] = {stride1_bytes, stride2_bytes};
    cuuint32_t box[3] = {b0, b1, b2};
    cuuint32_t estr[3] = {1, 1, 1};
    CUtensorMapSwizzle sw = swizzle_bytes == 128 ? CU_TENSOR_MAP_SWIZZLE_128B
                          : swizzle_bytes == 64  ? CU_TENSOR_MAP_SWIZZLE_64B
                          : swizzle_bytes == 32  ? CU_TENSOR_MAP_SWIZZLE_32B
                                                 : CU_TENSOR_MAP_SWIZZLE_NONE;
    CUresult r = fn(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<void *>(base), dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, sw, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return (int)r;
}

// 4D uint8 tensor map, 128-byte swizzle (the correlator's voltage tiles).  dims / box in BYTES-as-elements, innermost
// first; strides in bytes for dims 1..3 (multiples of 16).
int encode_tensor_map_4d_u8(CUtensorMap *out, const void *base, const uint64_t dims[4], const uint64_t strides[3],
                            const uint32_t box[4], int swizzle_bytes)
{
    EncodeTiledFn fn = encode_fn();
    if (!fn) return -1;
    cuuint64_t d[4] = {dims[0], dims[1], dims[2], dims[3]};
    cuuint64_t st[3] = {strides[0], strides[1], strides[2]};
    cuuint32_t b[4] = {box[0], box[1], box[2], box[3]};
    cuuint32_t estr[4] = {1, 1, 1, 1};
    CUresult r = fn(out, CU_TENSOR_MAP_DATA_TYPE_UINT8, 4, const_cast<void *>(base), d, st, b, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE,
                    swizzle_bytes == 32 ? CU_TENSOR_MAP_SWIZZLE_32B : swizzle_bytes == 64 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_128B,
                    CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return (int)r;
}

}  // namespace blink

extern "C" const char *blink_strerror(int code)
{
    switch (code) {
        case BLINK_OK: return "ok";
        case BLINK_ERR_INVALID_ARG: return "invalid argument";
        case BLINK_ERR_UNSUPPORTED: return "unsupported size";
        case BLINK_ERR_WORKSPACE: return "workspace too small";
        case BLINK_ERR_CUDA: return "CUDA error";
        default: return "unknown error code";
    }
}
extern "C" const char *blink_last_cuda_error(void) { return blink::g_err; }
extern "C" unsigned long long blink_kernel_launches(void) { return blink::g_launches.load(); }
extern "C" int blink_set_option(int key, int value)
{
    if (key < 0 || key >= 8) return BLINK_ERR_INVALID_ARG;
    blink::g_opts[key] = value;
    return BLINK_OK;
}
extern "C" int blink_get_option(int key, int *value)
{
    if (key < 0 || key >= 8 || !value) return BLINK_ERR_INVALID_ARG;
    *value = blink::g_opts[key];
    return BLINK_OK;
}
