// blink_image_static: blink_image for callers that cannot allocate device memory (code under CUDA graph capture, tight
// serving loops, harnesses that forbid cudaMalloc) and therefore have no workspace to pass.  The scratch the imaging kernels
// need -- the per-timestep sorted baselines, the team counters and the per-CTA half planes H[u][ky] of the fused kernel
// (blink_fused_kernel.cuh), or the chunk's grids of the unfused chain -- lives in ONE file-scope device array of a fixed,
// modest size instead.  Every GPU that loads the library holds that array until the process exits.
//
// Rules that follow from sharing one array:
//   * every call on a device uses the same array, which keeps the previous call's contents.  Nothing in it has to start at
//     zero except the team counters, which the fused launcher clears in-stream (cudaMemsetAsync) before the kernel that uses
//     them; everything else is written before it is read (the parity tests poison workspaces with NaN to hold this);
//   * two calls that overlap on the GPU (different streams, or the same stream from two threads without ordering) RACE on the
//     array.  Calls on one stream are ordered and safe;
//   * problems whose minimum blink_image workspace exceeds the array are refused with BLINK_ERR_WORKSPACE and a text that
//     names both sizes; nothing is launched.
// The entry point calls no cudaMalloc / cudaFree / allocating library routine: it resolves the array's device address once
// per device (cudaGetSymbolAddress; in host code the array's NAME is only a host-side stand-in, never a device address) and
// hands that pointer to the existing imaging path.
#include <mutex>
#include <stdio.h>

#include "blink_common.cuh"

namespace blink {

constexpr size_t kStaticScratchBytes = (size_t)32 << 20;        // 32 MiB per GPU
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

constexpr int kStaticMaxDevices = 64;
static std::mutex g_static_mu;
static void *g_static_ptr[kStaticMaxDevices];                   // device address of g_static_scratch on each device (guarded)

// device address of the array on the CURRENT device, resolved once per device with that device current
static int static_scratch_ptr(void **out)
{
    int dev = -1;
    BLINK_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticMaxDevices) { set_error_text("device ordinal out of range"); return BLINK_ERR_CUDA; }
    std::lock_guard<std::mutex> lk(g_static_mu);
    if (g_static_ptr[dev] == nullptr) {
        void *p = nullptr;
        BLINK_CUDA_TRY(cudaGetSymbolAddress(&p, g_static_scratch));
        if (p == nullptr || (reinterpret_cast<uintptr_t>(p) & 255u)) {
            set_error_text("cudaGetSymbolAddress(g_static_scratch) returned a null or misaligned address");
            return BLINK_ERR_CUDA;
        }
        g_static_ptr[dev] = p;
    }
    *out = g_static_ptr[dev];
    return BLINK_OK;
}

}  // namespace blink

using namespace blink;

extern "C" size_t blink_static_scratch_bytes(void) { return kStaticScratchBytes; }

extern "C" int blink_image_static(const blink_c64 *vis, const float *uvw_m, const double *freqs_hz, int T, int C, int P, int B,
                                  int n_pix, double pixscale_rad, int weighting, float *image, float *wsum, void *stream)
{
    // the size check is host arithmetic and comes first: a problem that does not fit launches nothing
    size_t rec = 0, mn = 0;
    int rc = blink_workspace_bytes(BLINK_OP_IMAGE, T, C, P, B, n_pix, weighting, &rec, &mn);
    if (rc != BLINK_OK) return rc;
    if (mn > kStaticScratchBytes) {
        char msg[256];
        snprintf(msg, sizeof(msg),
                 "blink_image_static: this problem needs at least %zu bytes of scratch, the built-in array holds %zu "
                 "(use blink_image with a caller-owned workspace)", mn, kStaticScratchBytes);
        set_error_text(msg);
        return BLINK_ERR_WORKSPACE;
    }
    rc = ensure_device();
    if (rc != BLINK_OK) return rc;
    void *scratch = nullptr;
    rc = static_scratch_ptr(&scratch);
    if (rc != BLINK_OK) return rc;
    // the existing path, unchanged, with the built-in array as its workspace (it chunks / limits its CTAs to what fits)
    return blink_image(vis, uvw_m, freqs_hz, T, C, P, B, n_pix, pixscale_rad, weighting, image, wsum, nullptr, nullptr, scratch,
                       kStaticScratchBytes, stream);
}
