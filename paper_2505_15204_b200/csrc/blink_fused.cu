// Fused imaging kernel (visibilities -> images without materialising the uv grid).  Placeholder in this
// revision: fused_supported() reports false and blink_image takes the unfused chain.
#include "blink_common.cuh"

namespace blink {

bool fused_supported(int, int, int, int) { return false; }
size_t fused_workspace_bytes(int, int) { return 0; }
int fused_default_ctas() { return sm_count() > 0 ? sm_count() : 148; }
int fused_image(const float2 *, const float *, const double *, double, int, int, int, int, int, int, int, int, float *,
                float *, int32_t *, void *, size_t, cudaStream_t)
{
    return BLINK_ERR_UNSUPPORTED;
}
int counts_only(const float *, const double *, double, int, int, int, int, int, int, uint32_t *, cudaStream_t)
{
    return BLINK_ERR_UNSUPPORTED;
}

}  // namespace blink
