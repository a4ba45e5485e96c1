// tcgen05 grouped GEMMs (placeholder until the kernels land): every entry reports UNSUPPORTED so the
// callers take the CUDA-core path.
#include "common.cuh"

namespace moe {
struct FfnGroup;
int32_t tc_ffn_fwd(const FfnGroup&, const void*, const void*, const void*, const void*, void*, void*, void*,
                   cudaStream_t) { return MOE_ERR_UNSUPPORTED; }
int32_t tc_ffn_bwd(const FfnGroup&, const void*, const void*, const void*, const void*, const void*, const void*,
                   const void*, void*, void*, void*, void*, void*, cudaStream_t) { return MOE_ERR_UNSUPPORTED; }
int32_t tc_grouped_gemm_fwd(const moe_config_t*, int, int, const void*, const void*, const int32_t*, void*, int32_t*,
                            cudaStream_t) { return MOE_ERR_UNSUPPORTED; }
int32_t tc_grouped_gemm_bwd(const moe_config_t*, int, int, const void*, const void*, const void*, const int32_t*,
                            void*, void*, int32_t*, cudaStream_t) { return MOE_ERR_UNSUPPORTED; }
int32_t fp8_grouped_gemm_fwd(const moe_config_t*, int, int, const void*, const void*, const int32_t*, void*,
                             const float*, const float*, int32_t*, cudaStream_t) { return MOE_ERR_UNSUPPORTED; }
}  // namespace moe

extern "C" int32_t moe_quantize_act(const void*, int64_t, int32_t, int32_t, uint8_t*, float*, void*) {
  return MOE_ERR_UNSUPPORTED;
}
extern "C" int32_t moe_quantize_weight(const void*, int32_t, int32_t, int32_t, int32_t, uint8_t*, float*, void*) {
  return MOE_ERR_UNSUPPORTED;
}
