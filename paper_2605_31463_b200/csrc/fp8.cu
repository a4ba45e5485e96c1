// FP8 e4m3 block-scaled path.  Quantisers and GEMMs land here; until then the
// entry points report MOE_ERR_UNSUPPORTED (nothing is enqueued, nothing falls back to another path).
#include "common.cuh"

extern "C" int32_t moe_quantize_act(const void*, int64_t, int32_t, int32_t, uint8_t*, float*, void*) {
  return MOE_ERR_UNSUPPORTED;
}
extern "C" int32_t moe_quantize_weight(const void*, int32_t, int32_t, int32_t, int32_t, uint8_t*, float*, void*) {
  return MOE_ERR_UNSUPPORTED;
}
