// Stand-alone SwiGLU forward / backward ("fused SwiGLU fwd/bwd").
// The tensor-core GEMMs fuse these into their epilogues; these kernels serve the fp32 path and the
// public moe_swiglu / moe_swiglu_bwd entry points.
#include "common.cuh"

namespace moe {
namespace {

template <typename T>
__global__ void __launch_bounds__(256) swiglu_kernel(const T* __restrict__ gu, T* __restrict__ a, int64_t rows, int F) {
  const int64_t n = rows * F;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t r = i / F;
    const int f = (int)(i - r * F);
    const float g = to_f(gu[r * 2 * F + f]);
    const float u = to_f(gu[r * 2 * F + F + f]);
    a[i] = from_f<T>(g * sigmoidf_acc(g) * u);
  }
}

template <typename T>
__global__ void __launch_bounds__(256) swiglu_bwd_kernel(const T* __restrict__ gu, const T* __restrict__ da,
                                                         T* __restrict__ dgu, int64_t rows, int F) {
  const int64_t n = rows * F;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t r = i / F;
    const int f = (int)(i - r * F);
    const float g = to_f(gu[r * 2 * F + f]);
    const float u = to_f(gu[r * 2 * F + F + f]);
    const float d = to_f(da[i]);
    const float s = sigmoidf_acc(g);
    dgu[r * 2 * F + f] = from_f<T>(d * u * s * (1.0f + g * (1.0f - s)));
    dgu[r * 2 * F + F + f] = from_f<T>(d * g * s);
  }
}

}  // namespace

int32_t swiglu_fwd(int dtype, const void* gu, void* a, int64_t rows, int F, cudaStream_t s) {
  if (rows <= 0) return MOE_OK;
  const unsigned grid = (unsigned)std::min<int64_t>(ceil_div(rows * F, 256), 148 * 16);
  if (dtype == 0)
    MOE_LAUNCH(swiglu_kernel<float>, grid, 256, 0, s, (const float*)gu, (float*)a, rows, F);
  else
    MOE_LAUNCH(swiglu_kernel<__nv_bfloat16>, grid, 256, 0, s, (const __nv_bfloat16*)gu, (__nv_bfloat16*)a, rows, F);
  return MOE_OK;
}

int32_t swiglu_bwd(int dtype, const void* gu, const void* da, void* dgu, int64_t rows, int F, cudaStream_t s) {
  if (rows <= 0) return MOE_OK;
  const unsigned grid = (unsigned)std::min<int64_t>(ceil_div(rows * F, 256), 148 * 16);
  if (dtype == 0)
    MOE_LAUNCH(swiglu_bwd_kernel<float>, grid, 256, 0, s, (const float*)gu, (const float*)da, (float*)dgu, rows, F);
  else
    MOE_LAUNCH(swiglu_bwd_kernel<__nv_bfloat16>, grid, 256, 0, s, (const __nv_bfloat16*)gu, (const __nv_bfloat16*)da,
               (__nv_bfloat16*)dgu, rows, F);
  return MOE_OK;
}

}  // namespace moe

extern "C" int32_t moe_swiglu(const moe_config_t* cfg, const void* gu, void* a, int64_t rows, void* stream) {
  using namespace moe;
  if (!cfg || !gu || !a || rows < 0) return MOE_ERR_INVALID_ARG;
  MOE_CHECK(validate(cfg));
  return swiglu_fwd(cfg->dtype, gu, a, rows, cfg->F, as_stream(stream));
}

extern "C" int32_t moe_swiglu_bwd(const moe_config_t* cfg, const void* gu, const void* da, void* dgu, int64_t rows,
                                  void* stream) {
  using namespace moe;
  if (!cfg || !gu || !da || !dgu || rows < 0) return MOE_ERR_INVALID_ARG;
  MOE_CHECK(validate(cfg));
  return swiglu_bwd(cfg->dtype, gu, da, dgu, rows, cfg->F, as_stream(stream));
}
