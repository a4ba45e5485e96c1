// Zero-computation experts (V2; "zero", "copy", "constant"): the last n_zero + n_copy + n_const
// router outputs own no FFN weights.  Their tokens are routed, permuted, combined and differentiated like any other
// expert's; only the expert function differs:  y = 0 | x | v_c.  These kernels fill the rows of those experts' groups
// (which the grouped GEMMs never visit) in the forward and in the backward.  HBM-bound row movers, 16-byte accesses.
#include "common.cuh"

namespace moe {
namespace {

constexpr int ZC_WARPS = 8;

// kind of zero-computation expert j (0-based among them): 0 = zero, 1 = copy, 2 = constant (+ index among constants)
__device__ __forceinline__ int zc_kind(int j, int n_zero, int n_copy, int& cidx) {
  cidx = j - n_zero - n_copy;
  return j < n_zero ? 0 : (j < n_zero + n_copy ? 1 : 2);
}

// grid (row chunks, n_zc).  Forward: y[r] = 0 | Xp[r] | v;  gu[r] = 0, a[r] = 0 (padding rows of the group included, so
// that every row below offsets[E] is defined).
__global__ void __launch_bounds__(ZC_WARPS * 32) zc_fwd_kernel(const int32_t* __restrict__ offsets,
                                                                const int32_t* __restrict__ counts, int E_ffn, int n_zero,
                                                                int n_copy, int nvecH, int nvecF, const int4* __restrict__ Xp,
                                                                const int4* __restrict__ v, int4* __restrict__ gu,
                                                                int4* __restrict__ a, int4* __restrict__ y) {
  const int j = blockIdx.y, e = E_ffn + j;
  int cidx;
  const int kind = zc_kind(j, n_zero, n_copy, cidx);
  const int lo = offsets[e], hi = offsets[e + 1], live = lo + counts[e];
  const int lane = threadIdx.x & 31;
  const int4 zero = make_int4(0, 0, 0, 0);
  for (int r = lo + blockIdx.x * ZC_WARPS + (threadIdx.x >> 5); r < hi; r += gridDim.x * ZC_WARPS) {
    const bool real = r < live;
    for (int c = lane; c < nvecH; c += 32) {
      int4 val = zero;
      if (real && kind == 1) val = Xp[(size_t)r * nvecH + c];
      if (real && kind == 2) val = v[(size_t)cidx * nvecH + c];
      y[(size_t)r * nvecH + c] = val;
    }
    for (int c = lane; c < 2 * nvecF; c += 32) gu[(size_t)r * 2 * nvecF + c] = zero;
    for (int c = lane; c < nvecF; c += 32) a[(size_t)r * nvecF + c] = zero;
  }
}

// Backward rows: dXp[r] = 0 | dy[r] | 0;  dgu[r] = 0.
__global__ void __launch_bounds__(ZC_WARPS * 32) zc_bwd_kernel(const int32_t* __restrict__ offsets,
                                                                const int32_t* __restrict__ counts, int E_ffn, int n_zero,
                                                                int n_copy, int nvecH, int nvecF, const int4* __restrict__ dy,
                                                                int4* __restrict__ dgu, int4* __restrict__ dXp) {
  const int j = blockIdx.y, e = E_ffn + j;
  int cidx;
  const int kind = zc_kind(j, n_zero, n_copy, cidx);
  const int lo = offsets[e], hi = offsets[e + 1], live = lo + counts[e];
  const int lane = threadIdx.x & 31;
  const int4 zero = make_int4(0, 0, 0, 0);
  for (int r = lo + blockIdx.x * ZC_WARPS + (threadIdx.x >> 5); r < hi; r += gridDim.x * ZC_WARPS) {
    for (int c = lane; c < nvecH; c += 32)
      dXp[(size_t)r * nvecH + c] = (r < live && kind == 1) ? dy[(size_t)r * nvecH + c] : zero;
    for (int c = lane; c < 2 * nvecF; c += 32) dgu[(size_t)r * 2 * nvecF + c] = zero;
  }
}

// dv[c, h] = sum over the constant expert's rows of dy[r, h]: one thread per column, rows in ascending order (fp32).
template <typename T>
__global__ void __launch_bounds__(256) zc_dconst_kernel(const int32_t* __restrict__ offsets,
                                                        const int32_t* __restrict__ counts, int e0, int H,
                                                        const T* __restrict__ dy, T* __restrict__ dv) {
  const int c = blockIdx.y, e = e0 + c;
  const int h = blockIdx.x * 256 + threadIdx.x;
  if (h >= H) return;
  const int lo = offsets[e], n = counts[e];
  float acc = 0.f;
  int i = 0;
  for (; i + 4 <= n; i += 4) {
    float x[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) x[u] = to_f(dy[(size_t)(lo + i + u) * H + h]);
#pragma unroll
    for (int u = 0; u < 4; ++u) acc += x[u];
  }
  for (; i < n; ++i) acc += to_f(dy[(size_t)(lo + i) * H + h]);
  dv[(size_t)c * H + h] = from_f<T>(acc);
}

}  // namespace

int32_t zc_forward(const moe_config_t* c, const int32_t* offsets, const int32_t* counts, const void* Xp, const void* zc_const,
                   void* gu, void* a, void* y, cudaStream_t s) {
  const int nz = n_zc(c);
  if (nz == 0) return MOE_OK;
  const size_t es = elem_bytes(c);
  if ((c->H * es) % 16 || (c->F * es) % 16) return MOE_ERR_UNSUPPORTED;
  MOE_LAUNCH(zc_fwd_kernel, dim3(64, (unsigned)nz), ZC_WARPS * 32, 0, s, offsets, counts, e_ffn(c), c->n_zero, c->n_copy,
             (int)(c->H * es / 16), (int)(c->F * es / 16), (const int4*)Xp, (const int4*)zc_const, (int4*)gu, (int4*)a,
             (int4*)y);
  return MOE_OK;
}

int32_t zc_backward(const moe_config_t* c, const int32_t* offsets, const int32_t* counts, const void* dy, void* dgu, void* dXp,
                    void* d_zc_const, cudaStream_t s) {
  const int nz = n_zc(c);
  if (nz == 0) return MOE_OK;
  const size_t es = elem_bytes(c);
  if ((c->H * es) % 16 || (c->F * es) % 16) return MOE_ERR_UNSUPPORTED;
  MOE_LAUNCH(zc_bwd_kernel, dim3(64, (unsigned)nz), ZC_WARPS * 32, 0, s, offsets, counts, e_ffn(c), c->n_zero, c->n_copy,
             (int)(c->H * es / 16), (int)(c->F * es / 16), (const int4*)dy, (int4*)dgu, (int4*)dXp);
  if (c->n_const > 0 && d_zc_const) {
    const dim3 grid((unsigned)ceil_div(c->H, 256), (unsigned)c->n_const);
    const int e0 = c->E - c->n_const;
    if (c->dtype == 0)
      MOE_LAUNCH(zc_dconst_kernel<float>, grid, 256, 0, s, offsets, counts, e0, c->H, (const float*)dy, (float*)d_zc_const);
    else
      MOE_LAUNCH(zc_dconst_kernel<__nv_bfloat16>, grid, 256, 0, s, offsets, counts, e0, c->H, (const __nv_bfloat16*)dy,
                 (__nv_bfloat16*)d_zc_const);
  }
  return MOE_OK;
}

}  // namespace moe
