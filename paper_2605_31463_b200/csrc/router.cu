// Router: logits z = X Wr^T (R1), and the router backward dw -> dz -> dWr (R8).  SURVEY.md §8c.
// dX += dz Wr is folded into the dX combine kernel (rows.cu).
#include <string.h>

#include "gemm_tc.cuh"

namespace moe {
namespace {

constexpr unsigned FULL = 0xffffffffu;

// z[t,e] = sum_h X[t,h] Wr[e,h]; fp32 accumulate, fp32 out.  64x64 tile, 4x4 per thread.
template <typename T>
__global__ void __launch_bounds__(256) logits_kernel(const T* __restrict__ X, const T* __restrict__ Wr, int Tn, int H,
                                                     int E, float* __restrict__ z) {
  __shared__ float sA[16][65];
  __shared__ float sB[16][65];
  const int m0 = blockIdx.x * 64, n0 = blockIdx.y * 64;
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  float acc[4][4] = {};
  for (int k0 = 0; k0 < H; k0 += 16) {
    for (int i = threadIdx.x; i < 1024; i += 256) {
      const int kk = i & 15, mm = i >> 4;
      const int k = k0 + kk;
      sA[kk][mm] = (m0 + mm < Tn && k < H) ? to_f(X[(size_t)(m0 + mm) * H + k]) : 0.f;
      sB[kk][mm] = (n0 + mm < E && k < H) ? to_f(Wr[(size_t)(n0 + mm) * H + k]) : 0.f;
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < 16; ++kk) {
      float a[4], b[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) a[i] = sA[kk][ty * 4 + i];
#pragma unroll
      for (int j = 0; j < 4; ++j) b[j] = sB[kk][tx * 4 + j];
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int m = m0 + ty * 4 + i, n = n0 + tx * 4 + j;
      if (m < Tn && n < E) z[(size_t)m * E + n] = acc[i][j];
    }
}

// dz over the selected experts (renormalised gating, R8):
//   softmax: dz_j = w_j (dw_j - sum_i w_i dw_i / c)
//   sigmoid: S = sum_i s_i + 1e-20; ds_j = c (dw_j / S - sum_i dw_i s_i / S^2); dz_j = ds_j s_j (1 - s_j)
//   no renorm, sigmoid: dz_j = c dw_j s_j (1 - s_j)
// One warp per token, lane j < K.  Also scatters dz to permuted-row order (dzp) for the dWr reduction.
__global__ void __launch_bounds__(128) dz_kernel(const float* __restrict__ z, const int32_t* __restrict__ idx,
                                                 const float* __restrict__ w, const float* __restrict__ dw,
                                                 const int32_t* __restrict__ f2p, int Tn, int E, int K, int score_fn,
                                                 int renorm, float c, float* __restrict__ dz,
                                                 float* __restrict__ dzp) {
  const int lane = threadIdx.x & 31;
  const int t = blockIdx.x * 4 + (threadIdx.x >> 5);
  if (t >= Tn) return;
  const bool act = lane < K;
  const size_t p = (size_t)t * K + lane;
  const float wj = act ? w[p] : 0.f;
  const float dwj = act ? dw[p] : 0.f;
  float out;
  if (score_fn == 0) {
    float inner = wj * dwj;
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) inner += __shfl_xor_sync(FULL, inner, off);
    out = (c != 0.f) ? wj * (dwj - inner / c) : 0.f;
  } else {
    const float zj = act ? z[(size_t)t * E + idx[p]] : 0.f;
    const float sj = act ? 1.0f / (1.0f + expf(-zj)) : 0.f;
    float ds;
    if (renorm) {
      float S = sj, D = dwj * sj;
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) {
        S += __shfl_xor_sync(FULL, S, off);
        D += __shfl_xor_sync(FULL, D, off);
      }
      S += 1e-20f;
      ds = c * (dwj / S - D / (S * S));
    } else {
      ds = c * dwj;
    }
    out = ds * sj * (1.0f - sj);
  }
  if (act) {
    dz[p] = out;
    dzp[f2p[p]] = out;
  }
}

// dWr[e,:] = sum_{i < counts[e]} dzp[off[e]+i] * Xp[off[e]+i,:]   (rows in ascending order, fp32)
template <typename T>
__global__ void __launch_bounds__(256) dwr_kernel(const float* __restrict__ dzp, const T* __restrict__ Xp,
                                                  const int32_t* __restrict__ offsets,
                                                  const int32_t* __restrict__ counts, int H, T* __restrict__ dWr) {
  const int e = blockIdx.x;
  const int h = blockIdx.y * 256 + threadIdx.x;
  if (h >= H) return;
  const int off = offsets[e], cnt = counts[e];
  float acc = 0.f;
  int i = 0;
  for (; i + 4 <= cnt; i += 4) {
    float x[4], d[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      x[u] = to_f(Xp[(size_t)(off + i + u) * H + h]);
      d[u] = dzp[off + i + u];
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) acc = fmaf(d[u], x[u], acc);
  }
  for (; i < cnt; ++i) acc = fmaf(dzp[off + i], to_f(Xp[(size_t)(off + i) * H + h]), acc);
  dWr[(size_t)e * H + h] = from_f<T>(acc);
}


// dWr on 128-row-aligned groups, in two deterministic passes that do not care how skewed the expert load is:
//  pass 1: one CTA per (128-row tile, 256-column slab): part[tile, h] = sum over the tile's live rows of dzp[r] * Xp[r, h]
//          (8 warps x 16 rows, 8 columns per lane with 16-byte loads, fixed-order shared-memory reduction);
//  pass 2: dWr[e, h] = sum of the expert's tile partials in ascending tile order.
__global__ void __launch_bounds__(256) dwr_tile_kernel(const float* __restrict__ dzp, const uint4* __restrict__ Xp,
                                                       const int32_t* __restrict__ mtile,
                                                       const int32_t* __restrict__ offsets,
                                                       const int32_t* __restrict__ counts, int H,
                                                       float* __restrict__ part) {
  __shared__ float red[8][256];
  const int tile = blockIdx.x;
  if (tile >= mtile[0]) return;
  const int e = mtile[1 + tile];
  const int live_end = offsets[e] + counts[e];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int col = blockIdx.y * 256 + lane * 8;
  float acc[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) acc[i] = 0.f;
  if (col < H) {
    const int r0 = tile * 128 + warp * 16;
#pragma unroll 4
    for (int i = 0; i < 16; ++i) {
      const int r = r0 + i;
      if (r >= live_end) break;
      const float d = dzp[r];
      const uint4 v = __ldg(Xp + ((size_t)r * H + col) / 8);
      const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        acc[2 * k] = fmaf(d, __uint_as_float(w[k] << 16), acc[2 * k]);
        acc[2 * k + 1] = fmaf(d, __uint_as_float(w[k] & 0xffff0000u), acc[2 * k + 1]);
      }
    }
  }
#pragma unroll
  for (int i = 0; i < 8; ++i) red[warp][lane * 8 + i] = acc[i];
  __syncthreads();
  const int h = blockIdx.y * 256 + threadIdx.x;
  if (h < H) {
    float s = 0.f;
#pragma unroll
    for (int w = 0; w < 8; ++w) s += red[w][threadIdx.x];
    part[(size_t)tile * H + h] = s;
  }
}

__global__ void __launch_bounds__(256) dwr_reduce_kernel(const float* __restrict__ part,
                                                         const int32_t* __restrict__ offsets, int H,
                                                         __nv_bfloat16* __restrict__ dWr) {
  const int e = blockIdx.x;
  const int h = blockIdx.y * 256 + threadIdx.x;
  if (h >= H) return;
  const int t0 = offsets[e] / 128, t1 = offsets[e + 1] / 128;
  float s = 0.f;
  for (int t = t0; t < t1; ++t) s += part[(size_t)t * H + h];
  dWr[(size_t)e * H + h] = __float2bfloat16_rn(s);
}

}  // namespace

int32_t router_logits(const moe_config_t* c, const void* X, const void* Wr, float* z, cudaStream_t s) {
  if (c->dtype != 0 && c->H % 64 == 0 && c->E % 4 == 0) {   // bf16: tcgen05 GEMM with fp32 output (one group of T rows)
    TcCall t;
    memset(&t, 0, sizeof(t));
    t.mode = TC_FWD_F32; t.E = 1; t.rows_cap = c->T; t.A = X; t.lda = c->H; t.B0 = Wr; t.b_rows = c->E; t.b_cols = c->H;
    t.N = c->E; t.Kd = c->H; t.out0 = z; t.ld0 = c->E;
    const int32_t st = tc_gemm(t, s);
    if (st != MOE_ERR_UNSUPPORTED) return st;
  }
  dim3 grid((unsigned)ceil_div(c->T, 64), (unsigned)ceil_div(c->E, 64));
  if (c->dtype == 0)
    MOE_LAUNCH(logits_kernel<float>, grid, 256, 0, s, (const float*)X, (const float*)Wr, c->T, c->H, c->E, z);
  else
    MOE_LAUNCH(logits_kernel<__nv_bfloat16>, grid, 256, 0, s, (const __nv_bfloat16*)X, (const __nv_bfloat16*)Wr, c->T,
               c->H, c->E, z);
  return MOE_OK;
}

int32_t router_bwd(const moe_config_t* c, const float* z, const int32_t* idx, const float* w, const float* dw,
                   const int32_t* f2p, const int32_t* offsets, const int32_t* counts, const int32_t* mtile,
                   const void* Xp, float* dz, float* dzp, float* part, void* dWr, cudaStream_t s) {
  if (c->score_fn == 0 && !c->renorm) return MOE_ERR_UNSUPPORTED;  // dense dz: not on any config's path
  MOE_LAUNCH(dz_kernel, (unsigned)ceil_div(c->T, 4), 128, 0, s, z, idx, w, dw, f2p, c->T, c->E, c->K, c->score_fn,
             c->renorm, c->routed_scale, dz, dzp);
  if (dWr && c->dtype != 0 && c->row_align % 128 == 0 && c->H % 8 == 0 && mtile && part) {
    const unsigned slabs = (unsigned)ceil_div(c->H, 256);
    MOE_LAUNCH(dwr_tile_kernel, dim3((unsigned)(padded_rows(c) / 128), slabs), 256, 0, s, dzp, (const uint4*)Xp, mtile,
               offsets, counts, c->H, part);
    MOE_LAUNCH(dwr_reduce_kernel, dim3((unsigned)c->E, slabs), 256, 0, s, part, offsets, c->H, (__nv_bfloat16*)dWr);
  } else if (dWr) {
    dim3 grid((unsigned)c->E, (unsigned)ceil_div(c->H, 256));
    if (c->dtype == 0)
      MOE_LAUNCH(dwr_kernel<float>, grid, 256, 0, s, dzp, (const float*)Xp, offsets, counts, c->H, (float*)dWr);
    else
      MOE_LAUNCH(dwr_kernel<__nv_bfloat16>, grid, 256, 0, s, dzp, (const __nv_bfloat16*)Xp, offsets, counts, c->H,
                 (__nv_bfloat16*)dWr);
  }
  return MOE_OK;
}

}  // namespace moe
