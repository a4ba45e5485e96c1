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
  const size_t p = (size_t)t * K + lane;
  const bool act = lane < K && idx[p] >= 0;        // an empty slot (variable-k routing) has no gradient and no row
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
  } else if (lane < K) {
    dz[p] = 0.f;
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
                                                       const int32_t* __restrict__ p2f, int K, int kshift,
                                                       float* __restrict__ part) {
  // p2f != nullptr: Xp is the TOKEN-major X [T,H] and permuted row r reads token row p2f[r] / K -- X (T H bytes) stays in
  // L2 across the K experts that touch each row, the row-grouped copy (K times larger) would stream from HBM
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
      // live rows only: p2f[r] >= 0; kshift >= 0: K = 2^kshift (no integer division per row and thread)
      const size_t src = p2f ? (size_t)(kshift >= 0 ? p2f[r] >> kshift : p2f[r] / K) : (size_t)r;
      const uint4 v = __ldg(Xp + (src * H + col) / 8);
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

// ---------------------------------------------------------------------------------------------------------
// A1..A2 auxiliary load-balancing loss: P_e = mean_t p[t,e], f_e, L = coef E sum eta f P
// ---------------------------------------------------------------------------------------------------------
// p over ALL experts for one token held by a warp (lane l owns experts l, l+32, ...): softmax(z), or s / sum s for
// sigmoid gates.  Also returns the per-lane derivative factor d_e with dp-ish meaning used by the backward:
// softmax: d = p;  sigmoid: d = s (1 - s) / S.
template <int VPT>
__device__ __forceinline__ void token_probs(const float* __restrict__ zrow, int E, int lane, bool softmax, float (&p)[VPT],
                                            float (&d)[VPT]) {
  float zr[VPT];
  float m = -INFINITY;
#pragma unroll
  for (int s = 0; s < VPT; ++s) {
    const int e = s * 32 + lane;
    zr[s] = e < E ? zrow[e] : -INFINITY;
    m = fmaxf(m, zr[s]);
  }
  float sum = 0.f;
  if (softmax) {
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) m = fmaxf(m, __shfl_xor_sync(FULL, m, off));
#pragma unroll
    for (int s = 0; s < VPT; ++s) {
      p[s] = (s * 32 + lane < E) ? expf(zr[s] - m) : 0.f;
      sum += p[s];
    }
  } else {
#pragma unroll
    for (int s = 0; s < VPT; ++s) {
      p[s] = (s * 32 + lane < E) ? 1.0f / (1.0f + expf(-zr[s])) : 0.f;
      sum += p[s];
    }
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) sum += __shfl_xor_sync(FULL, sum, off);
  const float inv = 1.0f / sum;
#pragma unroll
  for (int s = 0; s < VPT; ++s) {
    const float raw = p[s];
    p[s] = raw * inv;
    d[s] = softmax ? p[s] : raw * (1.0f - raw) * inv;
  }
}

// part[cta, e] = sum over the CTA's AUX_TOKENS_PER_CTA tokens of p[t, e]  (fixed order: warp w owns tokens w, w+8, ...;
// the 8 warps' sums are added in warp order), so P is deterministic.
template <int VPT>
__global__ void __launch_bounds__(256) aux_part_kernel(const float* __restrict__ z, int Tn, int E, int softmax,
                                                       float* __restrict__ part) {
  extern __shared__ float red[];   // [8][E]
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  float acc[VPT];
#pragma unroll
  for (int s = 0; s < VPT; ++s) acc[s] = 0.f;
  const int t0 = blockIdx.x * AUX_TOKENS_PER_CTA;
  for (int i = warp; i < AUX_TOKENS_PER_CTA; i += 8) {
    const int t = t0 + i;
    if (t >= Tn) break;
    float p[VPT], d[VPT];
    token_probs<VPT>(z + (size_t)t * E, E, lane, softmax != 0, p, d);
#pragma unroll
    for (int s = 0; s < VPT; ++s) acc[s] += p[s];
  }
#pragma unroll
  for (int s = 0; s < VPT; ++s)
    if (s * 32 + lane < E) red[warp * E + s * 32 + lane] = acc[s];
  __syncthreads();
  for (int e = threadIdx.x; e < E; e += blockDim.x) {
    float sum = 0.f;
#pragma unroll
    for (int w = 0; w < 8; ++w) sum += red[w * E + e];
    part[(size_t)blockIdx.x * E + e] = sum;
  }
}

// One CTA: P_e = (sum of the partials in CTA order) / T;  f_e = f_global[e] or counts[e] / sum counts;
// L = coef * E * sum_e eta_e f_e P_e (summed in expert order by thread 0 after a fixed-order block reduction).
__global__ void __launch_bounds__(1024) aux_final_kernel(const float* __restrict__ part, int nparts, int Tn, int E, int nzc,
                                                         float coef, float zc_weight, const int32_t* __restrict__ counts,
                                                         const float* __restrict__ f_global, float* __restrict__ aux_f,
                                                         float* __restrict__ aux_P, float* __restrict__ aux_loss,
                                                         float* __restrict__ loss_out) {
  __shared__ float sh[1024];
  __shared__ int total_sh;
  const int e = threadIdx.x;
  int cnt = (e < E && !f_global) ? counts[e] : 0;
  // total assignments (integer, exact)
  int v = cnt;
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(FULL, v, off);
  __shared__ int wsum[32];
  if ((e & 31) == 0) wsum[e >> 5] = v;
  __syncthreads();
  if (e == 0) {
    int tot = 0;
    for (int w = 0; w < 32; ++w) tot += wsum[w];
    total_sh = tot;
  }
  __syncthreads();
  float term = 0.f;
  if (e < E) {
    float P = 0.f;
    for (int i = 0; i < nparts; ++i) P += part[(size_t)i * E + e];
    P /= (float)Tn;
    const float f = f_global ? f_global[e] : (float)cnt / (float)max(total_sh, 1);
    aux_f[e] = f;
    aux_P[e] = P;
    term = (e >= E - nzc ? zc_weight : 1.0f) * f * P;
  }
  sh[e] = term;
  __syncthreads();
  if (e == 0) {
    float sum = 0.f;
    for (int i = 0; i < E; ++i) sum += sh[i];
    const float L = coef * (float)E * sum;
    aux_loss[0] = L;
    if (loss_out) loss_out[0] = L;
  }
}

// ---------------------------------------------------------------------------------------------------------
// dense router backward: dz over ALL experts (A3, softmax without renormalisation, V2)
// ---------------------------------------------------------------------------------------------------------
// One warp per token.  dzd[t, :] (fp32) = main term (R8, confined to the selected experts except for softmax without
// renorm) + balance term (A3);  dzb = its bf16 copy, row pitch Ep (zero beyond E);  dz_sel[t, j] = dzd[t, idx[t, j]].
template <int VPT, typename TB>
__global__ void __launch_bounds__(128) dz_dense_kernel(const float* __restrict__ z, const int32_t* __restrict__ idx,
                                                       const float* __restrict__ w, const float* __restrict__ dw,
                                                       const float* __restrict__ aux_f, int Tn, int E, int Ep, int K,
                                                       int score_fn, int renorm, int route_mode, float c, float aux_c,
                                                       int nzc, float zc_weight, float* __restrict__ dz_sel,
                                                       float* __restrict__ dzd, TB* __restrict__ dzb) {
  const int lane = threadIdx.x & 31;
  const int t = blockIdx.x * 4 + (threadIdx.x >> 5);
  if (t >= Tn) return;
  const bool softmax = score_fn == 0 && route_mode == 0;
  float p[VPT], d[VPT], out[VPT];
  token_probs<VPT>(z + (size_t)t * E, E, lane, softmax, p, d);
#pragma unroll
  for (int s = 0; s < VPT; ++s) out[s] = 0.f;
  // ---- A3: (coef E / T) d_e (g_e - sum_e' g_e' p_e'),  g = eta * f ----
  if (aux_f != nullptr && aux_c != 0.f) {
    float g[VPT], inner = 0.f;
#pragma unroll
    for (int s = 0; s < VPT; ++s) {
      const int e = s * 32 + lane;
      g[s] = e < E ? (e >= E - nzc ? zc_weight : 1.0f) * aux_f[e] : 0.f;
      inner += g[s] * p[s];
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) inner += __shfl_xor_sync(FULL, inner, off);
#pragma unroll
    for (int s = 0; s < VPT; ++s) out[s] = aux_c * d[s] * (g[s] - inner);
  }
  // ---- R8 main term on the selected experts (lane j < K holds slot j) ----
  const size_t q = (size_t)t * K + lane;
  const int ej = lane < K ? idx[q] : -1;
  const bool act = ej >= 0;
  const float wj = act ? w[q] : 0.f, dwj = act ? dw[q] : 0.f;
  float val;
  if (softmax) {
    float inner = wj * dwj;
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) inner += __shfl_xor_sync(FULL, inner, off);
    if (renorm) {
      val = (c != 0.f) ? wj * (dwj - inner / c) : 0.f;
    } else {
      val = wj * dwj;                                   // + the dense part -p_e * sum_i w_i dw_i below
#pragma unroll
      for (int s = 0; s < VPT; ++s) out[s] -= p[s] * inner;
    }
  } else {
    const float zj = act ? z[(size_t)t * E + ej] : 0.f;
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
    val = ds * sj * (1.0f - sj);
  }
  // scatter the K slot values to the lanes that own those experts (fixed slot order)
  for (int j = 0; j < K; ++j) {
    const int e = __shfl_sync(FULL, ej, j);
    const float vj = __shfl_sync(FULL, val, j);
    if (e < 0) continue;
#pragma unroll
    for (int s = 0; s < VPT; ++s)
      if (s == (e >> 5) && lane == (e & 31)) out[s] += vj;
  }
  // gather the final values of the selected experts back to their slots
  float mine = 0.f;
  for (int j = 0; j < K; ++j) {
    const int e = __shfl_sync(FULL, ej, j);
    float vv = 0.f;
#pragma unroll
    for (int s = 0; s < VPT; ++s)
      if (e >= 0 && s == (e >> 5)) vv = out[s];
    vv = __shfl_sync(FULL, vv, e >= 0 ? (e & 31) : 0);
    if (lane == j) mine = e >= 0 ? vv : 0.f;
  }
  if (lane < K) dz_sel[q] = mine;
#pragma unroll
  for (int s = 0; s < VPT; ++s) {
    const int e = s * 32 + lane;
    if (e < E) dzd[(size_t)t * E + e] = out[s];
    if (dzb != nullptr && e < Ep) dzb[(size_t)t * Ep + e] = from_f<TB>(e < E ? out[s] : 0.f);
  }
}

}  // namespace

int32_t aux_forward(const moe_config_t* c, const float* z, const int32_t* counts, const float* f_global, float* part,
                    float* aux_f, float* aux_P, float* aux_loss, float* loss_out, cudaStream_t s) {
  if (c->E > 1024) return MOE_ERR_UNSUPPORTED;
  const int nparts = (int)ceil_div(c->T, AUX_TOKENS_PER_CTA);
  const int softmax = (c->score_fn == 0 && c->route_mode == 0) ? 1 : 0;
  const size_t smem = (size_t)8 * c->E * sizeof(float);
  const int vpt = (int)ceil_div(c->E, 32);
#define MOE_AUX(V) MOE_LAUNCH(aux_part_kernel<V>, nparts, 256, smem, s, z, c->T, c->E, softmax, part)
  if (vpt <= 1) MOE_AUX(1); else if (vpt <= 2) MOE_AUX(2); else if (vpt <= 4) MOE_AUX(4); else if (vpt <= 8) MOE_AUX(8);
  else if (vpt <= 16) MOE_AUX(16); else MOE_AUX(32);
#undef MOE_AUX
  MOE_LAUNCH(aux_final_kernel, 1, 1024, 0, s, part, nparts, c->T, c->E, n_zc(c), c->aux_coef, c->aux_zc_weight, counts,
             f_global, aux_f, aux_P, aux_loss, loss_out);
  return MOE_OK;
}

int32_t router_bwd_dense(const moe_config_t* c, const float* z, const int32_t* idx, const float* w, const float* dw,
                         const float* aux_f, const void* X, const void* Wr, const int32_t* off_one, float* dz_sel,
                         float* dzd, void* dzb, void* dWr, void* dXr, cudaStream_t s) {
  if (c->E > 1024 || c->K > 32) return MOE_ERR_UNSUPPORTED;
  const int E = c->E, Ep = (E + 63) / 64 * 64, vpt = (int)ceil_div(Ep, 32);
  const float aux_c = c->aux_coef * (float)E / (float)c->T;
  const unsigned grid = (unsigned)ceil_div(c->T, 4);
  const bool bf = c->dtype != 0;
#define MOE_DZD(V)                                                                                                          do {                                                                                                                        if (bf) MOE_LAUNCH((dz_dense_kernel<V, __nv_bfloat16>), grid, 128, 0, s, z, idx, w, dw, aux_f, c->T, E, Ep, c->K,                             c->score_fn, c->renorm, c->route_mode, c->routed_scale, aux_c, n_zc(c), c->aux_zc_weight, dz_sel,                         dzd, (__nv_bfloat16*)dzb);                                                                             else MOE_LAUNCH((dz_dense_kernel<V, float>), grid, 128, 0, s, z, idx, w, dw, aux_f, c->T, E, Ep, c->K, c->score_fn,                        c->renorm, c->route_mode, c->routed_scale, aux_c, n_zc(c), c->aux_zc_weight, dz_sel, dzd,                                 (float*)nullptr);                                                                                       } while (0)
  if (vpt <= 2) MOE_DZD(2); else if (vpt <= 4) MOE_DZD(4); else if (vpt <= 8) MOE_DZD(8); else if (vpt <= 16) MOE_DZD(16);
  else MOE_DZD(32);
#undef MOE_DZD
  // dWr[e, h] = sum_t dz[t, e] X[t, h];  dXr[t, h] = sum_e dz[t, e] Wr[e, h]: one group of T rows
  const bool tc = bf && c->H % 64 == 0 && E % 64 == 0;
  if (tc) {
    TcCall g;
    if (dWr) {
      memset(&g, 0, sizeof(g));
      g.mode = TC_WGRAD; g.opt_pair = c->opt_pair; g.E = 1; g.rows_cap = c->T; g.A = dzb; g.lda = Ep; g.M = E; g.A2 = X; g.lda2 = c->H; g.N = c->H;
      g.out0 = dWr; g.ld0 = c->H;
      MOE_CHECK(tc_gemm(g, s));
    }
    memset(&g, 0, sizeof(g));
    g.mode = TC_DGRAD; g.opt_pair = c->opt_pair; g.E = 1; g.rows_cap = c->T; g.A = dzb; g.lda = Ep; g.B0 = Wr; g.b_rows = E; g.b_cols = c->H;
    g.N = c->H; g.out0 = dXr; g.ld0 = c->H;
    return tc_gemm(g, s);
  }
  // CUDA-core path (fp32, or shapes the tensor-core kernels do not take): dz in the activation type, one group {0, T}
  const void* dzc = bf ? (const void*)dzb : (const void*)dzd;
  const int lddz = bf ? Ep : E;
  if (dWr) MOE_CHECK(simt_grouped_gemm(2, c->dtype, 1, E, c->H, X, c->H, nullptr, dzc, lddz, off_one, dWr, 0, c->T, 0, s));
  return simt_grouped_gemm(1, c->dtype, 1, E, c->H, nullptr, 0, Wr, dzc, lddz, off_one, dXr, c->H, c->T, 0, s);
}

int32_t router_logits(const moe_config_t* c, const void* X, const void* Wr, float* z, cudaStream_t s) {
  if (c->dtype != 0 && c->H % 64 == 0 && c->E % 4 == 0) {   // bf16: tcgen05 GEMM with fp32 output (one group of T rows)
    TcCall t;
    memset(&t, 0, sizeof(t));
    t.mode = TC_FWD_F32; t.opt_pair = c->opt_pair; t.E = 1; t.rows_cap = c->T; t.A = X; t.lda = c->H; t.B0 = Wr; t.b_rows = c->E; t.b_cols = c->H;
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
                   const void* Xp, const void* X, const int32_t* p2f, float* dz, float* dzp, float* part, void* dWr,
                   cudaStream_t s) {
  if (c->score_fn == 0 && !c->renorm) return MOE_ERR_UNSUPPORTED;  // dense dz: not on any config's path
  MOE_LAUNCH(dz_kernel, (unsigned)ceil_div(c->T, 4), 128, 0, s, z, idx, w, dw, f2p, c->T, c->E, c->K, c->score_fn,
             c->renorm, c->routed_scale, dz, dzp);
  if (dWr && c->dtype != 0 && c->row_align % 128 == 0 && c->H % 8 == 0 && mtile && part) {
    const unsigned slabs = (unsigned)ceil_div(c->H, 256);
    const bool tok = X != nullptr && p2f != nullptr;     // read the token-major X through the map
    int kshift = -1;
    for (int sh = 0; sh < 31; ++sh)
      if ((1 << sh) == c->K) kshift = sh;
    MOE_LAUNCH(dwr_tile_kernel, dim3((unsigned)(padded_rows(c) / 128), slabs), 256, 0, s, dzp, (const uint4*)(tok ? X : Xp),
               mtile, offsets, counts, c->H, tok ? p2f : nullptr, c->K, kshift, part);
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
