// moe_route: top-k gating from fp32 logits.
// One warp per token; lane l holds experts l, l+32, ... in registers; K rounds of warp arg-max by
// shuffle with the (key desc, index asc) order, so ties go to the lower expert index.
#include <math.h>

#include "common.cuh"

namespace moe {
namespace {

constexpr unsigned FULL = 0xffffffffu;

struct RouteParams {
  int T, E, K, n_group, topk_group, score_fn, group_score, renorm, has_bias, route_mode;
  float routed_scale;
};

template <int VPT>
__global__ void __launch_bounds__(128) route_kernel(RouteParams p, const float* __restrict__ logits,
                                                    const float* __restrict__ bias,
                                                    const float* __restrict__ threshold, int32_t* __restrict__ topk_idx,
                                                    float* __restrict__ topk_w, int32_t* __restrict__ idx_copy,
                                                    float* __restrict__ w_copy) {
  const int lane = threadIdx.x & 31;
  const int t = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (t >= p.T) return;
  const float NEG = -INFINITY;
  const float* zrow = logits + (size_t)t * p.E;

  float z[VPT], key[VPT];
#pragma unroll
  for (int s = 0; s < VPT; ++s) {
    const int e = s * 32 + lane;
    if (e < p.E) {
      const float zv = zrow[e];
      z[s] = zv;
      float k;
      if (p.score_fn == 0) {
        k = zv;
      } else {
        // the (integer) selection is taken on fp32(sigmoid evaluated in fp64) + b, one fp32 add (R2)
        k = (float)(1.0 / (1.0 + exp(-(double)zv)));
      }
      if (p.has_bias) k = k + bias[e];
      key[s] = k;
    } else {
      z[s] = NEG;
      key[s] = NEG;
    }
  }

  // ---- R3 group-limited selection ----
  if (p.n_group > 1 && p.topk_group < p.n_group) {
    const int per = p.E / p.n_group;
    float gscore = NEG;  // lane g holds the score of group g
    for (int g = 0; g < p.n_group; ++g) {
      float m1 = NEG, m2 = NEG;
#pragma unroll
      for (int s = 0; s < VPT; ++s) {
        const int e = s * 32 + lane;
        if (e < p.E && e / per == g) {
          const float v = key[s];
          if (v > m1) { m2 = m1; m1 = v; } else if (v > m2) { m2 = v; }
        }
      }
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) {
        const float o1 = __shfl_xor_sync(FULL, m1, off);
        const float o2 = __shfl_xor_sync(FULL, m2, off);
        const float n1 = fmaxf(m1, o1);
        const float n2 = fmaxf(fminf(m1, o1), fmaxf(m2, o2));
        m1 = n1; m2 = n2;
      }
      const float sc = (p.group_score == 1 && per > 1) ? (m1 + m2) : m1;
      if (lane == g) gscore = sc;
    }
    unsigned keep = 0;
    for (int r = 0; r < p.topk_group; ++r) {
      const bool avail = lane < p.n_group && !((keep >> lane) & 1u);
      float v = avail ? gscore : NEG;
      int gi = avail ? lane : 0x7fffffff;
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) {
        const float ov = __shfl_xor_sync(FULL, v, off);
        const int og = __shfl_xor_sync(FULL, gi, off);
        const bool take = (og != 0x7fffffff) && (gi == 0x7fffffff || ov > v || (ov == v && og < gi));
        if (take) { v = ov; gi = og; }
      }
      keep |= 1u << gi;
    }
#pragma unroll
    for (int s = 0; s < VPT; ++s) {
      const int e = s * 32 + lane;
      if (e < p.E && !((keep >> (e / per)) & 1u)) key[s] = NEG;
    }
  }

  // ---- V1 threshold gating: only experts whose gate exceeds their threshold stay selectable; the
  // number of filled slots is min(K, #active), or 1 (the best gate) when no expert admits the token ----
  int n_fill = p.K;
  if (p.route_mode == 1) {
    int n_act = 0;
    float masked[VPT];
#pragma unroll
    for (int s = 0; s < VPT; ++s) {
      const int e = s * 32 + lane;
      const bool a = e < p.E && key[s] > threshold[e];
      masked[s] = a ? key[s] : NEG;
      n_act += __popc(__ballot_sync(FULL, a));
    }
    if (n_act > 0) {
#pragma unroll
      for (int s = 0; s < VPT; ++s) key[s] = masked[s];
    }
    n_fill = n_act == 0 ? 1 : min(n_act, p.K);
  }

  // ---- R4 top-k: K rounds of arg-max, ties -> lower expert index ----
  // Keys are mapped to order-preserving unsigned integers (-0 folded into +0 first, so equal floats stay equal);
  // a round is two hardware warp reductions: redux.max of the lanes' best keys, then redux.min of the expert
  // indices that hold that key -- exactly the (key desc, index asc) order of the oracle's arg-max.
  uint32_t ukey[VPT];
#pragma unroll
  for (int s = 0; s < VPT; ++s) {
    const uint32_t u = __float_as_uint(key[s] + 0.0f);
    ukey[s] = (u & 0x80000000u) ? ~u : (u | 0x80000000u);
    if (s * 32 + lane >= p.E) ukey[s] = 0u;          // below every real key (-inf maps to 0x007fffff)
  }
  int sel_e = 0;
  float sel_z = 0.f;
  for (int j = 0; j < p.K; ++j) {
    uint32_t best = 0u;
    int be = 0x7fffffff;
#pragma unroll
    for (int s = 0; s < VPT; ++s)
      if (ukey[s] > best) { best = ukey[s]; be = s * 32 + lane; }     // strict >: the lower slot wins a tie inside the lane
    const uint32_t m = __reduce_max_sync(FULL, best);
    const int e = (int)__reduce_min_sync(FULL, (best == m && be != 0x7fffffff) ? (unsigned)be : 0x7fffffffu);
    float zsel = 0.f;
#pragma unroll
    for (int s = 0; s < VPT; ++s)
      if (s == (e >> 5)) {
        zsel = z[s];
        if (lane == (e & 31)) ukey[s] = 0u;           // taken
      }
    zsel = __shfl_sync(FULL, zsel, e & 31);
    if (lane == j) { sel_e = e; sel_z = zsel; }
  }

  // ---- R5 gating weights (fp32); slots >= n_fill are empty (idx -1, weight 0) ----
  const bool act = lane < n_fill;
  float wj;
  if (p.score_fn == 0) {
    float m, den;
    if (p.renorm) {
      m = act ? sel_z : NEG;
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) m = fmaxf(m, __shfl_xor_sync(FULL, m, off));
      den = act ? expf(sel_z - m) : 0.f;
    } else {
      m = NEG;
#pragma unroll
      for (int s = 0; s < VPT; ++s) m = fmaxf(m, z[s]);
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) m = fmaxf(m, __shfl_xor_sync(FULL, m, off));
      den = 0.f;
#pragma unroll
      for (int s = 0; s < VPT; ++s)
        if (s * 32 + lane < p.E) den += expf(z[s] - m);
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) den += __shfl_xor_sync(FULL, den, off);
    wj = p.routed_scale * (expf(sel_z - m) / den);
  } else {
    const float sj = 1.0f / (1.0f + expf(-sel_z));
    if (p.renorm) {
      float sum = act ? sj : 0.f;
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) sum += __shfl_xor_sync(FULL, sum, off);
      wj = p.routed_scale * (sj / (sum + 1e-20f));
    } else {
      wj = p.routed_scale * sj;
    }
  }
  if (lane < p.K) {
    if (!act) { sel_e = -1; wj = 0.f; }
    topk_idx[(size_t)t * p.K + lane] = sel_e;
    topk_w[(size_t)t * p.K + lane] = wj;
    if (idx_copy) {                                   // the copy moe_layer_fwd keeps in ctx for the backward
      idx_copy[(size_t)t * p.K + lane] = sel_e;
      w_copy[(size_t)t * p.K + lane] = wj;
    }
  }
}

}  // namespace

}  // namespace moe

namespace moe {
int32_t route_impl(const moe_config_t* cfg, const float* logits, const float* bias, const float* threshold,
                   int32_t* topk_idx, float* topk_w, int32_t* idx_copy, float* w_copy, void* stream) {
  if (!cfg || !logits || !topk_idx || !topk_w) return MOE_ERR_INVALID_ARG;
  MOE_CHECK(validate(cfg));
  if (cfg->has_bias && !bias) return MOE_ERR_INVALID_ARG;
  if (cfg->route_mode == 1 && !threshold) return MOE_ERR_INVALID_ARG;
  if (cfg->E > 1024 || cfg->K > 32 || cfg->n_group > 32) return MOE_ERR_UNSUPPORTED;
  RouteParams p{cfg->T, cfg->E, cfg->K, cfg->n_group, cfg->topk_group, cfg->score_fn, cfg->group_score,
                cfg->renorm, cfg->has_bias, cfg->route_mode, cfg->routed_scale};
  const int warps = 4;
  dim3 grid((unsigned)ceil_div(cfg->T, warps)), block(warps * 32);
  cudaStream_t s = as_stream(stream);
  const int vpt = (int)ceil_div(cfg->E, 32);
  if (vpt <= 1) MOE_LAUNCH(route_kernel<1>, grid, block, 0, s, p, logits, bias, threshold, topk_idx, topk_w, idx_copy, w_copy);
  else if (vpt <= 2) MOE_LAUNCH(route_kernel<2>, grid, block, 0, s, p, logits, bias, threshold, topk_idx, topk_w, idx_copy, w_copy);
  else if (vpt <= 4) MOE_LAUNCH(route_kernel<4>, grid, block, 0, s, p, logits, bias, threshold, topk_idx, topk_w, idx_copy, w_copy);
  else if (vpt <= 8) MOE_LAUNCH(route_kernel<8>, grid, block, 0, s, p, logits, bias, threshold, topk_idx, topk_w, idx_copy, w_copy);
  else if (vpt <= 16) MOE_LAUNCH(route_kernel<16>, grid, block, 0, s, p, logits, bias, threshold, topk_idx, topk_w, idx_copy, w_copy);
  else MOE_LAUNCH(route_kernel<32>, grid, block, 0, s, p, logits, bias, threshold, topk_idx, topk_w, idx_copy, w_copy);
  return MOE_OK;
}
}  // namespace moe

extern "C" int32_t moe_route(const moe_config_t* cfg, const float* logits, const float* bias, int32_t* topk_idx,
                             float* topk_w, void* stream) {
  if (cfg && cfg->route_mode != 0) return MOE_ERR_INVALID_ARG;   // thresholds go through moe_route_threshold
  return moe::route_impl(cfg, logits, bias, nullptr, topk_idx, topk_w, nullptr, nullptr, stream);
}

extern "C" int32_t moe_route_threshold(const moe_config_t* cfg, const float* logits, const float* threshold,
                                       int32_t* topk_idx, float* topk_w, void* stream) {
  if (!cfg || cfg->route_mode != 1 || !threshold) return MOE_ERR_INVALID_ARG;
  return moe::route_impl(cfg, logits, nullptr, threshold, topk_idx, topk_w, nullptr, nullptr, stream);
}
