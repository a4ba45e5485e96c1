// Row movers on the permutation maps: gather (moe_permute), weighted combine (moe_unpermute_combine,
// also the dX reduction) and combine-backward.  SURVEY.md §8c R6/R7/R8.  All HBM-bound: one warp per
// token, 16-byte vector accesses, each source row read once, fixed j order, fp32 accumulation.
#include <algorithm>

#include "common.cuh"

namespace moe {
namespace {

constexpr unsigned FULL = 0xffffffffu;
constexpr int ROW_WARPS = 8;
constexpr int COMBINE_CTAS = 4096; // aim of the combine's grid: about seven waves of 4 resident CTAs per SM

__device__ __forceinline__ int4 ldg_stream(const int4* p) {
  int4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}
__device__ __forceinline__ void stg_stream(int4* p, const int4& v) {
  asm volatile("st.global.L1::no_allocate.v4.s32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z),
               "r"(v.w));
}

// Xp[f2p[t*K+j]] = X[t] for j < K: token-major, the source row is read once and written K times.  The CTAs past the token
// range zero the padding rows of the expert groups instead (pad_blocks = E x PAD_CTAS of them; see zero_pad_rows).
constexpr int PAD_CTAS = 16;       // x ROW_WARPS warps = 128 candidate rows per expert and pass
__device__ __forceinline__ void zero_pad_rows(const int32_t* __restrict__ p2f, const int32_t* __restrict__ offsets, int e, int sub,
                                              int v0, int v1, int nvec, int4* __restrict__ Xp) {
  // the padding rows are the tail of the group (perm_to_flat[r] < 0): one warp per candidate row counted back from its end
  const int lane = threadIdx.x & 31;
  const int begin = offsets[e], end = offsets[e + 1];
  for (int r = end - 1 - (sub * ROW_WARPS + (int)(threadIdx.x >> 5)); r >= begin && p2f[r] < 0; r -= ROW_WARPS * PAD_CTAS) {
    int4* dst = Xp + (size_t)r * nvec;
    for (int v = v0 + lane; v < v1; v += 32) dst[v] = make_int4(0, 0, 0, 0);
  }
}

template <int KT>
__global__ void __launch_bounds__(ROW_WARPS * 32) gather_kernel(const int4* __restrict__ X, int T, int Krt, int nvec,
                                                                 const int32_t* __restrict__ f2p,
                                                                 const int32_t* __restrict__ p2f,
                                                                 const int32_t* __restrict__ offsets, int tok_blocks,
                                                                 int4* __restrict__ Xp) {
  const int K = KT > 0 ? KT : Krt;
  const int lane = threadIdx.x & 31;
  // blockIdx.y = 2 KB column slab of the row: enough CTAs for several waves even when T / 8 is about one wave
  const int v_lo = blockIdx.y * 128, v_hi = min(nvec, (int)(blockIdx.y + 1) * 128);
  if ((int)blockIdx.x >= tok_blocks) {
    const int pb = blockIdx.x - tok_blocks;
    zero_pad_rows(p2f, offsets, pb / PAD_CTAS, pb % PAD_CTAS, v_lo, v_hi, nvec, Xp);
    return;
  }
  const int t = blockIdx.x * ROW_WARPS + (threadIdx.x >> 5);
  if (t >= T) return;
  const int4* src = X + (size_t)t * nvec;
  const int32_t* rows = f2p + (size_t)t * K;
  for (int v0 = v_lo; v0 < v_hi; v0 += 128) {
    int4 buf[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int v = v0 + u * 32 + lane;
      if (v < nvec) buf[u] = ldg_stream(src + v);
    }
#pragma unroll
    for (int j = 0; j < K; ++j) {
      if (rows[j] < 0) continue;                    // empty slot (variable-k routing): no row
      int4* dst = Xp + (size_t)rows[j] * nvec;
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int v = v0 + u * 32 + lane;
        if (v < nvec) stg_stream(dst + v, buf[u]);
      }
    }
  }
}

// The same padding-row zeroing as a kernel of its own (after combine-backward): blockIdx = (expert, sub-range).
__global__ void __launch_bounds__(ROW_WARPS * 32) zero_pad_kernel(const int32_t* __restrict__ p2f,
                                                                   const int32_t* __restrict__ offsets, int nvec,
                                                                   int4* __restrict__ Xp) {
  zero_pad_rows(p2f, offsets, blockIdx.x, blockIdx.y, 0, nvec, nvec, Xp);
}

template <typename T>
struct Vec;
template <>
struct Vec<float> {
  static constexpr int N = 4;
  __device__ static void unpack(const int4& v, float (&f)[4]) {
    f[0] = __int_as_float(v.x); f[1] = __int_as_float(v.y); f[2] = __int_as_float(v.z); f[3] = __int_as_float(v.w);
  }
  __device__ static int4 pack(const float (&f)[4]) {
    return make_int4(__float_as_int(f[0]), __float_as_int(f[1]), __float_as_int(f[2]), __float_as_int(f[3]));
  }
};
template <>
struct Vec<__nv_bfloat16> {
  static constexpr int N = 8;
  __device__ static void unpack(const int4& v, float (&f)[8]) {
    const int w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      f[2 * i] = __int_as_float(w[i] << 16);
      f[2 * i + 1] = __int_as_float(w[i] & 0xffff0000);
    }
  }
  __device__ static int4 pack(const float (&f)[8]) {
    int w[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const __nv_bfloat162 h = __floats2bfloat162_rn(f[2 * i], f[2 * i + 1]);
      w[i] = *reinterpret_cast<const int*>(&h);
    }
    return make_int4(w[0], w[1], w[2], w[3]);
  }
};

// Y[t] = sum_j w[t,j] * y[f2p[t*K+j]]  (+ add0[t]) (+ add1[t])  (+ sum_j dz[t,j] * Wr[idx[t,j]]);  w == NULL -> 1.
// Empty slots (f2p = -1, variable-k routing) contribute nothing.
// K = 8: capped at 40 registers so that 6 CTAs (48 warps) are resident per SM -- the kernel waits on its row loads, and more
// warps in flight moved configs[1] from 71 to 50 us and configs[2] from 135 to 104 us (K = 4 was slower that way).
template <typename T, int KT, bool SLABBED>
__global__ void __launch_bounds__(ROW_WARPS * 32, KT == 8 ? 6 : 1) combine_kernel(const int4* __restrict__ y, const float* __restrict__ w,
                                                                  const int32_t* __restrict__ f2p,
                                                                  const int4* __restrict__ add0,
                                                                  const int4* __restrict__ add1,
                                                                  const float* __restrict__ dz,
                                                                  const int32_t* __restrict__ idx,
                                                                  const int4* __restrict__ Wr, int Tn, int Krt, int nvec,
                                                                  int slab, int4* __restrict__ Y) {
  constexpr int N = Vec<T>::N;
  const int K = KT > 0 ? KT : Krt;
  const int lane = threadIdx.x & 31;
  const int t = blockIdx.x * ROW_WARPS + (threadIdx.x >> 5);
  if (t >= Tn) return;
  const int32_t* rows = f2p + (size_t)t * K;
  // SLABBED: blockIdx.y = column slab of `slab` 16-byte vectors (a multiple of 32); else whole rows
  const int v0 = SLABBED ? (int)blockIdx.y * slab : 0;
  const int v1 = SLABBED ? min(nvec, v0 + slab) : nvec;
  for (int v = v0 + lane; v < v1; v += 32) {
    float acc[N];
#pragma unroll
    for (int i = 0; i < N; ++i) acc[i] = 0.f;
    if (KT > 0) {                       // all K row loads in flight before the first use
      int4 q[KT > 0 ? KT : 1];
#pragma unroll
      for (int j = 0; j < KT; ++j) q[j] = rows[j] >= 0 ? ldg_stream(y + (size_t)rows[j] * nvec + v) : make_int4(0, 0, 0, 0);
#pragma unroll
      for (int j = 0; j < KT; ++j) {
        const float wj = w ? w[(size_t)t * K + j] : 1.0f;
        float f[N];
        Vec<T>::unpack(q[j], f);
#pragma unroll
        for (int i = 0; i < N; ++i) acc[i] = fmaf(wj, f[i], acc[i]);
      }
    } else {
      for (int j = 0; j < K; ++j) {
        if (rows[j] < 0) continue;
        const float wj = w ? w[(size_t)t * K + j] : 1.0f;
        float f[N];
        Vec<T>::unpack(ldg_stream(y + (size_t)rows[j] * nvec + v), f);
#pragma unroll
        for (int i = 0; i < N; ++i) acc[i] = fmaf(wj, f[i], acc[i]);
      }
    }
    if (add0) {
      float f[N];
      Vec<T>::unpack(ldg_stream(add0 + (size_t)t * nvec + v), f);
#pragma unroll
      for (int i = 0; i < N; ++i) acc[i] += f[i];
    }
    if (add1) {
      float f[N];
      Vec<T>::unpack(ldg_stream(add1 + (size_t)t * nvec + v), f);
#pragma unroll
      for (int i = 0; i < N; ++i) acc[i] += f[i];
    }
    if (dz) {
      for (int j = 0; j < K; ++j) {
        const int ej = idx[(size_t)t * K + j];
        if (ej < 0) continue;
        const float d = dz[(size_t)t * K + j];
        float f[N];
        Vec<T>::unpack(__ldg(Wr + (size_t)ej * nvec + v), f);
#pragma unroll
        for (int i = 0; i < N; ++i) acc[i] = fmaf(d, f[i], acc[i]);
      }
    }
    Y[(size_t)t * nvec + v] = Vec<T>::pack(acc);
  }
}

// dy[f2p[t*K+j]] = w[t,j] * dY[t];   dw[t,j] = <dY[t], y[f2p[t*K+j]]>.
// One warp per token; per 16-byte column chunk the K rows of y are loaded together (KT > 0) and the K dot products are
// kept in registers; lane partials are reduced by shuffles in a fixed order at the end.
template <typename T, int KT>
__global__ void __launch_bounds__(ROW_WARPS * 32) combine_bwd_kernel(const int4* __restrict__ dY,
                                                                      const int4* __restrict__ y,
                                                                      const float* __restrict__ w,
                                                                      const int32_t* __restrict__ f2p, int Tn, int Krt,
                                                                      int nvec, int4* __restrict__ dy,
                                                                      float* __restrict__ dw) {
  constexpr int N = Vec<T>::N;
  const int K = KT > 0 ? KT : Krt;
  const int lane = threadIdx.x & 31;
  const int t = blockIdx.x * ROW_WARPS + (threadIdx.x >> 5);
  if (t >= Tn) return;
  if (KT > 0) {
    int r[KT > 0 ? KT : 1];
    float wj[KT > 0 ? KT : 1], dot[KT > 0 ? KT : 1];
#pragma unroll
    for (int j = 0; j < KT; ++j) {
      r[j] = f2p[(size_t)t * K + j];
      wj[j] = w[(size_t)t * K + j];
      dot[j] = 0.f;
    }
    for (int v = lane; v < nvec; v += 32) {
      float g[N];
      Vec<T>::unpack(ldg_stream(dY + (size_t)t * nvec + v), g);
      int4 q[KT > 0 ? KT : 1];
#pragma unroll
      for (int j = 0; j < KT; ++j) q[j] = r[j] >= 0 ? ldg_stream(y + (size_t)r[j] * nvec + v) : make_int4(0, 0, 0, 0);
#pragma unroll
      for (int j = 0; j < KT; ++j) {
        float f[N], o[N];
        Vec<T>::unpack(q[j], f);
#pragma unroll
        for (int i = 0; i < N; ++i) {
          dot[j] = fmaf(g[i], f[i], dot[j]);
          o[i] = wj[j] * g[i];
        }
        if (r[j] >= 0) stg_stream(dy + (size_t)r[j] * nvec + v, Vec<T>::pack(o));   // empty slot: no row, dw = 0
      }
    }
#pragma unroll
    for (int j = 0; j < KT; ++j) {
      float d = dot[j];
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) d += __shfl_xor_sync(FULL, d, off);
      if (lane == 0) dw[(size_t)t * K + j] = d;
    }
  } else {
    for (int j = 0; j < K; ++j) {
      const int r = f2p[(size_t)t * K + j];
      const float wj = w[(size_t)t * K + j];
      float dot = 0.f;
      for (int v = lane; r >= 0 && v < nvec; v += 32) {
        float g[N], f[N], o[N];
        Vec<T>::unpack(__ldg(dY + (size_t)t * nvec + v), g);
        Vec<T>::unpack(ldg_stream(y + (size_t)r * nvec + v), f);
#pragma unroll
        for (int i = 0; i < N; ++i) {
          dot = fmaf(g[i], f[i], dot);
          o[i] = wj * g[i];
        }
        stg_stream(dy + (size_t)r * nvec + v, Vec<T>::pack(o));
      }
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) dot += __shfl_xor_sync(FULL, dot, off);
      if (lane == 0) dw[(size_t)t * K + j] = dot;
    }
  }
}

// dw[p] = sum_k part[k, f2p[p]] in ascending k (deterministic); an empty slot (f2p < 0) gets 0.
__global__ void __launch_bounds__(256) dw_reduce_kernel(const float* __restrict__ part, int nparts, int64_t R,
                                                        const int32_t* __restrict__ f2p, int64_t TK,
                                                        float* __restrict__ dw) {
  const int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
  if (i >= TK) return;
  const int r = f2p[i];
  float s = 0.f;
  if (r >= 0)
    for (int k = 0; k < nparts; ++k) s += part[(int64_t)k * R + r];
  dw[i] = s;
}

}  // namespace

int32_t dw_reduce(const moe_config_t* c, const float* part, int nparts, const int32_t* f2p, float* dw, cudaStream_t s) {
  const int64_t TK = (int64_t)c->T * c->K;
  MOE_LAUNCH(dw_reduce_kernel, (unsigned)ceil_div(TK, 256), 256, 0, s, part, nparts, padded_rows(c), f2p, TK, dw);
  return MOE_OK;
}

int32_t gather_rows(const moe_config_t* c, const void* X, int cols, size_t esz, const int32_t* f2p, const int32_t* p2f,
                    const int32_t* offsets, void* Xp, cudaStream_t s) {
  if ((cols * esz) % 16 != 0) return MOE_ERR_UNSUPPORTED;
  const int nvec = (int)(cols * esz / 16);
  const int tok_blocks = (int)ceil_div(c->T, ROW_WARPS);
  const int pad_blocks = c->row_align > 1 ? c->E * PAD_CTAS : 0;      // padding rows exist only with aligned groups
#define MOE_GATHER(KT)                                                                                              \
  MOE_LAUNCH(gather_kernel<KT>, dim3((unsigned)(tok_blocks + pad_blocks), (unsigned)ceil_div(nvec, 128)), ROW_WARPS * 32, 0, s, \
             (const int4*)X, c->T, c->K, nvec, f2p, p2f, offsets, tok_blocks, (int4*)Xp)
  switch (c->K) {
    case 2: MOE_GATHER(2); break;
    case 4: MOE_GATHER(4); break;
    case 8: MOE_GATHER(8); break;
    default: MOE_GATHER(0); break;
  }
#undef MOE_GATHER
  return MOE_OK;
}

int32_t combine(const moe_config_t* c, const void* y, const float* w, const int32_t* f2p, const void* add0,
                const void* add1, const float* dz, const int32_t* idx, const void* Wr, void* Y, cudaStream_t s) {
  const size_t esz = elem_bytes(c);
  if ((c->H * esz) % 16 != 0) return MOE_ERR_UNSUPPORTED;
  const int nvec = (int)(c->H * esz / 16);
  // Rows are cut into column slabs only when whole rows give fewer than ~3.5 waves of CTAs (4 resident per SM), where the
  // ragged last wave costs more than the split: measured configs[1] (1024 CTAs) 85 -> 70 us, configs[2] (512) 165 -> 133 us
  // with slabs, but configs[4] (2048 CTAs, 5.8 KB rows) 92 -> 108 us, so it keeps whole rows.
  const int64_t base_ctas = ceil_div(c->T, ROW_WARPS);
  const int slabs = base_ctas >= COMBINE_CTAS / 2
                        ? 1 : (int)std::max<int64_t>(1, std::min<int64_t>(ceil_div(nvec, 64), COMBINE_CTAS / base_ctas));
  const int slab = (int)round_up(ceil_div(nvec, slabs), 32);
  const dim3 grid((unsigned)base_ctas, (unsigned)ceil_div(nvec, slab));
#define MOE_COMBINE(TY, KT)                                                                                       \
  do {                                                                                                            \
    if (slabs > 1)                                                                                                \
      MOE_LAUNCH((combine_kernel<TY, KT, true>), grid, ROW_WARPS * 32, 0, s, (const int4*)y, w, f2p, (const int4*)add0,        \
                 (const int4*)add1, dz, idx, (const int4*)Wr, c->T, c->K, nvec, slab, (int4*)Y);                  \
    else                                                                                                          \
      MOE_LAUNCH((combine_kernel<TY, KT, false>), grid, ROW_WARPS * 32, 0, s, (const int4*)y, w, f2p, (const int4*)add0,       \
                 (const int4*)add1, dz, idx, (const int4*)Wr, c->T, c->K, nvec, slab, (int4*)Y);                  \
  } while (0)
  if (c->dtype == 0) {
    MOE_COMBINE(float, 0);
  } else {
    switch (c->K) {
      case 2: MOE_COMBINE(__nv_bfloat16, 2); break;
      case 4: MOE_COMBINE(__nv_bfloat16, 4); break;
      case 8: MOE_COMBINE(__nv_bfloat16, 8); break;
      default: MOE_COMBINE(__nv_bfloat16, 0); break;
    }
  }
#undef MOE_COMBINE
  return MOE_OK;
}

int32_t combine_bwd(const moe_config_t* c, const void* dY, const void* y, const float* w, const int32_t* f2p,
                    const int32_t* p2f, const int32_t* offsets, void* dy, float* dw, cudaStream_t s) {
  const size_t esz = elem_bytes(c);
  if ((c->H * esz) % 16 != 0) return MOE_ERR_UNSUPPORTED;
  const int nvec = (int)(c->H * esz / 16);
  const unsigned grid = (unsigned)ceil_div(c->T, ROW_WARPS);
#define MOE_COMBINE_BWD(TY, KT)                                                                                   \
  MOE_LAUNCH((combine_bwd_kernel<TY, KT>), grid, ROW_WARPS * 32, 0, s, (const int4*)dY, (const int4*)y, w, f2p, c->T, \
             c->K, nvec, (int4*)dy, dw)
  if (c->dtype == 0) {
    MOE_COMBINE_BWD(float, 0);
  } else {
    switch (c->K) {
      case 2: MOE_COMBINE_BWD(__nv_bfloat16, 2); break;
      case 4: MOE_COMBINE_BWD(__nv_bfloat16, 4); break;
      case 8: MOE_COMBINE_BWD(__nv_bfloat16, 8); break;
      default: MOE_COMBINE_BWD(__nv_bfloat16, 0); break;
    }
  }
#undef MOE_COMBINE_BWD
  if (c->row_align > 1)
    MOE_LAUNCH(zero_pad_kernel, dim3((unsigned)c->E, PAD_CTAS), ROW_WARPS * 32, 0, s, p2f, offsets, nvec, (int4*)dy);
  return MOE_OK;
}

}  // namespace moe

extern "C" int32_t moe_permute(const moe_config_t* cfg, const void* X, const int32_t* topk_idx, int32_t* counts,
                               int32_t* offsets, int32_t* perm_to_flat, int32_t* flat_to_perm, void* Xp, void* ws,
                               void* stream) {
  using namespace moe;
  if (!cfg || !topk_idx || !counts || !offsets || !perm_to_flat || !flat_to_perm || !ws) return MOE_ERR_INVALID_ARG;
  MOE_CHECK(validate(cfg));
  if (X && !Xp) return MOE_ERR_INVALID_ARG;
  cudaStream_t s = as_stream(stream);
  const WsLayout L = ws_layout(cfg);
  int32_t* hist = reinterpret_cast<int32_t*>((char*)ws + L.hist);
  int32_t* mtile = reinterpret_cast<int32_t*>((char*)ws + L.tmp);
  MOE_CHECK(build_maps(cfg, topk_idx, counts, offsets, perm_to_flat, flat_to_perm, mtile, hist, s));
  if (X) MOE_CHECK(gather_rows(cfg, X, cfg->H, elem_bytes(cfg), flat_to_perm, perm_to_flat, offsets, Xp, s));
  return MOE_OK;
}

extern "C" int32_t moe_unpermute_combine(const moe_config_t* cfg, const void* y, const float* topk_w,
                                         const int32_t* flat_to_perm, const void* shared_out, void* Y, void* stream) {
  using namespace moe;
  if (!cfg || !y || !topk_w || !flat_to_perm || !Y) return MOE_ERR_INVALID_ARG;
  MOE_CHECK(validate(cfg));
  return combine(cfg, y, topk_w, flat_to_perm, shared_out, nullptr, nullptr, nullptr, nullptr, Y, as_stream(stream));
}
