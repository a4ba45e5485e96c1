// Shared host/device helpers of libmoe_b200 (sm_100a only).  Not part of the public ABI.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/moe_b200.h"

namespace moe {

extern long long g_launches;  // kernels launched since load (moe_launch_count)

// Stage timing (moe_profile_*): a mark attributes the stream time since the previous mark to `stage`.
enum Stage { ST_BEGIN = 0, ST_ROUTER_GEMM, ST_ROUTE, ST_MAPS, ST_PERMUTE, ST_GEMM1_SWIGLU, ST_GEMM2, ST_COMBINE,
             ST_COMBINE_BWD, ST_DGRAD_DOWN_SWIGLU, ST_DGRAD_GATEUP, ST_WGRAD, ST_ROUTER_BWD, ST_DX_COMBINE,
             ST_SHARED_FWD, ST_SHARED_BWD, ST_QUANT, ST_COUNT };
extern int g_prof_on;
void prof_mark_impl(int stage, cudaStream_t s);
inline void prof_mark(int stage, cudaStream_t s) { if (g_prof_on) prof_mark_impl(stage, s); }

inline cudaStream_t as_stream(void* s) { return reinterpret_cast<cudaStream_t>(s); }

// Every kernel launch in the library goes through this so that launches are counted and launch
// errors become MOE_ERR_CUDA instead of being dropped.
#define MOE_LAUNCH(kernel, grid, block, smem, stream, ...)                 \
  do {                                                                     \
    kernel<<<(grid), (block), (smem), (stream)>>>(__VA_ARGS__);            \
    ++::moe::g_launches;                                                   \
    if (cudaPeekAtLastError() != cudaSuccess) {                            \
      cudaGetLastError();                                                  \
      return MOE_ERR_CUDA;                                                 \
    }                                                                      \
  } while (0)

#define MOE_CHECK(expr)                         \
  do {                                          \
    int32_t _s = (expr);                        \
    if (_s != MOE_OK) return _s;                \
  } while (0)

#define MOE_CUDA(expr)                          \
  do {                                          \
    if ((expr) != cudaSuccess) {                \
      cudaGetLastError();                       \
      return MOE_ERR_CUDA;                      \
    }                                           \
  } while (0)

inline int64_t round_up(int64_t x, int64_t a) { return (x + a - 1) / a * a; }
inline int64_t ceil_div(int64_t x, int64_t a) { return (x + a - 1) / a; }

int32_t validate(const moe_config_t* c);
// The limits include/moe_b200.h lists for moe_layer_fwd / bwd / wgrad (validate() + the routing kernel's E, K, n_group
// bounds + FP8 row alignment), checked BEFORE the first launch so that those UNSUPPORTED cases enqueue nothing.  It does
// not mirror every shape predicate of tc_gemm / fp8_gemm: the layer picks the CUDA-core GEMM for shapes the tensor-core
// path does not take, and a tensor-map creation failure inside a stage can still surface after earlier stages ran.
// `backward` is unused today (both directions share the limits).
int32_t layer_preflight(const moe_config_t* c, bool backward);

// Lazily filled per-device caches (function attributes, SM counts) are indexed by the CURRENT device, so a process
// that drives several GPUs (or several contexts) through the library gets each device set up once.
constexpr int MAX_DEVICES = 64;
inline int current_device() {
  int d = 0;
  if (cudaGetDevice(&d) != cudaSuccess) { cudaGetLastError(); return -1; }
  return (d >= 0 && d < MAX_DEVICES) ? d : -1;
}
int device_sm_count();   // SM count of the current device (cached per device); <= 0 on error
inline int64_t padded_rows(const moe_config_t* c) {
  int64_t tk = (int64_t)c->T * c->K;
  if (c->row_align <= 1) return tk;
  return round_up(tk + (int64_t)c->E * (c->row_align - 1), c->row_align);
}
inline size_t elem_bytes(const moe_config_t* c) { return c->dtype == 0 ? 4 : 2; }
// V2: zero-computation experts are the last n_zc of the E router outputs; the first E - n_zc own FFN weights.
inline int n_zc(const moe_config_t* c) { return c->n_zero + c->n_copy + c->n_const; }
inline int e_ffn(const moe_config_t* c) { return c->E - n_zc(c); }
// The router backward runs densely (dz [T,E] -> two GEMMs) when dz is not confined to the selected experts: the balance
// loss (A3), softmax gating without renormalisation; zero-computation experts use it too (their rows lie outside the
// FFN tile tables the sparse dWr reduction walks).
inline bool dense_router_bwd(const moe_config_t* c) {
  return c->aux_coef != 0.f || n_zc(c) > 0 || (c->score_fn == 0 && !c->renorm && c->route_mode == 0);
}

// Routing weights FUSED into the grouped GEMMs' epilogues (north_star (3)), for bf16 tensor-core layers:
//  1 (default): GEMM-1 writes a = w silu(g) u, so y = w y and the combine is a plain sum; the backward replaces the
//     combine-backward pass (reads y and dY, writes dy = w dY) by a plain row gather of dY (ws "dy" = UNWEIGHTED rows),
//     dgrad-down applies w in its epilogue and produces dw[t,j] = <da_r, a_r> there, so y is never read again.
//  2: as 1, and GEMM-1 / dgrad-down gather their A rows from the token-major X / dY themselves (TMA tile::gather4 through
//     perm_to_flat, gather-warp kernel variants), writing Xp / dy as a by-product of the staged tiles: no row-mover pass at
//     all.  Measured slower than 1 (the by-product stores cost the GEMMs more than the passes they
//     replace), kept selectable with cfg->opt_rows_fused = 3.
//  0 (cfg->opt_rows_fused = 1, and every other dtype / layout): w in the combine, dy = w dY from combine-backward.
int rows_fused(const moe_config_t* c);   // layout.cu
bool rows_fusable(const moe_config_t* c);  // the config admits levels 1 / 2 (decides the ws layout; the knob does not)

// ---- byte layout of ctx / ws ---------------------------------------------------------------
struct CtxLayout {
  size_t z, idx, w, counts, offsets, p2f, f2p, mtile, Xp, gu, a, y, gu_s, a_s, y_s;
  size_t aux_f, aux_P, aux_loss;   // A1: fp32 [E], [E], [1]
  // fp8 (dtype 2): codes + scales of the quantised activations / weights kept for the backward
  size_t Xq, Xq_s, Xpq, Xpq_s, aq, aq_s, Wgq, Wgq_s, Wuq, Wuq_s, Wdq, Wdq_s;
  size_t asq, asq_s, Wgsq, Wgsq_s, Wusq, Wusq_s, Wdsq, Wdsq_s;
  size_t total;
};
struct WsLayout {
  size_t hist, tmp, dw, dz, dzp, dwr_part, dy, dgu, dXp, dgu_s, dXs, dYq, dYq_s, dyq, dyq_s, dguq, dguq_s, dgusq, dgusq_s;
  size_t dwpart;                    // fused rows: fp32 [2 ceil(F/256), R] partial <da, a> sums of the dgrad-down epilogue
  size_t dzd, dzb, dXr, aux_part;  // dense router backward: dz fp32 [T,E], its bf16 copy [T,Ep], dz Wr [T,H]; aux partials
  size_t total;
};
CtxLayout ctx_layout(const moe_config_t* c);
WsLayout ws_layout(const moe_config_t* c);

constexpr int PERM_CHUNK = 1024;  // flat positions per counting-sort chunk (one CTA)

// ---- internal entry points shared between translation units ---------------------------------------
// permute.cu
int32_t build_maps(const moe_config_t* c, const int32_t* idx, int32_t* counts, int32_t* offsets, int32_t* p2f,
                   int32_t* f2p, int32_t* mtile_expert, int32_t* hist, cudaStream_t s);
constexpr int AUX_TOKENS_PER_CTA = 64;   // tokens per partial sum of P_e (A2)
int32_t gather_rows(const moe_config_t* c, const void* X, int cols, size_t esz, const int32_t* f2p, const int32_t* p2f,
                    const int32_t* offsets, void* Xp, cudaStream_t s);
int32_t combine(const moe_config_t* c, const void* y, const float* w, const int32_t* f2p, const void* add0,
                const void* add1, const float* dz, const int32_t* idx, const void* Wr, void* Y, cudaStream_t s);
// dw[p] = sum_k part[k, f2p[p]] (fixed order; an empty slot gets 0): the routing-weight gradient from the dgrad-down epilogue
int32_t dw_reduce(const moe_config_t* c, const float* part, int nparts, const int32_t* f2p, float* dw, cudaStream_t s);
int32_t combine_bwd(const moe_config_t* c, const void* dY, const void* y, const float* w, const int32_t* f2p,
                    const int32_t* p2f, const int32_t* offsets, void* dy, float* dw, cudaStream_t s);
// route.cu: moe_route with an optional second copy of the outputs
int32_t route_impl(const moe_config_t* c, const float* logits, const float* bias, const float* threshold,
                   int32_t* topk_idx, float* topk_w, int32_t* idx_copy, float* w_copy, void* stream);
// router.cu
int32_t router_logits(const moe_config_t* c, const void* X, const void* Wr, float* z, cudaStream_t s);
int32_t router_bwd(const moe_config_t* c, const float* z, const int32_t* idx, const float* w, const float* dw,
                   const int32_t* f2p, const int32_t* offsets, const int32_t* counts, const int32_t* mtile,
                   const void* Xp, const void* X /* token-major, with p2f: read instead of Xp; or NULL */, const int32_t* p2f,
                   float* dz, float* dzp, float* part, void* dWr, cudaStream_t s);
// dense router backward (A3 / softmax without renorm / V2): dz [T,E] fp32 (+ bf16 copy), dWr = dz^T X, dXr = dz Wr
int32_t router_bwd_dense(const moe_config_t* c, const float* z, const int32_t* idx, const float* w, const float* dw,
                         const float* aux_f, const void* X, const void* Wr, const int32_t* off_one /* device {0, T} */,
                         float* dz_sel, float* dzd, void* dzb, void* dWr, void* dXr, cudaStream_t s);
// A1..A2: f (from counts, or f_global), P, L_aux -> ctx fields; loss also to loss_out if not NULL
int32_t aux_forward(const moe_config_t* c, const float* z, const int32_t* counts, const float* f_global, float* part,
                    float* aux_f, float* aux_P, float* aux_loss, float* loss_out, cudaStream_t s);
// zc.cu (V2): rows of the zero-computation experts' groups
int32_t zc_forward(const moe_config_t* c, const int32_t* offsets, const int32_t* counts, const void* Xp, const void* zc_const,
                   void* gu, void* a, void* y, cudaStream_t s);
int32_t zc_backward(const moe_config_t* c, const int32_t* offsets, const int32_t* counts, const void* dy, void* dgu, void* dXp,
                    void* d_zc_const, cudaStream_t s);
// gemm_simt.cu: reference-free fallback GEMMs for fp32 (and any shape the tensor-core path rejects)
//   mode 0: C[r,n]    = sum_k A[r,k] B[e][n,k]           (rows grouped by offsets)
//   mode 1: dA[r,k]   = sum_n dC[r,n] B[e][n,k]
//   mode 2: dB[e][n,k]= sum_{r in e} dC[r,n] A[r,k]
int32_t simt_grouped_gemm(int mode, int dtype, int E, int N, int Kdim, const void* A, int lda, const void* B,
                          const void* dC, int lddc, const int32_t* offsets, void* out, int ldo, int64_t rows_cap,
                          int accumulate, cudaStream_t s);
// gemm_tc.cu: tcgen05 grouped GEMMs (bf16)
struct TcGemmArgs;
int32_t tc_prepare_tiles(const int32_t* offsets, int E, int64_t rows_cap, int32_t* mtile_expert, cudaStream_t s);
// elementwise.cu
int32_t swiglu_fwd(int dtype, const void* gu, void* a, int64_t rows, int F, cudaStream_t s);
int32_t swiglu_bwd(int dtype, const void* gu, const void* da, void* dgu, int64_t rows, int F, cudaStream_t s);

// ---- device helpers --------------------------------------------------------------------------------
__device__ __forceinline__ float bf16_to_f(__nv_bfloat16 v) { return __bfloat162float(v); }

template <typename T>
__device__ __forceinline__ float to_f(T v);
template <>
__device__ __forceinline__ float to_f<float>(float v) { return v; }
template <>
__device__ __forceinline__ float to_f<__nv_bfloat16>(__nv_bfloat16 v) { return __bfloat162float(v); }
template <typename T>
__device__ __forceinline__ T from_f(float v);
template <>
__device__ __forceinline__ float from_f<float>(float v) { return v; }
template <>
__device__ __forceinline__ __nv_bfloat16 from_f<__nv_bfloat16>(float v) { return __float2bfloat16_rn(v); }

__device__ __forceinline__ float sigmoidf_acc(float x) { return 1.0f / (1.0f + expf(-x)); }

}  // namespace moe
