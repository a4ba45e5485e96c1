// moe_layer_fwd / moe_layer_bwd: composition of the hot path (SURVEY.md §3 call stack, §8c R1..R8),
// plus the public grouped-GEMM entry points.  Single stream, no host synchronisation anywhere:
// per-expert counts stay on the device.
#include <stdlib.h>
#include <string.h>

#include "fp8.cuh"
#include "gemm_tc.cuh"
#include "tile_tables.cuh"

namespace moe {

// One SwiGLU FFN over grouped rows: the routed experts (E groups from the permutation) or the
// shared expert (one group holding every token).
struct FfnGroup {
  int dtype, E, H, F;
  int64_t rows_cap;        // upper bound on rows (buffer height)
  const int32_t* offsets;  // [E+1] device
  const int32_t* counts;   // [E] device or nullptr (then offsets differences are used)
  const int32_t* mtile;    // M-tile -> expert table (tensor-core path) or nullptr
  int row_align;
  int st_fwd1, st_fwd2, st_bwd1, st_bwd2, st_wgrad;  // profile stages of the five GEMM groups
  // rows_fused(cfg) >= 1 (routed experts only): w (by flat position, rows mapped through gidx = perm_to_flat) is applied in
  // the GEMM-1 / dgrad-down epilogues, so a holds w a and the copy called dy holds the UNWEIGHTED rows of dY;
  // rows_fused(cfg) == 2: those two GEMMs also gather their A rows from the TOKEN-major tok_in (X / dY) themselves and
  // write the row-grouped copies (Xp / dy) as a by-product
  const int32_t* gidx = nullptr;
  const void* tok_in = nullptr;
  int gK = 1;
  int64_t g_rows = 0;
  const float* roww = nullptr;
  float* dwpart = nullptr;
  int opt_pair = 0, opt_wide = 0, opt_fq = 0;   // moe_config_t::opt_pair / opt_fp8_wide / opt_fp8_fused_quant
};

inline void set_opts(FfnGroup& g, const moe_config_t* c) {
  g.opt_pair = c->opt_pair; g.opt_wide = c->opt_fp8_wide; g.opt_fq = c->opt_fp8_fused_quant;
}

namespace {

__global__ void set2_kernel(int32_t* p, int32_t a, int32_t b) {
  p[0] = a;
  p[1] = b;
}

// tcgen05 path: bf16, H and F multiples of 64, and either 128-row-aligned groups or a single group.
bool use_tc(const FfnGroup& g) {
  return g.dtype == 1 && g.H % 64 == 0 && g.F % 64 == 0 && (g.mtile != nullptr || g.E == 1);
}

TcCall tc_base(const FfnGroup& g, int mode) {
  TcCall c;
  memset(&c, 0, sizeof(c));
  c.mode = mode;
  c.opt_pair = g.opt_pair;
  c.E = g.E;
  c.rows_cap = g.rows_cap;
  c.offsets = g.offsets;
  c.counts = g.mtile ? g.counts : nullptr;
  c.mtile = g.mtile;
  if (g.mtile) {            // the pair / unpaired lists sit behind the M-tile table (tile_tables.cuh)
    c.plist = g.mtile + tile_plist_off(g.rows_cap);
    c.olist = g.mtile + tile_olist_off(g.rows_cap);
  }
  c.F = g.F;
  return c;
}

int32_t ffn_fwd(const FfnGroup& g, const void* Xp, const void* Wg, const void* Wu, const void* Wd, void* gu, void* a,
                void* y, cudaStream_t s) {
  if (use_tc(g)) {
    TcCall c = tc_base(g, TC_FWD_SWIGLU);   // gu = [Xp Wg^T | Xp Wu^T], a = silu(g) * u
    c.A = Xp; c.lda = g.H; c.B0 = Wg; c.B1 = Wu; c.b_rows = g.F; c.b_cols = g.H; c.N = g.F; c.Kd = g.H;
    c.out0 = gu; c.ld0 = 2 * g.F; c.out1 = a; c.ld1 = g.F;
    if (g.gidx) { c.gidx = g.gidx; c.roww = g.roww; }   // a = w silu(g) u
    if (g.tok_in) {                         // A = X [T,H] gathered in the kernel; Xp is its by-product
      c.A = g.tok_in; c.gat = 1; c.gK = g.gK; c.g_rows = g.g_rows; c.copy_out = const_cast<void*>(Xp); c.ld_copy = g.H;
    }
    MOE_CHECK(tc_gemm(c, s));
    prof_mark(g.st_fwd1, s);
    c = tc_base(g, TC_FWD);                 // y = a Wd^T
    c.A = a; c.lda = g.F; c.B0 = Wd; c.b_rows = g.H; c.b_cols = g.F; c.N = g.H; c.Kd = g.F; c.out0 = y; c.ld0 = g.H;
    MOE_CHECK(tc_gemm(c, s));
    prof_mark(g.st_fwd2, s);
    return MOE_OK;
  }
  const size_t es = g.dtype == 0 ? 4 : 2;
  MOE_CHECK(simt_grouped_gemm(0, g.dtype, g.E, g.F, g.H, Xp, g.H, Wg, nullptr, 0, g.offsets, gu, 2 * g.F, g.rows_cap, 0, s));
  MOE_CHECK(simt_grouped_gemm(0, g.dtype, g.E, g.F, g.H, Xp, g.H, Wu, nullptr, 0, g.offsets, (char*)gu + g.F * es,
                              2 * g.F, g.rows_cap, 0, s));
  MOE_CHECK(swiglu_fwd(g.dtype, gu, a, g.rows_cap, g.F, s));
  prof_mark(g.st_fwd1, s);
  MOE_CHECK(simt_grouped_gemm(0, g.dtype, g.E, g.H, g.F, a, g.F, Wd, nullptr, 0, g.offsets, y, g.H, g.rows_cap, 0, s));
  prof_mark(g.st_fwd2, s);
  return MOE_OK;
}

// The three weight gradients of one FFN group from the bf16 tensors (R8; R9: wgrad stays in bf16):
//   dWd[e] = dy_e^T a_e,  dWg[e] = dg_e^T Xp_e,  dWu[e] = du_e^T Xp_e.
// acc_f32: the outputs are fp32 buffers that the tiles are ADDED to (tensor-core path only).
int32_t ffn_wgrad(const FfnGroup& g, const void* dy, const void* Xp, const void* a, const void* dgu, void* dWg, void* dWu,
                  void* dWd, int acc_f32, cudaStream_t s) {
  const bool tc_ok = g.dtype != 0 && g.H % 64 == 0 && g.F % 64 == 0 && (g.mtile != nullptr || g.E == 1);
  if (tc_ok) {
    TcCall c = tc_base(g, TC_WGRAD);
    c.acc_f32 = acc_f32;
    c.A = dy; c.lda = g.H; c.M = g.H; c.A2 = a; c.lda2 = g.F; c.N = g.F; c.out0 = dWd; c.ld0 = g.F;
    MOE_CHECK(tc_gemm(c, s));
    c = tc_base(g, TC_WGRAD);
    c.acc_f32 = acc_f32;
    c.A = dgu; c.lda = 2 * g.F; c.M = g.F; c.A2 = Xp; c.lda2 = g.H; c.N = g.H; c.out0 = dWg; c.ld0 = g.H;
    MOE_CHECK(tc_gemm(c, s));
    c.a_col0 = g.F; c.out0 = dWu;
    MOE_CHECK(tc_gemm(c, s));
    prof_mark(g.st_wgrad, s);
    return MOE_OK;
  }
  if (acc_f32 || g.dtype == 2) return MOE_ERR_UNSUPPORTED;
  const size_t es = g.dtype == 0 ? 4 : 2;
  const void* dgu_u = (const char*)dgu + g.F * es;
  MOE_CHECK(simt_grouped_gemm(2, g.dtype, g.E, g.H, g.F, a, g.F, nullptr, dy, g.H, g.offsets, dWd, 0, g.rows_cap, 0, s));
  MOE_CHECK(simt_grouped_gemm(2, g.dtype, g.E, g.F, g.H, Xp, g.H, nullptr, dgu, 2 * g.F, g.offsets, dWg, 0, g.rows_cap, 0, s));
  MOE_CHECK(simt_grouped_gemm(2, g.dtype, g.E, g.F, g.H, Xp, g.H, nullptr, dgu_u, 2 * g.F, g.offsets, dWu, 0, g.rows_cap, 0, s));
  prof_mark(g.st_wgrad, s);
  return MOE_OK;
}

// dy [rows,H] -> dgu, dXp and (optionally) dWg, dWu, dWd.  da_tmp [rows,F] is scratch (CUDA-core path only).
int32_t ffn_bwd(const FfnGroup& g, const void* dy, const void* Xp, const void* gu, const void* a, const void* Wg,
                const void* Wu, const void* Wd, void* da_tmp, void* dgu, void* dXp, void* dWg, void* dWu, void* dWd,
                cudaStream_t s) {
  const size_t es = g.dtype == 0 ? 4 : 2;
  const void* dgu_u = (const char*)dgu + g.F * es;
  if (use_tc(g)) {
    TcCall c = tc_base(g, TC_DGRAD_SWIGLU);   // dgu = swiglu'(gu) * (dy Wd[e])
    c.A = dy; c.lda = g.H; c.B0 = Wd; c.b_rows = g.H; c.b_cols = g.F; c.N = g.F; c.gu = gu; c.ldgu = 2 * g.F;
    c.out0 = dgu; c.ld0 = 2 * g.F;
    if (g.gidx) { c.gidx = g.gidx; c.roww = g.roww; c.dwpart = g.dwpart; }   // dgu = w swiglu'(gu) da; dwpart = <da, a>
    if (g.tok_in) {                           // A = dY [T,H] gathered in the kernel; dy = its unweighted by-product copy
      c.A = g.tok_in; c.gat = 1; c.gK = g.gK; c.g_rows = g.g_rows; c.copy_out = const_cast<void*>(dy); c.ld_copy = g.H;
    }
    MOE_CHECK(tc_gemm(c, s));
    prof_mark(g.st_bwd1, s);
    c = tc_base(g, TC_DGRAD);                 // dXp = dg Wg[e] + du Wu[e]: one contraction over [dg|du]
    c.A = dgu; c.lda = 2 * g.F; c.B0 = Wg; c.B1 = Wu; c.b_rows = g.F; c.b_cols = g.H; c.N = g.H; c.out0 = dXp; c.ld0 = g.H;
    MOE_CHECK(tc_gemm(c, s));
    prof_mark(g.st_bwd2, s);
    if (dWd) MOE_CHECK(ffn_wgrad(g, dy, Xp, a, dgu, dWg, dWu, dWd, 0, s));
    return MOE_OK;
  }
  // da = dy Wd[e]            (B = Wd [E,H,F]: N = H, Kdim = F)
  MOE_CHECK(simt_grouped_gemm(1, g.dtype, g.E, g.H, g.F, nullptr, 0, Wd, dy, g.H, g.offsets, da_tmp, g.F, g.rows_cap, 0, s));
  MOE_CHECK(swiglu_bwd(g.dtype, gu, da_tmp, dgu, g.rows_cap, g.F, s));
  prof_mark(g.st_bwd1, s);
  // dXp = dg Wg[e] + du Wu[e]  (B = Wg [E,F,H]: N = F, Kdim = H)
  MOE_CHECK(simt_grouped_gemm(1, g.dtype, g.E, g.F, g.H, nullptr, 0, Wg, dgu, 2 * g.F, g.offsets, dXp, g.H, g.rows_cap, 0, s));
  MOE_CHECK(simt_grouped_gemm(1, g.dtype, g.E, g.F, g.H, nullptr, 0, Wu, dgu_u, 2 * g.F, g.offsets, dXp, g.H, g.rows_cap, 1, s));
  prof_mark(g.st_bwd2, s);
  if (dWd) MOE_CHECK(ffn_wgrad(g, dy, Xp, a, dgu, dWg, dWu, dWd, 0, s));
  return MOE_OK;
}

// Quantised operands of one FFN group on the fp8 path (R9): e4m3 codes + fp32 block scales.
struct Fp8Bufs {
  const uint8_t* Aq; const float* Aq_s;        // GEMM1 input rows [rows, H] (1x128)
  uint8_t* aq; float* aq_s;                    // a [rows, F] (1x128)
  const uint8_t *Wgq, *Wuq, *Wdq;              // weights (128x128)
  const float *Wgq_s, *Wuq_s, *Wdq_s;
  const uint8_t* dyq; const float* dyq_s;      // rows of Q(dY) [rows, H]
  uint8_t* dguq; float* dguq_s;                // [dg|du] [rows, 2F]
  const int32_t* p2f; const float* w;          // row weight of the dgrad-down epilogue (nullptr = 1)
  int mode;
};

// Quantise-in-epilogue vs the stand-alone quantiser passes for Q-a / Q-dgu.  Both give the same bits
// (tests/test_gpu_fp8.py).  With power-of-two scales the epilogue quantises by an exact multiplication and is the
// default; with fp32 scales (mode 0) every code needs an IEEE division on the promotion warps' critical path, which costs
// the two GEMMs more (+0.55 / +0.76 ms on configs[3]) than the two HBM passes it removes (-0.65 ms), so the stand-alone
// passes stay the default there.  moe_config_t::opt_fp8_fused_quant = 1 / 2 forces off / on.
bool fused_quant(const FfnGroup& g, int scale_mode) {
  if (g.opt_fq) return g.opt_fq == 2;
  return scale_mode == 1;
}

F8Call f8_base(const FfnGroup& g, int mode) {
  F8Call c;
  memset(&c, 0, sizeof(c));
  c.mode = mode;
  c.opt_wide = g.opt_wide;
  c.E = g.E;
  c.rows_cap = g.rows_cap;
  c.mtile = g.mtile;
  c.F = g.F;
  return c;
}

int32_t ffn_fwd_fp8(const FfnGroup& g, const Fp8Bufs& q, void* gu, void* a, void* y, cudaStream_t s) {
  F8Call c = f8_base(g, F8_FWD_SWIGLU);   // gu = [Q(X) Q(Wg)^T | Q(X) Q(Wu)^T], a = silu(g) * u
  c.A = q.Aq; c.lda = g.H; c.a_scales = q.Aq_s; c.B0 = q.Wgq; c.b0_scales = q.Wgq_s; c.B1 = q.Wuq; c.b1_scales = q.Wuq_s;
  c.b_rows = g.F; c.b_cols = g.H; c.N = g.F; c.out0 = gu; c.ld0 = 2 * g.F; c.out1 = a; c.ld1 = g.F;
  const bool fused = fused_quant(g, q.mode);
  if (fused) { c.q_codes = q.aq; c.q_scales = q.aq_s; c.q_mode = q.mode; }   // Q-a on the bf16 a, in the epilogue
  MOE_CHECK(fp8_gemm(c, s));
  prof_mark(g.st_fwd1, s);
  if (!fused) {
    MOE_CHECK(fp8_quantize_act(a, g.rows_cap, g.F, q.mode, q.aq, q.aq_s, s));   // Q-a as a stand-alone pass
    prof_mark(ST_QUANT, s);
  }
  c = f8_base(g, F8_FWD);                 // y = Q(a) Q(Wd)^T
  c.A = q.aq; c.lda = g.F; c.a_scales = q.aq_s; c.B0 = q.Wdq; c.b0_scales = q.Wdq_s; c.b_rows = g.H; c.b_cols = g.F;
  c.N = g.H; c.out0 = y; c.ld0 = g.H;
  MOE_CHECK(fp8_gemm(c, s));
  prof_mark(g.st_fwd2, s);
  return MOE_OK;
}

// dgrad in fp8 (codes of dY rows, dg, du), wgrad in bf16 from dy, a, dgu, Xp (R9).
int32_t ffn_bwd_fp8(const FfnGroup& g, const Fp8Bufs& q, const void* dy, const void* Xp, const void* gu, const void* a,
                    void* dgu, void* dXp, void* dWg, void* dWu, void* dWd, cudaStream_t s) {
  F8Call c = f8_base(g, F8_DGRAD_SWIGLU);  // dgu = swiglu'(gu) * w_r * (Q(dY)[t_r] Q(Wd)[e])
  c.A = q.dyq; c.lda = g.H; c.a_scales = q.dyq_s; c.B0 = q.Wdq; c.b0_scales = q.Wdq_s; c.b_rows = g.H; c.b_cols = g.F;
  c.N = g.F; c.gu = gu; c.ldgu = 2 * g.F; c.out0 = dgu; c.ld0 = 2 * g.F; c.p2f = q.p2f; c.w = q.w;
  const bool fused = fused_quant(g, q.mode);
  if (fused) { c.q_codes = q.dguq; c.q_scales = q.dguq_s; c.q_mode = q.mode; }   // Q-dgu in the epilogue
  MOE_CHECK(fp8_gemm(c, s));
  prof_mark(g.st_bwd1, s);
  if (!fused) {
    MOE_CHECK(fp8_quantize_act(dgu, g.rows_cap, 2 * g.F, q.mode, q.dguq, q.dguq_s, s));   // Q-dgu as a stand-alone pass
    prof_mark(ST_QUANT, s);
  }
  c = f8_base(g, F8_DGRAD);                // dXp = Q(dg) Q(Wg)[e] + Q(du) Q(Wu)[e]
  c.A = q.dguq; c.lda = 2 * g.F; c.a_scales = q.dguq_s; c.B0 = q.Wgq; c.b0_scales = q.Wgq_s; c.B1 = q.Wuq;
  c.b1_scales = q.Wuq_s; c.b_rows = g.F; c.b_cols = g.H; c.N = g.H; c.out0 = dXp; c.ld0 = g.H;
  MOE_CHECK(fp8_gemm(c, s));
  prof_mark(g.st_bwd2, s);
  if (dWd) MOE_CHECK(ffn_wgrad(g, dy, Xp, a, dgu, dWg, dWu, dWd, 0, s));
  return MOE_OK;
}

template <typename T>
T* at(const void* base, size_t off) {
  return reinterpret_cast<T*>((char*)base + off);
}

}  // namespace
}  // namespace moe

using namespace moe;

extern "C" int32_t moe_fp8_quantize_weights(const moe_config_t* cfg, const void* Wg, const void* Wu, const void* Wd,
                                            const void* Wg_s, const void* Wu_s, const void* Wd_s, void* ctx,
                                            void* stream) {
  if (!cfg || !Wg || !Wu || !Wd || !ctx) return MOE_ERR_INVALID_ARG;
  MOE_CHECK(validate(cfg));
  if (cfg->dtype != 2) return MOE_ERR_INVALID_ARG;
  const bool shared = cfg->F_shared > 0;
  if (shared && (!Wg_s || !Wu_s || !Wd_s)) return MOE_ERR_INVALID_ARG;
  cudaStream_t s = as_stream(stream);
  const CtxLayout C = ctx_layout(cfg);
  const int m = cfg->fp8_scale_mode, E = e_ffn(cfg), H = cfg->H, F = cfg->F, Fs = cfg->F_shared;
  MOE_CHECK(fp8_quantize_weight(Wg, E, F, H, m, at<uint8_t>(ctx, C.Wgq), at<float>(ctx, C.Wgq_s), s));
  MOE_CHECK(fp8_quantize_weight(Wu, E, F, H, m, at<uint8_t>(ctx, C.Wuq), at<float>(ctx, C.Wuq_s), s));
  MOE_CHECK(fp8_quantize_weight(Wd, E, H, F, m, at<uint8_t>(ctx, C.Wdq), at<float>(ctx, C.Wdq_s), s));
  if (shared) {
    MOE_CHECK(fp8_quantize_weight(Wg_s, 1, Fs, H, m, at<uint8_t>(ctx, C.Wgsq), at<float>(ctx, C.Wgsq_s), s));
    MOE_CHECK(fp8_quantize_weight(Wu_s, 1, Fs, H, m, at<uint8_t>(ctx, C.Wusq), at<float>(ctx, C.Wusq_s), s));
    MOE_CHECK(fp8_quantize_weight(Wd_s, 1, H, Fs, m, at<uint8_t>(ctx, C.Wdsq), at<float>(ctx, C.Wdsq_s), s));
  }
  return MOE_OK;
}

extern "C" int32_t moe_layer_fwd(const moe_config_t* cfg, const void* X, const void* Wr, const float* bias,
                                 const void* Wg, const void* Wu, const void* Wd, const void* Wg_s, const void* Wu_s,
                                 const void* Wd_s, void* Y, int32_t* topk_idx, float* topk_w, void* ctx, void* ws,
                                 void* stream) {
  return moe_layer_fwd_ex(cfg, X, Wr, bias, Wg, Wu, Wd, Wg_s, Wu_s, Wd_s, Y, topk_idx, topk_w, ctx, ws, nullptr, stream);
}

extern "C" int32_t moe_layer_fwd_ex(const moe_config_t* cfg, const void* X, const void* Wr, const float* bias,
                                    const void* Wg, const void* Wu, const void* Wd, const void* Wg_s, const void* Wu_s,
                                    const void* Wd_s, void* Y, int32_t* topk_idx, float* topk_w, void* ctx, void* ws,
                                    const moe_extras_t* ex, void* stream) {
  if (!cfg || !X || !Wr || !Y || !topk_idx || !topk_w || !ctx || !ws) return MOE_ERR_INVALID_ARG;
  MOE_CHECK(layer_preflight(cfg, false));
  if (cfg->has_bias && !bias) return MOE_ERR_INVALID_ARG;
  if (cfg->route_mode == 1 && !(ex && ex->threshold)) return MOE_ERR_INVALID_ARG;     // V1 needs the gate thresholds
  if (cfg->n_const > 0 && !(ex && ex->zc_const)) return MOE_ERR_INVALID_ARG;          // V2 needs the constant vectors
  const bool shared = cfg->F_shared > 0;
  const bool fp8 = cfg->dtype == 2;
  // fp8: Wg == Wu == Wd == NULL means "use the e4m3 codes already in ctx" (the FP8 weight cache, PAPER.md:116,
  // filled by an earlier moe_layer_fwd with weights or by moe_fp8_quantize_weights).
  const bool cached = fp8 && !Wg && !Wu && !Wd;
  if (!cached && (!Wg || !Wu || !Wd)) return MOE_ERR_INVALID_ARG;
  if (shared && !cached && (!Wg_s || !Wu_s || !Wd_s)) return MOE_ERR_INVALID_ARG;
  if (fp8 && cfg->row_align % 128 != 0) return MOE_ERR_UNSUPPORTED;
  cudaStream_t s = as_stream(stream);
  const CtxLayout C = ctx_layout(cfg);
  const WsLayout W = ws_layout(cfg);
  float* z = at<float>(ctx, C.z);
  int32_t* counts = at<int32_t>(ctx, C.counts);
  int32_t* offsets = at<int32_t>(ctx, C.offsets);
  int32_t* p2f = at<int32_t>(ctx, C.p2f);
  int32_t* f2p = at<int32_t>(ctx, C.f2p);
  int32_t* mtile = at<int32_t>(ctx, C.mtile);
  void* Xp = at<char>(ctx, C.Xp);
  void* gu = at<char>(ctx, C.gu);
  void* a = at<char>(ctx, C.a);
  void* y = at<char>(ctx, C.y);

  prof_mark(ST_BEGIN, s);
  MOE_CHECK(router_logits(cfg, X, Wr, z, s));                                              // R1
  prof_mark(ST_ROUTER_GEMM, s);
  MOE_CHECK(route_impl(cfg, z, bias, ex ? ex->threshold : nullptr, topk_idx, topk_w, at<int32_t>(ctx, C.idx),
                       at<float>(ctx, C.w), stream));                                                         // R2..R5 / V1
  prof_mark(ST_ROUTE, s);
  MOE_CHECK(build_maps(cfg, topk_idx, counts, offsets, p2f, f2p, mtile, at<int32_t>(ws, W.hist), s));  // R6
  prof_mark(ST_MAPS, s);
  const int fused = rows_fused(cfg);       // 2: X is gathered inside GEMM-1, which also writes Xp: no permute pass
  if (fused < 2) MOE_CHECK(gather_rows(cfg, X, cfg->H, elem_bytes(cfg), f2p, p2f, offsets, Xp, s));
  prof_mark(ST_PERMUTE, s);
  // the FFN runs over the experts that own weights (all of them unless zero-computation experts are configured, V2)
  FfnGroup g{cfg->dtype, e_ffn(cfg), cfg->H, cfg->F, padded_rows(cfg), offsets, counts,
             (cfg->row_align % 128 == 0) ? mtile : nullptr, cfg->row_align,
             ST_GEMM1_SWIGLU, ST_GEMM2, ST_DGRAD_DOWN_SWIGLU, ST_DGRAD_GATEUP, ST_WGRAD};
  set_opts(g, cfg);
  if (fused) { g.gidx = p2f; g.gK = cfg->K; g.g_rows = cfg->T; g.roww = topk_w; }
  if (fused == 2) g.tok_in = X;
  Fp8Bufs q, qs;
  memset(&q, 0, sizeof(q));
  memset(&qs, 0, sizeof(qs));
  if (fp8) {                                                                               // R9 quantisation points
    const int mode = cfg->fp8_scale_mode;
    uint8_t* Xq = at<uint8_t>(ctx, C.Xq);
    float* Xq_s = at<float>(ctx, C.Xq_s);
    MOE_CHECK(fp8_quantize_act(X, cfg->T, cfg->H, mode, Xq, Xq_s, s));                     // Q-X once per token
    MOE_CHECK(gather_rows(cfg, Xq, cfg->H, 1, f2p, p2f, offsets, at<uint8_t>(ctx, C.Xpq), s));
    MOE_CHECK(fp8_gather_scales(Xq_s, p2f, offsets, cfg->E, cfg->K, cfg->H / 128, at<float>(ctx, C.Xpq_s), s));
    if (!cached) MOE_CHECK(moe_fp8_quantize_weights(cfg, Wg, Wu, Wd, Wg_s, Wu_s, Wd_s, ctx, stream));   // Q-W
    prof_mark(ST_QUANT, s);
    q.Aq = at<uint8_t>(ctx, C.Xpq); q.Aq_s = at<float>(ctx, C.Xpq_s);
    q.aq = at<uint8_t>(ctx, C.aq); q.aq_s = at<float>(ctx, C.aq_s);
    q.Wgq = at<uint8_t>(ctx, C.Wgq); q.Wgq_s = at<float>(ctx, C.Wgq_s);
    q.Wuq = at<uint8_t>(ctx, C.Wuq); q.Wuq_s = at<float>(ctx, C.Wuq_s);
    q.Wdq = at<uint8_t>(ctx, C.Wdq); q.Wdq_s = at<float>(ctx, C.Wdq_s);
    q.mode = mode;
    qs = q;
    qs.Aq = Xq; qs.Aq_s = Xq_s;
    qs.aq = at<uint8_t>(ctx, C.asq); qs.aq_s = at<float>(ctx, C.asq_s);
    qs.Wgq = at<uint8_t>(ctx, C.Wgsq); qs.Wgq_s = at<float>(ctx, C.Wgsq_s);
    qs.Wuq = at<uint8_t>(ctx, C.Wusq); qs.Wuq_s = at<float>(ctx, C.Wusq_s);
    qs.Wdq = at<uint8_t>(ctx, C.Wdsq); qs.Wdq_s = at<float>(ctx, C.Wdsq_s);
    MOE_CHECK(ffn_fwd_fp8(g, q, gu, a, y, s));                                             // R7 on the codes
  } else {
    MOE_CHECK(ffn_fwd(g, Xp, Wg, Wu, Wd, gu, a, y, s));                                    // R7
  }
  MOE_CHECK(zc_forward(cfg, offsets, counts, Xp, ex ? ex->zc_const : nullptr, gu, a, y, s));   // V2: y = 0 | x | v
  if (cfg->aux_coef != 0.f)                                                                // A1..A2 balance loss
    MOE_CHECK(aux_forward(cfg, z, counts, ex ? ex->aux_f_global : nullptr, at<float>(ws, W.aux_part), at<float>(ctx, C.aux_f),
                          at<float>(ctx, C.aux_P), at<float>(ctx, C.aux_loss), ex ? ex->aux_loss : nullptr, s));
  const void* shared_out = nullptr;
  if (shared || dense_router_bwd(cfg)) MOE_LAUNCH(set2_kernel, 1, 1, 0, s, offsets + cfg->E + 1, 0, cfg->T);   // group {0, T}
  if (shared) {
    int32_t* off_s = offsets + cfg->E + 1;
    FfnGroup gs{cfg->dtype, 1, cfg->H, cfg->F_shared, cfg->T, off_s, nullptr, nullptr, 1,
                ST_SHARED_FWD, ST_SHARED_FWD, ST_SHARED_BWD, ST_SHARED_BWD, ST_SHARED_BWD};
    set_opts(gs, cfg);
    if (fp8)
      MOE_CHECK(ffn_fwd_fp8(gs, qs, at<char>(ctx, C.gu_s), at<char>(ctx, C.a_s), at<char>(ctx, C.y_s), s));
    else
      MOE_CHECK(ffn_fwd(gs, X, Wg_s, Wu_s, Wd_s, at<char>(ctx, C.gu_s), at<char>(ctx, C.a_s), at<char>(ctx, C.y_s), s));
    shared_out = at<char>(ctx, C.y_s);
  }
  // R7 combine (fused rows: y already carries w, so a plain sum over the K rows)
  MOE_CHECK(combine(cfg, y, fused ? nullptr : topk_w, f2p, shared_out, nullptr, nullptr, nullptr, nullptr, Y, s));
  prof_mark(ST_COMBINE, s);
  return MOE_OK;
}

extern "C" int32_t moe_layer_bwd(const moe_config_t* cfg, const void* dY, const void* X, const void* Wr,
                                 const void* Wg, const void* Wu, const void* Wd, const void* Wg_s, const void* Wu_s,
                                 const void* Wd_s, const void* ctx, void* dX, void* dWr, void* dWg, void* dWu,
                                 void* dWd, void* dWg_s, void* dWu_s, void* dWd_s, void* ws, void* stream) {
  return moe_layer_bwd_ex(cfg, dY, X, Wr, Wg, Wu, Wd, Wg_s, Wu_s, Wd_s, ctx, dX, dWr, dWg, dWu, dWd, dWg_s, dWu_s, dWd_s, ws,
                          nullptr, stream);
}

extern "C" int32_t moe_layer_bwd_ex(const moe_config_t* cfg, const void* dY, const void* X, const void* Wr,
                                    const void* Wg, const void* Wu, const void* Wd, const void* Wg_s, const void* Wu_s,
                                    const void* Wd_s, const void* ctx, void* dX, void* dWr, void* dWg, void* dWu,
                                    void* dWd, void* dWg_s, void* dWu_s, void* dWd_s, void* ws, const moe_extras_t* ex,
                                    void* stream) {
  if (!cfg || !dY || !X || !Wr || !ctx || !dX || !ws) return MOE_ERR_INVALID_ARG;
  MOE_CHECK(layer_preflight(cfg, true));
  const bool shared = cfg->F_shared > 0;
  const bool fp8 = cfg->dtype == 2;   // fp8: the dgrad reads the codes saved in ctx; the bf16 weights are not touched
  if (!fp8 && (!Wg || !Wu || !Wd)) return MOE_ERR_INVALID_ARG;
  if (!fp8 && shared && (!Wg_s || !Wu_s || !Wd_s)) return MOE_ERR_INVALID_ARG;
  if (fp8 && cfg->row_align % 128 != 0) return MOE_ERR_UNSUPPORTED;
  const bool wgrad = dWg || dWu || dWd;
  if (wgrad && !(dWg && dWu && dWd)) return MOE_ERR_INVALID_ARG;
  const bool wgrad_s = dWg_s || dWu_s || dWd_s;
  if (wgrad_s && !(shared && dWg_s && dWu_s && dWd_s)) return MOE_ERR_INVALID_ARG;
  cudaStream_t s = as_stream(stream);
  const CtxLayout C = ctx_layout(cfg);
  const WsLayout W = ws_layout(cfg);
  const float* z = at<float>(ctx, C.z);
  const int32_t* counts = at<int32_t>(ctx, C.counts);
  const int32_t* offsets = at<int32_t>(ctx, C.offsets);
  const int32_t* p2f = at<int32_t>(ctx, C.p2f);
  const int32_t* f2p = at<int32_t>(ctx, C.f2p);
  const int32_t* mtile = at<int32_t>(ctx, C.mtile);
  const int32_t* idx = at<int32_t>(ctx, C.idx);
  const float* w = at<float>(ctx, C.w);
  const void* Xp = at<char>(ctx, C.Xp);
  const void* gu = at<char>(ctx, C.gu);
  const void* a = at<char>(ctx, C.a);
  const void* y = at<char>(ctx, C.y);
  float* dw = at<float>(ws, W.dw);
  float* dz = at<float>(ws, W.dz);
  float* dzp = at<float>(ws, W.dzp);
  void* dy = at<char>(ws, W.dy);
  void* dgu = at<char>(ws, W.dgu);
  void* dXp = at<char>(ws, W.dXp);
  void* tmp = at<char>(ws, W.tmp);

  prof_mark(ST_BEGIN, s);
  // fused rows: no combine-bwd pass (no read of y): dy = the UNWEIGHTED rows of dY (a plain gather, or with 2 the by-product
  // of dgrad-down's own gather); dgrad-down applies w and produces dw in its epilogue
  const int fused = rows_fused(cfg);
  if (!fused) MOE_CHECK(combine_bwd(cfg, dY, y, w, f2p, p2f, offsets, dy, dw, s));         // R8 combine-bwd
  if (fused == 1) MOE_CHECK(gather_rows(cfg, dY, cfg->H, elem_bytes(cfg), f2p, p2f, offsets, dy, s));
  prof_mark(ST_COMBINE_BWD, s);
  FfnGroup g{cfg->dtype, e_ffn(cfg), cfg->H, cfg->F, padded_rows(cfg), offsets, counts,
             (cfg->row_align % 128 == 0) ? mtile : nullptr, cfg->row_align,
             ST_GEMM1_SWIGLU, ST_GEMM2, ST_DGRAD_DOWN_SWIGLU, ST_DGRAD_GATEUP, ST_WGRAD};
  set_opts(g, cfg);
  if (fused) { g.gidx = p2f; g.gK = cfg->K; g.g_rows = cfg->T; g.roww = w; g.dwpart = at<float>(ws, W.dwpart); }
  if (fused == 2) g.tok_in = dY;
  Fp8Bufs q, qs;
  memset(&q, 0, sizeof(q));
  memset(&qs, 0, sizeof(qs));
  if (fp8) {
    const int mode = cfg->fp8_scale_mode;
    uint8_t* dYq = at<uint8_t>(ws, W.dYq);
    float* dYq_s = at<float>(ws, W.dYq_s);
    MOE_CHECK(fp8_quantize_act(dY, cfg->T, cfg->H, mode, dYq, dYq_s, s));                  // Q-dY (w applied after the GEMM)
    MOE_CHECK(gather_rows(cfg, dYq, cfg->H, 1, f2p, p2f, offsets, at<uint8_t>(ws, W.dyq), s));
    MOE_CHECK(fp8_gather_scales(dYq_s, p2f, offsets, cfg->E, cfg->K, cfg->H / 128, at<float>(ws, W.dyq_s), s));
    prof_mark(ST_QUANT, s);
    q.Wgq = at<uint8_t>(ctx, C.Wgq); q.Wgq_s = at<float>(ctx, C.Wgq_s);
    q.Wuq = at<uint8_t>(ctx, C.Wuq); q.Wuq_s = at<float>(ctx, C.Wuq_s);
    q.Wdq = at<uint8_t>(ctx, C.Wdq); q.Wdq_s = at<float>(ctx, C.Wdq_s);
    q.dyq = at<uint8_t>(ws, W.dyq); q.dyq_s = at<float>(ws, W.dyq_s);
    q.dguq = at<uint8_t>(ws, W.dguq); q.dguq_s = at<float>(ws, W.dguq_s);
    q.p2f = p2f; q.w = w; q.mode = mode;
    qs = q;
    qs.Wgq = at<uint8_t>(ctx, C.Wgsq); qs.Wgq_s = at<float>(ctx, C.Wgsq_s);
    qs.Wuq = at<uint8_t>(ctx, C.Wusq); qs.Wuq_s = at<float>(ctx, C.Wusq_s);
    qs.Wdq = at<uint8_t>(ctx, C.Wdsq); qs.Wdq_s = at<float>(ctx, C.Wdsq_s);
    qs.dyq = dYq; qs.dyq_s = dYq_s;
    qs.dguq = at<uint8_t>(ws, W.dgusq); qs.dguq_s = at<float>(ws, W.dgusq_s);
    qs.p2f = nullptr; qs.w = nullptr;
    MOE_CHECK(ffn_bwd_fp8(g, q, dy, Xp, gu, a, dgu, dXp, dWg, dWu, dWd, s));               // R8 expert FFN on the codes
  } else {
    MOE_CHECK(ffn_bwd(g, dy, Xp, gu, a, Wg, Wu, Wd, tmp, dgu, dXp, dWg, dWu, dWd, s));     // R8 expert FFN
    if (fused) {
      MOE_CHECK(dw_reduce(cfg, g.dwpart, 2 * (int)ceil_div(cfg->F, 256), f2p, dw, s));     // dw[t,j] = <da_r, a_r>
      prof_mark(ST_COMBINE_BWD, s);
    }
  }
  MOE_CHECK(zc_backward(cfg, offsets, counts, dy, dgu, dXp, ex ? ex->d_zc_const : nullptr, s));      // V2: dXp = 0 | dy | 0
  const bool dense = dense_router_bwd(cfg);
  if (dense)                                                                                          // R8 router + A3
    MOE_CHECK(router_bwd_dense(cfg, z, idx, w, dw, cfg->aux_coef != 0.f ? at<float>(ctx, C.aux_f) : nullptr, X, Wr,
                               offsets + cfg->E + 1, dz, at<float>(ws, W.dzd), at<char>(ws, W.dzb), dWr, at<char>(ws, W.dXr),
                               s));
  else
    MOE_CHECK(router_bwd(cfg, z, idx, w, dw, f2p, offsets, counts, (cfg->row_align % 128 == 0) ? mtile : nullptr,
                         Xp, X, p2f, dz, dzp, at<float>(ws, W.dwr_part), dWr, s));                                    // R8 router
  prof_mark(ST_ROUTER_BWD, s);
  const void* dXs = nullptr;
  if (shared) {
    const int32_t* off_s = offsets + cfg->E + 1;
    FfnGroup gs{cfg->dtype, 1, cfg->H, cfg->F_shared, cfg->T, off_s, nullptr, nullptr, 1,
                ST_SHARED_FWD, ST_SHARED_FWD, ST_SHARED_BWD, ST_SHARED_BWD, ST_SHARED_BWD};
    set_opts(gs, cfg);
    if (fp8)
      MOE_CHECK(ffn_bwd_fp8(gs, qs, dY, X, at<char>(ctx, C.gu_s), at<char>(ctx, C.a_s), at<char>(ws, W.dgu_s),
                            at<char>(ws, W.dXs), dWg_s, dWu_s, dWd_s, s));
    else
      MOE_CHECK(ffn_bwd(gs, dY, X, at<char>(ctx, C.gu_s), at<char>(ctx, C.a_s), Wg_s, Wu_s, Wd_s, tmp,
                        at<char>(ws, W.dgu_s), at<char>(ws, W.dXs), dWg_s, dWu_s, dWd_s, s));
    dXs = at<char>(ws, W.dXs);
  }
  // dX[t] = sum_j dXp[f2p[tK+j]] + dXs[t] + sum_j dz[t,j] Wr[idx[t,j]]   (dense router backward: + (dz Wr)[t] instead)
  if (dense)
    MOE_CHECK(combine(cfg, dXp, nullptr, f2p, dXs, at<char>(ws, W.dXr), nullptr, nullptr, nullptr, dX, s));
  else
    MOE_CHECK(combine(cfg, dXp, nullptr, f2p, dXs, nullptr, dz, idx, Wr, dX, s));
  prof_mark(ST_DX_COMBINE, s);
  return MOE_OK;
}

// The weight-gradient half of the backward on its own (the layer-level piece of a delayed wgrad):
// reads what moe_layer_fwd left in ctx (Xp, a) and what a preceding moe_layer_bwd (called with NULL weight gradients)
// left in ws (dy, dgu), which therefore must not be reused in between.
extern "C" int32_t moe_layer_wgrad(const moe_config_t* cfg, const void* X, const void* dY, const void* ctx, const void* ws,
                                   void* dWg, void* dWu, void* dWd, void* dWg_s, void* dWu_s, void* dWd_s,
                                   int32_t accumulate_fp32, void* stream) {
  if (!cfg || !X || !dY || !ctx || !ws || !dWg || !dWu || !dWd) return MOE_ERR_INVALID_ARG;
  MOE_CHECK(layer_preflight(cfg, true));
  {   // the fp32-accumulate and fp8 weight gradients exist on the tensor-core path only: say so before any launch
    const bool tc_ok = cfg->dtype != 0 && cfg->H % 64 == 0 && cfg->F % 64 == 0 && cfg->row_align % 128 == 0 &&
                       (cfg->F_shared % 64 == 0);
    if ((accumulate_fp32 || cfg->dtype == 2) && !tc_ok) return MOE_ERR_UNSUPPORTED;
  }
  const bool shared = cfg->F_shared > 0;
  const bool wgrad_s = dWg_s || dWu_s || dWd_s;
  if (wgrad_s && !(shared && dWg_s && dWu_s && dWd_s)) return MOE_ERR_INVALID_ARG;
  cudaStream_t s = as_stream(stream);
  const CtxLayout C = ctx_layout(cfg);
  const WsLayout W = ws_layout(cfg);
  const int32_t* offsets = at<int32_t>(ctx, C.offsets);
  FfnGroup g{cfg->dtype, e_ffn(cfg), cfg->H, cfg->F, padded_rows(cfg), offsets, at<int32_t>(ctx, C.counts),
             (cfg->row_align % 128 == 0) ? at<int32_t>(ctx, C.mtile) : nullptr, cfg->row_align,
             ST_GEMM1_SWIGLU, ST_GEMM2, ST_DGRAD_DOWN_SWIGLU, ST_DGRAD_GATEUP, ST_WGRAD};
  set_opts(g, cfg);
  prof_mark(ST_BEGIN, s);
  MOE_CHECK(ffn_wgrad(g, at<char>(ws, W.dy), at<char>(ctx, C.Xp), at<char>(ctx, C.a), at<char>(ws, W.dgu), dWg, dWu, dWd,
                      accumulate_fp32 ? 1 : 0, s));
  if (wgrad_s) {
    FfnGroup gs{cfg->dtype, 1, cfg->H, cfg->F_shared, cfg->T, offsets + cfg->E + 1, nullptr, nullptr, 1,
                ST_SHARED_FWD, ST_SHARED_FWD, ST_SHARED_BWD, ST_SHARED_BWD, ST_SHARED_BWD};
    set_opts(gs, cfg);
    MOE_CHECK(ffn_wgrad(gs, dY, X, at<char>(ctx, C.a_s), at<char>(ws, W.dgu_s), dWg_s, dWu_s, dWd_s, accumulate_fp32 ? 1 : 0, s));
  }
  return MOE_OK;
}
