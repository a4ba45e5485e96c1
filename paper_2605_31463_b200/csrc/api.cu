// Public grouped-GEMM entry points and the host-buffer step (include/moe_b200.h).
#include <new>
#include <string.h>

#include "fp8.cuh"
#include "gemm_tc.cuh"
#include "tile_tables.cuh"

using namespace moe;

extern "C" int32_t moe_grouped_gemm_fwd(const moe_config_t* cfg, int32_t N, int32_t Kdim, const void* A,
                                        const void* B, const int32_t* offsets, void* C, const void* a_scales,
                                        const void* b_scales, void* ws, void* stream) {
  if (!cfg || !A || !B || !offsets || !C || !ws || N <= 0 || Kdim <= 0) return MOE_ERR_INVALID_ARG;
  MOE_CHECK(validate(cfg));
  cudaStream_t s = as_stream(stream);
  int32_t* mtile = reinterpret_cast<int32_t*>((char*)ws + ws_layout(cfg).tmp);
  if (cfg->dtype == 2) {   // e4m3 codes + block scales (R9)
    if (!a_scales || !b_scales) return MOE_ERR_INVALID_ARG;
    if (cfg->row_align % 128 != 0 || Kdim % 128 != 0 || N % 128 != 0) return MOE_ERR_UNSUPPORTED;
    MOE_CHECK(tc_prepare_tiles(offsets, cfg->E, padded_rows(cfg), mtile, s));
    F8Call c;
    memset(&c, 0, sizeof(c));
    c.mode = F8_FWD; c.opt_wide = cfg->opt_fp8_wide; c.E = cfg->E; c.rows_cap = padded_rows(cfg); c.mtile = mtile;
    c.A = (const uint8_t*)A; c.lda = Kdim; c.a_scales = (const float*)a_scales;
    c.B0 = (const uint8_t*)B; c.b0_scales = (const float*)b_scales; c.b_rows = N; c.b_cols = Kdim; c.N = N;
    c.out0 = C; c.ld0 = N;
    return fp8_gemm(c, s);
  }
  if (cfg->dtype == 1 && cfg->row_align % 128 == 0 && Kdim % 64 == 0 && N % 8 == 0) {
    MOE_CHECK(tc_prepare_tiles(offsets, cfg->E, padded_rows(cfg), mtile, s));
    TcCall c;
    memset(&c, 0, sizeof(c));
    c.mode = TC_FWD; c.opt_pair = cfg->opt_pair; c.E = cfg->E; c.rows_cap = padded_rows(cfg); c.offsets = offsets; c.mtile = mtile;
    c.plist = mtile + tile_plist_off(c.rows_cap); c.olist = mtile + tile_olist_off(c.rows_cap);
    c.A = A; c.lda = Kdim; c.B0 = B; c.b_rows = N; c.b_cols = Kdim; c.N = N; c.Kd = Kdim; c.out0 = C; c.ld0 = N;
    const int32_t st = tc_gemm(c, s);
    if (st != MOE_ERR_UNSUPPORTED) return st;
  }
  return simt_grouped_gemm(0, cfg->dtype, cfg->E, N, Kdim, A, Kdim, B, nullptr, 0, offsets, C, N, padded_rows(cfg), 0,
                           s);
}

extern "C" int32_t moe_grouped_gemm_bwd(const moe_config_t* cfg, int32_t N, int32_t Kdim, const void* dC,
                                        const void* A, const void* B, const int32_t* offsets, void* dA, void* dB,
                                        void* ws, void* stream) {
  if (!cfg || !dC || !offsets || !ws || N <= 0 || Kdim <= 0) return MOE_ERR_INVALID_ARG;
  if ((dA && !B) || (dB && !A)) return MOE_ERR_INVALID_ARG;
  MOE_CHECK(validate(cfg));
  if (cfg->dtype == 2) return MOE_ERR_UNSUPPORTED;
  cudaStream_t s = as_stream(stream);
  int32_t* mtile = reinterpret_cast<int32_t*>((char*)ws + ws_layout(cfg).tmp);
  if (cfg->dtype == 1 && cfg->row_align % 128 == 0 && N % 64 == 0 && Kdim % 8 == 0) {
    MOE_CHECK(tc_prepare_tiles(offsets, cfg->E, padded_rows(cfg), mtile, s));
    TcCall c;
    memset(&c, 0, sizeof(c));
    c.opt_pair = cfg->opt_pair; c.E = cfg->E; c.rows_cap = padded_rows(cfg); c.offsets = offsets; c.mtile = mtile;
    c.plist = mtile + tile_plist_off(c.rows_cap); c.olist = mtile + tile_olist_off(c.rows_cap);
    if (dA) {   // dA = dC B[e]: contraction over B's rows
      c.mode = TC_DGRAD; c.A = dC; c.lda = N; c.B0 = B; c.B1 = nullptr; c.b_rows = N; c.b_cols = Kdim; c.N = Kdim;
      c.out0 = dA; c.ld0 = Kdim;
      MOE_CHECK(tc_gemm(c, s));
    }
    if (dB) {   // dB[e] = dC_e^T A_e
      c.mode = TC_WGRAD; c.A = dC; c.lda = N; c.a_col0 = 0; c.M = N; c.A2 = A; c.lda2 = Kdim; c.N = Kdim;
      c.out0 = dB; c.ld0 = Kdim;
      MOE_CHECK(tc_gemm(c, s));
    }
    return MOE_OK;
  }
  const int64_t R = padded_rows(cfg);
  if (dA) MOE_CHECK(simt_grouped_gemm(1, cfg->dtype, cfg->E, N, Kdim, nullptr, 0, B, dC, N, offsets, dA, Kdim, R, 0, s));
  if (dB) MOE_CHECK(simt_grouped_gemm(2, cfg->dtype, cfg->E, N, Kdim, A, Kdim, nullptr, dC, N, offsets, dB, 0, R, 0, s));
  return MOE_OK;
}

// Everything moe_layer_fwd / moe_layer_bwd would refuse about a host step's arguments, decided BEFORE the first copy or
// event wait is enqueued, so that an INVALID_ARG / UNSUPPORTED host step leaves the streams (and the pipeline object)
// untouched.  The host steps take no moe_extras_t: configs that need one (threshold routing, constant experts) are
// rejected here; run those through moe_layer_fwd_ex / moe_layer_bwd_ex.
static int32_t host_step_preflight(const moe_config_t* cfg, const void* Wr, const float* bias, const void* Wg,
                                   const void* Wu, const void* Wd, const void* Wg_s, const void* Wu_s, const void* Wd_s,
                                   const void* dWg, const void* dWu, const void* dWd, const void* dWg_s,
                                   const void* dWu_s, const void* dWd_s, const int32_t* topk_idx, const float* topk_w,
                                   const void* ctx, const void* ws) {
  MOE_CHECK(layer_preflight(cfg, true));
  if (!Wr || !topk_idx || !topk_w || !ctx || !ws) return MOE_ERR_INVALID_ARG;
  if (cfg->has_bias && !bias) return MOE_ERR_INVALID_ARG;
  if (cfg->route_mode == 1 || cfg->n_const > 0) return MOE_ERR_INVALID_ARG;      // need moe_extras_t
  const bool shared = cfg->F_shared > 0;
  const bool cached = cfg->dtype == 2 && !Wg && !Wu && !Wd;                      // FP8 weight cache in ctx
  if (!cached && (!Wg || !Wu || !Wd)) return MOE_ERR_INVALID_ARG;
  if (shared && !cached && (!Wg_s || !Wu_s || !Wd_s)) return MOE_ERR_INVALID_ARG;
  const bool wgrad = dWg || dWu || dWd;
  if (wgrad && !(dWg && dWu && dWd)) return MOE_ERR_INVALID_ARG;
  const bool wgrad_s = dWg_s || dWu_s || dWd_s;
  if (wgrad_s && !(shared && dWg_s && dWu_s && dWd_s)) return MOE_ERR_INVALID_ARG;
  return MOE_OK;
}

extern "C" int32_t moe_layer_step_host(const moe_config_t* cfg, const void* X_host, const void* dY_host, void* Y_host,
                                       void* dX_host, void* X_dev, void* dY_dev, void* Y_dev, void* dX_dev,
                                       const void* Wr, const float* bias, const void* Wg, const void* Wu,
                                       const void* Wd, const void* Wg_s, const void* Wu_s, const void* Wd_s, void* dWr,
                                       void* dWg, void* dWu, void* dWd, void* dWg_s, void* dWu_s, void* dWd_s,
                                       int32_t* topk_idx, float* topk_w, void* ctx, void* ws, void* stream) {
  if (!cfg || !X_host || !dY_host || !Y_host || !dX_host || !X_dev || !dY_dev || !Y_dev || !dX_dev)
    return MOE_ERR_INVALID_ARG;
  MOE_CHECK(host_step_preflight(cfg, Wr, bias, Wg, Wu, Wd, Wg_s, Wu_s, Wd_s, dWg, dWu, dWd, dWg_s, dWu_s, dWd_s, topk_idx,
                                topk_w, ctx, ws));
  cudaStream_t s = as_stream(stream);
  const size_t bytes = (size_t)cfg->T * cfg->H * elem_bytes(cfg);
  MOE_CUDA(cudaMemcpyAsync(X_dev, X_host, bytes, cudaMemcpyHostToDevice, s));
  MOE_CUDA(cudaMemcpyAsync(dY_dev, dY_host, bytes, cudaMemcpyHostToDevice, s));
  MOE_CHECK(moe_layer_fwd(cfg, X_dev, Wr, bias, Wg, Wu, Wd, Wg_s, Wu_s, Wd_s, Y_dev, topk_idx, topk_w, ctx, ws, stream));
  MOE_CHECK(moe_layer_bwd(cfg, dY_dev, X_dev, Wr, Wg, Wu, Wd, Wg_s, Wu_s, Wd_s, ctx, dX_dev, dWr, dWg, dWu, dWd, dWg_s,
                          dWu_s, dWd_s, ws, stream));
  MOE_CUDA(cudaMemcpyAsync(Y_host, Y_dev, bytes, cudaMemcpyDeviceToHost, s));
  MOE_CUDA(cudaMemcpyAsync(dX_host, dX_dev, bytes, cudaMemcpyDeviceToHost, s));
  return MOE_OK;
}

// Pipelined host-buffer step: H2D of the step's inputs, fwd+bwd and D2H of its results run on three caller streams
// so that copy-in of step i+1 and copy-out of step i-1 overlap the compute of step i.  `slot` (0/1) selects which of
// the caller's two sets of device staging buffers this step uses; the six events that order the reuse of a slot
// (copy-in waits for the compute that last read the slot's inputs, compute waits for the copy-out that last read the
// slot's outputs) live in a CALLER-OWNED pipeline object created on the caller's current device, so the library
// itself holds no state for this call.
namespace {
struct Pipeline {
  uint32_t magic;
  int device;
  cudaEvent_t ev[2][3];
  bool used[2];
};
constexpr uint32_t PIPE_MAGIC = 0x4d6f4550u;   // "MoEP"
}  // namespace

extern "C" int32_t moe_pipeline_create(void** pipeline) {
  if (!pipeline) return MOE_ERR_INVALID_ARG;
  *pipeline = nullptr;
  const int dev = current_device();
  if (dev < 0) return MOE_ERR_CUDA;
  Pipeline* p = new (std::nothrow) Pipeline();
  if (!p) return MOE_ERR_WORKSPACE;
  p->magic = PIPE_MAGIC;
  p->device = dev;
  p->used[0] = p->used[1] = false;
  int made = 0;
  for (int i = 0; i < 2; ++i)
    for (int j = 0; j < 3; ++j, ++made)
      if (cudaEventCreateWithFlags(&p->ev[i][j], cudaEventDisableTiming) != cudaSuccess) {
        cudaGetLastError();
        for (int k = 0; k < made; ++k) cudaEventDestroy(p->ev[k / 3][k % 3]);
        delete p;
        return MOE_ERR_CUDA;
      }
  *pipeline = p;
  return MOE_OK;
}

extern "C" int32_t moe_pipeline_destroy(void* pipeline) {
  Pipeline* p = static_cast<Pipeline*>(pipeline);
  if (!p || p->magic != PIPE_MAGIC) return MOE_ERR_INVALID_ARG;
  for (int i = 0; i < 2; ++i)
    for (int j = 0; j < 3; ++j) cudaEventDestroy(p->ev[i][j]);
  cudaGetLastError();
  p->magic = 0;
  delete p;
  return MOE_OK;
}

extern "C" int32_t moe_layer_step_host_pipelined(
    void* pipeline, const moe_config_t* cfg, int32_t slot, const void* X_host, const void* dY_host, void* Y_host,
    void* dX_host, void* X_dev, void* dY_dev, void* Y_dev, void* dX_dev, const void* Wr, const float* bias, const void* Wg,
    const void* Wu, const void* Wd, const void* Wg_s, const void* Wu_s, const void* Wd_s, void* dWr, void* dWg, void* dWu,
    void* dWd, void* dWg_s, void* dWu_s, void* dWd_s, int32_t* topk_idx, float* topk_w, void* ctx, void* ws,
    void* stream_in, void* stream_compute, void* stream_out) {
  Pipeline* pl = static_cast<Pipeline*>(pipeline);
  if (!pl || pl->magic != PIPE_MAGIC) return MOE_ERR_INVALID_ARG;
  if (!cfg || !X_host || !dY_host || !Y_host || !dX_host || !X_dev || !dY_dev || !Y_dev || !dX_dev || slot < 0 || slot > 1)
    return MOE_ERR_INVALID_ARG;
  MOE_CHECK(host_step_preflight(cfg, Wr, bias, Wg, Wu, Wd, Wg_s, Wu_s, Wd_s, dWg, dWu, dWd, dWg_s, dWu_s, dWd_s, topk_idx,
                                topk_w, ctx, ws));
  if (current_device() != pl->device) return MOE_ERR_INVALID_ARG;   // the events belong to the device they were made on
  cudaStream_t si = as_stream(stream_in), sc = as_stream(stream_compute), so = as_stream(stream_out);
  cudaEvent_t ev_in = pl->ev[slot][0], ev_comp = pl->ev[slot][1], ev_out = pl->ev[slot][2];
  const size_t bytes = (size_t)cfg->T * cfg->H * elem_bytes(cfg);
  if (pl->used[slot]) MOE_CUDA(cudaStreamWaitEvent(si, ev_comp, 0));
  MOE_CUDA(cudaMemcpyAsync(X_dev, X_host, bytes, cudaMemcpyHostToDevice, si));
  MOE_CUDA(cudaMemcpyAsync(dY_dev, dY_host, bytes, cudaMemcpyHostToDevice, si));
  MOE_CUDA(cudaEventRecord(ev_in, si));
  MOE_CUDA(cudaStreamWaitEvent(sc, ev_in, 0));
  if (pl->used[slot]) MOE_CUDA(cudaStreamWaitEvent(sc, ev_out, 0));
  MOE_CHECK(moe_layer_fwd(cfg, X_dev, Wr, bias, Wg, Wu, Wd, Wg_s, Wu_s, Wd_s, Y_dev, topk_idx, topk_w, ctx, ws, stream_compute));
  MOE_CHECK(moe_layer_bwd(cfg, dY_dev, X_dev, Wr, Wg, Wu, Wd, Wg_s, Wu_s, Wd_s, ctx, dX_dev, dWr, dWg, dWu, dWd, dWg_s,
                          dWu_s, dWd_s, ws, stream_compute));
  MOE_CUDA(cudaEventRecord(ev_comp, sc));
  MOE_CUDA(cudaStreamWaitEvent(so, ev_comp, 0));
  MOE_CUDA(cudaMemcpyAsync(Y_host, Y_dev, bytes, cudaMemcpyDeviceToHost, so));
  MOE_CUDA(cudaMemcpyAsync(dX_host, dX_dev, bytes, cudaMemcpyDeviceToHost, so));
  MOE_CUDA(cudaEventRecord(ev_out, so));
  pl->used[slot] = true;
  return MOE_OK;
}
