// Config validation, ctx / ws byte layouts and the small query entry points of the C ABI.
#include <string.h>

#include "common.cuh"
#include "tile_tables.cuh"

namespace moe {

long long g_launches = 0;

int32_t validate(const moe_config_t* c) {
  if (!c) return MOE_ERR_INVALID_ARG;
  if (c->T <= 0 || c->H <= 0 || c->E <= 0 || c->K <= 0 || c->F <= 0) return MOE_ERR_INVALID_ARG;
  if (c->n_group < 1 || c->topk_group < 1 || c->topk_group > c->n_group) return MOE_ERR_INVALID_ARG;
  if (c->score_fn < 0 || c->score_fn > 1 || c->group_score < 0 || c->group_score > 1) return MOE_ERR_INVALID_ARG;
  if (c->dtype < 0 || c->dtype > 2 || c->fp8_scale_mode < 0 || c->fp8_scale_mode > 1) return MOE_ERR_INVALID_ARG;
  if (c->row_align < 1 || c->F_shared < 0) return MOE_ERR_INVALID_ARG;
  if (c->K > c->E) return MOE_ERR_UNSUPPORTED;
  if (c->E % c->n_group != 0) return MOE_ERR_UNSUPPORTED;
  if ((int64_t)c->K > (int64_t)c->topk_group * (c->E / c->n_group)) return MOE_ERR_UNSUPPORTED;
  if ((int64_t)c->T * c->K >= (1ll << 31) || padded_rows(c) >= (1ll << 31)) return MOE_ERR_UNSUPPORTED;
  const int a = c->dtype == 0 ? 4 : 8;  // 16-byte rows
  if (c->H % a != 0 || c->F % a != 0 || c->F_shared % a != 0) return MOE_ERR_UNSUPPORTED;
  if (c->dtype == 2 && (c->H % 128 != 0 || c->F % 128 != 0 || c->F_shared % 128 != 0)) return MOE_ERR_UNSUPPORTED;
  // widened rows
  if (c->route_mode < 0 || c->route_mode > 1 || c->n_zero < 0 || c->n_copy < 0 || c->n_const < 0) return MOE_ERR_INVALID_ARG;
  if (c->route_mode == 1 && (c->score_fn != 1 || c->n_group != 1 || c->has_bias)) return MOE_ERR_INVALID_ARG;
  if (n_zc(c) >= c->E) return MOE_ERR_INVALID_ARG;              // at least one FFN expert
  if (!(c->aux_coef == c->aux_coef) || !(c->aux_zc_weight == c->aux_zc_weight)) return MOE_ERR_INVALID_ARG;   // NaN
  if (c->opt_rows_fused < 0 || c->opt_rows_fused > 3 || c->opt_pair < 0 || c->opt_pair > 3 || c->opt_fp8_wide < 0 ||
      c->opt_fp8_wide > 3 || c->opt_fp8_fused_quant < 0 || c->opt_fp8_fused_quant > 2)
    return MOE_ERR_INVALID_ARG;
  return MOE_OK;
}

int32_t layer_preflight(const moe_config_t* c, bool backward) {
  MOE_CHECK(validate(c));
  // moe_route (route.cu): one warp per token holds E/32 keys per lane, K <= 32 output slots, one lane per group
  if (c->E > 1024 || c->K > 32 || c->n_group > 32) return MOE_ERR_UNSUPPORTED;
  // fp8 expert GEMMs need 128-row tiles that belong to one expert
  if (c->dtype == 2 && c->row_align % 128 != 0) return MOE_ERR_UNSUPPORTED;
  (void)backward;
  return MOE_OK;
}

bool rows_fusable(const moe_config_t* c) {
  return c->dtype == 1 && c->H % 64 == 0 && c->F % 64 == 0 && c->row_align % 128 == 0 && n_zc(c) == 0;
}

int rows_fused(const moe_config_t* c) {
  if (!rows_fusable(c)) return 0;
  return c->opt_rows_fused ? c->opt_rows_fused - 1 : 1;
}

int device_sm_count() {
  static int sm[MAX_DEVICES] = {0};
  const int d = current_device();
  if (d < 0) return 0;
  if (sm[d] == 0 && cudaDeviceGetAttribute(&sm[d], cudaDevAttrMultiProcessorCount, d) != cudaSuccess) {
    cudaGetLastError();
    sm[d] = 0;
  }
  return sm[d];
}

namespace {
struct Carver {
  size_t cur = 0;
  size_t take(size_t bytes) {
    const size_t at = cur;
    cur += (bytes + 255) / 256 * 256;
    return at;
  }
};
}  // namespace

CtxLayout ctx_layout(const moe_config_t* c) {
  CtxLayout L;
  memset(&L, 0, sizeof(L));
  Carver k;
  const size_t es = elem_bytes(c);
  const size_t R = (size_t)padded_rows(c), T = c->T, H = c->H, F = c->F, E = c->E, Fs = c->F_shared;
  L.z = k.take(T * E * 4);
  L.idx = k.take(T * c->K * 4);
  L.w = k.take(T * c->K * 4);
  L.counts = k.take(E * 4);
  L.offsets = k.take((E + 1) * 4 + 16);  // + {0, T} for the shared expert's single group
  L.p2f = k.take(R * 4);
  L.f2p = k.take(T * c->K * 4);
  L.mtile = k.take(tile_table_ints((int64_t)R, c->E) * 4);   // mtile | plist | olist (tile_tables.cuh)
  L.Xp = k.take(R * H * es);
  L.gu = k.take(R * 2 * F * es);
  L.a = k.take(R * F * es);
  L.y = k.take(R * H * es);
  if (Fs) {
    L.gu_s = k.take(T * 2 * Fs * es);
    L.a_s = k.take(T * Fs * es);
    L.y_s = k.take(T * H * es);
  }
  if (c->aux_coef != 0.f) {
    L.aux_f = k.take(E * 4);
    L.aux_P = k.take(E * 4);
    L.aux_loss = k.take(4);
  }
  if (c->dtype == 2) {
    L.Xq = k.take(T * H); L.Xq_s = k.take(T * (H / 128) * 4);
    L.Xpq = k.take(R * H); L.Xpq_s = k.take(R * (H / 128) * 4);
    L.aq = k.take(R * F); L.aq_s = k.take(R * (F / 128) * 4);
    L.Wgq = k.take(E * F * H); L.Wgq_s = k.take(E * (F / 128) * (H / 128) * 4);
    L.Wuq = k.take(E * F * H); L.Wuq_s = k.take(E * (F / 128) * (H / 128) * 4);
    L.Wdq = k.take(E * H * F); L.Wdq_s = k.take(E * (H / 128) * (F / 128) * 4);
    if (Fs) {
      L.asq = k.take(T * Fs); L.asq_s = k.take(T * (Fs / 128) * 4);
      L.Wgsq = k.take(Fs * H); L.Wgsq_s = k.take((Fs / 128) * (H / 128) * 4);
      L.Wusq = k.take(Fs * H); L.Wusq_s = k.take((Fs / 128) * (H / 128) * 4);
      L.Wdsq = k.take(H * Fs); L.Wdsq_s = k.take((H / 128) * (Fs / 128) * 4);
    }
  }
  L.total = k.cur;
  return L;
}

WsLayout ws_layout(const moe_config_t* c) {
  WsLayout L;
  memset(&L, 0, sizeof(L));
  Carver k;
  const size_t es = elem_bytes(c);
  const size_t R = (size_t)padded_rows(c), T = c->T, H = c->H, F = c->F, E = c->E, Fs = c->F_shared;
  const size_t nchunks = (T * c->K + PERM_CHUNK - 1) / PERM_CHUNK;
  L.hist = k.take(nchunks * E * 4);
  // tmp: M-tile table for stand-alone calls, or da [R,F] / da_s [T,Fs] on the CUDA-core path
  size_t tmp = tile_table_ints((int64_t)R, c->E) * 4;
  if (R * F * es > tmp) tmp = R * F * es;
  if (T * Fs * es > tmp) tmp = T * Fs * es;
  L.tmp = k.take(tmp);
  L.dw = k.take(T * c->K * 4);
  L.dz = k.take(T * c->K * 4);
  L.dzp = k.take(R * 4);
  L.dwr_part = k.take((R / 128 + 1) * H * 4);   // per-tile partial sums of dWr (fp32)
  L.dy = k.take(R * H * es);                                 // fused rows: the UNWEIGHTED gathered dY
  // reserved whenever the config COULD fuse, whatever cfg->opt_rows_fused says: every offset below must be the same for
  // the sizing query, moe_layer_bwd and a later moe_layer_wgrad even if the caller changes the selector between them
  if (rows_fusable(c)) L.dwpart = k.take(2 * ((F + 255) / 256) * R * 4);
  L.dgu = k.take(R * 2 * F * es);
  L.dXp = k.take(R * H * es);
  if (Fs) {
    L.dgu_s = k.take(T * 2 * Fs * es);
    L.dXs = k.take(T * H * es);
  }
  if (c->dtype == 2) {
    L.dYq = k.take(T * H); L.dYq_s = k.take(T * (H / 128) * 4);
    L.dyq = k.take(R * H); L.dyq_s = k.take(R * (H / 128) * 4);
    L.dguq = k.take(R * 2 * F); L.dguq_s = k.take(R * (2 * F / 128) * 4);
    if (Fs) { L.dgusq = k.take(T * 2 * Fs); L.dgusq_s = k.take(T * (2 * Fs / 128) * 4); }
  }
  if (dense_router_bwd(c)) {
    const size_t Ep = (E + 63) / 64 * 64;       // bf16 copy padded so that it is a legal TMA / UMMA operand
    L.dzd = k.take(T * E * 4);
    L.dzb = k.take(T * Ep * 2);
    L.dXr = k.take(T * H * es);
  }
  if (c->aux_coef != 0.f) L.aux_part = k.take(((T + AUX_TOKENS_PER_CTA - 1) / AUX_TOKENS_PER_CTA) * E * 4);
  L.total = k.cur;
  return L;
}

}  // namespace moe

using namespace moe;

extern "C" const char* moe_status_string(int32_t status) {
  switch (status) {
    case MOE_OK: return "ok";
    case MOE_ERR_INVALID_ARG: return "invalid argument";
    case MOE_ERR_UNSUPPORTED: return "unsupported configuration";
    case MOE_ERR_WORKSPACE: return "workspace error";
    case MOE_ERR_CUDA: return "CUDA error";
    case MOE_ERR_TOO_LARGE: return "problem exceeds the built-in scratch (MOE_PERMUTE_STATIC_WS_BYTES) of moe_permute_static_ws";
    default: return "unknown status";
  }
}

extern "C" int32_t moe_version(void) { return 100; }

extern "C" int64_t moe_launch_count(void) { return g_launches; }

extern "C" int32_t moe_layer_rows_fused(const moe_config_t* cfg) {
  if (validate(cfg) != MOE_OK) return MOE_ERR_INVALID_ARG;
  return rows_fused(cfg);
}

extern "C" int64_t moe_padded_rows(const moe_config_t* cfg) {
  if (validate(cfg) != MOE_OK) return -1;
  return padded_rows(cfg);
}

extern "C" int32_t moe_workspace_bytes(const moe_config_t* cfg, size_t* ws_bytes, size_t* ctx_bytes) {
  MOE_CHECK(validate(cfg));
  if (ws_bytes) *ws_bytes = ws_layout(cfg).total;
  if (ctx_bytes) *ctx_bytes = ctx_layout(cfg).total;
  return MOE_OK;
}

extern "C" int32_t moe_ctx_field(const moe_config_t* cfg, const char* name, size_t* byte_offset, size_t* byte_len) {
  MOE_CHECK(validate(cfg));
  if (!name || !byte_offset || !byte_len) return MOE_ERR_INVALID_ARG;
  const CtxLayout L = ctx_layout(cfg);
  const size_t es = elem_bytes(cfg);
  const size_t R = (size_t)padded_rows(cfg), T = cfg->T, H = cfg->H, F = cfg->F, E = cfg->E, Fs = cfg->F_shared;
  struct { const char* n; size_t off, len; } tab[] = {
      {"z", L.z, T * E * 4}, {"counts", L.counts, E * 4}, {"offsets", L.offsets, (E + 1) * 4},
      {"perm_to_flat", L.p2f, R * 4}, {"flat_to_perm", L.f2p, T * cfg->K * 4}, {"Xp", L.Xp, R * H * es},
      {"gu", L.gu, R * 2 * F * es}, {"a", L.a, R * F * es}, {"y", L.y, R * H * es},
      {"gu_s", L.gu_s, T * 2 * Fs * es}, {"a_s", L.a_s, T * Fs * es}, {"y_s", L.y_s, T * H * es},
      {"aux_f", L.aux_f, E * 4}, {"aux_P", L.aux_P, E * 4}, {"aux_loss", L.aux_loss, 4},
      {"aq", L.aq, R * F}, {"aq_s", L.aq_s, R * (F / 128) * 4}};
  for (auto& t : tab)
    if (strcmp(t.n, name) == 0) {
      const size_t nl = strlen(name);
      if (nl > 2 && strcmp(name + nl - 2, "_s") == 0 && !Fs) return MOE_ERR_INVALID_ARG;
      if (strncmp(name, "aux_", 4) == 0 && cfg->aux_coef == 0.f) return MOE_ERR_INVALID_ARG;
      if (strncmp(name, "aq", 2) == 0 && cfg->dtype != 2) return MOE_ERR_INVALID_ARG;
      *byte_offset = t.off;
      *byte_len = t.len;
      return MOE_OK;
    }
  return MOE_ERR_INVALID_ARG;
}

extern "C" int32_t moe_ws_field(const moe_config_t* cfg, const char* name, size_t* byte_offset, size_t* byte_len) {
  MOE_CHECK(validate(cfg));
  if (!name || !byte_offset || !byte_len) return MOE_ERR_INVALID_ARG;
  const WsLayout L = ws_layout(cfg);
  const size_t es = elem_bytes(cfg);
  const size_t R = (size_t)padded_rows(cfg), T = cfg->T, H = cfg->H, F = cfg->F;
  struct { const char* n; size_t off, len; } tab[] = {
      {"dw", L.dw, T * cfg->K * 4}, {"dz", L.dz, T * cfg->K * 4}, {"dy", L.dy, R * H * es},
      {"dgu", L.dgu, R * 2 * F * es}, {"dXp", L.dXp, R * H * es}, {"dz_dense", L.dzd, T * (size_t)cfg->E * 4},
      {"dguq", L.dguq, R * 2 * F}, {"dguq_s", L.dguq_s, R * (2 * F / 128) * 4}};
  for (auto& t : tab)
    if (strcmp(t.n, name) == 0) {
      if (strcmp(name, "dz_dense") == 0 && !dense_router_bwd(cfg)) return MOE_ERR_INVALID_ARG;
      if (strncmp(name, "dguq", 4) == 0 && cfg->dtype != 2) return MOE_ERR_INVALID_ARG;
      *byte_offset = t.off;
      *byte_len = t.len;
      return MOE_OK;
    }
  return MOE_ERR_INVALID_ARG;
}

// ---- stage timing -------------------------------------------------------------------------------------
namespace moe {
int g_prof_on = 0;
namespace {
constexpr int MAX_MARKS = 8192;
cudaEvent_t g_ev[MAX_MARKS];
int g_ev_stage[MAX_MARKS];
int g_ev_created = 0, g_ev_used = 0, g_ev_device = -1;
bool g_ev_overflow = false;
const char* const kStageNames[ST_COUNT] = {"begin", "router_gemm", "route", "maps", "permute", "gemm1_swiglu", "gemm2",
                                           "combine", "combine_bwd", "dgrad_down_swiglu", "dgrad_gateup", "wgrad",
                                           "router_bwd", "dx_combine", "shared_fwd", "shared_bwd", "quant"};
}  // namespace
void prof_mark_impl(int stage, cudaStream_t s) {
  if (g_ev_used >= MAX_MARKS) { g_ev_overflow = true; return; }   // reported by moe_profile_stage_ms, never silently dropped
  const int dev = current_device();
  if (dev != g_ev_device) {            // events belong to the device they were created on: start over on a new one
    for (int i = 0; i < g_ev_created; ++i) cudaEventDestroy(g_ev[i]);
    cudaGetLastError();
    g_ev_created = g_ev_used = 0;
    g_ev_device = dev;
  }
  if (g_ev_used >= g_ev_created) {
    if (cudaEventCreate(&g_ev[g_ev_created]) != cudaSuccess) { cudaGetLastError(); return; }
    ++g_ev_created;
  }
  g_ev_stage[g_ev_used] = stage;
  cudaEventRecord(g_ev[g_ev_used++], s);
}
}  // namespace moe

extern "C" int32_t moe_profile_enable(int32_t on) {
  g_prof_on = on ? 1 : 0;
  g_ev_used = 0;
  g_ev_overflow = false;
  return MOE_OK;
}

extern "C" int32_t moe_profile_stage_ms(const char* stage, double* total_ms, int64_t* segments) {
  if (!stage || !total_ms || !segments) return MOE_ERR_INVALID_ARG;
  int want = -1;
  for (int i = 1; i < ST_COUNT; ++i)
    if (strcmp(kStageNames[i], stage) == 0) want = i;
  if (want < 0) return MOE_ERR_INVALID_ARG;
  if (g_ev_overflow) return MOE_ERR_WORKSPACE;   // more than MAX_MARKS marks since moe_profile_enable: totals would be truncated
  double sum = 0;
  int64_t n = 0;
  for (int i = 1; i < g_ev_used; ++i) {
    if (g_ev_stage[i] != want) continue;
    if (cudaEventSynchronize(g_ev[i]) != cudaSuccess) { cudaGetLastError(); return MOE_ERR_CUDA; }
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, g_ev[i - 1], g_ev[i]) != cudaSuccess) { cudaGetLastError(); return MOE_ERR_CUDA; }
    sum += ms;
    ++n;
  }
  *total_ms = sum;
  *segments = n;
  return MOE_OK;
}
