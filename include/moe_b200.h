/* moe_b200.h -- C ABI of the B200-native (sm_100a) routed-expert MoE layer, forward and backward.
 *
 * What is computed: the hot path of PithTrain's MoE training step on one GPU
 * (BASELINE.json:north_star; §3.2 "MoE fwd/bwd have data-dependent
 * per-expert shapes", "fused SwiGLU fwd/bwd", "FP8 quantization"; App. B.2 "the
 * top-k expert IDs and their gating weights", "non-negative and sum to 1 over the top-k").  The paper
 * prints no equation for the layer; the exact arithmetic is the reading R1..R9 of SURVEY.md §8(c),
 * restated in DESIGN.md, and each entry point below names the R-step it implements.
 *
 * Conventions (all entry points)
 *  - Every pointer is a DEVICE pointer owned by the caller unless its name ends in `_host`.
 *    The library allocates no device memory.  Its only process-wide state is host-side and per device: lazily
 *    resolved driver entry points, "function attribute already raised" flags and the SM count, each indexed by
 *    the current device, plus the optional profiling marks of moe_profile_*.  Scratch comes from the caller
 *    (`ws`), sized by moe_workspace_bytes; the pipelined host step keeps its events in a caller-owned object.
 *  - Work is enqueued on `stream` (a cudaStream_t passed as void*; NULL = legacy default stream);
 *    calls return without synchronising.  Per-expert counts never visit the host.
 *  - Row-major, innermost dimension contiguous, base pointers 16-byte aligned.
 *  - Return value: MOE_OK or a negative moe_status.  INVALID_ARG, and UNSUPPORTED for every limit this header lists
 *    (the config checks, E <= 1024, K <= 32, n_group <= 32, FP8 needs row_align % 128 == 0), are decided before the
 *    first launch, so on those nothing has been enqueued and no output buffer has been touched.  MOE_ERR_CUDA (a failed
 *    launch or runtime call) can occur mid-way, and so can an UNSUPPORTED that only a later stage can discover (the
 *    driver refusing a tensor map for an exotic leading dimension): after either, ctx / ws / outputs are undefined.
 *    No exceptions, no aborts, no printing.  Inputs must be finite.
 *  - Activation / weight element type follows cfg->dtype: 0 = fp32, 1 = bf16, 2 = bf16 I/O with
 *    e4m3 block-scaled expert GEMMs.  Logits, gating weights and their gradients are always fp32.
 *  - Permuted-row tensors have TK_pad = moe_padded_rows(cfg) rows: expert group e occupies rows
 *    [offsets[e], offsets[e] + counts[e]) and starts at a multiple of cfg->row_align; padding rows
 *    map to -1 in perm_to_flat and hold zeros.  The tensor-core (bf16 / fp8) GEMMs require
 *    row_align to be a multiple of 128; the fp32 path accepts any row_align >= 1.
 */
#ifndef MOE_B200_H
#define MOE_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct moe_config_t {
  int32_t T, H, E, K, F;       /* tokens, hidden, routed experts, top-k, expert FFN width             */
  int32_t n_group, topk_group; /* 1,1 = no group limiting (R3); E % n_group == 0; n_group <= 32        */
  int32_t score_fn;            /* 0 = softmax, 1 = sigmoid (R2)                                        */
  int32_t group_score;         /* 0 = max, 1 = sum of the two largest keys in the group (R3)           */
  int32_t renorm;              /* 1 = divide the selected weights by their sum (R5)                    */
  float routed_scale;          /* multiplies w after renormalisation (R5)                              */
  int32_t has_bias;            /* selection-only per-expert bias b[E], no gradient (R2)                */
  int32_t F_shared;            /* 0 = no shared expert (R7)                                            */
  int32_t dtype;               /* 0 = fp32, 1 = bf16, 2 = fp8-e4m3 block-scaled GEMMs with bf16 I/O    */
  int32_t fp8_scale_mode;      /* 0 = fp32 amax/448, 1 = power of two (R9)                             */
  int32_t row_align;           /* expert groups start at multiples of this many rows (>= 1)            */
  /* ---- widened rows; all zero = the plain top-k layer ---- */
  int32_t route_mode;          /* 0 = top-k (R2..R5); 1 = threshold-gated variable-k on sigmoid gates (V1,
                                  PAPER.md:456): needs score_fn = 1, n_group = 1, thresholds in moe_extras_t    */
  int32_t n_zero, n_copy, n_const; /* zero-computation experts (V2): the LAST n_zero + n_copy +
                                  n_const of the E router outputs, in this order; they own no FFN weights:
                                  Wg, Wu, Wd and their gradients hold E - n_zero - n_copy - n_const experts    */
  float aux_coef;              /* auxiliary load-balancing loss coefficient (A1); 0 = off    */
  float aux_zc_weight;         /* weight of the zero-computation experts in the balance term    */
  /* ---- kernel-variant selectors.  All 0 = the library's defaults (the measured, documented path).  The library reads
   * NO environment variables; these fields are the only way to reach the non-default variants, which exist so that the
   * tests can hold every variant to the same oracle.  Value v > 0 forces level v - 1. ---- */
  int32_t opt_rows_fused;      /* levels 0 / 1 / 2 of moe_layer_rows_fused (ignored where the config cannot fuse)      */
  int32_t opt_pair;            /* cta_group::2 pair kernel: level 0 never, 1 weight gradients + single-group GEMMs
                                  (default), 2 ragged expert GEMMs as M-tile pairs too                                 */
  int32_t opt_fp8_wide;        /* FP8 128 x 256 tiles: level 0 never, 1 plain-epilogue GEMMs (default), 2 all modes    */
  int32_t opt_fp8_fused_quant; /* Q-a / Q-dgu in the GEMM epilogues: level 0 off, 1 on (default: on iff
                                  fp8_scale_mode == 1)                                                                 */
} moe_config_t;

/* Optional inputs / outputs of the widened rows, passed to moe_layer_fwd_ex / moe_layer_bwd_ex (NULL members that the
 * config does not need are ignored).  All device pointers. */
typedef struct moe_extras_t {
  const float* threshold;    /* [E] fp32 gate thresholds, required iff route_mode == 1 (no gradient)              */
  const void* zc_const;      /* [n_const, H] constant experts' vectors (activation type), required iff n_const > 0 */
  void* d_zc_const;          /* bwd: [n_const, H] their gradient, overwritten; NULL = not wanted                   */
  const float* aux_f_global; /* [E] fp32 or NULL: assignment fractions f_e of the GLOBAL batch (e.g. counts
                                all-reduced over data-parallel ranks and normalised); NULL = this batch's own     */
  float* aux_loss;           /* fwd: device scalar that receives L_aux, or NULL                                    */
} moe_extras_t;

enum moe_status {
  MOE_OK = 0,
  MOE_ERR_INVALID_ARG = -1, /* NULL where a pointer is required, non-positive size, bad enum    */
  MOE_ERR_UNSUPPORTED = -2, /* valid in principle, not implemented for this shape / dtype        */
  MOE_ERR_WORKSPACE = -3,   /* reserved                                                          */
  MOE_ERR_CUDA = -4,        /* a CUDA runtime / driver call failed (launch error, no sm_100 GPU) */
  MOE_ERR_TOO_LARGE = -5    /* moe_permute_static_ws: the problem needs more than the built-in scratch */
};

/* Text for a status code (static storage). */
const char* moe_status_string(int32_t status);

/* Library version as major*10000 + minor*100 + patch. */
int32_t moe_version(void);

/* Upper bound on permuted rows: T*K if row_align == 1, else (T*K + E*(row_align-1)) rounded up to
 * row_align.  Returns < 0 on an invalid config. */
int64_t moe_padded_rows(const moe_config_t* cfg);

/* How moe_layer_fwd / bwd / wgrad fold the routing weight and the permutation into the grouped GEMMs for this config
 * (< 0: invalid config).  PAPER.md:116 ("fused ... token scatter"); BASELINE.json north_star (3) "routing-weight scaling
 * fused into the epilogues".
 *  0  nothing fused (fp32, FP8, unaligned groups, zero-computation experts; or cfg->opt_rows_fused = 1): w is applied in the
 *     combine, the backward starts with a combine-backward pass writing dy = w dY and dw.
 *  1  (default for bf16 with H, F multiples of 64 and row_align a multiple of 128): the routing weight is applied in the
 *     GEMM-1 epilogue (ctx "a" holds w_r a_r, ctx "y" holds w_r y_r, the combine is a plain sum over the K rows) and in the
 *     dgrad-down epilogue, which also produces dw[t,j] = <da_r, a_r> (= <dY_t, y_r>, R8).  The combine-backward pass is
 *     replaced by a plain row gather of dY: ws "dy" holds the UNWEIGHTED rows of dY, y is not read by the backward.
 *  2  (cfg->opt_rows_fused = 3) as 1, and GEMM-1 gathers the rows of X, dgrad-down the rows of dY, inside the kernel (TMA
 *     tile::gather4 through perm_to_flat), each writing the row-grouped copy ("Xp", "dy") that the weight gradients contract
 *     over as a by-product of its staged tiles: no row-mover pass at all.
 * The layer's results (Y, dX, dW*, dWr, topk_*) mean the same in all three.  The stand-alone moe_permute /
 * moe_unpermute_combine are not affected. */
int32_t moe_layer_rows_fused(const moe_config_t* cfg);

/* Bytes of scratch (`ws`, contents undefined between calls) and of saved-for-backward context
 * (`ctx`, written by moe_layer_fwd, read by moe_layer_bwd) for this config.  Both 256-byte multiples. */
int32_t moe_workspace_bytes(const moe_config_t* cfg, size_t* ws_bytes, size_t* ctx_bytes);

/* R2..R5.  Top-k routing from fp32 logits.
 *   logits [T,E] fp32; bias [E] fp32 or NULL (required iff cfg->has_bias)
 *   topk_idx [T,K] int32: slot j holds the j-th largest selection key, ties -> lower expert index
 *   topk_w   [T,K] fp32 gating weights (bias never enters w)
 * Selection key: softmax -> z (+ b); sigmoid -> fp32(1/(1+exp(-z)) evaluated in fp64) + b in fp32.
 * Group limiting: keep topk_group of n_group contiguous groups by group score; others -> -inf.
 * UNSUPPORTED: E > 1024, K > 32, n_group > 32, K > topk_group * E / n_group. */
int32_t moe_route(const moe_config_t* cfg, const float* logits, const float* bias, int32_t* topk_idx,
                  float* topk_w, void* stream);

/* V1: threshold-gated variable-k routing.  s = sigmoid(z) (evaluated as in moe_route);
 * expert e is active for a token iff s[e] > threshold[e]; the active experts fill the K slots in (s desc, index asc)
 * order (more than K active: the K largest stay), unused slots hold topk_idx = -1 and topk_w = 0; a token no expert
 * admits keeps its single best expert.  Weights: routed_scale * s_j / (sum of the selected s + 1e-20) (renorm) or
 * routed_scale * s_j.  Every other entry point accepts the -1 slots (they own no permuted row). */
int32_t moe_route_threshold(const moe_config_t* cfg, const float* logits, const float* threshold, int32_t* topk_idx,
                            float* topk_w, void* stream);

/* R6.  Histogram, exclusive scan, stable counting sort of flat positions
 * p = t*K + j by expert (no atomics; deterministic), then the row gather Xp[r] = X[perm_to_flat[r] / K].
 *   X [T,H] (cfg->dtype element type) or NULL to build the maps only (then Xp is ignored)
 *   topk_idx [T,K]; counts [E]; offsets [E+1]; perm_to_flat [TK_pad] (-1 on padding rows and on rows
 *   >= offsets[E]); flat_to_perm [T*K]; Xp [TK_pad,H] (padding rows zero; rows >= offsets[E] untouched)
 *   ws: scratch of at least moe_workspace_bytes().  */
int32_t moe_permute(const moe_config_t* cfg, const void* X, const int32_t* topk_idx, int32_t* counts,
                    int32_t* offsets, int32_t* perm_to_flat, int32_t* flat_to_perm, void* Xp, void* ws,
                    void* stream);

/* moe_permute for callers that cannot supply `ws` because they cannot allocate device memory at all: a plug-in inside
 * a runtime that owns the GPU's memory and passes only input / output tensors, a process that forbids cudaMalloc after
 * start-up (it synchronises the device and can fail on a nearly full GPU), a loop that must stay clear of the allocator.
 * Same arguments, results and limits as moe_permute minus `ws`; the scratch (the chunk histograms) is a fixed array of
 * MOE_PERMUTE_STATIC_WS_BYTES built into the library image, so every GPU that loads libmoe_b200.so gives up that much
 * memory until the process exits.  The call allocates nothing (no cudaMalloc / cudaFree / allocating library routine).
 *   Limit: ceil(T*K / 1024) * E * 4 <= MOE_PERMUTE_STATIC_WS_BYTES, else MOE_ERR_TOO_LARGE and nothing is enqueued
 *   (all five BASELINE.json configs need 32 KiB; T*K = 1M positions with E = 256 is the largest that fits).
 *   First call on each device: looks up the array's device address (cudaGetSymbolAddress, with that device current)
 *   and caches it; make that first call before any stream capture begins.
 *   One array per GPU, shared by all calls, contents left over from the last call.  Nothing needs clearing (every entry
 *   that is read is written first by the same call).  Calls that overlap on one GPU -- two streams, two threads -- race
 *   on the array and corrupt each other's maps: serialise them (one stream, or events).
 *   The GEMM tile tables moe_permute leaves in `ws` as a by-product are not produced. */
#define MOE_PERMUTE_STATIC_WS_BYTES (1u << 20)
int32_t moe_permute_static_ws(const moe_config_t* cfg, const void* X, const int32_t* topk_idx, int32_t* counts,
                              int32_t* offsets, int32_t* perm_to_flat, int32_t* flat_to_perm, void* Xp,
                              void* stream);

/* R7, one grouped GEMM: for every expert e and row r in [offsets[e], offsets[e+1]):
 *   C[r, n] = sum_k A[r, k] * B[e][n, k]         A [TK_pad,Kdim], B [E,N,Kdim], C [TK_pad,N]
 * fp32 accumulation; C in the element type of A.  dtype 2: A and B are e4m3 codes (uint8) with
 * a_scales [TK_pad, Kdim/128] fp32 and b_scales [E, ceil(N/128), Kdim/128] fp32, C is bf16.
 * Rows >= offsets[E] are not touched.  Requirements for dtype 1: row_align % 128 == 0, Kdim % 64 == 0, N % 8 == 0
 * (other bf16 shapes run on CUDA cores); dtype 2: row_align % 128 == 0, Kdim % 128 == 0, N % 128 == 0.  */
int32_t moe_grouped_gemm_fwd(const moe_config_t* cfg, int32_t N, int32_t Kdim, const void* A, const void* B,
                             const int32_t* offsets, void* C, const void* a_scales, const void* b_scales,
                             void* ws, void* stream);

/* R8, the two gradients of C = A * B[e]^T (either output may be NULL = skipped; this is the split
 * that a delayed weight-gradient schedule needs):
 *   dA[r, k]    = sum_n dC[r, n] * B[e][n, k]                       (dgrad)   dA [TK_pad,Kdim]
 *   dB[e][n, k] = sum_{r in e} dC[r, n] * A[r, k]                   (wgrad)   dB [E,N,Kdim], overwritten;
 *                                                                   an empty expert gets exact zeros
 * Padding rows of dC and A must be zero (they are when produced by this library).  bf16 / fp32 only. */
int32_t moe_grouped_gemm_bwd(const moe_config_t* cfg, int32_t N, int32_t Kdim, const void* dC, const void* A,
                             const void* B, const int32_t* offsets, void* dA, void* dB, void* ws,
                             void* stream);

/* R7 SwiGLU ([34]):  a[r,f] = silu(gu[r,f]) * gu[r,F+f],  gu [rows,2F] = [gate | up]. */
int32_t moe_swiglu(const moe_config_t* cfg, const void* gu, void* a, int64_t rows, void* stream);

/* R8 SwiGLU backward: dgu[r,f] = da*u*s*(1+g*(1-s)), dgu[r,F+f] = da*g*s with s = sigmoid(g). */
int32_t moe_swiglu_bwd(const moe_config_t* cfg, const void* gu, const void* da, void* dgu, int64_t rows,
                       void* stream);

/* R7 combine:  Y[t,:] = sum_{j=0..K-1} topk_w[t,j] * y[flat_to_perm[t*K+j],:]  (+ shared_out[t,:]),
 * fp32 accumulation in ascending j, one rounding to the output type. */
int32_t moe_unpermute_combine(const moe_config_t* cfg, const void* y, const float* topk_w,
                              const int32_t* flat_to_perm, const void* shared_out, void* Y, void* stream);

/* R9 quantisers ([22]).  Input is the bf16 tensor; codes are e4m3fn (RNE, saturating
 * at +-448) of v/scale in fp32; scale = amax/448 (mode 0) or 2^ceil(log2(amax/448)) (mode 1); an all-zero
 * block has scale 1.  1x128 blocks along the last axis / 128x128 blocks over the last two axes.
 *   moe_quantize_act:    v [rows, cols] bf16 -> codes [rows, cols] u8, scales [rows, ceil(cols/128)] fp32
 *   moe_quantize_weight: w [batch, rows, cols] bf16 -> codes u8, scales [batch, ceil(rows/128), ceil(cols/128)] */
int32_t moe_quantize_act(const void* v, int64_t rows, int32_t cols, int32_t scale_mode, uint8_t* codes,
                         float* scales, void* stream);
int32_t moe_quantize_weight(const void* w, int32_t batch, int32_t rows, int32_t cols, int32_t scale_mode,
                            uint8_t* codes, float* scales, void* stream);

/* FP8 weight cache ("FP8 weight cache"; R9 Q-W): quantise the bf16 expert weights (and the shared
 * expert's, if any) to e4m3 codes + 128x128 block scales inside `ctx`.  moe_layer_fwd does this itself when it is
 * given weights; call this once per optimiser step and pass Wg = Wu = Wd = NULL (and NULL shared weights) to
 * moe_layer_fwd for the following micro-batches to reuse the codes.  cfg->dtype must be 2. */
int32_t moe_fp8_quantize_weights(const moe_config_t* cfg, const void* Wg, const void* Wu, const void* Wd,
                                 const void* Wg_s, const void* Wu_s, const void* Wd_s, void* ctx, void* stream);

/* R1..R7: the whole forward.  X [T,H]; Wr [E,H]; bias [E] or NULL; Wg, Wu [E,F,H]; Wd [E,H,F];
 * shared expert Wg_s, Wu_s [F_shared,H], Wd_s [H,F_shared] or NULL (iff F_shared == 0).
 * Outputs Y [T,H], topk_idx [T,K], topk_w [T,K]; ctx receives what the backward needs.
 * dtype 2 (R9): X, a are quantised 1x128 and the weights 128x128 on the fly (codes kept in ctx); Wg = Wu = Wd = NULL
 * reuses the weight codes already in ctx; requires row_align % 128 == 0 and H, F, F_shared multiples of 128. */
int32_t moe_layer_fwd(const moe_config_t* cfg, const void* X, const void* Wr, const float* bias,
                      const void* Wg, const void* Wu, const void* Wd, const void* Wg_s, const void* Wu_s,
                      const void* Wd_s, void* Y, int32_t* topk_idx, float* topk_w, void* ctx, void* ws,
                      void* stream);

/* The forward with the widened rows' extras (`ex` may be NULL when the config needs none; moe_layer_fwd is this call
 * with ex = NULL):  route_mode 1 routes with ex->threshold (V1);  zero-computation experts (V2) contribute
 * w * 0 / w * X[t] / w * zc_const[c] and run no GEMM;  aux_coef != 0 (A1..A2) also computes
 *   L_aux = aux_coef * E * sum_e eta_e f_e P_e,   f_e = fraction of the routed assignments on expert e (ex->aux_f_global
 *   if given, else this batch's counts / assignments made),   P_e = mean over tokens of p[t,e]  (p = softmax(z) for
 *   score_fn 0, s / sum_e s for sigmoid gates),   eta_e = aux_zc_weight for zero-computation experts, else 1,
 * stores f in ctx for the backward and writes L_aux to ex->aux_loss (also readable as ctx field "aux_loss"). */
int32_t moe_layer_fwd_ex(const moe_config_t* cfg, const void* X, const void* Wr, const float* bias,
                         const void* Wg, const void* Wu, const void* Wd, const void* Wg_s, const void* Wu_s,
                         const void* Wd_s, void* Y, int32_t* topk_idx, float* topk_w, void* ctx, void* ws,
                         const moe_extras_t* ex, void* stream);

/* R8: the whole backward for L = <Y, dY>.  Weight gradients are overwritten, in the weights' type.
 * Any of dWr / dWg / dWu / dWd (and the shared triple) may be NULL together with the others of its
 * group to skip the weight-gradient GEMMs (dX is always produced).
 * dtype 2 (R9): dgrad runs on e4m3 codes (Q(dY), Q(dg), Q(du), the weight codes in ctx; the bf16 weight pointers are
 * not read and may be NULL), wgrad on the bf16 tensors. */
int32_t moe_layer_bwd(const moe_config_t* cfg, const void* dY, const void* X, const void* Wr, const void* Wg,
                      const void* Wu, const void* Wd, const void* Wg_s, const void* Wu_s, const void* Wd_s,
                      const void* ctx, void* dX, void* dWr, void* dWg, void* dWu, void* dWd, void* dWg_s,
                      void* dWu_s, void* dWd_s, void* ws, void* stream);

/* The backward with the extras: L = <Y, dY> + L_aux.  The balance term adds the dense gradient
 *   dz[t,j] += (aux_coef E / T) d_j (g_j - sum_e g_e p[t,e]),  g = eta * f,  d_j = p_j (softmax) or s_j (1 - s_j) / sum_e s_e
 * (A3; f carries no gradient) to the router backward, which then runs as two dense GEMMs (dWr = dz^T X, dX += dz Wr);
 * the same dense path serves softmax gating without renormalisation.  ex->d_zc_const receives sum_r dy[r] per constant
 * expert.  moe_layer_bwd is this call with ex = NULL. */
int32_t moe_layer_bwd_ex(const moe_config_t* cfg, const void* dY, const void* X, const void* Wr, const void* Wg,
                         const void* Wu, const void* Wd, const void* Wg_s, const void* Wu_s, const void* Wd_s,
                         const void* ctx, void* dX, void* dWr, void* dWg, void* dWu, void* dWd, void* dWg_s,
                         void* dWu_s, void* dWd_s, void* ws, const moe_extras_t* ex, void* stream);

/* R8, weight gradients only -- the separately schedulable half of the backward that a delayed weight-gradient
 * schedule needs (PAPER.md:116 "wgrad delay", :239).  Call moe_layer_bwd with NULL weight gradients first (dgrad, dX,
 * dWr), then this at any later point of the same stream order; `ctx` and `ws` must be the untouched buffers of those
 * calls (it reads Xp, a from ctx and dy, dgu from ws).  X, dY are the layer input and output gradient (used by the
 * shared expert).  accumulate_fp32 = 0: gradients in the weights' type, overwritten (as moe_layer_bwd);
 * accumulate_fp32 = 1: dW* are fp32 tensors of the weights' shapes and the new gradient is ADDED to them (fp32 main
 * gradients across micro-batches); tensor-core path only (dtype 1 or 2, row_align % 128 == 0), else UNSUPPORTED. */
int32_t moe_layer_wgrad(const moe_config_t* cfg, const void* X, const void* dY, const void* ctx, const void* ws,
                        void* dWg, void* dWu, void* dWd, void* dWg_s, void* dWu_s, void* dWd_s,
                        int32_t accumulate_fp32, void* stream);

/* End-to-end step with HOST activations: copies X_host and dY_host [T,H] to the device buffers
 * X_dev / dY_dev, runs moe_layer_fwd + moe_layer_bwd, copies Y and dX back to Y_host / dX_host, all on
 * `stream` (host buffers should be pinned; returns without synchronising).  Weights, gradients, ctx,
 * ws and the staging buffers X_dev, dY_dev, Y_dev, dX_dev are device memory.  The host steps take no moe_extras_t:
 * a config that needs one (route_mode == 1, n_const > 0) is INVALID_ARG here; every argument check of moe_layer_fwd /
 * moe_layer_bwd is made before the first copy is enqueued. */
int32_t moe_layer_step_host(const moe_config_t* cfg, const void* X_host, const void* dY_host, void* Y_host,
                            void* dX_host, void* X_dev, void* dY_dev, void* Y_dev, void* dX_dev,
                            const void* Wr, const float* bias, const void* Wg, const void* Wu, const void* Wd,
                            const void* Wg_s, const void* Wu_s, const void* Wd_s, void* dWr, void* dWg,
                            void* dWu, void* dWd, void* dWg_s, void* dWu_s, void* dWd_s, int32_t* topk_idx,
                            float* topk_w, void* ctx, void* ws, void* stream);

/* The same step, software-pipelined over three caller streams: the H2D copies go to `stream_in`, fwd+bwd to
 * `stream_compute`, the D2H copies to `stream_out`, ordered by the events of a caller-owned pipeline object, so that
 * consecutive calls overlap copy-in of step i+1 and copy-out of step i-1 with the compute of step i.
 *   moe_pipeline_create:  makes the object (six events, timing disabled) on the CURRENT device; *pipeline receives it.
 *   moe_pipeline_destroy: destroys it; the caller must have synchronised the three streams first.
 * `slot` is 0 or 1 and names which of the caller's TWO sets of staging buffers (X_dev, dY_dev, Y_dev, dX_dev) this call
 * uses; alternate it between calls.  ctx, ws, weights and gradients are shared by both slots (compute is serial on
 * stream_compute).  The host input buffers may be changed once stream_in has passed this call's copies; the host
 * outputs are valid once stream_out has.  One pipeline object serves one (device, stream triple, buffer set); it is not
 * thread-safe.  INVALID_ARG if `pipeline` is not a live object of the current device. */
int32_t moe_pipeline_create(void** pipeline);
int32_t moe_pipeline_destroy(void* pipeline);
int32_t moe_layer_step_host_pipelined(void* pipeline, const moe_config_t* cfg, int32_t slot, const void* X_host,
                                      const void* dY_host, void* Y_host, void* dX_host, void* X_dev, void* dY_dev,
                                      void* Y_dev, void* dX_dev, const void* Wr, const float* bias, const void* Wg,
                                      const void* Wu, const void* Wd, const void* Wg_s, const void* Wu_s, const void* Wd_s,
                                      void* dWr, void* dWg, void* dWu, void* dWd, void* dWg_s, void* dWu_s, void* dWd_s,
                                      int32_t* topk_idx, float* topk_w, void* ctx, void* ws, void* stream_in,
                                      void* stream_compute, void* stream_out);

/* Read-only view of buffers inside ctx after moe_layer_fwd (for tests and tracing):
 * name in {"z","counts","offsets","perm_to_flat","flat_to_perm","Xp","gu","a","y","gu_s","a_s","y_s",
 *          "aux_f","aux_P","aux_loss" (fp32 [E], [E], [1]; aux_coef != 0),
 *          "aq","aq_s" (dtype 2: e4m3 codes [TK_pad,F] and fp32 scales [TK_pad,F/128] of a, written by the GEMM-1 epilogue)}.
 * With moe_layer_rows_fused(cfg) >= 1 "a" and "y" carry the row's routing weight (w_r a_r, w_r y_r).
 * Writes the byte offset inside ctx and the byte length.  */
int32_t moe_ctx_field(const moe_config_t* cfg, const char* name, size_t* byte_offset, size_t* byte_len);
/* Same for ws after moe_layer_bwd: {"dw","dz","dy","dgu","dXp","dz_dense" (fp32 [T,E]; dense router backward only),
 * "dguq","dguq_s" (dtype 2: codes [TK_pad,2F] / scales [TK_pad,2F/128] of [dg|du], written by the dgrad-down epilogue)}.
 * "dy" is w_r dY[t_r] with moe_layer_rows_fused(cfg) == 0 and the unweighted row dY[t_r] otherwise. */
int32_t moe_ws_field(const moe_config_t* cfg, const char* name, size_t* byte_offset, size_t* byte_len);

/* Stage timing for bench.py: while enabled, moe_layer_fwd / moe_layer_bwd record a CUDA event on
 * their stream after every stage; moe_profile_stage_ms synchronises on those events and returns the summed
 * device time and the number of recorded segments of one stage since the last moe_profile_enable call.  Stages:
 * "router_gemm","route","maps","permute","gemm1_swiglu","gemm2","combine","combine_bwd","dgrad_down_swiglu",
 * "dgrad_gateup","wgrad","router_bwd","dx_combine","shared_fwd","shared_bwd","quant".  Host-side state, not
 * thread-safe; at most 8192 marks are kept between two enable calls -- past that moe_profile_stage_ms returns
 * MOE_ERR_WORKSPACE instead of a truncated total. */
int32_t moe_profile_enable(int32_t on);
int32_t moe_profile_stage_ms(const char* stage, double* total_ms, int64_t* segments);

/* Number of kernels this library has launched since load (for bench.py's gpu_launches). */
int64_t moe_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* MOE_B200_H */
