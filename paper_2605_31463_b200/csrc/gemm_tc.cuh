// Host-side description of one tcgen05 grouped-GEMM launch (gemm_tc.cu).  Not part of the public ABI.
#pragma once
#include "common.cuh"

namespace moe {

// What one launch computes (bf16 operands, fp32 accumulation in TMEM, bf16 outputs):
//  TC_FWD          C[r,n]      = sum_k A[r,k] B[e][n,k]                 A [rows,Kd], B [E,N,Kd]
//  TC_FWD_SWIGLU   g = A Wg[e]^T, u = A Wu[e]^T  ->  gu[r,:] = [g|u], a = silu(g)*u      (R7)
//  TC_DGRAD        dA[r,k]     = sum_n dC[r,n] B[e][n,k]                B read MN-major; the contraction may
//                  run over two (dC-half, B) pairs: dXp = dg Wg[e] + du Wu[e]            (R8)
//  TC_DGRAD_SWIGLU da = dy Wd[e]; dgu = swiglu'(gu) * da                                   (R8)
//  TC_WGRAD        dB[e][n,k]  = sum_{r in e} dC[r,n] A[r,k]            both operands MN-major, the contraction
//                  length is the expert's (padded) row count; an empty expert gets zeros   (R8)
//  TC_FWD_F32      as TC_FWD with fp32 output (router logits z = X Wr^T, R1)
enum TcMode { TC_FWD = 0, TC_FWD_SWIGLU = 1, TC_DGRAD = 2, TC_DGRAD_SWIGLU = 3, TC_WGRAD = 4, TC_FWD_F32 = 5 };

struct TcCall {
  int mode;
  int opt_pair;            // moe_config_t::opt_pair (0 = default level 1)
  int E;                   // groups
  int64_t rows_cap;        // height of the row-grouped buffers (TMA bound; rows >= it read as zero)
  const int32_t* counts;   // [E] device or nullptr: real rows per group (WGRAD trims its contraction to them)
  const int32_t* offsets;  // [E+1] device; group e = rows [offsets[e], offsets[e+1]), multiples of 128 if mtile != nullptr
  const int32_t* mtile;    // device {n_tiles, expert of tile 0, ...} or nullptr: one group of rows_cap rows at row 0
  const int32_t* plist;    // device pair / unpaired M-tile lists (tile_tables.cuh) belonging to mtile, or nullptr:
  const int32_t* olist;    //   then every tile runs on the 1-CTA kernel
  // --- operands (device, bf16) ---
  const void* A;  int lda;   // row-grouped left operand            [rows_cap, lda]
  const void* B0; const void* B1;  // weights [E, b_rows, b_cols] (B1: Wu for FWD_SWIGLU / second half of split DGRAD)
  int b_rows, b_cols;        // per-expert weight matrix shape (row-major)
  const void* A2; int lda2;  // WGRAD: the other row-grouped operand (fwd activations) [rows_cap, lda2]
  int a_col0;                // WGRAD: first column of A used as output rows (dWu: F)
  // --- problem sizes ---
  int N;                     // output columns (FWD: b_rows; FWD_SWIGLU: F; DGRAD*: b_cols; WGRAD: lda2 columns used)
  int Kd;                    // contraction length (FWD*: b_cols; DGRAD*: b_rows (x2 if split)); WGRAD: ignored
  int M;                     // WGRAD: output rows per expert
  // --- outputs (device, bf16) ---
  void* out0; int ld0;       // C / gu / dA / dgu / dB[E,M,N] (ld0 = N for WGRAD)
  void* out1; int ld1;       // FWD_SWIGLU: a
  const void* gu; int ldgu;  // DGRAD_SWIGLU: saved [g|u]
  int F;                     // SwiGLU width
  int acc_f32;               // WGRAD: out0 is fp32 [E,M,N] and the tile is ADDED to it (ld0 in fp32 elements)
  // --- fused permutation (PAPER.md:116 fused token scatter; optional; FWD_SWIGLU and DGRAD_SWIGLU of grouped launches) ---
  const int32_t* gidx;       // perm_to_flat [rows_cap] (device): flat position t*K+j of each row, -1 = padding row
  int gat;                   // 1: A is the TOKEN-major tensor [g_rows, lda]; its rows are gathered by TMA (tile::gather4)
                             // through gidx inside the kernel; 0: A is row-grouped already
  int gK;                    // top-k: token row = flat position / gK
  int64_t g_rows;            // rows of the token-major tensor (T)
  void* copy_out; int ld_copy;   // gat: the gathered rows are also written here, row-grouped [rows_cap, ld_copy] (padding rows
                             // as zeros): Xp from GEMM-1, the gathered dY from dgrad-down, for the weight gradients.  NULL = off
  const float* roww;         // routing weights by flat position [T*K] (needs gidx): FWD_SWIGLU writes a = w silu(g) u,
                             // DGRAD_SWIGLU writes dgu = w swiglu'(gu) da
  float* dwpart;             // DGRAD_SWIGLU: fp32 [2 * ceil(F / 256), rows_cap] partial sums of <da, silu(g) u> (dw, R8)
};

// Returns MOE_ERR_UNSUPPORTED (nothing enqueued) if the shape does not fit the tensor-core path.
int32_t tc_gemm(const TcCall& c, cudaStream_t s);

}  // namespace moe
