// Internal interface of the FP8 e4m3 block-scaled path (fp8.cu: quantisers, gemm_fp8.cu: grouped GEMM).
// Not part of the public ABI.
#pragma once
#include "common.cuh"

namespace moe {

// R9 quantisers (bf16 in; e4m3 codes + fp32 scales out).
int32_t fp8_quantize_act(const void* v, int64_t rows, int cols, int mode, uint8_t* codes, float* scales,
                         cudaStream_t s);
int32_t fp8_quantize_weight(const void* w, int batch, int rows, int cols, int mode, uint8_t* codes, float* scales,
                            cudaStream_t s);
// scales of permuted rows: dst[r, :] = src[perm_to_flat[r] / K, :], zero on padding rows.
int32_t fp8_gather_scales(const float* src, const int32_t* p2f, const int32_t* offsets, int E, int K, int nblk,
                          float* dst, cudaStream_t s);

// What one fp8 grouped-GEMM launch computes (e4m3 codes, 1x128 scales on the row-grouped operand, 128x128 scales on
// the weights, fp32 accumulation, bf16 outputs).  Dequantisation is fused into the main loop.
//  F8_FWD           C[r,n]  = sum_k A[r,k] B[e][n,k]                                 (gemm2: y = a Wd^T)
//  F8_FWD_SWIGLU    g = A Wg[e]^T, u = A Wu[e]^T -> gu = [g|u], a = silu(g) * u      (gemm1)
//  F8_DGRAD         dA[r,k] = sum_n dC[r,n] B[e][n,k]; the contraction may run over two (dC-half, B) pairs
//                   (dXp = dg Wg[e] + du Wu[e]); weights read MN-major
//  F8_DGRAD_SWIGLU  da = roww[r] * (dYq[r] Wd[e]); dgu = swiglu'(gu) * da             (dgrad-down)
enum F8Mode { F8_FWD = 0, F8_FWD_SWIGLU = 1, F8_DGRAD = 2, F8_DGRAD_SWIGLU = 3 };

struct F8Call {
  int mode;
  int E;
  int64_t rows_cap;        // height of the row-grouped buffers
  const int32_t* mtile;    // device {n_tiles, expert of tile 0, ...} or nullptr: one group of rows_cap rows
  const uint8_t* A;        // [rows_cap, lda] codes
  int lda;
  const float* a_scales;   // [rows_cap, lda / 128]
  const uint8_t* B0; const float* b0_scales;   // weights [E, b_rows, b_cols] codes, scales [E, b_rows/128, b_cols/128]
  const uint8_t* B1; const float* b1_scales;   // Wu (FWD_SWIGLU) / second half of a split DGRAD, or nullptr
  int b_rows, b_cols;
  int N;                   // output columns (FWD: b_rows; FWD_SWIGLU: F; DGRAD*: b_cols)
  void* out0; int ld0;     // C / gu / dA / dgu (bf16)
  void* out1; int ld1;     // FWD_SWIGLU: a (bf16)
  const void* gu; int ldgu;            // DGRAD_SWIGLU: saved [g|u] (bf16)
  const int32_t* p2f; const float* w;  // DGRAD_SWIGLU: row weight = w[p2f[r]] (0 on padding rows); nullptr = 1
  int F;
};

int32_t fp8_gemm(const F8Call& c, cudaStream_t s);

}  // namespace moe
