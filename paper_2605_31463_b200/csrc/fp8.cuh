// Internal interface of the FP8 e4m3 block-scaled path (fp8.cu: quantisers, gemm_fp8.cu: grouped GEMM).
// Not part of the public ABI.
#pragma once
#include <cuda_fp8.h>

#include "common.cuh"

namespace moe {

#ifdef __CUDACC__
// R9 quantiser arithmetic, shared by the stand-alone quantisers (fp8.cu) and the quantise-in-epilogue of the fp8 GEMMs
// (gemm_fp8.cu), so that fused and stand-alone codes are the same bits:
//   scale = amax / 448 in fp32 (mode 0) or the next power of two (mode 1); an all-zero block has scale 1;
//   code  = e4m3fn(RNE, saturating) of v / scale computed in fp32.
__device__ __forceinline__ float fp8_block_scale(float amax, int mode) {
  if (amax == 0.f) return 1.f;
  float r = __fdiv_rn(amax, 448.0f);
  if (mode == 1) {                       // 2^ceil(log2 r): r = m 2^ex, m in [0.5, 1)
    int ex;
    const float m = frexpf(r, &ex);
    r = ldexpf(1.0f, m == 0.5f ? ex - 1 : ex);
  }
  return r;
}
__device__ __forceinline__ uint32_t fp8_encode4(float a, float b, float c, float d, float scale) {
  // cvt.rn.satfinite.e4m3x2.f32 packs two codes per instruction (.x -> low byte)
  const uint32_t lo = __nv_cvt_float2_to_fp8x2(make_float2(__fdiv_rn(a, scale), __fdiv_rn(b, scale)), __NV_SATFINITE, __NV_E4M3);
  const uint32_t hi = __nv_cvt_float2_to_fp8x2(make_float2(__fdiv_rn(c, scale), __fdiv_rn(d, scale)), __NV_SATFINITE, __NV_E4M3);
  return lo | (hi << 16);
}
// Power-of-two scales (mode 1): v / scale == v * (1 / scale) exactly, so the quantise-in-epilogue multiplies.
__device__ __forceinline__ uint32_t fp8_encode4_pow2(float a, float b, float c, float d, float inv_scale) {
  const uint32_t lo = __nv_cvt_float2_to_fp8x2(make_float2(a * inv_scale, b * inv_scale), __NV_SATFINITE, __NV_E4M3);
  const uint32_t hi = __nv_cvt_float2_to_fp8x2(make_float2(c * inv_scale, d * inv_scale), __NV_SATFINITE, __NV_E4M3);
  return lo | (hi << 16);
}
#endif

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
  int opt_wide;            // moe_config_t::opt_fp8_wide (0 = default level 1)
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
  // fused quantise-in-epilogue (R9 Q-a / Q-dgu): when q_codes != nullptr the SwiGLU modes also emit the
  // e4m3 codes and 1x128 scales of the bf16 tensor they write -- FWD_SWIGLU: a [rows, F] -> q_codes [rows, F],
  // q_scales [rows, F/128];  DGRAD_SWIGLU: dgu [rows, 2F] -> q_codes [rows, 2F], q_scales [rows, 2F/128] -- the same
  // bits as fp8_quantize_act on that tensor, without re-reading it from HBM.
  uint8_t* q_codes; float* q_scales; int q_mode;
};

int32_t fp8_gemm(const F8Call& c, cudaStream_t s);

}  // namespace moe
