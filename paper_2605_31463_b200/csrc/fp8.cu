// FP8 e4m3 block-scaled path ("FP8 training", "FP8 quantization").
//  * quantisers: 1x128 activation blocks, 128x128 weight blocks; bit-exact against the oracle's definition
//    (scale = amax/448 in fp32 or the next power of two; v/scale in fp32; e4m3fn RNE, saturating at +-448)
//  * the fp8 grouped GEMM: tcgen05 kind::f8f6f4 on TMA-fed 128x128x128 tiles; every 128-deep k-block's partial
//    product lands in its own TMEM buffer and is promoted into fp32 register accumulators with the block scales
//    (sa[row, kb] * sb[n-block, kb]) by eight epilogue warps -- the dequantisation is fused into the main loop.
#include <string.h>

#include <algorithm>

#include "fp8.cuh"
#include "tc_ptx.cuh"

namespace moe {
namespace {

constexpr unsigned FULL = 0xffffffffu;

// ---------------------------------------------------------------------------------------------
// quantisers
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ float block_scale(float amax, int mode) { return fp8_block_scale(amax, mode); }
__device__ __forceinline__ uint32_t encode4(float a, float b, float c, float d, float scale) {
  return fp8_encode4(a, b, c, d, scale);
}

__device__ __forceinline__ void unpack8(const uint4& v, float (&f)[8]) {
  const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    f[2 * i] = __uint_as_float(w[i] << 16);
    f[2 * i + 1] = __uint_as_float(w[i] & 0xffff0000u);
  }
}

__device__ __forceinline__ float amax8(const float (&f)[8]) {
  float m = 0.f;
#pragma unroll
  for (int i = 0; i < 8; ++i) m = fmaxf(m, fabsf(f[i]));
  return m;
}

// 1x128 blocks along the last axis: 16 lanes x 8 elements per block, two blocks per warp.
__global__ void __launch_bounds__(256) quant_act_kernel(const uint4* __restrict__ v, int64_t rows, int cols, int nblk,
                                                        int mode, uint2* __restrict__ codes,
                                                        float* __restrict__ scales) {
  const int64_t gid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t blk = gid >> 4;          // (row, block) index
  const int sub = (int)(gid & 15);
  const bool in_range = blk < rows * nblk;
  const int64_t row = in_range ? blk / nblk : 0;
  const int b = in_range ? (int)(blk - row * nblk) : 0;
  const int col = b * 128 + sub * 8;
  const bool ok = in_range && col < cols;
  float f[8];
  if (ok) {
    unpack8(v[(row * cols + col) >> 3], f);
  } else {
#pragma unroll
    for (int i = 0; i < 8; ++i) f[i] = 0.f;
  }
  float m = amax8(f);
#pragma unroll
  for (int off = 8; off > 0; off >>= 1) m = fmaxf(m, __shfl_xor_sync(FULL, m, off));
  const float s = block_scale(m, mode);
  if (ok) codes[(row * cols + col) >> 3] = make_uint2(encode4(f[0], f[1], f[2], f[3], s), encode4(f[4], f[5], f[6], f[7], s));
  if (in_range && sub == 0) scales[blk] = s;
}

// 128x128 blocks over the last two axes: one CTA of 1024 threads per block, 2 passes x 8 elements per thread kept in
// registers between the amax reduction and the encode (each element is read from HBM once); few registers per thread so
// that two CTAs (64 warps) stay resident per SM and the load phase of one overlaps the encode phase of the other.
constexpr int QW_THREADS = 1024;
__global__ void __launch_bounds__(QW_THREADS, 2) quant_weight_kernel(const uint4* __restrict__ w, int rows, int cols,
                                                                     int rb, int cb, int mode,
                                                                     uint2* __restrict__ codes,
                                                                     float* __restrict__ scales) {
  __shared__ float red[QW_THREADS / 32];
  __shared__ float s_scale;
  const int bc = blockIdx.x % cb;
  const int br = (blockIdx.x / cb) % rb;
  const int64_t batch = blockIdx.x / (cb * rb);
  const int sub = threadIdx.x & 15, r0 = threadIdx.x >> 4;   // 64 row-lanes per pass
  const int col = bc * 128 + sub * 8;
  uint4 raw[2];
  float m = 0.f;
#pragma unroll
  for (int p = 0; p < 2; ++p) {
    const int row = br * 128 + p * 64 + r0;
    raw[p] = make_uint4(0u, 0u, 0u, 0u);
    if (row < rows && col < cols) raw[p] = __ldg(w + (((batch * rows + row) * cols + col) >> 3));
    float f[8];
    unpack8(raw[p], f);
    m = fmaxf(m, amax8(f));
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) m = fmaxf(m, __shfl_xor_sync(FULL, m, off));
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
  __syncthreads();
  if (threadIdx.x < 32) {
    float mm = red[threadIdx.x];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) mm = fmaxf(mm, __shfl_xor_sync(FULL, mm, off));
    if (threadIdx.x == 0) {
      const float s = block_scale(mm, mode);
      s_scale = s;
      scales[blockIdx.x] = s;            // [batch, rb, cb] == blockIdx order
    }
  }
  __syncthreads();
  const float s = s_scale;
#pragma unroll
  for (int p = 0; p < 2; ++p) {
    const int row = br * 128 + p * 64 + r0;
    if (row < rows && col < cols) {
      float f[8];
      unpack8(raw[p], f);
      codes[((batch * rows + row) * cols + col) >> 3] =
          make_uint2(encode4(f[0], f[1], f[2], f[3], s), encode4(f[4], f[5], f[6], f[7], s));
    }
  }
}

// scales_p[r, :] = scales[perm_to_flat[r] / K, :] (0 on padding rows); rows < offsets[E] only.
__global__ void __launch_bounds__(256) gather_scales_kernel(const float* __restrict__ src, const int32_t* __restrict__ p2f,
                                                            const int32_t* __restrict__ offsets, int E, int K, int nblk,
                                                            float* __restrict__ dst) {
  const int64_t total = (int64_t)offsets[E] * nblk;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t r = i / nblk;
    const int b = (int)(i - r * nblk);
    const int p = p2f[r];
    dst[i] = p >= 0 ? src[(int64_t)(p / K) * nblk + b] : 0.f;
  }
}

}  // namespace

int32_t fp8_quantize_act(const void* v, int64_t rows, int cols, int mode, uint8_t* codes, float* scales,
                         cudaStream_t s) {
  if (rows == 0) return MOE_OK;
  if (cols % 8 != 0) return MOE_ERR_UNSUPPORTED;
  const int nblk = (cols + 127) / 128;
  const int64_t threads = rows * nblk * 16;
  MOE_LAUNCH(quant_act_kernel, (unsigned)ceil_div(threads, 256), 256, 0, s, (const uint4*)v, rows, cols, nblk, mode,
             (uint2*)codes, scales);
  return MOE_OK;
}

int32_t fp8_quantize_weight(const void* w, int batch, int rows, int cols, int mode, uint8_t* codes, float* scales,
                            cudaStream_t s) {
  if (cols % 8 != 0) return MOE_ERR_UNSUPPORTED;
  const int rb = (rows + 127) / 128, cb = (cols + 127) / 128;
  const int64_t blocks = (int64_t)batch * rb * cb;
  if (blocks >= (1ll << 31)) return MOE_ERR_UNSUPPORTED;
  MOE_LAUNCH(quant_weight_kernel, (unsigned)blocks, QW_THREADS, 0, s, (const uint4*)w, rows, cols, rb, cb, mode, (uint2*)codes,
             scales);
  return MOE_OK;
}

int32_t fp8_gather_scales(const float* src, const int32_t* p2f, const int32_t* offsets, int E, int K, int nblk,
                          float* dst, cudaStream_t s) {
  MOE_LAUNCH(gather_scales_kernel, 148 * 4, 256, 0, s, src, p2f, offsets, E, K, nblk, dst);
  return MOE_OK;
}

}  // namespace moe

extern "C" int32_t moe_quantize_act(const void* v, int64_t rows, int32_t cols, int32_t scale_mode, uint8_t* codes,
                                    float* scales, void* stream) {
  if (!v || !codes || !scales || rows < 0 || cols <= 0 || scale_mode < 0 || scale_mode > 1) return MOE_ERR_INVALID_ARG;
  return moe::fp8_quantize_act(v, rows, cols, scale_mode, codes, scales, moe::as_stream(stream));
}

extern "C" int32_t moe_quantize_weight(const void* w, int32_t batch, int32_t rows, int32_t cols, int32_t scale_mode,
                                       uint8_t* codes, float* scales, void* stream) {
  if (!w || !codes || !scales || batch <= 0 || rows <= 0 || cols <= 0 || scale_mode < 0 || scale_mode > 1)
    return MOE_ERR_INVALID_ARG;
  return moe::fp8_quantize_weight(w, batch, rows, cols, scale_mode, codes, scales, moe::as_stream(stream));
}
