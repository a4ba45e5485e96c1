// CUDA-core grouped GEMMs with generic strides: the fp32 path (configs[0]) and the path for shapes the
// tcgen05 kernels reject.  fp32 accumulation in ascending contraction order inside a thread.
//   mode 0: C[r,n]     = sum_k A[r,k]  * B[e][n,k]
//   mode 1: dA[r,k]    = sum_n dC[r,n] * B[e][n,k]
//   mode 2: dB[e][n,k] = sum_{r in e} dC[r,n] * A[r,k]     (an empty expert writes exact zeros)
// SURVEY.md §8c R7/R8.
#include "common.cuh"

namespace moe {
namespace {

constexpr int TS = 64;  // output tile
constexpr int KS = 16;  // contraction tile

struct SimtArgs {
  int mode, E, N, Kdim, lda, lddc, ldo;
  const void *A, *B, *dC;
  void* out;
  const int32_t* offsets;
  int max_row_tiles;  // grid.x for modes 0/1
  int accumulate;     // 1: out += result (second half of a split contraction)
};

template <typename T>
__global__ void __launch_bounds__(256) simt_kernel(SimtArgs p) {
  __shared__ float sA[KS][TS + 1];
  __shared__ float sB[KS][TS + 1];
  __shared__ int s_e, s_m0;
  // ---- which problem does this CTA work on ----
  int e, m0, M, Ncols, Kc;
  if (p.mode == 2) {
    e = blockIdx.z;
    m0 = blockIdx.x * TS;
    M = p.N;
    Ncols = p.Kdim;
    Kc = p.offsets[e + 1] - p.offsets[e];
    if (m0 >= M) return;
  } else {
    if (threadIdx.x == 0) {
      int b = blockIdx.x, found = -1, fm = 0;
      for (int i = 0; i < p.E; ++i) {
        const int c = p.offsets[i + 1] - p.offsets[i];
        const int tiles = (c + TS - 1) / TS;
        if (b < tiles) { found = i; fm = b * TS; break; }
        b -= tiles;
      }
      s_e = found;
      s_m0 = fm;
    }
    __syncthreads();
    e = s_e;
    m0 = s_m0;
    if (e < 0) return;
    M = p.offsets[e + 1] - p.offsets[e];
    Ncols = (p.mode == 0) ? p.N : p.Kdim;
    Kc = (p.mode == 0) ? p.Kdim : p.N;
  }
  const int n0 = blockIdx.y * TS;
  const int64_t off = p.offsets[e];
  // element accessors: A'(m,c), B'(j,c)
  const T* Ap;
  const T* Bp;
  int64_t sam, sak, sbn, sbk;
  if (p.mode == 0) {
    Ap = (const T*)p.A + off * p.lda; sam = p.lda; sak = 1;
    Bp = (const T*)p.B + (int64_t)e * p.N * p.Kdim; sbn = p.Kdim; sbk = 1;
  } else if (p.mode == 1) {
    Ap = (const T*)p.dC + off * p.lddc; sam = p.lddc; sak = 1;
    Bp = (const T*)p.B + (int64_t)e * p.N * p.Kdim; sbn = 1; sbk = p.Kdim;
  } else {
    Ap = (const T*)p.dC + off * p.lddc; sam = 1; sak = p.lddc;
    Bp = (const T*)p.A + off * p.lda; sbn = 1; sbk = p.lda;
  }
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  float acc[4][4];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;

  for (int k0 = 0; k0 < Kc; k0 += KS) {
    for (int i = threadIdx.x; i < KS * TS; i += 256) {
      int kk, mm;
      if (sak == 1) { kk = i % KS; mm = i / KS; } else { mm = i % TS; kk = i / TS; }
      const int m = m0 + mm, k = k0 + kk;
      sA[kk][mm] = (m < M && k < Kc) ? to_f(Ap[m * sam + k * sak]) : 0.f;
    }
    for (int i = threadIdx.x; i < KS * TS; i += 256) {
      int kk, nn;
      if (sbk == 1) { kk = i % KS; nn = i / KS; } else { nn = i % TS; kk = i / TS; }
      const int n = n0 + nn, k = k0 + kk;
      sB[kk][nn] = (n < Ncols && k < Kc) ? to_f(Bp[n * sbn + k * sbk]) : 0.f;
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < KS; ++kk) {
      float a[4], b[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) a[i] = sA[kk][ty * 4 + i];
#pragma unroll
      for (int j = 0; j < 4; ++j) b[j] = sB[kk][tx * 4 + j];
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
    }
    __syncthreads();
  }
  T* out;
  int64_t ldo;
  if (p.mode == 2) { out = (T*)p.out + (int64_t)e * p.N * p.Kdim; ldo = p.Kdim; }
  else { out = (T*)p.out + off * p.ldo; ldo = p.ldo; }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int m = m0 + ty * 4 + i;
    if (m >= M) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int n = n0 + tx * 4 + j;
      if (n < Ncols) out[m * ldo + n] = from_f<T>(acc[i][j] + (p.accumulate ? to_f(out[m * ldo + n]) : 0.f));
    }
  }
}

}  // namespace

int32_t simt_grouped_gemm(int mode, int dtype, int E, int N, int Kdim, const void* A, int lda, const void* B,
                          const void* dC, int lddc, const int32_t* offsets, void* out, int ldo, int64_t rows_cap,
                          int accumulate, cudaStream_t s) {
  SimtArgs p{mode, E, N, Kdim, lda, lddc, ldo, A, B, dC, out, offsets, 0, accumulate};
  dim3 grid;
  if (mode == 2) {
    grid = dim3((unsigned)ceil_div(N, TS), (unsigned)ceil_div(Kdim, TS), (unsigned)E);
  } else {
    p.max_row_tiles = (int)(ceil_div(rows_cap, TS) + E);
    grid = dim3((unsigned)p.max_row_tiles, (unsigned)ceil_div(mode == 0 ? N : Kdim, TS), 1);
  }
  if (dtype == 0)
    MOE_LAUNCH(simt_kernel<float>, grid, 256, 0, s, p);
  else
    MOE_LAUNCH(simt_kernel<__nv_bfloat16>, grid, 256, 0, s, p);
  return MOE_OK;
}

}  // namespace moe
