// FP8 e4m3 block-scaled grouped GEMM for sm_100a (SURVEY.md §8a a5/a6/a9/a11 in configs[3]; §8c R9).
//
// Persistent, warp-specialised: warp 0 = TMA producer, warp 1 = MMA issuer (tcgen05.mma kind::f8f6f4, M 128 x N 128
// x K 32, four per 128-deep k-block), warps 2..9 = promotion + epilogue.  A k-block's partial product is written to
// one of four 128-column TMEM buffers (never accumulated across k-blocks in TMEM); the promotion warps read it with
// tcgen05.ld, multiply by sa[row, kb] * sb[n-block, kb] and add into fp32 register accumulators -- the block-scale
// dequantisation of R9 fused into the main loop, exact up to fp32 rounding of the scaled sums.  Tiles are
// 128 rows x 128 output columns, so every tile sees exactly one weight-scale scalar per k-block (two for the
// gate/up pair of the fused SwiGLU forward, whose tile is 64 gate + 64 up columns).
#include <stdlib.h>
#include <string.h>

#include <algorithm>

#include "fp8.cuh"
#include "tc_ptx.cuh"

namespace moe {
namespace {

constexpr int BM = 128, BN = 128, BK = 128, UK = 32;
constexpr int STAGES = 6;
constexpr int A_BYTES = BM * BK, B_BYTES = BN * BK, STAGE_BYTES = A_BYTES + B_BYTES;   // 16 + 16 KB
constexpr int NBUF = 4;                                                                  // TMEM partial-product ring
constexpr int XCH_BYTES = 2 * 2 * BM * 2 * 4;   // amax exchange of the fused quantisers: [parity][g|u][row][column half] fp32
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + XCH_BYTES + 1024 + 256;
constexpr int EPI_WARPS = 8;
constexpr int NTHREADS = 64 + EPI_WARPS * 32;
constexpr int TMEM_COLS = NBUF * BN;   // 512

__device__ __forceinline__ void umma_f8(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f8f6f4 [%0], %1, %2, %3, p;\n\t"
      "}" ::"r"(d_tmem),
      "l"(adesc), "l"(bdesc), "r"(idesc), "r"(acc)
      : "memory");
}

struct F8Params {
  int E, n_tiles, nkb, kb_split, b_rows, N, F;
  int nb_b_cols;            // b_cols / 128 (scale row pitch of the weights)
  int a_nblk;               // lda / 128 (scale row pitch of A)
  int64_t rows_valid;
  const int32_t* mtile;
  const float* a_scales;
  const float* b0_scales;
  const float* b1_scales;
  __nv_bfloat16* out0;
  int64_t ld0;
  __nv_bfloat16* out1;
  int64_t ld1;
  const __nv_bfloat16* gu;
  int64_t ldgu;
  const int32_t* p2f;
  const float* w;
  uint8_t* q_codes;         // fused Q-a / Q-dgu output (nullptr: not fused)
  float* q_scales;
  int q_mode;
};

struct Tile {
  int e, m0, n0;
};

// i = sequence number of the tile inside this CTA's persistent loop.  F8_FWD_SWIGLU walks the 64-column n-tiles in
// PAIRS (i = 2q, 2q+1 are the two halves of one 128-column block of `a` on the SAME CTA), so that the fused Q-a sees a
// whole 1x128 quantisation block; the other modes take one tile per step.
template <int MODE>
__device__ __forceinline__ bool decode_tile(const F8Params& p, int64_t i, int64_t total, Tile& tl) {
  int64_t t;
  if (MODE == F8_FWD_SWIGLU) {
    const int64_t unit = blockIdx.x + (i >> 1) * (int64_t)gridDim.x;    // (M-tile, n-pair)
    t = unit * 2 + (i & 1);
  } else {
    t = blockIdx.x + i * (int64_t)gridDim.x;
  }
  if (t >= total) return false;
  const int mt = (int)(t / p.n_tiles);
  tl.n0 = (int)(t - (int64_t)mt * p.n_tiles) * (MODE == F8_FWD_SWIGLU ? BN / 2 : BN);
  tl.m0 = mt * BM;
  tl.e = p.mtile ? p.mtile[1 + mt] : 0;
  return true;
}

__device__ __forceinline__ int64_t total_tiles(const F8Params& p) {
  const int64_t mt = p.mtile ? p.mtile[0] : (p.rows_valid + BM - 1) / BM;
  return mt * p.n_tiles;
}

// weight-scale scalar(s) of k-block kb for this tile.  K-major weights [E, N, Kd]: scales [E, N/128, Kd/128];
// MN-major use (dgrad) of weights [E, b_rows, b_cols]: the contraction runs over b_rows, the output over b_cols.
template <int MODE>
__device__ __forceinline__ void weight_scales(const F8Params& p, const Tile& tl, int kb, float& s0, float& s1) {
  if (MODE == F8_FWD) {
    s0 = s1 = __ldg(p.b0_scales + ((int64_t)tl.e * (p.b_rows / 128) + tl.n0 / 128) * p.nb_b_cols + kb);
  } else if (MODE == F8_FWD_SWIGLU) {
    const int64_t i = ((int64_t)tl.e * (p.b_rows / 128) + tl.n0 / 128) * p.nb_b_cols + kb;
    s0 = __ldg(p.b0_scales + i);
    s1 = __ldg(p.b1_scales + i);
  } else {
    const bool second = kb >= p.kb_split;
    const float* sc = second ? p.b1_scales : p.b0_scales;
    const int kbl = second ? kb - p.kb_split : kb;
    s0 = s1 = __ldg(sc + ((int64_t)tl.e * (p.b_rows / 128) + kbl) * p.nb_b_cols + tl.n0 / 128);
  }
}

__device__ __forceinline__ uint4 pack8(const float* v) {
  uint4 o;
  o.x = pack_bf16(v[0], v[1]);
  o.y = pack_bf16(v[2], v[3]);
  o.z = pack_bf16(v[4], v[5]);
  o.w = pack_bf16(v[6], v[7]);
  return o;
}

__device__ __forceinline__ float fast_sigmoid8(float x) { return 1.0f / (1.0f + __expf(-x)); }

// four e4m3 codes of v / scale (R9): IEEE division for fp32 scales, an exact multiplication for power-of-two scales
__device__ __forceinline__ uint32_t enc4(float a, float b, float c, float d, float scale, float inv, int mode) {
  return mode == 1 ? fp8_encode4_pow2(a, b, c, d, inv) : fp8_encode4(a, b, c, d, scale);
}

// ---------------------------------------------------------------------------------------------
// the kernel
// ---------------------------------------------------------------------------------------------
template <int MODE>
__global__ void __launch_bounds__(NTHREADS, 1)
f8_gemm_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB0,
               const __grid_constant__ CUtensorMap tmB1, const F8Params p) {
  constexpr bool B_MN = (MODE == F8_DGRAD || MODE == F8_DGRAD_SWIGLU);
  extern __shared__ uint8_t smem_raw[];
  const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  float* const xch = reinterpret_cast<float*>(smem_raw + (base - smem_u32(smem_raw)) + STAGES * STAGE_BYTES);
  const uint32_t bars = base + STAGES * STAGE_BYTES + XCH_BYTES;
  const uint32_t full0 = bars, empty0 = bars + 8 * STAGES, pfull0 = bars + 16 * STAGES, pempty0 = pfull0 + 8 * NBUF;
  const uint32_t tmem_slot = pempty0 + 8 * NBUF;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmA);
    tma_prefetch_desc(&tmB0);
    tma_prefetch_desc(&tmB1);
    for (int s = 0; s < STAGES; ++s) {
      mbar_init(full0 + 8 * s, 1);
      mbar_init(empty0 + 8 * s, 1);
    }
    for (int b = 0; b < NBUF; ++b) {
      mbar_init(pfull0 + 8 * b, 1);
      mbar_init(pempty0 + 8 * b, EPI_WARPS);
    }
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc(tmem_slot, TMEM_COLS);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

  const int64_t total = total_tiles(p);

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      Tile tl;
      for (int64_t t = 0; decode_tile<MODE>(p, t, total, tl); ++t) {
        for (int kb = 0; kb < p.nkb; ++kb) {
          mbar_wait(empty0 + 8 * stage, phase ^ 1);
          const uint32_t fb = full0 + 8 * stage;
          const uint32_t sa = base + stage * STAGE_BYTES, sb = sa + A_BYTES;
          mbar_expect_tx(fb, STAGE_BYTES);
          tma_load_2d(sa, &tmA, fb, kb * BK, tl.m0);                                   // 128 B x 128 rows
          if (MODE == F8_FWD) {
            tma_load_2d(sb, &tmB0, fb, kb * BK, tl.e * p.b_rows + tl.n0);              // 128 B x 128 rows
          } else if (MODE == F8_FWD_SWIGLU) {
            tma_load_2d(sb, &tmB0, fb, kb * BK, tl.e * p.b_rows + tl.n0);              // 128 B x 64 rows (Wg)
            tma_load_2d(sb + B_BYTES / 2, &tmB1, fb, kb * BK, tl.e * p.b_rows + tl.n0);  // (Wu)
          } else {
            const bool second = kb >= p.kb_split;
            tma_load_2d(sb, second ? &tmB1 : &tmB0, fb, tl.n0,
                        tl.e * p.b_rows + (second ? kb - p.kb_split : kb) * BK);       // 128 cols x 128 k-rows
          }
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (lane == 0) {
      constexpr uint32_t idesc = instr_desc(0, 0, B_MN ? 1 : 0, BN);
      int stage = 0, buf = 0;
      uint32_t phase = 0, bphase = 0;
      Tile tl;
      for (int64_t t = 0; decode_tile<MODE>(p, t, total, tl); ++t) {
        for (int kb = 0; kb < p.nkb; ++kb) {
          mbar_wait(pempty0 + 8 * buf, bphase ^ 1);
          mbar_wait(full0 + 8 * stage, phase);
          tc_fence_after();
          const uint32_t sa = base + stage * STAGE_BYTES, sb = sa + A_BYTES;
          const uint32_t dacc = tmem_base + buf * BN;
#pragma unroll
          for (int k = 0; k < BK / UK; ++k) {
            const uint64_t ad = smem_desc(sa + k * UK, 16, 1024);
            const uint64_t bd = B_MN ? smem_desc(sb + k * UK * 128, B_BYTES, 1024) : smem_desc(sb + k * UK, 16, 1024);
            umma_f8(dacc, ad, bd, idesc, k != 0);
          }
          umma_commit(empty0 + 8 * stage);
          umma_commit(pfull0 + 8 * buf);
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
          if (++buf == NBUF) { buf = 0; bphase ^= 1; }
        }
      }
    }
  } else {
    // ===================== promotion + epilogue warps 2..9 =====================
    const int lg = warp & 3;                   // TMEM lane group of this warp
    const int ch = (warp - 2) >> 2;            // column half
    const int row_in_tile = lg * 32 + lane;
    const int c0 = (MODE == F8_FWD_SWIGLU) ? ch * 32 : ch * 64;
    const int c1 = (MODE == F8_FWD_SWIGLU) ? 64 + ch * 32 : ch * 64 + 32;
    int buf = 0;
    uint32_t bphase = 0;
    float amax_prev = 0.f;                     // fused Q-a: |a| max of this thread's 32 columns in the pair's first half
    Tile tl;
    for (int64_t t = 0; decode_tile<MODE>(p, t, total, tl); ++t) {
      const int64_t row = (int64_t)tl.m0 + row_in_tile;
      const bool row_ok = row < p.rows_valid;
      const float* sa_row = p.a_scales + (row_ok ? row : 0) * p.a_nblk;
      float acc0[32], acc1[32];
#pragma unroll
      for (int i = 0; i < 32; ++i) acc0[i] = acc1[i] = 0.f;
      float sa_n = __ldg(sa_row), s0_n, s1_n;
      weight_scales<MODE>(p, tl, 0, s0_n, s1_n);
      for (int kb = 0; kb < p.nkb; ++kb) {
        const float f0 = sa_n * s0_n, f1 = sa_n * s1_n;
        if (kb + 1 < p.nkb) {
          sa_n = __ldg(sa_row + kb + 1);
          weight_scales<MODE>(p, tl, kb + 1, s0_n, s1_n);
        }
        mbar_wait(pfull0 + 8 * buf, bphase);
        tc_fence_after();
        const uint32_t tacc = tmem_base + ((uint32_t)(lg * 32) << 16) + buf * BN;
        uint32_t v0[32], v1[32];
        tmem_ld32(tacc + c0, v0);
        tmem_ld32(tacc + c1, v1);
        tmem_ld_wait();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(pempty0 + 8 * buf);
#pragma unroll
        for (int i = 0; i < 32; ++i) {
          acc0[i] = fmaf(f0, __uint_as_float(v0[i]), acc0[i]);
          acc1[i] = fmaf(f1, __uint_as_float(v1[i]), acc1[i]);
        }
        if (++buf == NBUF) { buf = 0; bphase ^= 1; }
      }
      // rows past the buffer (row_ok false) store nothing, but still take part in the fused quantisers' barriers
      if (MODE == F8_FWD || MODE == F8_DGRAD) {
        __nv_bfloat16* dst = p.out0 + row * p.ld0 + tl.n0;
        if (row_ok) {
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            *reinterpret_cast<uint4*>(dst + c0 + q * 8) = pack8(acc0 + q * 8);
            *reinterpret_cast<uint4*>(dst + c1 + q * 8) = pack8(acc1 + q * 8);
          }
        }
      } else if (MODE == F8_FWD_SWIGLU) {
        const int col = tl.n0 + ch * 32;
        __nv_bfloat16* gdst = p.out0 + row * p.ld0 + col;
        __nv_bfloat16* udst = gdst + p.F;
        __nv_bfloat16* adst = p.out1 + row * p.ld1 + col;
        if (row_ok) {
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            *reinterpret_cast<uint4*>(gdst + q * 8) = pack8(acc0 + q * 8);
            *reinterpret_cast<uint4*>(udst + q * 8) = pack8(acc1 + q * 8);
          }
        }
#pragma unroll
        for (int i = 0; i < 32; ++i) acc0[i] = acc0[i] * fast_sigmoid8(acc0[i]) * acc1[i];
        uint4 ab[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          ab[q] = pack8(acc0 + q * 8);
          if (row_ok) *reinterpret_cast<uint4*>(adst + q * 8) = ab[q];
        }
        if (p.q_codes) {
          // fused Q-a (R9): quantise the bf16 a just written, 1 x 128 along F.  A block = the two 64-column halves this
          // CTA computes back to back (t even, odd) x the two column-half warps of this lane group.
          float am = 0.f;
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            const uint32_t wv[4] = {ab[q].x, ab[q].y, ab[q].z, ab[q].w};
#pragma unroll
            for (int i = 0; i < 4; ++i) am = fmaxf(am, fmaxf(fabsf(bf16_lo(wv[i])), fabsf(bf16_hi(wv[i]))));
          }
          if ((t & 1) == 0) {
            amax_prev = am;                                            // first half: wait for the second
          } else {
            am = fmaxf(am, amax_prev);
            float* slot = xch + (((t >> 1) & 1) * 2 * BM + row_in_tile) * 2;
            slot[ch] = am;
            named_bar_sync(1 + lg, 64);                                // the two warps that share these 128 rows' blocks
            const float sc = fp8_block_scale(fmaxf(slot[0], slot[1]), p.q_mode);
            const float isc = 1.0f / sc;
            if (row_ok) {
            const int blk0 = tl.n0 - BN / 2;                           // first column of the 128-column block
            uint8_t* cdst = p.q_codes + row * (int64_t)p.F + blk0 + ch * 32;
            // first half: this thread's own earlier bf16 stores, read back (L2-hot, same thread: program order)
            const volatile uint4* prev = reinterpret_cast<const volatile uint4*>(adst - BN / 2);
            uint32_t c0w[8], c1w[8];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
              uint4 pv;
              pv.x = prev[q].x; pv.y = prev[q].y; pv.z = prev[q].z; pv.w = prev[q].w;
              const uint32_t w0[4] = {pv.x, pv.y, pv.z, pv.w}, w1[4] = {ab[q].x, ab[q].y, ab[q].z, ab[q].w};
#pragma unroll
              for (int h = 0; h < 2; ++h) {
                c0w[q * 2 + h] = enc4(bf16_lo(w0[2 * h]), bf16_hi(w0[2 * h]), bf16_lo(w0[2 * h + 1]), bf16_hi(w0[2 * h + 1]), sc, isc, p.q_mode);
                c1w[q * 2 + h] = enc4(bf16_lo(w1[2 * h]), bf16_hi(w1[2 * h]), bf16_lo(w1[2 * h + 1]), bf16_hi(w1[2 * h + 1]), sc, isc, p.q_mode);
              }
            }
            *reinterpret_cast<uint4*>(cdst) = make_uint4(c0w[0], c0w[1], c0w[2], c0w[3]);
            *reinterpret_cast<uint4*>(cdst + 16) = make_uint4(c0w[4], c0w[5], c0w[6], c0w[7]);
            *reinterpret_cast<uint4*>(cdst + BN / 2) = make_uint4(c1w[0], c1w[1], c1w[2], c1w[3]);
            *reinterpret_cast<uint4*>(cdst + BN / 2 + 16) = make_uint4(c1w[4], c1w[5], c1w[6], c1w[7]);
            if (ch == 0) p.q_scales[row * (int64_t)(p.F / 128) + blk0 / 128] = sc;
            }
          }
        }
      } else {  // F8_DGRAD_SWIGLU: this thread owns the 64 columns [ch * 64, ch * 64 + 64) of dg and of du of its row
        float rw = 1.0f;
        if (p.w && row_ok) {
          const int pf = p.p2f[row];
          rw = pf >= 0 ? p.w[pf] : 0.f;
        }
        uint4 dgp[8], dup[8];               // bf16 dg / du, 8 columns per uint4 (kept for the fused quantiser)
#pragma unroll
        for (int half = 0; half < 2; ++half) {
          const int col = tl.n0 + (half ? c1 : c0);
          const float* acc = half ? acc1 : acc0;
          const __nv_bfloat16* gsrc = p.gu + row * p.ldgu + col;
          __nv_bfloat16* dgdst = p.out0 + row * p.ld0 + col;
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            uint4 gq = make_uint4(0u, 0u, 0u, 0u), uq = gq;
            if (row_ok) {
              gq = *reinterpret_cast<const uint4*>(gsrc + q * 8);
              uq = *reinterpret_cast<const uint4*>(gsrc + p.F + q * 8);
            }
            const uint32_t gw[4] = {gq.x, gq.y, gq.z, gq.w}, uw[4] = {uq.x, uq.y, uq.z, uq.w};
            float og[8], ou[8];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              const float g0 = bf16_lo(gw[i]), g1 = bf16_hi(gw[i]), u0 = bf16_lo(uw[i]), u1 = bf16_hi(uw[i]);
              const float d0 = rw * acc[q * 8 + 2 * i], d1 = rw * acc[q * 8 + 2 * i + 1];
              const float s0 = fast_sigmoid8(g0), s1 = fast_sigmoid8(g1);
              og[2 * i] = d0 * u0 * s0 * (1.0f + g0 * (1.0f - s0));
              og[2 * i + 1] = d1 * u1 * s1 * (1.0f + g1 * (1.0f - s1));
              ou[2 * i] = d0 * g0 * s0;
              ou[2 * i + 1] = d1 * g1 * s1;
            }
            dgp[half * 4 + q] = pack8(og);
            dup[half * 4 + q] = pack8(ou);
            if (row_ok) {
              *reinterpret_cast<uint4*>(dgdst + q * 8) = dgp[half * 4 + q];
              *reinterpret_cast<uint4*>(dgdst + p.F + q * 8) = dup[half * 4 + q];
            }
          }
        }
        if (p.q_codes) {
          // fused Q-dgu (R9): 1 x 128 blocks of [dg | du] along 2F; this tile's 128 columns are exactly one block of dg and
          // one of du, shared with the other column-half warp of the lane group.
          float amg = 0.f, amu = 0.f;
#pragma unroll
          for (int q = 0; q < 8; ++q) {
            const uint32_t wg[4] = {dgp[q].x, dgp[q].y, dgp[q].z, dgp[q].w}, wu[4] = {dup[q].x, dup[q].y, dup[q].z, dup[q].w};
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              amg = fmaxf(amg, fmaxf(fabsf(bf16_lo(wg[i])), fabsf(bf16_hi(wg[i]))));
              amu = fmaxf(amu, fmaxf(fabsf(bf16_lo(wu[i])), fabsf(bf16_hi(wu[i]))));
            }
          }
          float* slot = xch + ((t & 1) * 2 * BM) * 2;                   // [parity][g|u][row][ch]
          slot[(0 * BM + row_in_tile) * 2 + ch] = amg;
          slot[(1 * BM + row_in_tile) * 2 + ch] = amu;
          named_bar_sync(1 + lg, 64);
          const float sg = fp8_block_scale(fmaxf(slot[(0 * BM + row_in_tile) * 2], slot[(0 * BM + row_in_tile) * 2 + 1]), p.q_mode);
          const float su = fp8_block_scale(fmaxf(slot[(1 * BM + row_in_tile) * 2], slot[(1 * BM + row_in_tile) * 2 + 1]), p.q_mode);
          const float isg = 1.0f / sg, isu = 1.0f / su;
          if (row_ok) {
            uint8_t* cg = p.q_codes + row * (int64_t)(2 * p.F) + tl.n0 + ch * 64;
            uint8_t* cu = cg + p.F;
#pragma unroll
            for (int q = 0; q < 8; q += 2) {
              uint32_t eg[4], eu[4];
#pragma unroll
              for (int h = 0; h < 2; ++h) {
                const uint4 vg = dgp[q + h], vu = dup[q + h];
                eg[2 * h] = enc4(bf16_lo(vg.x), bf16_hi(vg.x), bf16_lo(vg.y), bf16_hi(vg.y), sg, isg, p.q_mode);
                eg[2 * h + 1] = enc4(bf16_lo(vg.z), bf16_hi(vg.z), bf16_lo(vg.w), bf16_hi(vg.w), sg, isg, p.q_mode);
                eu[2 * h] = enc4(bf16_lo(vu.x), bf16_hi(vu.x), bf16_lo(vu.y), bf16_hi(vu.y), su, isu, p.q_mode);
                eu[2 * h + 1] = enc4(bf16_lo(vu.z), bf16_hi(vu.z), bf16_lo(vu.w), bf16_hi(vu.w), su, isu, p.q_mode);
              }
              *reinterpret_cast<uint4*>(cg + q * 8) = make_uint4(eg[0], eg[1], eg[2], eg[3]);
              *reinterpret_cast<uint4*>(cu + q * 8) = make_uint4(eu[0], eu[1], eu[2], eu[3]);
            }
            if (ch == 0) {
              float* sc = p.q_scales + row * (int64_t)(2 * p.F / 128);
              sc[tl.n0 / 128] = sg;
              sc[(p.F + tl.n0) / 128] = su;
            }
          }
        }
      }
      __syncwarp();
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem_base, TMEM_COLS);
}

// ---------------------------------------------------------------------------------------------
// the wide kernel: F8_FWD / F8_DGRAD on 128 x 256 tiles
// ---------------------------------------------------------------------------------------------
// All four modes when the output width allows.  Same roles and the same two-level accumulation as above, but a tile is
// 256 accumulator columns wide (the fused SwiGLU forward: 128 gate + 128 up columns = one whole 1 x 128 block of a): 48 KB of operands per 128-deep k-block feed twice
// the MACs of a 128 x 128 tile's 32 KB (the narrow kernel is bound by that feed), the partial product
// of a k-block lands in one of two 256-column TMEM buffers, and a promotion thread owns one row x 128 columns = exactly one
// weight-scale column block (128 fp32 accumulators in registers).
constexpr int WBN = 256, WSTAGES = 4, WB_BYTES = WBN * BK, WSTAGE_BYTES = A_BYTES + WB_BYTES, WNBUF = 2;
static_assert(WSTAGES * WSTAGE_BYTES <= STAGES * STAGE_BYTES, "fits the same shared-memory allocation");

template <int MODE>
__device__ __forceinline__ bool wide_tile(const F8Params& p, int64_t i, int64_t total, Tile& tl) {
  const int64_t t = blockIdx.x + i * (int64_t)gridDim.x;
  if (t >= total) return false;
  const int mt = (int)(t / p.n_tiles);
  tl.n0 = (int)(t - (int64_t)mt * p.n_tiles) * (MODE == F8_FWD_SWIGLU ? WBN / 2 : WBN);   // SwiGLU: 128 gate + 128 up
  tl.m0 = mt * BM;
  tl.e = p.mtile ? p.mtile[1 + mt] : 0;
  return true;
}

template <int MODE>
__global__ void __launch_bounds__(NTHREADS, 1)
f8_wide_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB0,
               const __grid_constant__ CUtensorMap tmB1, const F8Params p) {
  constexpr bool B_MN = (MODE == F8_DGRAD || MODE == F8_DGRAD_SWIGLU);
  extern __shared__ uint8_t smem_raw[];
  const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  float* const xch = reinterpret_cast<float*>(smem_raw + (base - smem_u32(smem_raw)) + WSTAGES * WSTAGE_BYTES);
  const uint32_t bars = base + WSTAGES * WSTAGE_BYTES + XCH_BYTES;
  const uint32_t full0 = bars, empty0 = bars + 8 * WSTAGES, pfull0 = bars + 16 * WSTAGES, pempty0 = pfull0 + 8 * WNBUF;
  const uint32_t tmem_slot = pempty0 + 8 * WNBUF;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmA);
    tma_prefetch_desc(&tmB0);
    tma_prefetch_desc(&tmB1);
    for (int s = 0; s < WSTAGES; ++s) {
      mbar_init(full0 + 8 * s, 1);
      mbar_init(empty0 + 8 * s, 1);
    }
    for (int b = 0; b < WNBUF; ++b) {
      mbar_init(pfull0 + 8 * b, 1);
      mbar_init(pempty0 + 8 * b, EPI_WARPS);
    }
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc(tmem_slot, WNBUF * WBN);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

  const int64_t total = total_tiles(p);

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      Tile tl;
      for (int64_t t = 0; wide_tile<MODE>(p, t, total, tl); ++t) {
        for (int kb = 0; kb < p.nkb; ++kb) {
          mbar_wait(empty0 + 8 * stage, phase ^ 1);
          const uint32_t fb = full0 + 8 * stage;
          const uint32_t sa = base + stage * WSTAGE_BYTES, sb = sa + A_BYTES;
          mbar_expect_tx(fb, WSTAGE_BYTES);
          tma_load_2d(sa, &tmA, fb, kb * BK, tl.m0);                                   // 128 B x 128 rows
          if (MODE == F8_FWD) {
            tma_load_2d(sb, &tmB0, fb, kb * BK, tl.e * p.b_rows + tl.n0);              // 128 B x 256 rows
          } else if (MODE == F8_FWD_SWIGLU) {
            tma_load_2d(sb, &tmB0, fb, kb * BK, tl.e * p.b_rows + tl.n0);              // 128 B x 128 rows (Wg)
            tma_load_2d(sb + WB_BYTES / 2, &tmB1, fb, kb * BK, tl.e * p.b_rows + tl.n0);   // (Wu)
          } else {
            const bool second = kb >= p.kb_split;
            const int kr = tl.e * p.b_rows + (second ? kb - p.kb_split : kb) * BK;
#pragma unroll
            for (int i = 0; i < WBN / 128; ++i)                                        // 128 cols x 128 k-rows each
              tma_load_2d(sb + i * (128 * BK), second ? &tmB1 : &tmB0, fb, tl.n0 + 128 * i, kr);
          }
          if (++stage == WSTAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (lane == 0) {
      constexpr uint32_t idesc = instr_desc(0, 0, B_MN ? 1 : 0, WBN);
      int stage = 0, buf = 0;
      uint32_t phase = 0, bphase = 0;
      Tile tl;
      for (int64_t t = 0; wide_tile<MODE>(p, t, total, tl); ++t) {
        for (int kb = 0; kb < p.nkb; ++kb) {
          mbar_wait(pempty0 + 8 * buf, bphase ^ 1);
          mbar_wait(full0 + 8 * stage, phase);
          tc_fence_after();
          const uint32_t sa = base + stage * WSTAGE_BYTES, sb = sa + A_BYTES;
          const uint32_t dacc = tmem_base + buf * WBN;
#pragma unroll
          for (int k = 0; k < BK / UK; ++k) {
            const uint64_t ad = smem_desc(sa + k * UK, 16, 1024);
            // MN-major B: two 128-column boxes, 128 * BK bytes apart (LBO)
            const uint64_t bd = B_MN ? smem_desc(sb + k * UK * 128, 128 * BK, 1024) : smem_desc(sb + k * UK, 16, 1024);
            umma_f8(dacc, ad, bd, idesc, k != 0);
          }
          umma_commit(empty0 + 8 * stage);
          umma_commit(pfull0 + 8 * buf);
          if (++stage == WSTAGES) { stage = 0; phase ^= 1; }
          if (++buf == WNBUF) { buf = 0; bphase ^= 1; }
        }
      }
    }
  } else {
    // ===================== promotion + epilogue warps 2..9 =====================
    // A thread owns one row and 128 accumulator columns: columns [ch * 128, + 128) of the tile, or for the fused SwiGLU
    // forward 64 gate columns [ch * 64, + 64) and the 64 up columns of the same outputs [128 + ch * 64, + 64).
    constexpr bool SW = (MODE == F8_FWD_SWIGLU);
    const int lg = warp & 3;                   // TMEM lane group of this warp
    const int ch = (warp - 2) >> 2;
    const int row_in_tile = lg * 32 + lane;
    const int c0 = SW ? ch * 64 : ch * 128;                 // first TMEM column of accumulators 0..63
    const int c1 = SW ? 128 + ch * 64 : ch * 128 + 64;      // ... and of accumulators 64..127
    int buf = 0;
    uint32_t bphase = 0;
    Tile tl;
    for (int64_t t = 0; wide_tile<MODE>(p, t, total, tl); ++t) {
      const int64_t row = (int64_t)tl.m0 + row_in_tile;
      const bool row_ok = row < p.rows_valid;
      const float* sa_row = p.a_scales + (row_ok ? row : 0) * p.a_nblk;
      const int nb = tl.n0 / 128 + (SW ? 0 : ch);             // weight-scale column block of this thread
      // weight scale(s) of k-block kb: one scalar, or the gate / up pair of the SwiGLU forward
      auto wscale = [&](int kb, float& s0, float& s1) {
        if (MODE == F8_FWD || SW) {
          const int64_t i = ((int64_t)tl.e * (p.b_rows / 128) + nb) * p.nb_b_cols + kb;
          s0 = __ldg(p.b0_scales + i);
          s1 = SW ? __ldg(p.b1_scales + i) : s0;
        } else {
          const bool second = kb >= p.kb_split;
          s0 = s1 = __ldg((second ? p.b1_scales : p.b0_scales) +
                          ((int64_t)tl.e * (p.b_rows / 128) + (second ? kb - p.kb_split : kb)) * p.nb_b_cols + nb);
        }
      };
      float acc[128];
#pragma unroll
      for (int i = 0; i < 128; ++i) acc[i] = 0.f;
      float sa_n = __ldg(sa_row), s0_n, s1_n;
      wscale(0, s0_n, s1_n);
      for (int kb = 0; kb < p.nkb; ++kb) {
        const float f0 = sa_n * s0_n, f1 = sa_n * s1_n;
        if (kb + 1 < p.nkb) {
          sa_n = __ldg(sa_row + kb + 1);
          wscale(kb + 1, s0_n, s1_n);
        }
        mbar_wait(pfull0 + 8 * buf, bphase);
        tc_fence_after();
        const uint32_t tacc = tmem_base + ((uint32_t)(lg * 32) << 16) + buf * WBN;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          uint32_t v[32];
          tmem_ld32(tacc + (j < 2 ? c0 + j * 32 : c1 + (j - 2) * 32), v);
          tmem_ld_wait();
          if (j == 3) {                        // the buffer is drained: the MMAs of k-block kb + 2 may overwrite it
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(pempty0 + 8 * buf);
          }
          const float f = j < 2 ? f0 : f1;
#pragma unroll
          for (int i = 0; i < 32; ++i) acc[j * 32 + i] = fmaf(f, __uint_as_float(v[i]), acc[j * 32 + i]);
        }
        if (++buf == WNBUF) { buf = 0; bphase ^= 1; }
      }
      if (MODE == F8_FWD || MODE == F8_DGRAD) {
        if (row_ok) {
          __nv_bfloat16* dst = p.out0 + row * p.ld0 + tl.n0 + ch * 128;
#pragma unroll
          for (int q = 0; q < 16; ++q) *reinterpret_cast<uint4*>(dst + q * 8) = pack8(acc + q * 8);
        }
      } else if (SW) {
        // g = acc[0..63], u = acc[64..127] of output columns n0 + ch * 64 ..; a = silu(g) * u
        const int col = tl.n0 + ch * 64;
        __nv_bfloat16* gdst = p.out0 + row * p.ld0 + col;
        __nv_bfloat16* adst = p.out1 + row * p.ld1 + col;
        if (row_ok) {
#pragma unroll
          for (int q = 0; q < 8; ++q) {
            *reinterpret_cast<uint4*>(gdst + q * 8) = pack8(acc + q * 8);
            *reinterpret_cast<uint4*>(gdst + p.F + q * 8) = pack8(acc + 64 + q * 8);
          }
        }
#pragma unroll
        for (int i = 0; i < 64; ++i) acc[i] = acc[i] * fast_sigmoid8(acc[i]) * acc[64 + i];
        uint4 ab[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) {
          ab[q] = pack8(acc + q * 8);
          if (row_ok) *reinterpret_cast<uint4*>(adst + q * 8) = ab[q];
        }
        if (p.q_codes) {
          // fused Q-a (R9): quantise the bf16 a just written, 1 x 128 along F = this tile's 128 columns, shared with the
          // other column-half warp of the lane group (amax exchanged through shared memory, double-buffered by tile parity)
          float am = 0.f;
#pragma unroll
          for (int q = 0; q < 8; ++q) {
            const uint32_t wv[4] = {ab[q].x, ab[q].y, ab[q].z, ab[q].w};
#pragma unroll
            for (int i = 0; i < 4; ++i) am = fmaxf(am, fmaxf(fabsf(bf16_lo(wv[i])), fabsf(bf16_hi(wv[i]))));
          }
          float* slot = xch + ((t & 1) * BM + row_in_tile) * 2;
          slot[ch] = am;
          named_bar_sync(1 + lg, 64);
          const float sc = fp8_block_scale(fmaxf(slot[0], slot[1]), p.q_mode);
          const float isc = 1.0f / sc;
          if (row_ok) {
            uint8_t* cdst = p.q_codes + row * (int64_t)p.F + col;
#pragma unroll
            for (int q = 0; q < 8; q += 2) {
              uint32_t e[4];
#pragma unroll
              for (int h = 0; h < 2; ++h) {
                const uint4 va = ab[q + h];
                e[2 * h] = enc4(bf16_lo(va.x), bf16_hi(va.x), bf16_lo(va.y), bf16_hi(va.y), sc, isc, p.q_mode);
                e[2 * h + 1] = enc4(bf16_lo(va.z), bf16_hi(va.z), bf16_lo(va.w), bf16_hi(va.w), sc, isc, p.q_mode);
              }
              *reinterpret_cast<uint4*>(cdst + q * 8) = make_uint4(e[0], e[1], e[2], e[3]);
            }
            if (ch == 0) p.q_scales[row * (int64_t)(p.F / 128) + tl.n0 / 128] = sc;
          }
        }
      } else {
        // F8_DGRAD_SWIGLU: acc = da of columns [n0 + ch * 128, + 128) of F: one whole 1 x 128 block of dg and one of du
        float rw = 1.0f;
        if (p.w && row_ok) {
          const int pf = p.p2f[row];
          rw = pf >= 0 ? p.w[pf] : 0.f;
        }
        const int col = tl.n0 + ch * 128;
        const __nv_bfloat16* gsrc = p.gu + row * p.ldgu + col;
        __nv_bfloat16* dgdst = p.out0 + row * p.ld0 + col;
        float amg = 0.f, amu = 0.f;
#pragma unroll
        for (int q = 0; q < 16; ++q) {
          uint4 gq = make_uint4(0u, 0u, 0u, 0u), uq = gq;
          if (row_ok) {
            gq = *reinterpret_cast<const uint4*>(gsrc + q * 8);
            uq = *reinterpret_cast<const uint4*>(gsrc + p.F + q * 8);
          }
          const uint32_t gw[4] = {gq.x, gq.y, gq.z, gq.w}, uw[4] = {uq.x, uq.y, uq.z, uq.w};
          float og[8], ou[8];
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const float g0 = bf16_lo(gw[i]), g1 = bf16_hi(gw[i]), u0 = bf16_lo(uw[i]), u1 = bf16_hi(uw[i]);
            const float d0 = rw * acc[q * 8 + 2 * i], d1 = rw * acc[q * 8 + 2 * i + 1];
            const float s0 = fast_sigmoid8(g0), s1 = fast_sigmoid8(g1);
            og[2 * i] = d0 * u0 * s0 * (1.0f + g0 * (1.0f - s0));
            og[2 * i + 1] = d1 * u1 * s1 * (1.0f + g1 * (1.0f - s1));
            ou[2 * i] = d0 * g0 * s0;
            ou[2 * i + 1] = d1 * g1 * s1;
          }
          const uint4 pg = pack8(og), pu = pack8(ou);
          if (row_ok) {
            *reinterpret_cast<uint4*>(dgdst + q * 8) = pg;
            *reinterpret_cast<uint4*>(dgdst + p.F + q * 8) = pu;
          }
          const uint32_t wg[4] = {pg.x, pg.y, pg.z, pg.w}, wu[4] = {pu.x, pu.y, pu.z, pu.w};
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            amg = fmaxf(amg, fmaxf(fabsf(bf16_lo(wg[i])), fabsf(bf16_hi(wg[i]))));
            amu = fmaxf(amu, fmaxf(fabsf(bf16_lo(wu[i])), fabsf(bf16_hi(wu[i]))));
          }
        }
        if (p.q_codes && row_ok) {
          // fused Q-dgu (R9): the thread holds the amax of its whole dg block and du block; the bf16 values are its own
          // stores of a moment ago, read back (L2-hot, same thread: program order) instead of 128 more live registers
          const float sg = fp8_block_scale(amg, p.q_mode), su = fp8_block_scale(amu, p.q_mode);
          const float isg = 1.0f / sg, isu = 1.0f / su;
          uint8_t* cg = p.q_codes + row * (int64_t)(2 * p.F) + col;
          const volatile uint4* rg = reinterpret_cast<const volatile uint4*>(dgdst);
          const volatile uint4* ru = reinterpret_cast<const volatile uint4*>(dgdst + p.F);
#pragma unroll
          for (int q = 0; q < 16; q += 2) {
            uint32_t eg[4], eu[4];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
              uint4 vg, vu;
              vg.x = rg[q + h].x; vg.y = rg[q + h].y; vg.z = rg[q + h].z; vg.w = rg[q + h].w;
              vu.x = ru[q + h].x; vu.y = ru[q + h].y; vu.z = ru[q + h].z; vu.w = ru[q + h].w;
              eg[2 * h] = enc4(bf16_lo(vg.x), bf16_hi(vg.x), bf16_lo(vg.y), bf16_hi(vg.y), sg, isg, p.q_mode);
              eg[2 * h + 1] = enc4(bf16_lo(vg.z), bf16_hi(vg.z), bf16_lo(vg.w), bf16_hi(vg.w), sg, isg, p.q_mode);
              eu[2 * h] = enc4(bf16_lo(vu.x), bf16_hi(vu.x), bf16_lo(vu.y), bf16_hi(vu.y), su, isu, p.q_mode);
              eu[2 * h + 1] = enc4(bf16_lo(vu.z), bf16_hi(vu.z), bf16_lo(vu.w), bf16_hi(vu.w), su, isu, p.q_mode);
            }
            *reinterpret_cast<uint4*>(cg + q * 8) = make_uint4(eg[0], eg[1], eg[2], eg[3]);
            *reinterpret_cast<uint4*>(cg + p.F + q * 8) = make_uint4(eu[0], eu[1], eu[2], eu[3]);
          }
          float* sc = p.q_scales + row * (int64_t)(2 * p.F / 128);
          sc[col / 128] = sg;
          sc[(p.F + col) / 128] = su;
        }
      }
      __syncwarp();
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem_base, WNBUF * WBN);
}

// ---------------------------------------------------------------------------------------------
// host
// ---------------------------------------------------------------------------------------------
bool g_attr_set[MAX_DEVICES][4];   // per device

template <int MODE>
int32_t launch(const CUtensorMap& a, const CUtensorMap& b0, const CUtensorMap& b1, const F8Params& p, int64_t max_tiles,
               cudaStream_t s) {
  const int dev = current_device();
  if (dev < 0) return MOE_ERR_CUDA;
  if (!g_attr_set[dev][MODE]) {
    MOE_CUDA(cudaFuncSetAttribute(f8_gemm_kernel<MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES));
    g_attr_set[dev][MODE] = true;
  }
  const int sms = tc_sm_count();
  if (sms <= 0) return MOE_ERR_CUDA;
  const unsigned grid = (unsigned)std::max<int64_t>(1, std::min<int64_t>(sms, max_tiles));
  MOE_LAUNCH(f8_gemm_kernel<MODE>, grid, NTHREADS, SMEM_BYTES, s, a, b0, b1, p);
  return MOE_OK;
}

bool g_wide_attr[MAX_DEVICES][4];

template <int MODE>
int32_t launch_wide(const CUtensorMap& a, const CUtensorMap& b0, const CUtensorMap& b1, const F8Params& p, int64_t max_tiles,
                    cudaStream_t s) {
  const int dev = current_device();
  if (dev < 0) return MOE_ERR_CUDA;
  if (!g_wide_attr[dev][MODE]) {
    MOE_CUDA(cudaFuncSetAttribute(f8_wide_kernel<MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES));
    g_wide_attr[dev][MODE] = true;
  }
  const int sms = tc_sm_count();
  if (sms <= 0) return MOE_ERR_CUDA;
  const unsigned grid = (unsigned)std::max<int64_t>(1, std::min<int64_t>(sms, max_tiles));
  MOE_LAUNCH(f8_wide_kernel<MODE>, grid, NTHREADS, SMEM_BYTES, s, a, b0, b1, p);
  return MOE_OK;
}

// 128 x 256 tiles when the output width allows.  Default (1): the plain-epilogue GEMMs (gemm2, dgrad gate/up: configs[3]
// 1.46 -> 1.16 ms, 2.71 -> 2.51 ms).  The fused-SwiGLU modes run on the wide kernel too (parity-tested) but slower (gemm1
// 2.66 -> 2.86 ms, dgrad-down 1.67 -> 1.78 ms): their long epilogues are not overlapped with the next tile's main loop, and
// two TMEM buffers give the MMAs less slack than four.  moe_config_t::opt_fp8_wide: level 0 (never) / 1 / 2 (all modes).
bool use_wide(const F8Call& c, int N, bool swiglu) {
  const int level = c.opt_wide ? c.opt_wide - 1 : 1;
  return level > (swiglu ? 1 : 0) && N % WBN == 0;
}

}  // namespace

int32_t fp8_gemm(const F8Call& c, cudaStream_t s) {
  if (c.mtile == nullptr && c.E != 1) return MOE_ERR_UNSUPPORTED;
  if (!c.A || !c.a_scales || !c.B0 || !c.b0_scales || !c.out0) return MOE_ERR_INVALID_ARG;
  if (c.lda % 128 || c.b_rows % 128 || c.b_cols % 128 || (c.ld0 & 7)) return MOE_ERR_UNSUPPORTED;
  F8Params p;
  memset(&p, 0, sizeof(p));
  p.E = c.E;
  p.rows_valid = c.rows_cap;
  p.mtile = c.mtile;
  p.a_scales = c.a_scales;
  p.a_nblk = c.lda / 128;
  p.b0_scales = c.b0_scales;
  p.b1_scales = c.b1_scales ? c.b1_scales : c.b0_scales;
  p.b_rows = c.b_rows;
  p.nb_b_cols = c.b_cols / 128;
  p.N = c.N;
  p.F = c.F;
  p.out0 = (__nv_bfloat16*)c.out0;
  p.ld0 = c.ld0;
  p.out1 = (__nv_bfloat16*)c.out1;
  p.ld1 = c.ld1;
  p.gu = (const __nv_bfloat16*)c.gu;
  p.ldgu = c.ldgu;
  p.p2f = c.p2f;
  p.w = c.w;
  p.q_codes = c.q_codes;
  p.q_scales = c.q_scales;
  p.q_mode = c.q_mode;
  if (c.q_codes && (!c.q_scales || c.F % 128 != 0)) return MOE_ERR_INVALID_ARG;
  CUtensorMap ta, tb0, tb1;
  const int64_t max_mtiles = ceil_div(c.rows_cap, BM);
  const int64_t wrows = (int64_t)c.E * c.b_rows;
  switch (c.mode) {
    case F8_FWD: {
      if (c.lda != c.b_cols || c.N != c.b_rows) return MOE_ERR_INVALID_ARG;
      p.nkb = c.b_cols / BK;
      const bool wide = use_wide(c, c.N, false);
      p.n_tiles = c.N / (wide ? WBN : BN);
      if (!tc_make_map(&ta, 1, c.A, c.lda, c.rows_cap, c.lda, BK, BM)) return MOE_ERR_UNSUPPORTED;
      if (!tc_make_map(&tb0, 1, c.B0, c.b_cols, wrows, c.b_cols, BK, wide ? WBN : BN)) return MOE_ERR_UNSUPPORTED;
      if (wide) return launch_wide<F8_FWD>(ta, tb0, tb0, p, max_mtiles * p.n_tiles, s);
      return launch<F8_FWD>(ta, tb0, tb0, p, max_mtiles * p.n_tiles, s);
    }
    case F8_FWD_SWIGLU: {
      if (!c.B1 || !c.b1_scales || !c.out1 || c.lda != c.b_cols || c.F != c.b_rows || (c.ld1 & 7)) return MOE_ERR_INVALID_ARG;
      p.nkb = c.b_cols / BK;
      const bool wide = use_wide(c, 2 * c.F, true);          // a wide tile = 128 gate + 128 up columns: F is a multiple of 128 already
      p.n_tiles = c.F / ((wide ? WBN : BN) / 2);
      if (!tc_make_map(&ta, 1, c.A, c.lda, c.rows_cap, c.lda, BK, BM)) return MOE_ERR_UNSUPPORTED;
      if (!tc_make_map(&tb0, 1, c.B0, c.b_cols, wrows, c.b_cols, BK, (wide ? WBN : BN) / 2)) return MOE_ERR_UNSUPPORTED;
      if (!tc_make_map(&tb1, 1, c.B1, c.b_cols, wrows, c.b_cols, BK, (wide ? WBN : BN) / 2)) return MOE_ERR_UNSUPPORTED;
      if (wide) return launch_wide<F8_FWD_SWIGLU>(ta, tb0, tb1, p, max_mtiles * p.n_tiles, s);
      return launch<F8_FWD_SWIGLU>(ta, tb0, tb1, p, max_mtiles * p.n_tiles, s);
    }
    case F8_DGRAD:
    case F8_DGRAD_SWIGLU: {
      const bool split = c.B1 != nullptr;
      if (c.N != c.b_cols || c.lda != (split ? 2 : 1) * c.b_rows) return MOE_ERR_INVALID_ARG;
      p.kb_split = c.b_rows / BK;
      p.nkb = split ? 2 * p.kb_split : p.kb_split;
      const bool wide = use_wide(c, c.N, c.mode == F8_DGRAD_SWIGLU);
      p.n_tiles = c.N / (wide ? WBN : BN);
      if (!tc_make_map(&ta, 1, c.A, c.lda, c.rows_cap, c.lda, BK, BM)) return MOE_ERR_UNSUPPORTED;
      if (!tc_make_map(&tb0, 1, c.B0, c.b_cols, wrows, c.b_cols, BN, BK)) return MOE_ERR_UNSUPPORTED;
      if (!tc_make_map(&tb1, 1, split ? c.B1 : c.B0, c.b_cols, wrows, c.b_cols, BN, BK)) return MOE_ERR_UNSUPPORTED;
      if (c.mode == F8_DGRAD) {
        if (wide) return launch_wide<F8_DGRAD>(ta, tb0, tb1, p, max_mtiles * p.n_tiles, s);
        return launch<F8_DGRAD>(ta, tb0, tb1, p, max_mtiles * p.n_tiles, s);
      }
      if (!c.gu || c.F != c.b_cols || (c.ldgu & 7)) return MOE_ERR_INVALID_ARG;
      if (wide) return launch_wide<F8_DGRAD_SWIGLU>(ta, tb0, tb1, p, max_mtiles * p.n_tiles, s);
      return launch<F8_DGRAD_SWIGLU>(ta, tb0, tb1, p, max_mtiles * p.n_tiles, s);
    }
  }
  return MOE_ERR_INVALID_ARG;
}

}  // namespace moe
