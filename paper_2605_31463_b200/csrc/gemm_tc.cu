// tcgen05 / TMEM / TMA grouped GEMMs for sm_100a (bf16 in, fp32 accumulate in tensor memory, bf16 out).
//
// One persistent, warp-specialised kernel template serves every expert GEMM of the layer (SURVEY.md §8a
// a5, a6, a9..a12): warp 0 = TMA producer, warp 1 = MMA issuer (one elected thread, tcgen05.mma
// cta_group::1, M=128 x N=256 x K=16 per instruction), warps 2..5 = epilogue (tcgen05.ld from a
// double-buffered 2 x 256-column TMEM accumulator).  Operands are staged by TMA into 128-byte-swizzled
// shared memory, 4 stages of (128 x 64 A tile + 256 x 64 B tile) = 192 KB.  The tile schedule is
// computed on the device from the per-expert row offsets (shapes are data dependent; the
// counts never visit the host): a 128-row M-tile belongs to exactly one expert because expert groups
// start at multiples of 128 rows.  SwiGLU forward / backward are fused into the epilogues.
// Both K-major and MN-major shared-memory operand layouts are used, so the dgrad (weights read
// "transposed") and wgrad (both operands contracted over rows) need no transposed copies in HBM.
#include <cuda.h>
#include <string.h>

#include <algorithm>

#include "gemm_tc.cuh"
#include "tc_ptx.cuh"

namespace moe {

// ---------------------------------------------------------------------------------------------
// TMA tensor maps (shared with fp8.cu)
// ---------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = nullptr;
  static bool tried = false;
  if (!tried) {
    tried = true;
    void* sym = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(sym);
    else
      cudaGetLastError();
  }
  return fn;
}

bool tc_make_map(CUtensorMap* m, int elem_bytes, const void* ptr, int64_t inner, int64_t outer, int64_t ld,
                 int box_inner, int box_outer) {
  EncodeTiledFn fn = encode_fn();
  if (!fn || !ptr || inner <= 0 || outer <= 0) return false;
  if ((reinterpret_cast<uintptr_t>(ptr) & 15) || ((ld * elem_bytes) & 15)) return false;
  const cuuint64_t dims[2] = {(cuuint64_t)inner, (cuuint64_t)outer};
  const cuuint64_t strides[1] = {(cuuint64_t)ld * elem_bytes};
  const cuuint32_t box[2] = {(cuuint32_t)box_inner, (cuuint32_t)box_outer};
  const cuuint32_t estr[2] = {1, 1};
  const CUtensorMapDataType dt = elem_bytes == 2 ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16 : CU_TENSOR_MAP_DATA_TYPE_UINT8;
  return fn(m, dt, 2, const_cast<void*>(ptr), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

bool tc_make_map3(CUtensorMap* m, int elem_bytes, const void* ptr, int64_t d0, int64_t d1, int64_t d2, int64_t ld, int box0,
                  int box1) {
  EncodeTiledFn fn = encode_fn();
  if (!fn || !ptr || d0 <= 0 || d1 <= 0 || d2 <= 0) return false;
  if ((reinterpret_cast<uintptr_t>(ptr) & 15) || ((ld * elem_bytes) & 15)) return false;
  const cuuint64_t dims[3] = {(cuuint64_t)d0, (cuuint64_t)d1, (cuuint64_t)d2};
  const cuuint64_t strides[2] = {(cuuint64_t)ld * elem_bytes, (cuuint64_t)d1 * ld * elem_bytes};
  const cuuint32_t box[3] = {(cuuint32_t)box0, (cuuint32_t)box1, 1};
  const cuuint32_t estr[3] = {1, 1, 1};
  return fn(m, elem_bytes == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3,
            const_cast<void*>(ptr), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            box0 * elem_bytes == 64 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_128B,
            CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

int tc_sm_count() { return device_sm_count(); }

namespace {

constexpr int BM = 128;      // tile rows  (UMMA M)
constexpr int BN = 256;      // tile cols  (UMMA N)
constexpr int BK = 64;       // k-block: 64 bf16 = 128 bytes = one swizzle span
constexpr int UK = 16;       // UMMA K for 16-bit operands
constexpr int STAGES = 4;
constexpr int A_BYTES = BM * BK * 2;   // 16 KB
constexpr int B_BYTES = BN * BK * 2;   // 32 KB
constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
constexpr int MN_BOX_BYTES = 64 * BK * 2;  // one 64(MN) x 64(K) box of an MN-major operand: 8 KB
constexpr int OBUF_BYTES = BM * 128;       // epilogue staging: 128 rows x 64 bf16 columns (one 128-byte-swizzled TMA box)
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 2 * OBUF_BYTES + 1024 /*align*/ + 256 /*barriers*/;
constexpr int EPI_WARPS = 8;            // two per TMEM lane group: column-chunk parity `ch` splits a tile between them
constexpr int NTHREADS = 64 + EPI_WARPS * 32;
constexpr int TMEM_COLS = 512;

// ---------------------------------------------------------------------------------------------
// kernel parameters
// ---------------------------------------------------------------------------------------------
struct TcParams {
  int E, n_tiles, m_tiles, nkb, kb_split, b_rows, N, M, F, a_col0, tma_out, acc_f32;
  int64_t rows_valid;
  const int32_t* mtile;
  const int32_t* offsets;
  __nv_bfloat16* out0;
  int64_t ld0;
  __nv_bfloat16* out1;
  int64_t ld1;
  const __nv_bfloat16* gu;
  int64_t ldgu;
};

struct Tile {
  int e, m0, n0, nkb, row0;
};

template <int MODE>
__device__ __forceinline__ bool decode_tile(const TcParams& p, int64_t t, int64_t total, Tile& tl) {
  if (t >= total) return false;
  if (MODE == TC_WGRAD) {
    const int per_e = p.m_tiles * p.n_tiles;
    tl.e = (int)(t / per_e);
    const int r = (int)(t - (int64_t)tl.e * per_e);
    tl.m0 = (r / p.n_tiles) * BM;
    tl.n0 = (r % p.n_tiles) * BN;
    if (p.mtile) {
      tl.row0 = p.offsets[tl.e];
      tl.nkb = (p.offsets[tl.e + 1] - tl.row0) / BK;
    } else {
      tl.row0 = 0;
      tl.nkb = (int)((p.rows_valid + BK - 1) / BK);
    }
  } else {
    // n fastest: consecutive CTAs share the 128-row activation tile
    const int mt = (int)(t / p.n_tiles);
    tl.n0 = (int)(t - (int64_t)mt * p.n_tiles) * (MODE == TC_FWD_SWIGLU ? BN / 2 : BN);
    tl.m0 = mt * BM;
    tl.e = p.mtile ? p.mtile[1 + mt] : 0;
    tl.nkb = p.nkb;
    tl.row0 = 0;
  }
  return true;
}

template <int MODE>
__device__ __forceinline__ int64_t total_tiles(const TcParams& p) {
  if (MODE == TC_WGRAD) return (int64_t)p.E * p.m_tiles * p.n_tiles;
  const int64_t mt = p.mtile ? p.mtile[0] : (p.rows_valid + BM - 1) / BM;
  return mt * p.n_tiles;
}

// ---------------------------------------------------------------------------------------------
// epilogues: thread = tile row (TMEM lane); 32-column chunks; direct 16-byte global stores
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void store_row_chunk(__nv_bfloat16* dst, const uint32_t (&v)[32], int ncols) {
  // dst: first of 32 output columns of this thread's row (16-byte aligned); ncols valid (multiple of 8)
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    if (q * 8 < ncols) {
      uint4 o;
      o.x = pack_bf16(__uint_as_float(v[q * 8 + 0]), __uint_as_float(v[q * 8 + 1]));
      o.y = pack_bf16(__uint_as_float(v[q * 8 + 2]), __uint_as_float(v[q * 8 + 3]));
      o.z = pack_bf16(__uint_as_float(v[q * 8 + 4]), __uint_as_float(v[q * 8 + 5]));
      o.w = pack_bf16(__uint_as_float(v[q * 8 + 6]), __uint_as_float(v[q * 8 + 7]));
      *reinterpret_cast<uint4*>(dst + q * 8) = o;
    }
  }
}

__device__ __forceinline__ float fast_sigmoid(float x) { return __fdividef(1.0f, 1.0f + __expf(-x)); }

template <int MODE>
__device__ __forceinline__ void epilogue_tile(const TcParams& p, const Tile& tl, uint32_t tacc, int row_in_tile,
                                              bool have_acc, int ch) {
  // tacc: TMEM address of this warp's lane group at the accumulator stage's first column
  if (MODE == TC_FWD || MODE == TC_DGRAD) {
    const int64_t row = (int64_t)tl.m0 + row_in_tile;
    const bool row_ok = row < p.rows_valid;
    __nv_bfloat16* dst = p.out0 + row * p.ld0 + tl.n0;
#pragma unroll 1
    for (int c = ch; c < BN / 32; c += 2) {
      const int ncols = p.N - (tl.n0 + c * 32);   // warp-uniform
      if (ncols <= 0) break;
      uint32_t v[32];
      tmem_ld32(tacc + c * 32, v);
      tmem_ld_wait();
      if (row_ok) store_row_chunk(dst + c * 32, v, ncols);
    }
  } else if (MODE == TC_FWD_F32) {
    const int64_t row = (int64_t)tl.m0 + row_in_tile;
    const bool row_ok = row < p.rows_valid;
    float* dst = reinterpret_cast<float*>(p.out0) + row * p.ld0 + tl.n0;
#pragma unroll 1
    for (int c = ch; c < BN / 32; c += 2) {
      const int ncols = p.N - (tl.n0 + c * 32);   // warp-uniform, multiple of 4
      if (ncols <= 0) break;
      uint32_t v[32];
      tmem_ld32(tacc + c * 32, v);
      tmem_ld_wait();
      if (row_ok) {
#pragma unroll
        for (int q = 0; q < 8; ++q)
          if (q * 4 < ncols)
            *reinterpret_cast<uint4*>(dst + c * 32 + q * 4) = make_uint4(v[q * 4], v[q * 4 + 1], v[q * 4 + 2], v[q * 4 + 3]);
      }
    }
  } else if (MODE == TC_FWD_SWIGLU) {
    // accumulator columns [0,128) = gate, [128,256) = up for output columns n0 .. n0+127
    const int64_t row = (int64_t)tl.m0 + row_in_tile;
    const bool row_ok = row < p.rows_valid;
    __nv_bfloat16* gdst = p.out0 + row * p.ld0 + tl.n0;
    __nv_bfloat16* udst = gdst + p.F;
    __nv_bfloat16* adst = p.out1 + row * p.ld1 + tl.n0;
#pragma unroll 1
    for (int c = ch; c < BN / 64; c += 2) {
      const int ncols = p.F - (tl.n0 + c * 32);
      if (ncols <= 0) break;
      uint32_t g[32], u[32];
      tmem_ld32(tacc + c * 32, g);
      tmem_ld32(tacc + BN / 2 + c * 32, u);
      tmem_ld_wait();
      if (row_ok) {
        store_row_chunk(gdst + c * 32, g, ncols);
        store_row_chunk(udst + c * 32, u, ncols);
      }
#pragma unroll
      for (int i = 0; i < 32; ++i) {
        const float gv = __uint_as_float(g[i]);
        g[i] = __float_as_uint(gv * fast_sigmoid(gv) * __uint_as_float(u[i]));
      }
      if (row_ok) store_row_chunk(adst + c * 32, g, ncols);
    }
  }
}

// TC_FWD_SWIGLU epilogue with F % 32 == 0: per 32-column chunk the warp group stages g and u (two 64-byte-swizzled
// 8 KB boxes) and stores them by TMA, then reuses the first box for a = silu(g) * u.
__device__ __forceinline__ void pack32_to_box(uint32_t rowaddr, int sw, const uint32_t (&v)[32]) {
#pragma unroll
  for (int q = 0; q < 4; ++q)
    st_shared_v4(rowaddr + ((q ^ sw) << 4), pack_bf16(__uint_as_float(v[q * 8 + 0]), __uint_as_float(v[q * 8 + 1])),
                 pack_bf16(__uint_as_float(v[q * 8 + 2]), __uint_as_float(v[q * 8 + 3])),
                 pack_bf16(__uint_as_float(v[q * 8 + 4]), __uint_as_float(v[q * 8 + 5])),
                 pack_bf16(__uint_as_float(v[q * 8 + 6]), __uint_as_float(v[q * 8 + 7])));
}

__device__ __forceinline__ void fwd_swiglu_tile_tma(const TcParams& p, const Tile& tl, uint32_t tacc, int row_in_tile,
                                                    uint32_t obuf, const CUtensorMap* tmGU, const CUtensorMap* tmAo,
                                                    bool issuer, int ch) {
  const uint32_t rowaddr = obuf + row_in_tile * 64;
  const int sw = (row_in_tile >> 1) & 3;
#pragma unroll 1
  for (int c = ch; c < BN / 64; c += 2) {
    if (p.F - (tl.n0 + c * 32) <= 0) break;     // warp-group uniform
    uint32_t g[32], u[32];
    tmem_ld32(tacc + c * 32, g);
    tmem_ld32(tacc + BN / 2 + c * 32, u);
    tmem_ld_wait();
    if (issuer) bulk_wait_read0();
    named_bar_sync(1 + ch, 128);
    pack32_to_box(rowaddr, sw, g);
    pack32_to_box(rowaddr + OBUF_BYTES / 2, sw, u);
    fence_proxy_async();
    named_bar_sync(1 + ch, 128);
    if (issuer) {
      tma_store_3d(tmGU, obuf, tl.n0 + c * 32, tl.m0, 0);
      tma_store_3d(tmGU, obuf + OBUF_BYTES / 2, p.F + tl.n0 + c * 32, tl.m0, 0);
      bulk_commit();
    }
#pragma unroll
    for (int i = 0; i < 32; ++i) {
      const float gv = __uint_as_float(g[i]);
      g[i] = __float_as_uint(gv * fast_sigmoid(gv) * __uint_as_float(u[i]));
    }
    if (issuer) bulk_wait_read0();
    named_bar_sync(1 + ch, 128);
    pack32_to_box(rowaddr, sw, g);
    fence_proxy_async();
    named_bar_sync(1 + ch, 128);
    if (issuer) {
      tma_store_3d(tmAo, obuf, tl.n0 + c * 32, tl.m0, 0);
      bulk_commit();
    }
  }
}

// TC_DGRAD_SWIGLU epilogue: acc = da [128 x 256 columns of F]; dgu = swiglu'(g, u) * da.  The saved g, u of this
// thread's row are fetched from HBM two 32-column chunks ahead of the TMEM drain (the first two before the
// accumulator is even complete), so their latency hides behind the main loop and the previous chunk's math.
struct GuChunk {
  uint4 g[4], u[4];
};

__device__ __forceinline__ void gu_load(const TcParams& p, const Tile& tl, int64_t row, bool row_ok, int c, GuChunk& k) {
  const int ncols = p.F - (tl.n0 + c * 32);
  if (!row_ok || ncols <= 0) return;
  const uint4* gp = reinterpret_cast<const uint4*>(p.gu + row * p.ldgu + tl.n0 + c * 32);
  const uint4* up = reinterpret_cast<const uint4*>(p.gu + row * p.ldgu + p.F + tl.n0 + c * 32);
#pragma unroll
  for (int q = 0; q < 4; ++q)
    if (q * 8 < ncols) {
      k.g[q] = __ldg(gp + q);
      k.u[q] = __ldg(up + q);
    }
}

// Output path: with F % 32 == 0 the chunk's dg and du (32 columns x 128 rows each) are staged in the warp group's two
// 64-byte-swizzled 8 KB boxes and written by TMA (full lines instead of 16-byte partial sectors per thread).
__device__ __forceinline__ void dgrad_swiglu_chunk(const TcParams& p, const Tile& tl, int64_t row, bool row_ok, int c,
                                                   uint32_t tacc, const GuChunk& k, uint32_t obuf, int row_in_tile,
                                                   const CUtensorMap* tmO, bool issuer, int ch) {
  const int ncols = p.F - (tl.n0 + c * 32);   // warp-uniform
  if (ncols <= 0) return;
  uint32_t d[32];
  tmem_ld32(tacc + c * 32, d);
  tmem_ld_wait();
  if (p.tma_out) {
    if (issuer) bulk_wait_read0();     // this group's previous stores have finished reading the boxes
    named_bar_sync(1 + ch, 128);
    const uint32_t rowaddr = obuf + row_in_tile * 64;
    const int sw = (row_in_tile >> 1) & 3;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const uint32_t gw[4] = {k.g[q].x, k.g[q].y, k.g[q].z, k.g[q].w}, uw[4] = {k.u[q].x, k.u[q].y, k.u[q].z, k.u[q].w};
      uint32_t og[4], ou[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const float g0 = bf16_lo(gw[i]), g1 = bf16_hi(gw[i]), u0 = bf16_lo(uw[i]), u1 = bf16_hi(uw[i]);
        const float d0 = __uint_as_float(d[q * 8 + 2 * i]), d1 = __uint_as_float(d[q * 8 + 2 * i + 1]);
        const float s0 = fast_sigmoid(g0), s1 = fast_sigmoid(g1);
        og[i] = pack_bf16(d0 * u0 * s0 * (1.0f + g0 * (1.0f - s0)), d1 * u1 * s1 * (1.0f + g1 * (1.0f - s1)));
        ou[i] = pack_bf16(d0 * g0 * s0, d1 * g1 * s1);
      }
      if (!row_ok) og[0] = og[1] = og[2] = og[3] = ou[0] = ou[1] = ou[2] = ou[3] = 0u;   // clipped by the map anyway
      st_shared_v4(rowaddr + ((q ^ sw) << 4), og[0], og[1], og[2], og[3]);
      st_shared_v4(rowaddr + OBUF_BYTES / 2 + ((q ^ sw) << 4), ou[0], ou[1], ou[2], ou[3]);
    }
    fence_proxy_async();
    named_bar_sync(1 + ch, 128);
    if (issuer) {
      tma_store_3d(tmO, obuf, tl.n0 + c * 32, tl.m0, 0);
      tma_store_3d(tmO, obuf + OBUF_BYTES / 2, p.F + tl.n0 + c * 32, tl.m0, 0);
      bulk_commit();
    }
    return;
  }
  if (!row_ok) return;
  __nv_bfloat16* dgdst = p.out0 + row * p.ld0 + tl.n0 + c * 32;
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    if (q * 8 < ncols) {
      const uint32_t gw[4] = {k.g[q].x, k.g[q].y, k.g[q].z, k.g[q].w}, uw[4] = {k.u[q].x, k.u[q].y, k.u[q].z, k.u[q].w};
      uint32_t og[4], ou[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const float g0 = bf16_lo(gw[i]), g1 = bf16_hi(gw[i]), u0 = bf16_lo(uw[i]), u1 = bf16_hi(uw[i]);
        const float d0 = __uint_as_float(d[q * 8 + 2 * i]), d1 = __uint_as_float(d[q * 8 + 2 * i + 1]);
        const float s0 = fast_sigmoid(g0), s1 = fast_sigmoid(g1);
        og[i] = pack_bf16(d0 * u0 * s0 * (1.0f + g0 * (1.0f - s0)), d1 * u1 * s1 * (1.0f + g1 * (1.0f - s1)));
        ou[i] = pack_bf16(d0 * g0 * s0, d1 * g1 * s1);
      }
      *reinterpret_cast<uint4*>(dgdst + q * 8) = make_uint4(og[0], og[1], og[2], og[3]);
      *reinterpret_cast<uint4*>(dgdst + p.F + q * 8) = make_uint4(ou[0], ou[1], ou[2], ou[3]);
    }
  }
}

// TC_DGRAD_SWIGLU chunk with F % 32 == 0: g, u of the chunk (two 32-column x 128-row boxes) were fetched by TMA into the
// warp group's two 64-byte-swizzled 8 KB boxes; every thread turns its own row into dg, du IN PLACE and the same boxes
// leave by TMA store.  No per-thread global loads or stores at all.
__device__ __forceinline__ void dgrad_swiglu_chunk_tma(const TcParams& p, const Tile& tl, int c, uint32_t tacc, uint32_t obuf,
                                                       int row_in_tile, uint32_t gbar, uint32_t& gphase,
                                                       const CUtensorMap* tmO, bool issuer, int ch) {
  uint32_t d[32];
  tmem_ld32(tacc + c * 32, d);
  mbar_wait(gbar, gphase);           // g, u of this chunk have landed
  gphase ^= 1;
  tmem_ld_wait();
  const uint32_t rowaddr = obuf + row_in_tile * 64;
  const int sw = (row_in_tile >> 1) & 3;
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    const uint32_t ga = rowaddr + ((q ^ sw) << 4), ua = ga + OBUF_BYTES / 2;
    const uint4 gq = ld_shared_v4(ga), uq = ld_shared_v4(ua);
    const uint32_t gw[4] = {gq.x, gq.y, gq.z, gq.w}, uw[4] = {uq.x, uq.y, uq.z, uq.w};
    uint32_t og[4], ou[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const float g0 = bf16_lo(gw[i]), g1 = bf16_hi(gw[i]), u0 = bf16_lo(uw[i]), u1 = bf16_hi(uw[i]);
      const float d0 = __uint_as_float(d[q * 8 + 2 * i]), d1 = __uint_as_float(d[q * 8 + 2 * i + 1]);
      const float s0 = fast_sigmoid(g0), s1 = fast_sigmoid(g1);
      og[i] = pack_bf16(d0 * u0 * s0 * (1.0f + g0 * (1.0f - s0)), d1 * u1 * s1 * (1.0f + g1 * (1.0f - s1)));
      ou[i] = pack_bf16(d0 * g0 * s0, d1 * g1 * s1);
    }
    st_shared_v4(ga, og[0], og[1], og[2], og[3]);
    st_shared_v4(ua, ou[0], ou[1], ou[2], ou[3]);
  }
  fence_proxy_async();
  named_bar_sync(1 + ch, 128);
  if (issuer) {
    tma_store_3d(tmO, obuf, tl.n0 + c * 32, tl.m0, 0);
    tma_store_3d(tmO, obuf + OBUF_BYTES / 2, p.F + tl.n0 + c * 32, tl.m0, 0);
    bulk_commit();
  }
}

// issuer thread of a warp group: once the group's previous stores have read the boxes, fetch g, u of chunk c into them
__device__ __forceinline__ void gu_tma_fetch(const TcParams& p, const Tile& tl, int c, uint32_t obuf, uint32_t gbar,
                                             const CUtensorMap* tmGU) {
  bulk_wait_read0();
  mbar_expect_tx(gbar, OBUF_BYTES);
  tma_load_3d(obuf, tmGU, gbar, tl.n0 + c * 32, tl.m0, 0);
  tma_load_3d(obuf + OBUF_BYTES / 2, tmGU, gbar, p.F + tl.n0 + c * 32, tl.m0, 0);
}

// TC_WGRAD epilogue.  An expert's contraction is short (its row count), so the weight-gradient tiles are bound by
// how fast 128 x 256 bf16 outputs leave the SM: each 64-column chunk is packed into a 128-byte-swizzled shared-memory
// box (thread = row, conflict-free 16-byte stores) and written with one TMA store (full 128-byte lines; rows past M
// and columns past N are clipped by the 3-D tensor map [E, M, N]).  The two column-parity warp groups own one box each
// and alternate, so one group's TMA store overlaps the other group's TMEM drain.
__device__ __forceinline__ void wgrad_store_tile(const TcParams& p, const Tile& tl, uint32_t tacc, int row_in_tile,
                                                 bool have_acc, uint32_t obuf, const CUtensorMap* tmO, bool issuer,
                                                 int ch, int ecoord) {
#pragma unroll 1
  for (int c = ch; c < BN / 64; c += 2) {
    const int ncols = p.N - (tl.n0 + c * 64);   // warp-uniform
    if (ncols <= 0) break;
    uint32_t v0[32], v1[32];
    if (have_acc) {
      tmem_ld32(tacc + c * 64, v0);
      tmem_ld32(tacc + c * 64 + 32, v1);
      tmem_ld_wait();
    } else {
#pragma unroll
      for (int i = 0; i < 32; ++i) v0[i] = v1[i] = 0u;   // empty expert: exact zeros
    }
    if (issuer) bulk_wait_read0();     // this group's previous TMA store has finished reading the box
    named_bar_sync(1 + ch, 128);
    const uint32_t rowaddr = obuf + row_in_tile * 128;
    const int sw = row_in_tile & 7;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      st_shared_v4(rowaddr + ((j ^ sw) << 4), pack_bf16(__uint_as_float(v0[j * 8 + 0]), __uint_as_float(v0[j * 8 + 1])),
                   pack_bf16(__uint_as_float(v0[j * 8 + 2]), __uint_as_float(v0[j * 8 + 3])),
                   pack_bf16(__uint_as_float(v0[j * 8 + 4]), __uint_as_float(v0[j * 8 + 5])),
                   pack_bf16(__uint_as_float(v0[j * 8 + 6]), __uint_as_float(v0[j * 8 + 7])));
      st_shared_v4(rowaddr + (((j + 4) ^ sw) << 4), pack_bf16(__uint_as_float(v1[j * 8 + 0]), __uint_as_float(v1[j * 8 + 1])),
                   pack_bf16(__uint_as_float(v1[j * 8 + 2]), __uint_as_float(v1[j * 8 + 3])),
                   pack_bf16(__uint_as_float(v1[j * 8 + 4]), __uint_as_float(v1[j * 8 + 5])),
                   pack_bf16(__uint_as_float(v1[j * 8 + 6]), __uint_as_float(v1[j * 8 + 7])));
    }
    fence_proxy_async();
    named_bar_sync(1 + ch, 128);
    if (issuer) {
      tma_store_3d(tmO, obuf, tl.n0 + c * 64, tl.m0, ecoord);
      bulk_commit();
    }
  }
}

// TC_WGRAD with fp32 accumulation into an existing gradient (dB += tile; PAPER.md:116 wgrad delay keeps fp32 main
// gradients across micro-batches): 32-column fp32 chunks (128-byte rows) staged like above and added by a TMA
// reduce-add store, so the old gradient is never read by the SM.  An empty expert adds nothing.
__device__ __forceinline__ void wgrad_accum_tile(const TcParams& p, const Tile& tl, uint32_t tacc, int row_in_tile,
                                                 uint32_t obuf, const CUtensorMap* tmO, bool issuer, int ch) {
#pragma unroll 1
  for (int c = ch; c < BN / 32; c += 2) {
    const int ncols = p.N - (tl.n0 + c * 32);   // warp-uniform
    if (ncols <= 0) break;
    uint32_t v[32];
    tmem_ld32(tacc + c * 32, v);
    tmem_ld_wait();
    if (issuer) bulk_wait_read0();
    named_bar_sync(1 + ch, 128);
    const uint32_t rowaddr = obuf + row_in_tile * 128;
    const int sw = row_in_tile & 7;
#pragma unroll
    for (int j = 0; j < 8; ++j) st_shared_v4(rowaddr + ((j ^ sw) << 4), v[j * 4], v[j * 4 + 1], v[j * 4 + 2], v[j * 4 + 3]);
    fence_proxy_async();
    named_bar_sync(1 + ch, 128);
    if (issuer) {
      tma_reduce_add_3d(tmO, obuf, tl.n0 + c * 32, tl.m0, tl.e);
      bulk_commit();
    }
  }
}

// ---------------------------------------------------------------------------------------------
// the kernel
// ---------------------------------------------------------------------------------------------
template <int MODE>
__global__ void __launch_bounds__(NTHREADS, 1)
tc_gemm_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB0,
               const __grid_constant__ CUtensorMap tmB1, const __grid_constant__ CUtensorMap tmO,
               const __grid_constant__ CUtensorMap tmO2, const TcParams p) {
  constexpr bool A_MN = (MODE == TC_WGRAD);
  constexpr bool B_MN = (MODE == TC_DGRAD || MODE == TC_DGRAD_SWIGLU || MODE == TC_WGRAD);
  extern __shared__ uint8_t smem_raw[];
  const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;   // 128-byte swizzle wants 1024-byte alignment
  const uint32_t obuf0 = base + STAGES * STAGE_BYTES;
  const uint32_t bars = obuf0 + 2 * OBUF_BYTES;
  // barrier addresses: full[s] = bars + 8 s; empty[s] = bars + 8 (STAGES + s); tfull[a] / tempty[a] follow
  const uint32_t full0 = bars, empty0 = bars + 8 * STAGES, tfull0 = bars + 16 * STAGES, tempty0 = tfull0 + 16;
  const uint32_t tmem_slot = tempty0 + 16;
  const uint32_t gbar0 = tempty0 + 24;   // two barriers: g, u boxes of the dgrad-down epilogue groups
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmA);
    tma_prefetch_desc(&tmB0);
    tma_prefetch_desc(&tmB1);
    tma_prefetch_desc(&tmO);
    tma_prefetch_desc(&tmO2);
    for (int s = 0; s < STAGES; ++s) {
      mbar_init(full0 + 8 * s, 1);
      mbar_init(empty0 + 8 * s, 1);
    }
    for (int a = 0; a < 2; ++a) {
      mbar_init(tfull0 + 8 * a, 1);
      mbar_init(tempty0 + 8 * a, EPI_WARPS);   // one arrive per epilogue warp
      mbar_init(gbar0 + 8 * a, 1);
    }
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc(tmem_slot, TMEM_COLS);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

  const int64_t total = total_tiles<MODE>(p);

  if (warp == 0) {
    // ===================== TMA producer (one thread) =====================
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      Tile tl;
      for (int64_t t = blockIdx.x; decode_tile<MODE>(p, t, total, tl); t += gridDim.x) {
        for (int kb = 0; kb < tl.nkb; ++kb) {
          mbar_wait(empty0 + 8 * stage, phase ^ 1);
          const uint32_t fb = full0 + 8 * stage;
          const uint32_t sa = base + stage * STAGE_BYTES, sb = sa + A_BYTES;
          mbar_expect_tx(fb, STAGE_BYTES);
          if (!A_MN) {
            tma_load_2d(sa, &tmA, fb, kb * BK, tl.m0);                              // box 64 x 128
          } else {
            const int kr = tl.row0 + kb * BK;
#pragma unroll
            for (int i = 0; i < BM / 64; ++i) tma_load_2d(sa + i * MN_BOX_BYTES, &tmA, fb, p.a_col0 + tl.m0 + 64 * i, kr);
          }
          if (MODE == TC_FWD || MODE == TC_FWD_F32) {
            tma_load_2d(sb, &tmB0, fb, kb * BK, tl.e * p.b_rows + tl.n0);            // box 64 x 256
          } else if (MODE == TC_FWD_SWIGLU) {
            tma_load_2d(sb, &tmB0, fb, kb * BK, tl.e * p.b_rows + tl.n0);            // box 64 x 128 (Wg)
            tma_load_2d(sb + B_BYTES / 2, &tmB1, fb, kb * BK, tl.e * p.b_rows + tl.n0);  // (Wu)
          } else if (MODE == TC_WGRAD) {
            const int kr = tl.row0 + kb * BK;
#pragma unroll
            for (int i = 0; i < BN / 64; ++i) tma_load_2d(sb + i * MN_BOX_BYTES, &tmB0, fb, tl.n0 + 64 * i, kr);
          } else {
            const bool second = kb >= p.kb_split;
            const CUtensorMap* bm = second ? &tmB1 : &tmB0;
            const int kr = tl.e * p.b_rows + (second ? kb - p.kb_split : kb) * BK;
#pragma unroll
            for (int i = 0; i < BN / 64; ++i) tma_load_2d(sb + i * MN_BOX_BYTES, bm, fb, tl.n0 + 64 * i, kr);
          }
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer (one thread) =====================
    if (lane == 0) {
      constexpr uint32_t idesc = instr_desc(1, A_MN ? 1 : 0, B_MN ? 1 : 0, BN);
      int stage = 0, as = 0;
      uint32_t phase = 0, aphase = 0;
      Tile tl;
      for (int64_t t = blockIdx.x; decode_tile<MODE>(p, t, total, tl); t += gridDim.x) {
        if (tl.nkb == 0) continue;
        mbar_wait(tempty0 + 8 * as, aphase ^ 1);
        tc_fence_after();
        const uint32_t dacc = tmem_base + as * BN;
        for (int kb = 0; kb < tl.nkb; ++kb) {
          mbar_wait(full0 + 8 * stage, phase);
          tc_fence_after();
          const uint32_t sa = base + stage * STAGE_BYTES, sb = sa + A_BYTES;
#pragma unroll
          for (int k = 0; k < BK / UK; ++k) {
            const uint64_t ad = A_MN ? smem_desc(sa + k * UK * 128, MN_BOX_BYTES, 1024) : smem_desc(sa + k * UK * 2, 16, 1024);
            const uint64_t bd = B_MN ? smem_desc(sb + k * UK * 128, MN_BOX_BYTES, 1024) : smem_desc(sb + k * UK * 2, 16, 1024);
            umma_bf16(dacc, ad, bd, idesc, (kb | k) != 0);
          }
          umma_commit(empty0 + 8 * stage);   // frees the smem stage once these MMAs have read it
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
        umma_commit(tfull0 + 8 * as);        // accumulator complete
        if (++as == 2) { as = 0; aphase ^= 1; }
      }
    }
  } else {
    // ===================== epilogue warps 2..5 =====================
    const int lg = warp & 3;                 // TMEM lane group this warp may access
    const int ch = (warp - 2) >> 2;          // which half of the column chunks this warp drains
    const int row_in_tile = lg * 32 + lane;
    int as = 0;
    uint32_t aphase = 0, gphase = 0;
    Tile tl;
    for (int64_t t = blockIdx.x; decode_tile<MODE>(p, t, total, tl); t += gridDim.x) {
      const bool have = tl.nkb > 0;
      const uint32_t tacc = tmem_base + ((uint32_t)(lg * 32) << 16) + as * BN;
      if (MODE == TC_DGRAD_SWIGLU) {
        const int64_t row = (int64_t)tl.m0 + row_in_tile;
        const bool row_ok = row < p.rows_valid;
        {   // pull the NEXT tile's g, u rows into L2 a whole tile ahead (ch 0 warps take g, ch 1 warps take u)
          Tile nx;
          if (decode_tile<MODE>(p, t + gridDim.x, total, nx)) {
            const int64_t nrow = (int64_t)nx.m0 + row_in_tile;
            if (nrow < p.rows_valid) {
              const __nv_bfloat16* src = p.gu + nrow * p.ldgu + (ch ? p.F : 0) + nx.n0;
              const int ncol = min(BN, p.F - nx.n0);
              for (int c = 0; c < ncol; c += 64) asm volatile("prefetch.global.L2 [%0];" ::"l"(src + c));
            }
          }
        }
        constexpr int NC = BN / 64;              // chunks per warp: this warp drains columns [ch * 128, ch * 128 + 128)
        if (p.tma_out) {
          const bool issuer = (threadIdx.x & 127) == 64;
          const uint32_t obuf = obuf0 + ch * OBUF_BYTES, gbar = gbar0 + 8 * ch;
          const int nvalid = min(NC, (p.F - tl.n0 - ch * (BN / 2) + 31) / 32);      // chunks of this group inside F
          if (issuer && nvalid > 0) gu_tma_fetch(p, tl, ch * NC, obuf, gbar, &tmB1);   // overlaps the rest of the main loop
          __syncwarp();
          mbar_wait(tfull0 + 8 * as, aphase);
          tc_fence_after();
          for (int i = 0; i < nvalid; ++i) {
            dgrad_swiglu_chunk_tma(p, tl, ch * NC + i, tacc, obuf, row_in_tile, gbar, gphase, &tmO, issuer, ch);
            if (issuer && i + 1 < nvalid) gu_tma_fetch(p, tl, ch * NC + i + 1, obuf, gbar, &tmB1);
            __syncwarp();
          }
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(tempty0 + 8 * as);
          if (++as == 2) { as = 0; aphase ^= 1; }
          continue;
        }
        GuChunk k[3];
        gu_load(p, tl, row, row_ok, ch * NC, k[0]);
        gu_load(p, tl, row, row_ok, ch * NC + 1, k[1]);
        mbar_wait(tfull0 + 8 * as, aphase);
        tc_fence_after();
#pragma unroll
        for (int i = 0; i < NC; ++i) {
          if (i + 2 < NC) gu_load(p, tl, row, row_ok, ch * NC + i + 2, k[(i + 2) % 3]);
          dgrad_swiglu_chunk(p, tl, row, row_ok, ch * NC + i, tacc, k[i % 3], obuf0 + ch * OBUF_BYTES, row_in_tile, &tmO,
                             (threadIdx.x & 127) == 64, ch);
        }
      } else if (MODE == TC_WGRAD || MODE == TC_FWD || MODE == TC_DGRAD) {
        if (have) {
          mbar_wait(tfull0 + 8 * as, aphase);
          tc_fence_after();
        }
        if (MODE == TC_WGRAD && p.acc_f32) {
          if (have) wgrad_accum_tile(p, tl, tacc, row_in_tile, obuf0 + ch * OBUF_BYTES, &tmO, (threadIdx.x & 127) == 64, ch);
        } else {
          wgrad_store_tile(p, tl, tacc, row_in_tile, have, obuf0 + ch * OBUF_BYTES, &tmO, (threadIdx.x & 127) == 64, ch,
                           MODE == TC_WGRAD ? tl.e : 0);
        }
      } else if (MODE == TC_FWD_SWIGLU && p.tma_out) {
        mbar_wait(tfull0 + 8 * as, aphase);
        tc_fence_after();
        fwd_swiglu_tile_tma(p, tl, tacc, row_in_tile, obuf0 + ch * OBUF_BYTES, &tmO, &tmO2, (threadIdx.x & 127) == 64, ch);
      } else {
        if (have) {
          mbar_wait(tfull0 + 8 * as, aphase);
          tc_fence_after();
        }
        epilogue_tile<MODE>(p, tl, tacc, row_in_tile, have, ch);
      }
      if (have) {
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(tempty0 + 8 * as);
        if (++as == 2) { as = 0; aphase ^= 1; }
      }
    }
    if ((MODE == TC_WGRAD || MODE == TC_FWD || MODE == TC_DGRAD || MODE == TC_DGRAD_SWIGLU || MODE == TC_FWD_SWIGLU) &&
        (threadIdx.x & 127) == 64)
      bulk_wait0();   // all TMA stores complete before the CTA retires
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem_base, TMEM_COLS);
}

// ---------------------------------------------------------------------------------------------
// host: tensor maps and launch
// ---------------------------------------------------------------------------------------------
// 2-D bf16 tensor [outer, inner] (inner contiguous, row pitch ld elements), box = box_outer x 64, 128-byte swizzle,
// out-of-bounds elements read as zero.
bool make_map(CUtensorMap* m, const void* ptr, int64_t inner, int64_t outer, int64_t ld, int box_outer) {
  return tc_make_map(m, 2, ptr, inner, outer, ld, BK, box_outer);
}

bool g_attr_set[MAX_DEVICES][6];   // per device: cudaFuncAttributeMaxDynamicSharedMemorySize raised for tc_gemm_kernel<MODE>

template <int MODE>
int32_t launch(const CUtensorMap& a, const CUtensorMap& b0, const CUtensorMap& b1, const CUtensorMap& o, const TcParams& p,
               int64_t max_tiles, cudaStream_t s, const CUtensorMap* o2 = nullptr) {
  const int dev = current_device();
  if (dev < 0) return MOE_ERR_CUDA;
  if (!g_attr_set[dev][MODE]) {
    MOE_CUDA(cudaFuncSetAttribute(tc_gemm_kernel<MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES));
    g_attr_set[dev][MODE] = true;
  }
  const int sms = device_sm_count();
  if (sms <= 0) return MOE_ERR_CUDA;
  const unsigned grid = (unsigned)std::max<int64_t>(1, std::min<int64_t>(sms, max_tiles));
  MOE_LAUNCH(tc_gemm_kernel<MODE>, grid, NTHREADS, SMEM_BYTES, s, a, b0, b1, o, o2 ? *o2 : o, p);
  return MOE_OK;
}

// mtile[0] = number of 128-row tiles below offsets[E]; mtile[1 + i] = expert owning tile i.
__global__ void prepare_tiles_kernel(const int32_t* __restrict__ offsets, int E, int32_t* __restrict__ mtile) {
  for (int e = threadIdx.x; e < E; e += blockDim.x) {
    const int lo = offsets[e] / BM, hi = offsets[e + 1] / BM;
    for (int t = lo; t < hi; ++t) mtile[1 + t] = e;
  }
  if (threadIdx.x == 0) mtile[0] = offsets[E] / BM;
}

}  // namespace

int32_t tc_prepare_tiles(const int32_t* offsets, int E, int64_t rows_cap, int32_t* mtile_expert, cudaStream_t s) {
  (void)rows_cap;
  MOE_LAUNCH(prepare_tiles_kernel, 1, 256, 0, s, offsets, E, mtile_expert);
  return MOE_OK;
}

int32_t tc_gemm(const TcCall& c, cudaStream_t s) {
  if (c.mtile == nullptr && c.E != 1) return MOE_ERR_UNSUPPORTED;
  TcParams p;
  memset(&p, 0, sizeof(p));
  p.E = c.E;
  p.rows_valid = c.rows_cap;
  p.mtile = c.mtile;
  p.offsets = c.offsets;
  p.out0 = (__nv_bfloat16*)c.out0;
  p.ld0 = c.ld0;
  p.out1 = (__nv_bfloat16*)c.out1;
  p.ld1 = c.ld1;
  p.gu = (const __nv_bfloat16*)c.gu;
  p.ldgu = c.ldgu;
  p.F = c.F;
  p.N = c.N;
  p.M = c.M;
  p.b_rows = c.b_rows;
  p.a_col0 = c.a_col0;
  CUtensorMap ta, tb0, tb1, to;
  const int64_t max_mtiles = ceil_div(c.rows_cap, BM);
  if (c.mode == TC_FWD_F32 ? ((c.N & 3) || (c.ld0 & 3)) : ((c.N & 7) || (c.ld0 & 7))) return MOE_ERR_UNSUPPORTED;
  switch (c.mode) {
    case TC_FWD_F32:
    case TC_FWD: {
      if (c.Kd % BK) return MOE_ERR_UNSUPPORTED;
      p.nkb = c.Kd / BK;
      p.n_tiles = (int)ceil_div(c.N, BN);
      if (!make_map(&ta, c.A, c.Kd, c.rows_cap, c.lda, BM)) return MOE_ERR_UNSUPPORTED;
      if (!make_map(&tb0, c.B0, c.b_cols, (int64_t)c.E * c.b_rows, c.b_cols, BN)) return MOE_ERR_UNSUPPORTED;
      if (c.mode == TC_FWD_F32) return launch<TC_FWD_F32>(ta, tb0, tb0, ta, p, max_mtiles * p.n_tiles, s);
      if (!tc_make_map3(&to, 2, c.out0, c.N, c.rows_cap, 1, c.ld0, 64, BM)) return MOE_ERR_UNSUPPORTED;   // C [rows, N]
      return launch<TC_FWD>(ta, tb0, tb0, to, p, max_mtiles * p.n_tiles, s);
    }
    case TC_FWD_SWIGLU: {
      if (c.Kd % BK || (c.F & 7) || (c.ld1 & 7)) return MOE_ERR_UNSUPPORTED;
      p.nkb = c.Kd / BK;
      p.n_tiles = (int)ceil_div(c.F, BN / 2);
      if (!make_map(&ta, c.A, c.Kd, c.rows_cap, c.lda, BM)) return MOE_ERR_UNSUPPORTED;
      if (!make_map(&tb0, c.B0, c.b_cols, (int64_t)c.E * c.b_rows, c.b_cols, BN / 2)) return MOE_ERR_UNSUPPORTED;
      if (!make_map(&tb1, c.B1, c.b_cols, (int64_t)c.E * c.b_rows, c.b_cols, BN / 2)) return MOE_ERR_UNSUPPORTED;
      p.tma_out = (c.F % 32 == 0) ? 1 : 0;   // g / u boxes of 32 columns must not straddle the [g|u] boundary
      CUtensorMap to2;
      if (p.tma_out && (!tc_make_map3(&to, 2, c.out0, 2 * (int64_t)c.F, c.rows_cap, 1, c.ld0, 32, BM) ||    // gu [rows, 2F]
                        !tc_make_map3(&to2, 2, c.out1, c.F, c.rows_cap, 1, c.ld1, 32, BM)))                  // a [rows, F]
        p.tma_out = 0;
      if (!p.tma_out) return launch<TC_FWD_SWIGLU>(ta, tb0, tb1, ta, p, max_mtiles * p.n_tiles, s);
      return launch<TC_FWD_SWIGLU>(ta, tb0, tb1, to, p, max_mtiles * p.n_tiles, s, &to2);
    }
    case TC_DGRAD:
    case TC_DGRAD_SWIGLU: {
      // contraction over the weights' rows (b_rows per source), output columns = b_cols
      if (c.b_rows % BK) return MOE_ERR_UNSUPPORTED;
      const bool split = c.B1 != nullptr;
      p.kb_split = c.b_rows / BK;
      p.nkb = split ? 2 * p.kb_split : p.kb_split;
      p.n_tiles = (int)ceil_div(c.N, BN);
      if (!make_map(&ta, c.A, (int64_t)p.nkb * BK, c.rows_cap, c.lda, BM)) return MOE_ERR_UNSUPPORTED;
      if (!make_map(&tb0, c.B0, c.b_cols, (int64_t)c.E * c.b_rows, c.b_cols, 64)) return MOE_ERR_UNSUPPORTED;
      if (!make_map(&tb1, split ? c.B1 : c.B0, c.b_cols, (int64_t)c.E * c.b_rows, c.b_cols, 64)) return MOE_ERR_UNSUPPORTED;
      if (c.mode == TC_DGRAD) {
        if (!tc_make_map3(&to, 2, c.out0, c.N, c.rows_cap, 1, c.ld0, 64, BM)) return MOE_ERR_UNSUPPORTED;   // dA [rows, N]
        return launch<TC_DGRAD>(ta, tb0, tb1, to, p, max_mtiles * p.n_tiles, s);
      }
      if ((c.F & 7) || (c.ldgu & 7)) return MOE_ERR_UNSUPPORTED;
      p.tma_out = (c.F % 32 == 0) ? 1 : 0;   // dg / du boxes of 32 columns must not straddle the [dg|du] boundary
      if (p.tma_out && !split &&                                                          // saved [g|u] rows, same boxes
          !tc_make_map3(&tb1, 2, c.gu, 2 * (int64_t)c.F, c.rows_cap, 1, c.ldgu, 32, BM))
        p.tma_out = 0;
      if (!tc_make_map3(&to, 2, c.out0, 2 * (int64_t)c.F, c.rows_cap, 1, c.ld0, 32, BM)) return MOE_ERR_UNSUPPORTED;   // dgu [rows, 2F]
      return launch<TC_DGRAD_SWIGLU>(ta, tb0, tb1, to, p, max_mtiles * p.n_tiles, s);
    }
    case TC_WGRAD: {
      p.m_tiles = (int)ceil_div(c.M, BM);
      p.n_tiles = (int)ceil_div(c.N, BN);
      // A: [rows_cap, lda] read MN-major (inner = columns = output rows); A2 likewise (inner = output columns)
      if (!make_map(&ta, c.A, c.lda, c.rows_cap, c.lda, 64)) return MOE_ERR_UNSUPPORTED;
      if (!make_map(&tb0, c.A2, c.N, c.rows_cap, c.lda2, 64)) return MOE_ERR_UNSUPPORTED;
      p.acc_f32 = c.acc_f32 ? 1 : 0;
      if (c.acc_f32 ? !tc_make_map3(&to, 4, c.out0, c.N, c.M, c.E, c.ld0, 32, BM)    // fp32 dB [E, M, N], reduce-add
                    : !tc_make_map3(&to, 2, c.out0, c.N, c.M, c.E, c.ld0, 64, BM))   // bf16 dB [E, M, N], overwrite
        return MOE_ERR_UNSUPPORTED;
      return launch<TC_WGRAD>(ta, tb0, tb0, to, p, (int64_t)c.E * p.m_tiles * p.n_tiles, s);
    }
  }
  return MOE_ERR_INVALID_ARG;
}

}  // namespace moe
