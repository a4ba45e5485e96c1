// tcgen05 / TMEM / TMA grouped GEMMs for sm_100a (bf16 in, fp32 accumulate in tensor memory, bf16 out).
//
// One persistent, warp-specialised kernel template serves every expert GEMM of the layer (SURVEY.md §8a
// a5, a6, a9..a12): warp 0 = TMA producer, warp 1 = MMA issuer (one elected thread, tcgen05.mma
// cta_group::1, M=128 x N=256 x K=16 per instruction), warps 2..9 = epilogue (EPI_WARPS = 8, two per TMEM lane group,
// each taking every other 64-column chunk; tcgen05.ld from a double-buffered 2 x 256-column TMEM accumulator).  Operands are staged by TMA into 128-byte-swizzled
// shared memory, 4 stages of (128 x 64 A tile + 256 x 64 B tile) = 192 KB.  The tile schedule is
// computed on the device from the per-expert row offsets (shapes are data dependent; the
// counts never visit the host): a 128-row M-tile belongs to exactly one expert because expert groups
// start at multiples of 128 rows.  SwiGLU forward / backward are fused into the epilogues.
// Both K-major and MN-major shared-memory operand layouts are used, so the dgrad (weights read
// "transposed") and wgrad (both operands contracted over rows) need no transposed copies in HBM.
#include <cuda.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>

#include "gemm_tc.cuh"
#include "tc_ptx.cuh"
#include "tile_tables.cuh"

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
constexpr int A_BYTES = BM * BK * 2;   // 16 KB: this CTA's 128 rows of the left operand
constexpr int B_BYTES = BN * BK * 2;   // 32 KB: all 256 columns of the right operand (a CTA of a pair holds half)
// Per-CTA operand ring.  1-CTA kernel: 4 stages of (A 16 KB + B 32 KB).  CTA-pair kernel (cta_group::2, M = 256): each
// CTA stages its own 128 A rows and HALF of B (the pair's tensor cores read both halves), 5 stages of 32 KB, so a
// k-block costs each SM 32 KB of L2 -> SM traffic instead of 48 KB for the same 128 x 256 x 64 MACs; the 32 KB this
// saves hold a second staging box per epilogue warp group (NOBUF), so a group fills one box while the TMA store of
// its other box is still reading shared memory.
// SHORT (1-CTA weight gradients): an expert's contraction is a handful of k-blocks and every tile ends with 64 KB of output,
// so a stage of the ring is traded for a second staging box per warp group (3 stages, NOBUF 2).
template <bool PAIR, bool SHORT = false> struct Ring {
  static constexpr int STAGES = PAIR ? 5 : (SHORT ? 3 : 4);
  static constexpr int B_CTA = PAIR ? B_BYTES / 2 : B_BYTES;
  static constexpr int STAGE_BYTES = A_BYTES + B_CTA;
  static constexpr int NOBUF = (PAIR || SHORT) ? 2 : 1;   // staging boxes per epilogue warp group
};
constexpr int MAX_STAGES = 6;
constexpr int MN_BOX_BYTES = 64 * BK * 2;  // one 64(MN) x 64(K) box of an MN-major operand: 8 KB
constexpr int OBUF_BYTES = BM * 128;       // epilogue staging: 128 rows x 64 bf16 columns (one 128-byte-swizzled TMA box)
constexpr int SMEM_BYTES = Ring<false>::STAGES * Ring<false>::STAGE_BYTES + 2 * OBUF_BYTES + 1024 /*align*/ + 256 /*barriers*/;
static_assert(Ring<false, true>::STAGES * Ring<false, true>::STAGE_BYTES + 2 * Ring<false, true>::NOBUF * OBUF_BYTES <=
              Ring<false>::STAGES * Ring<false>::STAGE_BYTES + 2 * Ring<false>::NOBUF * OBUF_BYTES, "fits the same allocation");
static_assert(Ring<true>::STAGES * Ring<true>::STAGE_BYTES + 2 * Ring<true>::NOBUF * OBUF_BYTES ==
              Ring<false>::STAGES * Ring<false>::STAGE_BYTES + 2 * Ring<false>::NOBUF * OBUF_BYTES, "same shared-memory footprint");
constexpr int EPI_WARPS = 8;            // two per TMEM lane group: column-chunk parity `ch` splits a tile between them
constexpr int NTHREADS = 64 + EPI_WARPS * 32;
constexpr int TMEM_COLS = 512;

// ---------------------------------------------------------------------------------------------
// kernel parameters
// ---------------------------------------------------------------------------------------------
struct TcParams {
  int E, n_tiles, m_tiles, nkb, kb_split, b_rows, N, M, F, a_col0, tma_out, acc_f32, short_ring;
  int64_t rows_valid;
  const int32_t* mtile;    // M-tile -> expert (nullptr: one group of rows_valid rows)
  const int32_t* tlist;    // which M-tiles this launch runs: pair kernel = plist, 1-CTA kernel = olist or nullptr (all)
  const int32_t* offsets;
  const int32_t* counts;   // WGRAD: real rows per expert (nullptr: contract over the whole 128-aligned group)
  __nv_bfloat16* out0;
  int64_t ld0;
  __nv_bfloat16* out1;
  int64_t ld1;
  const __nv_bfloat16* gu;
  int64_t ldgu;
  // fused permutation ("fused token scatter"; north_star: routing weights in the epilogues)
  const int32_t* gidx;     // perm_to_flat [rows]: flat position t*K+j of a permuted row, -1 = padding row; nullptr = off
  int gat;                 // 1: the K-major A operand is GATHERED through gidx from token-major rows (gather-warp kernels)
  int copy_out;            // gathered A tiles are also stored to the row-grouped copy behind tmC (Xp / dy), each k-block once
  int gshift, gK;          // flat position -> token row: p >> gshift (K a power of two) or p / gK (gshift < 0)
  const float* roww;       // routing weights by flat position [T*K] (nullptr = 1): FWD_SWIGLU a *= w; DGRAD_SWIGLU dgu *= w
  float* dwpart;           // DGRAD_SWIGLU: [2 * n_tiles, rows_valid] partial sums of <da, silu(g) u> per row (nullptr = off)
};

struct Tile {
  int e, m0, n0, nkb, row0;
};

// Tile t of this launch for the CTA of pair-rank `rank` (0 in the 1-CTA kernel).  A pair works on two consecutive
// M-tiles of one expert (rows m0 = first tile + 128 rank) and the same 256 output columns.
template <int MODE, bool PAIR>
__device__ __forceinline__ bool decode_tile(const TcParams& p, int64_t t, int64_t total, int rank, Tile& tl) {
  if (t >= total) return false;
  if (MODE == TC_WGRAD) {
    const int per_e = p.m_tiles * p.n_tiles;
    tl.e = (int)(t / per_e);
    const int r = (int)(t - (int64_t)tl.e * per_e);
    tl.m0 = (r / p.n_tiles) * (PAIR ? 2 * BM : BM) + rank * BM;
    tl.n0 = (r % p.n_tiles) * BN;
    if (p.mtile) {
      // k-blocks of 64 rows up to the expert's last real row: the 128-row alignment padding (zero rows) is skipped
      tl.row0 = p.offsets[tl.e];
      tl.nkb = p.counts ? (p.counts[tl.e] + BK - 1) / BK : (p.offsets[tl.e + 1] - tl.row0) / BK;
    } else {
      tl.row0 = 0;
      tl.nkb = (int)((p.rows_valid + BK - 1) / BK);
    }
  } else {
    // n fastest: consecutive CTAs / pairs share the activation rows
    const int mi = (int)(t / p.n_tiles);
    tl.n0 = (int)(t - (int64_t)mi * p.n_tiles) * (MODE == TC_FWD_SWIGLU ? BN / 2 : BN);
    const int mt = p.tlist ? p.tlist[1 + mi] : (PAIR ? 2 * mi : mi);
    tl.m0 = (mt + rank) * BM;
    tl.e = p.mtile ? p.mtile[1 + mt] : 0;
    tl.nkb = p.nkb;
    tl.row0 = 0;
  }
  return true;
}

template <int MODE, bool PAIR>
__device__ __forceinline__ int64_t total_tiles(const TcParams& p) {
  if (MODE == TC_WGRAD) return (int64_t)p.E * p.m_tiles * p.n_tiles;
  int64_t mt;
  if (p.tlist) mt = p.tlist[0];
  else if (p.mtile) mt = PAIR ? 0 : p.mtile[0];
  else mt = (p.rows_valid + (PAIR ? 2 * BM : BM) - 1) / (PAIR ? 2 * BM : BM);
  return mt * p.n_tiles;
}

// Token rows of the four permuted rows r .. r+3 (r a multiple of 4): the TMA gather coordinates of one lane.  A padding
// row keeps a negative coordinate, which is out of bounds and therefore reads as zeros.
__device__ __forceinline__ void gather_rows4(const TcParams& p, int64_t r, int (&t)[4]) {
  const int4 v = __ldg(reinterpret_cast<const int4*>(p.gidx + r));
  const int f[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
  for (int i = 0; i < 4; ++i) t[i] = f[i] < 0 ? -1 : (p.gshift >= 0 ? f[i] >> p.gshift : f[i] / p.gK);
}
// routing weight of permuted row r (0 for a padding row); 1 when the launch carries no weights
__device__ __forceinline__ float row_weight(const TcParams& p, int64_t r) {
  if (!p.roww) return 1.0f;
  const int f = r < p.rows_valid ? __ldg(p.gidx + r) : -1;
  return f >= 0 ? __ldg(p.roww + f) : 0.0f;
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
                                                    bool issuer, int ch, float wrow) {
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
      g[i] = __float_as_uint(gv * fast_sigmoid(gv) * __uint_as_float(u[i]) * wrow);   // wrow = 1 unless w is folded into a
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
                                                       const CUtensorMap* tmO, bool issuer, int ch, float wrow, float& dwacc) {
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
      const float a0 = g0 * s0, a1 = g1 * s1;                          // silu(g)
      dwacc = fmaf(d0, a0 * u0, fmaf(d1, a1 * u1, dwacc));             // <da, a>: the routing weight's gradient (R8)
      const float e0 = wrow * d0, e1 = wrow * d1;                      // da of the weighted row (wrow = 1: w not folded)
      og[i] = pack_bf16(e0 * u0 * s0 * (1.0f + g0 * (1.0f - s0)), e1 * u1 * s1 * (1.0f + g1 * (1.0f - s1)));
      ou[i] = pack_bf16(e0 * a0, e1 * a1);
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
// `rel` = what releases the accumulator (called by every thread right after the tile's last TMEM load, before the
// last chunk is staged); `seq` = running chunk counter of this warp group, selecting which of its NB staging boxes
// a chunk uses.
template <int NB, typename Rel>
__device__ __forceinline__ void wgrad_store_tile(const TcParams& p, const Tile& tl, uint32_t tacc, int row_in_tile,
                                                 bool have_acc, uint32_t obuf0g, const CUtensorMap* tmO, bool issuer,
                                                 int ch, int ecoord, uint32_t& seq, Rel rel) {
  const int nch = min(BN / 64, (p.N - tl.n0 + 63) / 64);   // 64-column chunks of this tile inside N (warp-uniform)
#pragma unroll 1
  for (int c = ch; c < nch; c += 2) {
    uint32_t v0[32], v1[32];
    if (have_acc) {
      tmem_ld32(tacc + c * 64, v0);
      tmem_ld32(tacc + c * 64 + 32, v1);
      tmem_ld_wait();
    } else {
#pragma unroll
      for (int i = 0; i < 32; ++i) v0[i] = v1[i] = 0u;   // empty expert: exact zeros
    }
    if (c + 2 >= nch) rel();           // accumulator drained: the next tile's MMAs may overwrite it
    const uint32_t obuf = obuf0g + (NB == 2 ? (seq & 1u) * OBUF_BYTES : 0u);
    ++seq;
    if (issuer) {                      // the TMA store that last used this box has finished reading it
      if (NB == 2) bulk_wait_read1();
      else bulk_wait_read0();
    }
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
  if (ch >= nch) rel();                // this warp group has no chunk in the tile (N tail): still one release per warp
}

// TC_WGRAD with fp32 accumulation into an existing gradient (dB += tile; PAPER.md:116 wgrad delay keeps fp32 main
// gradients across micro-batches): 32-column fp32 chunks (128-byte rows) staged like above and added by a TMA
// reduce-add store, so the old gradient is never read by the SM.  An empty expert adds nothing.
template <int NB, typename Rel>
__device__ __forceinline__ void wgrad_accum_tile(const TcParams& p, const Tile& tl, uint32_t tacc, int row_in_tile,
                                                 uint32_t obuf0g, const CUtensorMap* tmO, bool issuer, int ch, uint32_t& seq,
                                                 Rel rel) {
  const int nch = min(BN / 32, (p.N - tl.n0 + 31) / 32);
#pragma unroll 1
  for (int c = ch; c < nch; c += 2) {
    uint32_t v[32];
    tmem_ld32(tacc + c * 32, v);
    tmem_ld_wait();
    if (c + 2 >= nch) rel();
    const uint32_t obuf = obuf0g + (NB == 2 ? (seq & 1u) * OBUF_BYTES : 0u);
    ++seq;
    if (issuer) {
      if (NB == 2) bulk_wait_read1();
      else bulk_wait_read0();
    }
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
  if (ch >= nch) rel();
}

// ---------------------------------------------------------------------------------------------
// the kernel
// ---------------------------------------------------------------------------------------------
// PAIR = false: one CTA per SM, tcgen05 cta_group::1, 128 x 256 tiles (the unpaired M-tiles, see tile_tables.cuh).
// PAIR = true : launched as clusters of two CTAs (one TPC).  The pair computes a 256 x 256 tile with cta_group::2 MMAs
//   issued by the leader (rank 0): each CTA stages its own 128 rows of A and one half of B; TMA bytes of both CTAs are
//   signalled on the leader's full barrier; tcgen05.commit multicasts "stage free" / "accumulator ready" to both CTAs;
//   each CTA's epilogue warps drain their own 128 TMEM lanes and release the accumulator on the leader's barrier.
template <int MODE, bool PAIR, int GW>
__global__ void __launch_bounds__(NTHREADS + (GW > 0 ? 32 * (GW + 1) : 0), 1)
tc_gemm_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB0,
               const __grid_constant__ CUtensorMap tmB1, const __grid_constant__ CUtensorMap tmO,
               const __grid_constant__ CUtensorMap tmO2, const __grid_constant__ CUtensorMap tmC, const TcParams p) {
  constexpr bool A_MN = (MODE == TC_WGRAD);
  constexpr bool B_MN = (MODE == TC_DGRAD || MODE == TC_DGRAD_SWIGLU || MODE == TC_WGRAD);
  using R = Ring<PAIR>;
  constexpr int STAGE_BYTES = R::STAGE_BYTES, B_CTA = R::B_CTA;
  // the 1-CTA weight-gradient kernel picks its ring at run time (p.short_ring): 3 stages + 2 staging boxes per warp group
  const bool short_ring = MODE == TC_WGRAD && !PAIR && p.short_ring;
  const int STAGES = short_ring ? Ring<false, true>::STAGES : R::STAGES;
  const int NOBUF = short_ring ? Ring<false, true>::NOBUF : R::NOBUF;
  const int GROUP_OBUF = NOBUF * OBUF_BYTES;   // staging bytes of one epilogue warp group
  extern __shared__ uint8_t smem_raw[];
  const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;   // 128-byte swizzle wants 1024-byte alignment
  const uint32_t obuf0 = base + STAGES * STAGE_BYTES;
  const uint32_t bars = obuf0 + 2 * GROUP_OBUF;
  // barrier addresses: full[s] = bars + 8 s; empty[s] = bars + 8 (MAX_STAGES + s); tfull[a] / tempty[a] follow
  const uint32_t full0 = bars, empty0 = bars + 8 * MAX_STAGES, tfull0 = bars + 16 * MAX_STAGES, tempty0 = tfull0 + 16;
  const uint32_t tmem_slot = tempty0 + 16;
  const uint32_t gbar0 = tempty0 + 24;   // two barriers: g, u boxes of the dgrad-down epilogue groups
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int rank = PAIR ? (int)cluster_ctarank() : 0;              // 0 = pair leader (issues the MMAs)
  const int64_t unit = PAIR ? (blockIdx.x >> 1) : blockIdx.x;      // index of this CTA / pair among the launch's workers
  const int64_t nunits = PAIR ? (gridDim.x >> 1) : gridDim.x;

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmA);
    tma_prefetch_desc(&tmB0);
    tma_prefetch_desc(&tmB1);
    tma_prefetch_desc(&tmO);
    tma_prefetch_desc(&tmO2);
    for (int s = 0; s < MAX_STAGES; ++s) {
      mbar_init(full0 + 8 * s, 1);
      mbar_init(empty0 + 8 * s, (GW > 0 && p.copy_out) ? 2 : 1);   // MMA commit (+ the copy-out warp's store has read the stage)
    }
    for (int a = 0; a < 2; ++a) {
      mbar_init(tfull0 + 8 * a, 1);
      mbar_init(tempty0 + 8 * a, PAIR ? 2 * EPI_WARPS : EPI_WARPS);   // one arrive per epilogue warp (of both CTAs)
      mbar_init(gbar0 + 8 * a, 1);
    }
    fence_barrier_init();
  }
  if (warp == 1) {
    if (PAIR) tmem_alloc_pair(tmem_slot, TMEM_COLS);
    else tmem_alloc(tmem_slot, TMEM_COLS);
  }
  tc_fence_before();
  __syncwarp();
  if (PAIR) cluster_sync_all();   // the peer's barriers are initialised before anything is signalled on them
  else __syncthreads();
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

  const int64_t total = total_tiles<MODE, PAIR>(p);

  if (warp == 0) {
    // ===================== TMA producer (one thread per CTA): every operand that is tiled in HBM =====================
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      // the next tile's schedule entry (two dependent global loads) is fetched while this tile's k-loop runs
      Tile tl, nx;
      bool ok = decode_tile<MODE, PAIR>(p, unit, total, rank, tl), okn = false;
      const bool a_tiled = !(GW > 0 && p.gat == 1);   // else: the gather warps' job
      for (int64_t t = unit; ok; t += nunits, tl = nx, ok = okn) {
        okn = decode_tile<MODE, PAIR>(p, t + nunits, total, rank, nx);
        const int bn0 = tl.n0 + (PAIR ? rank * (BN / 2) : 0);   // first of the B columns this CTA stages
        for (int kb = 0; kb < tl.nkb; ++kb) {
          mbar_wait(empty0 + 8 * stage, phase ^ 1);
          const uint32_t sa = base + stage * STAGE_BYTES, sb = sa + A_BYTES;
          uint32_t fb = full0 + 8 * stage;
          if (PAIR) {
            if (rank == 0) mbar_expect_tx(fb, 2 * STAGE_BYTES);   // both CTAs' boxes complete on the leader's barrier
            fb = mapa_shared(fb, 0);
          } else {
            mbar_expect_tx(fb, STAGE_BYTES);
          }
          auto load = [&](uint32_t dst, const CUtensorMap* m, int c0, int c1) {
            if (PAIR) tma_load_2d_pair(dst, m, fb, c0, c1);
            else tma_load_2d(dst, m, fb, c0, c1);
          };
          if (a_tiled) {
            if (!A_MN) {
              load(sa, &tmA, kb * BK, tl.m0);                                        // box 64 x 128
            } else {
              const int kr = tl.row0 + kb * BK;
#pragma unroll
              for (int i = 0; i < BM / 64; ++i) load(sa + i * MN_BOX_BYTES, &tmA, p.a_col0 + tl.m0 + 64 * i, kr);
            }
          }
          if (MODE == TC_FWD || MODE == TC_FWD_F32) {
            load(sb, &tmB0, kb * BK, tl.e * p.b_rows + bn0);                       // box 64 x 256 (pair: 64 x 128)
          } else if (MODE == TC_FWD_SWIGLU) {
            if (PAIR) {                                                             // leader stages Wg, its peer Wu
              load(sb, rank == 0 ? &tmB0 : &tmB1, kb * BK, tl.e * p.b_rows + tl.n0);
            } else {
              load(sb, &tmB0, kb * BK, tl.e * p.b_rows + tl.n0);                   // box 64 x 128 (Wg)
              load(sb + B_BYTES / 2, &tmB1, kb * BK, tl.e * p.b_rows + tl.n0);     // (Wu)
            }
          } else if (MODE == TC_WGRAD) {
            const int kr = tl.row0 + kb * BK;
#pragma unroll
            for (int i = 0; i < B_CTA / MN_BOX_BYTES; ++i) load(sb + i * MN_BOX_BYTES, &tmB0, bn0 + 64 * i, kr);
          } else {
            const bool second = kb >= p.kb_split;
            const CUtensorMap* bm = second ? &tmB1 : &tmB0;
            const int kr = tl.e * p.b_rows + (second ? kb - p.kb_split : kb) * BK;
#pragma unroll
            for (int i = 0; i < B_CTA / MN_BOX_BYTES; ++i) load(sb + i * MN_BOX_BYTES, bm, bn0 + 64 * i, kr);
          }
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer (one thread; in a pair only the leader's) =====================
    if (lane == 0 && rank == 0) {
      constexpr uint32_t idesc = instr_desc(1, A_MN ? 1 : 0, B_MN ? 1 : 0, BN, PAIR ? 2 * BM : BM);
      int stage = 0, as = 0;
      uint32_t phase = 0, aphase = 0;
      Tile tl, nx;
      bool ok = decode_tile<MODE, PAIR>(p, unit, total, rank, tl), okn = false;
      for (int64_t t = unit; ok; t += nunits, tl = nx, ok = okn) {
        okn = decode_tile<MODE, PAIR>(p, t + nunits, total, rank, nx);
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
            if (PAIR) umma_bf16_pair(dacc, ad, bd, idesc, (kb | k) != 0);
            else umma_bf16(dacc, ad, bd, idesc, (kb | k) != 0);
          }
          // frees the smem stage (in both CTAs of a pair) once these MMAs have read it
          if (PAIR) umma_commit_pair(empty0 + 8 * stage);
          else umma_commit(empty0 + 8 * stage);
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
        if (PAIR) umma_commit_pair(tfull0 + 8 * as);   // accumulator complete
        else umma_commit(tfull0 + 8 * as);
        if (++as == 2) { as = 0; aphase ^= 1; }
      }
    }
  } else if (warp < 2 + EPI_WARPS) {
    // ===================== epilogue warps 2..9 =====================
    const int lg = warp & 3;                 // TMEM lane group this warp may access
    const int ch = (warp - 2) >> 2;          // which half of the column chunks this warp drains
    const int row_in_tile = lg * 32 + lane;
    int as = 0;
    uint32_t aphase = 0, gphase = 0, oseq = 0;
    Tile tl;
    // accumulator released: one arrive per epilogue warp, in a pair on the LEADER's barrier (it gates the next MMAs)
    auto release_acc = [&](int a) {
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        if (PAIR) mbar_arrive_cluster(mapa_shared(tempty0 + 8 * a, 0));
        else mbar_arrive(tempty0 + 8 * a);
      }
    };
    Tile nx;
    bool ok = decode_tile<MODE, PAIR>(p, unit, total, rank, tl), okn = false;
    for (int64_t t = unit; ok; t += nunits, tl = nx, ok = okn) {
      okn = decode_tile<MODE, PAIR>(p, t + nunits, total, rank, nx);
      const bool have = tl.nkb > 0;
      const uint32_t tacc = tmem_base + ((uint32_t)(lg * 32) << 16) + as * BN;
      if (MODE == TC_DGRAD_SWIGLU) {
        const int64_t row = (int64_t)tl.m0 + row_in_tile;
        const bool row_ok = row < p.rows_valid;
        constexpr int NC = BN / 64;              // chunks per warp: this warp drains columns [ch * 128, ch * 128 + 128)
        if (GW > 0 || p.tma_out) {
          const bool issuer = (threadIdx.x & 127) == 64;
          const uint32_t obuf = obuf0 + ch * GROUP_OBUF, gbar = gbar0 + 8 * ch;
          const int nvalid = min(NC, (p.F - tl.n0 - ch * (BN / 2) + 31) / 32);      // chunks of this group inside F
          if (issuer && nvalid > 0) gu_tma_fetch(p, tl, ch * NC, obuf, gbar, &tmB1);   // overlaps the rest of the main loop
          __syncwarp();
          const float wrow = row_weight(p, row);
          float dwacc = 0.f;
          mbar_wait(tfull0 + 8 * as, aphase);
          tc_fence_after();
          for (int i = 0; i < nvalid; ++i) {
            dgrad_swiglu_chunk_tma(p, tl, ch * NC + i, tacc, obuf, row_in_tile, gbar, gphase, &tmO, issuer, ch, wrow, dwacc);
            if (issuer && i + 1 < nvalid) gu_tma_fetch(p, tl, ch * NC + i + 1, obuf, gbar, &tmB1);
            __syncwarp();
          }
          release_acc(as);
          // this warp group's share of <da, a> over its 128 columns: part (2 n-tile + ch), summed later in fixed order
          if (p.dwpart && row_ok) p.dwpart[(int64_t)(2 * (tl.n0 / BN) + ch) * p.rows_valid + row] = dwacc;
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
          dgrad_swiglu_chunk(p, tl, row, row_ok, ch * NC + i, tacc, k[i % 3], obuf0 + ch * GROUP_OBUF, row_in_tile, &tmO,
                             (threadIdx.x & 127) == 64, ch);
        }
      } else if (MODE == TC_WGRAD || MODE == TC_FWD || MODE == TC_DGRAD) {
        if (have) {
          mbar_wait(tfull0 + 8 * as, aphase);
          tc_fence_after();
        }
        // the accumulator is released inside, right after its last TMEM load (one arrive per warp)
        auto rel = [&]() { if (have) release_acc(as); };
        if (MODE == TC_WGRAD && p.acc_f32) {
          if (have) {
            if (NOBUF == 2) wgrad_accum_tile<2>(p, tl, tacc, row_in_tile, obuf0 + ch * GROUP_OBUF, &tmO, (threadIdx.x & 127) == 64, ch, oseq, rel);
            else wgrad_accum_tile<1>(p, tl, tacc, row_in_tile, obuf0 + ch * GROUP_OBUF, &tmO, (threadIdx.x & 127) == 64, ch, oseq, rel);
          }
        } else {
          if (NOBUF == 2)
            wgrad_store_tile<2>(p, tl, tacc, row_in_tile, have, obuf0 + ch * GROUP_OBUF, &tmO, (threadIdx.x & 127) == 64, ch,
                                MODE == TC_WGRAD ? tl.e : 0, oseq, rel);
          else
            wgrad_store_tile<1>(p, tl, tacc, row_in_tile, have, obuf0 + ch * GROUP_OBUF, &tmO, (threadIdx.x & 127) == 64, ch,
                                MODE == TC_WGRAD ? tl.e : 0, oseq, rel);
        }
        if (have && ++as == 2) { as = 0; aphase ^= 1; }
        continue;
      } else if (MODE == TC_FWD_SWIGLU && (GW > 0 || p.tma_out)) {
        const float wrow = row_weight(p, (int64_t)tl.m0 + row_in_tile);
        mbar_wait(tfull0 + 8 * as, aphase);
        tc_fence_after();
        fwd_swiglu_tile_tma(p, tl, tacc, row_in_tile, obuf0 + ch * GROUP_OBUF, &tmO, &tmO2, (threadIdx.x & 127) == 64, ch, wrow);
      } else {
        if (have) {
          mbar_wait(tfull0 + 8 * as, aphase);
          tc_fence_after();
        }
        epilogue_tile<MODE>(p, tl, tacc, row_in_tile, have, ch);
      }
      if (have) {
        release_acc(as);
        if (++as == 2) { as = 0; aphase ^= 1; }
      }
    }
    if ((MODE == TC_WGRAD || MODE == TC_FWD || MODE == TC_DGRAD || MODE == TC_DGRAD_SWIGLU || MODE == TC_FWD_SWIGLU) &&
        (threadIdx.x & 127) == 64)
      bulk_wait0();   // all TMA stores complete before the CTA retires
  } else if (GW > 0 && !A_MN && warp < 2 + EPI_WARPS + GW) {
    // ===================== gather warps (GW > 0): the A operand, rows addressed through the permutation map =====================
    // A's 16 KB per k-block (128 permuted rows x 64 columns) is 32 units of one tile::gather4 = four token rows x 128 bytes;
    // the 128-byte swizzle follows the shared-memory address, so the units build the same tile a tiled load would.  A warp
    // issues one gather4 per ~66 cycles whatever its lane count and the TMA unit accepts one per ~14 cycles (measured), so
    // the units are dealt round-robin to GW warps (unit = warp + GW * lane).  Padding rows carry a negative (out-of-bounds)
    // coordinate and read as zeros.
    const int gw = warp - (2 + EPI_WARPS);
    const int u0 = gw + lane * GW;
    if (u0 < 32) {
      int stage = 0;
      uint32_t phase = 0;
      Tile tl, nx;
      bool ok = decode_tile<MODE, PAIR>(p, unit, total, rank, tl), okn = false;
      for (int64_t t = unit; ok; t += nunits, tl = nx, ok = okn) {
        okn = decode_tile<MODE, PAIR>(p, t + nunits, total, rank, nx);
        int gr[4] = {-1, -1, -1, -1};
        if (tl.nkb > 0) gather_rows4(p, tl.m0 + 4 * u0, gr);
        for (int kb = 0; kb < tl.nkb; ++kb) {
          mbar_wait(empty0 + 8 * stage, phase ^ 1);
          const uint32_t sa = base + stage * STAGE_BYTES;
          if (PAIR) tma_gather4_pair(sa + u0 * 512, &tmA, mapa_shared(full0 + 8 * stage, 0), kb * BK, gr[0], gr[1], gr[2], gr[3]);
          else tma_gather4(sa + u0 * 512, &tmA, full0 + 8 * stage, kb * BK, gr[0], gr[1], gr[2], gr[3]);
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (GW > 0 && !A_MN && !PAIR && warp == 2 + EPI_WARPS + GW) {
    // ===================== copy-out warp (GW > 0): the permuted copy as a by-product =====================
    // The gathered A tile of a k-block sits in shared memory in exactly the layout of a tiled TMA box, so it is also stored to
    // the row-grouped copy (Xp from GEMM-1, the gathered dY from dgrad-down) that the weight gradients contract over -- no
    // separate permute pass, no second read of X / dY.  The n_tiles CTAs that work on one M-tile share the job: n-tile j
    // stores the k-blocks with kb % n_tiles == j (each block exactly once, the store traffic spread evenly over all tiles).
    // A stage is released to the producer once the MMAs (tcgen05.commit) AND its store have read it; two stores in flight.
    if (lane == 0 && p.copy_out) {
      int stage = 0, pending = -1;
      uint32_t phase = 0;
      Tile tl, nx;
      bool ok = decode_tile<MODE, PAIR>(p, unit, total, rank, tl), okn = false;
      for (int64_t t = unit; ok; t += nunits, tl = nx, ok = okn) {
        okn = decode_tile<MODE, PAIR>(p, t + nunits, total, rank, nx);
        const int nt = tl.n0 / (MODE == TC_FWD_SWIGLU ? BN / 2 : BN);    // this tile's n-tile index
        for (int kb = 0; kb < tl.nkb; ++kb) {
          mbar_wait(full0 + 8 * stage, phase);
          if (kb % p.n_tiles == nt) {
            tma_store_2d(&tmC, base + stage * STAGE_BYTES, kb * BK, tl.m0);
            bulk_commit();
            if (pending >= 0) {
              bulk_wait_read1();                       // the store before this one has read its stage
              mbar_arrive(empty0 + 8 * pending);
            }
            pending = stage;
          } else {
            if (pending >= 0) {
              bulk_wait_read0();
              mbar_arrive(empty0 + 8 * pending);
              pending = -1;
            }
            mbar_arrive(empty0 + 8 * stage);
          }
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
      }
      if (pending >= 0) {
        bulk_wait_read0();
        mbar_arrive(empty0 + 8 * pending);
      }
      bulk_wait0();                                    // all stores complete before the CTA retires
    }
  }
  tc_fence_before();
  __syncwarp();
  if (PAIR) cluster_sync_all();   // neither CTA retires (nor frees tensor memory) while its peer may still use it
  else __syncthreads();
  if (warp == 1) {
    if (PAIR) tmem_dealloc_pair(tmem_base, TMEM_COLS);
    else tmem_dealloc(tmem_base, TMEM_COLS);
  }
}

// ---------------------------------------------------------------------------------------------
// host: tensor maps and launch
// ---------------------------------------------------------------------------------------------
// 2-D bf16 tensor [outer, inner] (inner contiguous, row pitch ld elements), box = box_outer x 64, 128-byte swizzle,
// out-of-bounds elements read as zero.
bool make_map(CUtensorMap* m, const void* ptr, int64_t inner, int64_t outer, int64_t ld, int box_outer) {
  return tc_make_map(m, 2, ptr, inner, outer, ld, BK, box_outer);
}

constexpr int GATHER_WARPS = 5;       // + 1 copy-out warp: 512 threads, 128 registers each
bool g_attr_set[MAX_DEVICES][6][2][2];   // per device: MaxDynamicSharedMemorySize raised for tc_gemm_kernel<MODE, PAIR, GW>

// max_units = upper bound on tiles (PAIR: pair-tiles).  PAIR launches clusters of two CTAs (one TPC each).
template <int MODE, bool PAIR, int GW>
int32_t launch_impl(const CUtensorMap& a, const CUtensorMap& b0, const CUtensorMap& b1, const CUtensorMap& o, const TcParams& p,
                    int64_t max_units, cudaStream_t s, const CUtensorMap* o2, const CUtensorMap* cp) {
  const int dev = current_device();
  if (dev < 0) return MOE_ERR_CUDA;
  if (!g_attr_set[dev][MODE][PAIR][GW > 0]) {
    MOE_CUDA(cudaFuncSetAttribute(tc_gemm_kernel<MODE, PAIR, GW>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES));
    g_attr_set[dev][MODE][PAIR][GW > 0] = true;
  }
  const int sms = device_sm_count();
  if (sms <= 0) return MOE_ERR_CUDA;
  constexpr int NT = NTHREADS + (GW > 0 ? 32 * (GW + 1) : 0);
  const CUtensorMap& cc = cp ? *cp : a;
  if (!PAIR) {
    const unsigned grid = (unsigned)std::max<int64_t>(1, std::min<int64_t>(sms, max_units));
    MOE_LAUNCH((tc_gemm_kernel<MODE, false, GW>), grid, NT, SMEM_BYTES, s, a, b0, b1, o, o2 ? *o2 : o, cc, p);
    return MOE_OK;
  }
  const unsigned pairs = (unsigned)std::max<int64_t>(1, std::min<int64_t>(sms / 2, max_units));
  cudaLaunchConfig_t cfg;
  memset(&cfg, 0, sizeof(cfg));
  cfg.gridDim = dim3(2 * pairs);
  cfg.blockDim = dim3(NT);
  cfg.dynamicSmemBytes = SMEM_BYTES;
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = 2;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  const CUtensorMap& oo2 = o2 ? *o2 : o;
  ++g_launches;
  if (cudaLaunchKernelEx(&cfg, tc_gemm_kernel<MODE, true, GW>, a, b0, b1, o, oo2, cc, p) != cudaSuccess) {
    cudaGetLastError();
    return MOE_ERR_CUDA;
  }
  return MOE_OK;
}

// A launch with a gathered A operand (p.gat) runs the 1-CTA variant with GATHER_WARPS gather warps + one copy-out warp;
// only the two ragged GEMMs the fused layer feeds from token-major rows (GEMM-1, dgrad-down) have one.
template <int MODE, bool PAIR>
int32_t launch(const CUtensorMap& a, const CUtensorMap& b0, const CUtensorMap& b1, const CUtensorMap& o, const TcParams& p,
               int64_t max_units, cudaStream_t s, const CUtensorMap* o2 = nullptr, const CUtensorMap* cp = nullptr) {
  constexpr bool CAN_GATHER = (MODE == TC_FWD_SWIGLU || MODE == TC_DGRAD_SWIGLU) && !PAIR;
  if (p.gat != 0) {
    if constexpr (CAN_GATHER) return launch_impl<MODE, PAIR, GATHER_WARPS>(a, b0, b1, o, p, max_units, s, o2, cp);
    else return MOE_ERR_UNSUPPORTED;
  }
  return launch_impl<MODE, PAIR, 0>(a, b0, b1, o, p, max_units, s, o2, nullptr);
}

// Which launches use the CTA-pair kernel.  Default 1: the weight gradients (no ragged dimension: every 256 x 256 tile
// is a full pair tile) and single-group GEMMs (shared expert, router); the ragged expert GEMMs stay on the 1-CTA kernel
// because the unpaired last M-tile of every other expert needs a second launch whose tail costs what the pairs save
// (measured).  Selected by moe_config_t::opt_pair: level 0 (never) / 1 / 2 (ragged GEMMs too).
int pair_mode(const TcCall& c) { return c.opt_pair ? c.opt_pair - 1 : 1; }

// One logical GEMM = the pair kernel over the paired M-tiles (or over everything: single group, wgrad) followed by the
// 1-CTA kernel over the unpaired M-tiles.  With `pl == nullptr` (no pair table) the 1-CTA kernel runs all tiles.
template <int MODE>
int32_t launch_both(const CUtensorMap& a, const CUtensorMap& b0, const CUtensorMap& b0_pair, const CUtensorMap& b1,
                    const CUtensorMap& o, TcParams p, const TcCall& c, cudaStream_t s, const CUtensorMap* o2 = nullptr,
                    const CUtensorMap* cp = nullptr) {
  const int64_t max_mtiles = ceil_div(c.rows_cap, BM);
  const bool grouped = c.mtile != nullptr;
  if (pair_mode(c) == 0 || p.gat || (grouped && (pair_mode(c) < 2 || !c.plist || !c.olist))) {   // gathered A: 1-CTA kernel
    p.tlist = nullptr;
    return launch<MODE, false>(a, b0, b1, o, p, max_mtiles * p.n_tiles, s, o2, cp);
  }
  if (!grouped) {       // one group of rows_cap rows from row 0: pairs of consecutive M-tiles cover it
    p.tlist = nullptr;
    return launch<MODE, true>(a, b0_pair, b1, o, p, ceil_div(c.rows_cap, 2 * BM) * p.n_tiles, s, o2);
  }
  p.tlist = c.plist;
  MOE_CHECK((launch<MODE, true>(a, b0_pair, b1, o, p, (max_mtiles / 2) * p.n_tiles, s, o2)));
  p.tlist = c.olist;
  return launch<MODE, false>(a, b0, b1, o, p, (int64_t)std::min<int64_t>(c.E, max_mtiles) * p.n_tiles, s, o2);
}

// Tile tables (tile_tables.cuh) from the row offsets alone, for the stand-alone grouped-GEMM entry points.
__global__ void __launch_bounds__(1024) prepare_tiles_kernel(const int32_t* __restrict__ offsets, int E,
                                                             int32_t* __restrict__ mtile, int32_t* __restrict__ plist,
                                                             int32_t* __restrict__ olist) {
  __shared__ int32_t wsum[32];
  const int e = threadIdx.x;
  const int excl = e < E ? offsets[e] : 0, incl = e < E ? offsets[e + 1] : 0;
  write_tile_tables(e, E, excl, incl, mtile, plist, olist, wsum);
}

}  // namespace

int32_t tc_prepare_tiles(const int32_t* offsets, int E, int64_t rows_cap, int32_t* mtile_expert, cudaStream_t s) {
  if (E > 1024) return MOE_ERR_UNSUPPORTED;
  MOE_LAUNCH(prepare_tiles_kernel, 1, 1024, 0, s, offsets, E, mtile_expert, mtile_expert + tile_plist_off(rows_cap),
             mtile_expert + tile_olist_off(rows_cap));
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
  p.counts = c.counts;
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
  p.gidx = c.gidx;
  p.gat = c.gat;
  p.gK = c.gK > 0 ? c.gK : 1;
  p.gshift = -1;
  for (int sh = 0; sh < 31; ++sh)
    if ((1 << sh) == p.gK) p.gshift = sh;
  p.roww = c.roww;
  p.dwpart = c.dwpart;
  p.copy_out = (c.gat && c.copy_out) ? 1 : 0;
  if (c.gat < 0 || c.gat > 1 || (c.gat && c.mode != TC_FWD_SWIGLU && c.mode != TC_DGRAD_SWIGLU)) return MOE_ERR_INVALID_ARG;
  if ((c.gat || c.roww) && (!c.gidx || !c.mtile)) return MOE_ERR_INVALID_ARG;
  if (c.gat && (c.g_rows <= 0 || (reinterpret_cast<uintptr_t>(c.gidx) & 15))) return MOE_ERR_INVALID_ARG;
  if (c.copy_out && !c.gat) return MOE_ERR_INVALID_ARG;
  const int64_t a_rows = c.gat == 1 ? c.g_rows : c.rows_cap;     // rows of the tensor behind the A map
  const int a_box = c.gat == 1 ? 1 : BM;                          // gathered: box = one row of 64 columns (x4 per gather4)
  CUtensorMap ta, tb0, tb0p, tb1, to, tc;
  if (c.mode == TC_FWD_F32 ? ((c.N & 3) || (c.ld0 & 3)) : ((c.N & 7) || (c.ld0 & 7))) return MOE_ERR_UNSUPPORTED;
  switch (c.mode) {
    case TC_FWD_F32:
    case TC_FWD: {
      if (c.Kd % BK) return MOE_ERR_UNSUPPORTED;
      p.nkb = c.Kd / BK;
      p.n_tiles = (int)ceil_div(c.N, BN);
      if (!make_map(&ta, c.A, c.Kd, a_rows, c.lda, a_box)) return MOE_ERR_UNSUPPORTED;
      if (!make_map(&tb0, c.B0, c.b_cols, (int64_t)c.E * c.b_rows, c.b_cols, BN)) return MOE_ERR_UNSUPPORTED;
      if (!make_map(&tb0p, c.B0, c.b_cols, (int64_t)c.E * c.b_rows, c.b_cols, BN / 2)) return MOE_ERR_UNSUPPORTED;   // a pair CTA's half
      if (c.mode == TC_FWD_F32) return launch_both<TC_FWD_F32>(ta, tb0, tb0p, tb0, ta, p, c, s);
      if (!tc_make_map3(&to, 2, c.out0, c.N, c.rows_cap, 1, c.ld0, 64, BM)) return MOE_ERR_UNSUPPORTED;   // C [rows, N]
      return launch_both<TC_FWD>(ta, tb0, tb0p, tb0, to, p, c, s);
    }
    case TC_FWD_SWIGLU: {
      if (c.Kd % BK || (c.F & 7) || (c.ld1 & 7)) return MOE_ERR_UNSUPPORTED;
      p.nkb = c.Kd / BK;
      p.n_tiles = (int)ceil_div(c.F, BN / 2);
      if (!make_map(&ta, c.A, c.Kd, a_rows, c.lda, a_box)) return MOE_ERR_UNSUPPORTED;
      if (!make_map(&tb0, c.B0, c.b_cols, (int64_t)c.E * c.b_rows, c.b_cols, BN / 2)) return MOE_ERR_UNSUPPORTED;
      if (!make_map(&tb1, c.B1, c.b_cols, (int64_t)c.E * c.b_rows, c.b_cols, BN / 2)) return MOE_ERR_UNSUPPORTED;
      p.tma_out = (c.F % 32 == 0) ? 1 : 0;   // g / u boxes of 32 columns must not straddle the [g|u] boundary
      CUtensorMap to2;
      if (p.tma_out && (!tc_make_map3(&to, 2, c.out0, 2 * (int64_t)c.F, c.rows_cap, 1, c.ld0, 32, BM) ||    // gu [rows, 2F]
                        !tc_make_map3(&to2, 2, c.out1, c.F, c.rows_cap, 1, c.ld1, 32, BM)))                  // a [rows, F]
        p.tma_out = 0;
      if (!p.tma_out && (c.roww || c.gat)) return MOE_ERR_UNSUPPORTED;   // weighted epilogue / gather variant: TMA-store path only
      if (p.copy_out && !make_map(&tc, c.copy_out, c.Kd, c.rows_cap, c.ld_copy, BM)) return MOE_ERR_UNSUPPORTED;   // Xp [rows, H]
      if (!p.tma_out) return launch_both<TC_FWD_SWIGLU>(ta, tb0, tb0, tb1, ta, p, c, s);
      return launch_both<TC_FWD_SWIGLU>(ta, tb0, tb0, tb1, to, p, c, s, &to2, p.copy_out ? &tc : nullptr);
    }
    case TC_DGRAD:
    case TC_DGRAD_SWIGLU: {
      // contraction over the weights' rows (b_rows per source), output columns = b_cols
      if (c.b_rows % BK) return MOE_ERR_UNSUPPORTED;
      const bool split = c.B1 != nullptr;
      p.kb_split = c.b_rows / BK;
      p.nkb = split ? 2 * p.kb_split : p.kb_split;
      p.n_tiles = (int)ceil_div(c.N, BN);
      if (!make_map(&ta, c.A, (int64_t)p.nkb * BK, a_rows, c.lda, a_box)) return MOE_ERR_UNSUPPORTED;
      if (!make_map(&tb0, c.B0, c.b_cols, (int64_t)c.E * c.b_rows, c.b_cols, 64)) return MOE_ERR_UNSUPPORTED;
      if (!make_map(&tb1, split ? c.B1 : c.B0, c.b_cols, (int64_t)c.E * c.b_rows, c.b_cols, 64)) return MOE_ERR_UNSUPPORTED;
      if (c.mode == TC_DGRAD) {
        if (!tc_make_map3(&to, 2, c.out0, c.N, c.rows_cap, 1, c.ld0, 64, BM)) return MOE_ERR_UNSUPPORTED;   // dA [rows, N]
        return launch_both<TC_DGRAD>(ta, tb0, tb0, tb1, to, p, c, s);
      }
      if ((c.F & 7) || (c.ldgu & 7)) return MOE_ERR_UNSUPPORTED;
      p.tma_out = (c.F % 32 == 0) ? 1 : 0;   // dg / du boxes of 32 columns must not straddle the [dg|du] boundary
      if (p.tma_out && !split &&                                                          // saved [g|u] rows, same boxes
          !tc_make_map3(&tb1, 2, c.gu, 2 * (int64_t)c.F, c.rows_cap, 1, c.ldgu, 32, BM))
        p.tma_out = 0;
      if (!p.tma_out && (c.roww || c.dwpart || c.gat)) return MOE_ERR_UNSUPPORTED;
      if (p.copy_out && !make_map(&tc, c.copy_out, (int64_t)p.nkb * BK, c.rows_cap, c.ld_copy, BM)) return MOE_ERR_UNSUPPORTED;
      if (!tc_make_map3(&to, 2, c.out0, 2 * (int64_t)c.F, c.rows_cap, 1, c.ld0, 32, BM)) return MOE_ERR_UNSUPPORTED;   // dgu [rows, 2F]
      return launch_both<TC_DGRAD_SWIGLU>(ta, tb0, tb0, tb1, to, p, c, s, nullptr, p.copy_out ? &tc : nullptr);
    }
    case TC_WGRAD: {
      // every (expert, 256 x 256 output tile) goes to a CTA pair: no ragged dimension, the contraction runs over the
      // expert's rows.  A: [rows_cap, lda] read MN-major (inner = columns = output rows); A2 likewise (output columns).
      // The pair kernel pays where operand traffic binds: contractions of >= 4 k-blocks (about 256 real rows per expert;
      // rows_cap counts 127 padding rows per expert) and an output height that 256-row tiles cover without extra padding.
      // Measured: configs[1] 690 -> 625 us; configs[2] (128 rows per expert: 2 k-blocks per 64 KB of
      // output per CTA, write-bound) 8.04 -> 8.75 ms and configs[4] (2880 = 11.25 x 256) 4.2 -> 4.5 ms, so those stay 1-CTA.
      const bool pair = pair_mode(c) > 0 && (c.mtile == nullptr || c.rows_cap >= 384 * (int64_t)c.E) &&
                        ceil_div(c.M, 2 * BM) * 2 == ceil_div(c.M, BM);
      p.m_tiles = (int)ceil_div(c.M, pair ? 2 * BM : BM);
      p.n_tiles = (int)ceil_div(c.N, BN);
      if (!make_map(&ta, c.A, c.lda, c.rows_cap, c.lda, 64)) return MOE_ERR_UNSUPPORTED;
      if (!make_map(&tb0, c.A2, c.N, c.rows_cap, c.lda2, 64)) return MOE_ERR_UNSUPPORTED;
      p.acc_f32 = c.acc_f32 ? 1 : 0;
      if (c.acc_f32 ? !tc_make_map3(&to, 4, c.out0, c.N, c.M, c.E, c.ld0, 32, BM)    // fp32 dB [E, M, N], reduce-add
                    : !tc_make_map3(&to, 2, c.out0, c.N, c.M, c.E, c.ld0, 64, BM))   // bf16 dB [E, M, N], overwrite
        return MOE_ERR_UNSUPPORTED;
      const int64_t units = (int64_t)c.E * p.m_tiles * p.n_tiles;
      // short contractions (about 256 real rows per expert or fewer): every tile is mostly its 64 KB of output, so the
      // 1-CTA kernel trades a ring stage for a second staging box per warp group (configs[2]: 7.30 -> 6.73 ms; with the
      // long contractions of configs[4] the 4-stage ring is 2 % faster)
      p.short_ring = (c.mtile != nullptr && c.rows_cap < 384 * (int64_t)c.E) ? 1 : 0;
      if (pair) return launch<TC_WGRAD, true>(ta, tb0, tb0, to, p, units, s);
      return launch<TC_WGRAD, false>(ta, tb0, tb0, to, p, units, s);
    }
  }
  return MOE_ERR_INVALID_ARG;
}

}  // namespace moe
