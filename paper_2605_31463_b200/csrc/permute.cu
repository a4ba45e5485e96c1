// Histogram + exclusive scan + stable counting sort of flat positions by expert, and the row movers
// built on the resulting maps (SURVEY.md §8c R6, R7 combine, R8 combine-bwd).
// No atomics anywhere: ranks come from warp match/ballot and per-chunk prefix tables, so the maps are
// deterministic and bit-exact against the oracle's stable counting sort.  Two launches: chunk histograms, then
// scan + scatter (no memset: the padding rows' -1 entries are written by the second kernel).
#include "common.cuh"
#include "tile_tables.cuh"

namespace moe {
namespace {

constexpr unsigned FULL = 0xffffffffu;
constexpr int CHUNK_WARPS = 8;                                   // 256 threads per chunk CTA
constexpr int CHUNK_ROUNDS = PERM_CHUNK / (CHUNK_WARPS * 32);    // rounds of 32 positions per warp

// Per-warp running histogram over this warp's contiguous slice of the chunk.
// rank[r] = number of earlier positions of the same expert inside this warp's slice.
__device__ __forceinline__ void warp_rank(const int32_t* __restrict__ idx, int64_t TK, int64_t warp_base, int lane,
                                          int32_t* wh, int (&ex)[CHUNK_ROUNDS], int (&rank)[CHUNK_ROUNDS]) {
#pragma unroll
  for (int r = 0; r < CHUNK_ROUNDS; ++r) {
    const int64_t p = warp_base + r * 32 + lane;
    const int e = (p < TK) ? idx[p] : -1;       // -1: past the end, or an empty slot of a variable-k router (V1)
    ex[r] = e;
    const unsigned m = __match_any_sync(FULL, e);
    const int before = __popc(m & ((1u << lane) - 1u));
    int base = 0;
    if (e >= 0) base = wh[e];
    rank[r] = base + before;
    __syncwarp();
    if (e >= 0 && before == 0) wh[e] = base + __popc(m);  // lowest lane of each match set updates
    __syncwarp();
  }
}

// Phase 1: hist[chunk][e] = number of positions of expert e in the chunk.
__global__ void __launch_bounds__(CHUNK_WARPS * 32) hist_kernel(const int32_t* __restrict__ idx, int64_t TK, int E,
                                                                 int32_t* __restrict__ hist) {
  extern __shared__ int32_t wh[];  // [CHUNK_WARPS][E]
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  for (int i = threadIdx.x; i < CHUNK_WARPS * E; i += blockDim.x) wh[i] = 0;
  __syncthreads();
  int ex[CHUNK_ROUNDS], rank[CHUNK_ROUNDS];
  const int64_t base = (int64_t)blockIdx.x * PERM_CHUNK + warp * (CHUNK_ROUNDS * 32);
  warp_rank(idx, TK, base, lane, wh + warp * E, ex, rank);
  __syncthreads();
  for (int e = threadIdx.x; e < E; e += blockDim.x) {
    int s = 0;
#pragma unroll
    for (int w = 0; w < CHUNK_WARPS; ++w) s += wh[w * E + e];
    hist[(size_t)blockIdx.x * E + e] = s;
  }
}

// Phase 1b, only for many chunks (nchunks > PREFIX_MIN_CHUNKS): turn each expert's column of chunk counts into an
// INCLUSIVE prefix over chunks, in place, so that phase 2 reads two entries per expert instead of the whole column
// (otherwise every one of the nchunks CTAs walks all nchunks rows: O(nchunks^2 E) loads, 1 GB of L2 reads at T*K = 1M).
// One CTA per expert, strided block scan with a running carry.
constexpr int PREFIX_MIN_CHUNKS = 256;
__global__ void __launch_bounds__(1024) hist_prefix_kernel(int32_t* __restrict__ hist, int E, int nchunks) {
  __shared__ int32_t wsum[32];
  __shared__ int32_t s_carry;
  const int e = blockIdx.x;
  if (threadIdx.x == 0) s_carry = 0;
  __syncthreads();
  for (int c0 = 0; c0 < nchunks; c0 += 1024) {
    const int c = c0 + threadIdx.x;
    const int v = c < nchunks ? hist[(size_t)c * E + e] : 0;
    const int incl = block_incl_scan_1024(v, wsum) + s_carry;
    if (c < nchunks) hist[(size_t)c * E + e] = incl;
    __syncthreads();
    if (threadIdx.x == 1023) s_carry = incl;
    __syncthreads();
  }
}

// Phase 2: scan + scatter in one launch (1024 threads per chunk CTA).  Every CTA rebuilds what it needs from the chunk
// histograms (E x nchunks ints, L2-resident): thread e sums expert e's column -> counts, aligned exclusive offsets by a block
// scan, and the chunk's base row of expert e = offsets[e] + positions of e in earlier chunks.  CTA 0 also publishes counts,
// offsets and the tile tables of the tensor-core GEMMs (tile_tables.cuh; row_align a multiple of 128); the padding rows of
// expert e get their -1 in perm_to_flat from CTA e % nchunks.  Then the first 8 warps scatter as before:
// flat_to_perm[p] = base[e] + rank of p among the chunk's positions of e.
__global__ void __launch_bounds__(1024) scan_scatter_kernel(const int32_t* __restrict__ idx, int64_t TK, int E, int E_tab,
                                                            int row_align, const int32_t* __restrict__ hist, int nchunks,
                                                            int32_t* __restrict__ counts, int32_t* __restrict__ offsets,
                                                            int32_t* __restrict__ mtile, int32_t* __restrict__ plist,
                                                            int32_t* __restrict__ olist, int32_t* __restrict__ p2f,
                                                            int32_t* __restrict__ f2p, int64_t rows_cap, int prefixed) {
  extern __shared__ int32_t sm[];          // [E] chunk bases, then [CHUNK_WARPS][E] per-warp histograms
  __shared__ int32_t wsum[32];
  __shared__ int32_t s_end;
  int32_t* cbase = sm;
  int32_t* wh = sm + E;
  const int e = threadIdx.x;
  int cnt = 0, before = 0;
  if (e < E) {
    if (prefixed) {   // hist holds inclusive prefixes over chunks (hist_prefix_kernel)
      cnt = hist[(size_t)(nchunks - 1) * E + e];
      before = blockIdx.x > 0 ? hist[(size_t)(blockIdx.x - 1) * E + e] : 0;
    } else {
      for (int c = 0; c < nchunks; ++c) {
        const int h = hist[(size_t)c * E + e];
        if (c < (int)blockIdx.x) before += h;
        cnt += h;
      }
    }
  }
  const int a = row_align < 1 ? 1 : row_align;
  const int padded = (e < E) ? (cnt + a - 1) / a * a : 0;
  const int incl = block_incl_scan_1024(padded, wsum);
  const int excl = incl - padded;
  if (e < E) {
    cbase[e] = excl + before;
    if (blockIdx.x == 0) {
      counts[e] = cnt;
      offsets[e] = excl;
      if (e == E - 1) offsets[E] = incl;
    }
    if (e % nchunks == (int)blockIdx.x)
      for (int r = excl + cnt; r < incl; ++r) p2f[r] = -1;      // padding rows of the group
    if (e == E - 1) s_end = incl;
  }
  // the GEMM tile tables cover the first E_tab experts (those that own FFN weights; V2: the rest compute nothing)
  if (blockIdx.x == 0 && mtile != nullptr) write_tile_tables(e, E_tab, excl, incl, mtile, plist, olist, wsum);
  for (int i = threadIdx.x; i < CHUNK_WARPS * E; i += blockDim.x) wh[i] = 0;
  __syncthreads();
  // rows past the last group (the slack of the worst-case buffer height) own no flat position either
  for (int64_t r = (int64_t)s_end + blockIdx.x * 1024 + threadIdx.x; r < rows_cap; r += (int64_t)gridDim.x * 1024) p2f[r] = -1;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  int ex[CHUNK_ROUNDS], rank[CHUNK_ROUNDS];
  const int64_t base = (int64_t)blockIdx.x * PERM_CHUNK + warp * (CHUNK_ROUNDS * 32);
  if (warp < CHUNK_WARPS) warp_rank(idx, TK, base, lane, wh + warp * E, ex, rank);
  __syncthreads();
  // turn per-warp totals into exclusive prefixes over warps, offset by the chunk base
  for (int x = threadIdx.x; x < E; x += blockDim.x) {
    int run = cbase[x];
#pragma unroll
    for (int w = 0; w < CHUNK_WARPS; ++w) {
      const int h = wh[w * E + x];
      wh[w * E + x] = run;
      run += h;
    }
  }
  __syncthreads();
  if (warp < CHUNK_WARPS) {
#pragma unroll
    for (int r = 0; r < CHUNK_ROUNDS; ++r) {
      const int64_t p = base + r * 32 + lane;
      if (ex[r] >= 0) {
        const int row = wh[warp * E + ex[r]] + rank[r];
        f2p[p] = row;
        p2f[row] = (int32_t)p;
      } else if (p < TK) {
        f2p[p] = -1;                              // an empty slot owns no permuted row
      }
    }
  }
}

}  // namespace

int32_t build_maps(const moe_config_t* c, const int32_t* idx, int32_t* counts, int32_t* offsets, int32_t* p2f,
                   int32_t* f2p, int32_t* mtile_expert, int32_t* hist, cudaStream_t s) {
  const int64_t TK = (int64_t)c->T * c->K;
  const int nchunks = (int)ceil_div(TK, PERM_CHUNK);
  if (c->E > 1024) return MOE_ERR_UNSUPPORTED;
  const size_t smem = (size_t)CHUNK_WARPS * c->E * sizeof(int32_t);
  MOE_LAUNCH(hist_kernel, nchunks, CHUNK_WARPS * 32, smem, s, idx, TK, c->E, hist);
  const int prefixed = nchunks > PREFIX_MIN_CHUNKS;
  if (prefixed) MOE_LAUNCH(hist_prefix_kernel, c->E, 1024, 0, s, hist, c->E, nchunks);
  int32_t* mt = (c->row_align % 128 == 0) ? mtile_expert : nullptr;
  const int64_t R = padded_rows(c);
  MOE_LAUNCH(scan_scatter_kernel, nchunks, 1024, smem + (size_t)c->E * sizeof(int32_t), s, idx, TK, c->E, e_ffn(c), c->row_align,
             hist, nchunks, counts, offsets, mt, mt ? mt + tile_plist_off(R) : nullptr, mt ? mt + tile_olist_off(R) : nullptr,
             p2f, f2p, R, prefixed);
  return MOE_OK;
}

}  // namespace moe
