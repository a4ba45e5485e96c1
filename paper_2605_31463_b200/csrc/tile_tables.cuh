// Tile tables of the tensor-core grouped GEMMs (expert groups start at multiples of 128 rows), built on the
// device from the per-expert row offsets (per-expert shapes are data dependent and never visit the
// host).  One int32 array, three tables:
//   mtile            mtile[0] = number of 128-row M-tiles below offsets[E];  mtile[1 + i] = expert of M-tile i
//   plist = mtile + tile_plist_off(R)
//                    plist[0] = number of M-tile PAIRS (two consecutive M-tiles of ONE expert: the unit of work of the
//                    cta_group::2 kernels, whose CTA pair shares the expert's weight tile);  plist[1 + i] = first M-tile of pair i
//   olist = mtile + tile_olist_off(R)
//                    olist[0] = number of UNPAIRED M-tiles (the last tile of an expert with an odd tile count; run by the
//                    1-CTA kernel);  olist[1 + i] = that M-tile
// Not part of the public ABI.
#pragma once
#include "common.cuh"

namespace moe {

inline size_t tile_plist_off(int64_t R) { return (size_t)(R / 128 + 4); }
inline size_t tile_olist_off(int64_t R) { return (size_t)(R / 128 + 4 + R / 256 + 4); }
inline size_t tile_table_ints(int64_t R, int E) { return tile_olist_off(R) + (size_t)E + 4; }

#ifdef __CUDACC__
// Inclusive prefix sum of `v` over a 1024-thread block (wsum: 32 ints of shared memory, reusable right after).
__device__ __forceinline__ int block_incl_scan_1024(int v, int32_t* wsum) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int off = 1; off < 32; off <<= 1) {
    const int o = __shfl_up_sync(0xffffffffu, v, off);
    if (lane >= off) v += o;
  }
  __syncthreads();   // a previous scan's readers are done with wsum
  if (lane == 31) wsum[warp] = v;
  __syncthreads();
  if (warp == 0) {
    int ws = wsum[lane];
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
      const int o = __shfl_up_sync(0xffffffffu, ws, off);
      if (lane >= off) ws += o;
    }
    wsum[lane] = ws;
  }
  __syncthreads();
  return v + (warp > 0 ? wsum[warp - 1] : 0);
}

// Called by all 1024 threads of the block; thread e < E owns expert e whose (128-aligned) row range is [excl, incl).
__device__ __forceinline__ void write_tile_tables(int e, int E, int excl, int incl, int32_t* mtile, int32_t* plist,
                                                  int32_t* olist, int32_t* wsum) {
  const int t0 = excl / 128, nt = (e < E) ? (incl - excl) / 128 : 0;
  const int np = nt >> 1, no = nt & 1;
  const int pincl = block_incl_scan_1024(np, wsum);
  const int oincl = block_incl_scan_1024(no, wsum);
  if (e < E) {
    for (int t = 0; t < nt; ++t) mtile[1 + t0 + t] = e;
    for (int i = 0; i < np; ++i) plist[1 + pincl - np + i] = t0 + 2 * i;
    if (no) olist[oincl] = t0 + nt - 1;       // 1 + (oincl - 1)
    if (e == E - 1) {
      mtile[0] = incl / 128;
      plist[0] = pincl;
      olist[0] = oincl;
    }
  }
}
#endif

}  // namespace moe
