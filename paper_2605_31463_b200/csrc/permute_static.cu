// moe_permute_static_ws: moe_permute (R6) for callers that cannot give the library a workspace.
//
// Who that is.  moe_permute needs a few KB of device scratch (the per-chunk expert histograms that its two kernels hand
// to each other) and asks the caller for it as `ws`.  Some callers have nowhere to get it from: an operator plug-in
// running inside a serving or training runtime that owns every byte of device memory and hands the plug-in nothing but
// its input and output tensors; a process whose memory pool was sized at start-up and which bans cudaMalloc afterwards
// (cudaMalloc / cudaFree synchronise the whole device and may fail when the 180 GB are nearly full); a latency-critical
// loop that must not touch the allocator at all.  For them this file keeps the scratch inside the library image: a
// fixed file-scope __device__ array.  The entry point below allocates nothing -- no cudaMalloc, no cudaFree, no
// library routine that allocates -- it only launches the same kernels moe_permute launches.
//
// What it costs.  MOE_PERMUTE_STATIC_WS_BYTES (1 MiB) of device memory on every GPU that loads libmoe_b200.so, held
// until the process exits, whether or not this entry point is ever called.  Problems whose histograms do not fit
// (ceil(T*K/1024) * E * 4 bytes > 1 MiB) are refused with MOE_ERR_TOO_LARGE; nothing is enqueued then.
//
// Sharing.  There is one array per GPU and every call on that GPU uses it.  It keeps whatever the previous call left
// there; that is harmless because the histogram kernel overwrites every entry the scan kernel later reads (nothing has
// to start at zero, so nothing is cleared).  Two calls that run at the same time on one GPU (different streams, or
// different host threads) race on the array and produce garbage maps: keep calls on one stream, or order them with
// events.
#include <mutex>

#include "common.cuh"

namespace moe {
namespace {

constexpr size_t STATIC_WS_INTS = MOE_PERMUTE_STATIC_WS_BYTES / sizeof(int32_t);

// The scratch itself.  In host code `g_static_hist` is only a handle the runtime knows the symbol by, NOT a device
// address: it must never be passed to a kernel as is.  device_scratch() below turns it into the address on the current
// GPU (each GPU has its own copy of the array, at its own address).
static __device__ __align__(256) int32_t g_static_hist[STATIC_WS_INTS];

std::mutex g_setup_mutex;
int32_t* g_scratch_addr[MAX_DEVICES];   // device address of g_static_hist on device d, nullptr until looked up

// Device address of the array on the CURRENT device, looked up once per device (with that device current) and cached.
int32_t device_scratch(int32_t** out) {
  const int dev = current_device();
  if (dev < 0) return MOE_ERR_CUDA;
  std::lock_guard<std::mutex> lock(g_setup_mutex);
  if (g_scratch_addr[dev] == nullptr) {
    void* p = nullptr;
    if (cudaGetSymbolAddress(&p, g_static_hist) != cudaSuccess || p == nullptr) {
      cudaGetLastError();
      return MOE_ERR_CUDA;
    }
    g_scratch_addr[dev] = static_cast<int32_t*>(p);
  }
  *out = g_scratch_addr[dev];
  return MOE_OK;
}

}  // namespace
}  // namespace moe

extern "C" int32_t moe_permute_static_ws(const moe_config_t* cfg, const void* X, const int32_t* topk_idx,
                                         int32_t* counts, int32_t* offsets, int32_t* perm_to_flat,
                                         int32_t* flat_to_perm, void* Xp, void* stream) {
  using namespace moe;
  if (!cfg || !topk_idx || !counts || !offsets || !perm_to_flat || !flat_to_perm) return MOE_ERR_INVALID_ARG;
  MOE_CHECK(validate(cfg));
  if (X && !Xp) return MOE_ERR_INVALID_ARG;
  if (cfg->E > 1024) return MOE_ERR_UNSUPPORTED;                       // same limit as moe_permute
  const int64_t nchunks = ceil_div((int64_t)cfg->T * cfg->K, PERM_CHUNK);
  if (nchunks * cfg->E > (int64_t)STATIC_WS_INTS) return MOE_ERR_TOO_LARGE;
  int32_t* hist = nullptr;
  MOE_CHECK(device_scratch(&hist));       // first call on a device: cudaGetSymbolAddress (do it before any capture)
  cudaStream_t s = as_stream(stream);
  // No tile tables here (mtile = nullptr): they are a by-product moe_permute leaves in `ws` for nobody; the grouped
  // GEMM entry points rebuild theirs from `offsets`.
  MOE_CHECK(build_maps(cfg, topk_idx, counts, offsets, perm_to_flat, flat_to_perm, nullptr, hist, s));
  if (X) MOE_CHECK(gather_rows(cfg, X, cfg->H, elem_bytes(cfg), flat_to_perm, perm_to_flat, offsets, Xp, s));
  return MOE_OK;
}
