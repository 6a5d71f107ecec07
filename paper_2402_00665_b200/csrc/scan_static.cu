// scan_static.cu -- bvh_scan_counts_static: the counts -> offsets scan (K7, scan.cu; reading G21) for callers that
// have no way to hand the library a scratch buffer.
//
// Who that is.  Every other entry point takes its working memory from the caller, which presumes the caller can get
// device memory at the moment of the call.  Some cannot: code that runs after the application has given its whole
// memory budget to a pool or an arena and has nothing left to carve the tile sums from; a plug-in or callback that the
// host framework forbids to touch the allocator (cudaMalloc synchronises the device and can stall every other stream,
// and it is illegal while a stream of the process is being captured); a real-time loop that must not take the
// allocator's lock.  For them the scan's one piece of scratch -- one int64 per tile of 4096 counts -- lives in a
// fixed array inside the library's device image.
//
// What it costs.  kStaticScanTiles * 8 bytes = 64 KB of device memory on EVERY GPU on which the library's module is
// loaded, from load until the process exits, whether or not this entry point is ever called.  The size is fixed at
// compile time, so a batch of more than BVH_SCAN_STATIC_MAX_Q counts is refused (BVH_ERR_STATIC_LIMIT) rather than
// overrun; use bvh_scan_counts with your own scratch for those.
//
// What is shared.  There is ONE array per GPU and every call on that GPU uses it, whatever the stream.  Two calls whose
// kernels may overlap on the GPU (different streams without an event between them, or two host threads) race on it
// and corrupt each other's offsets: keep the calls of one device on one stream or order them yourself.  The array
// keeps what the last call left there; that is harmless, because the first kernel of a scan writes the tile sums of
// all the tiles the later kernels read (nothing has to start at zero, so nothing is cleared).
//
// The kernels are the ones bvh_scan_counts launches (scan.cu, through launch_scan); only where the tile sums live
// differs, so the offsets are the same bits.
#include <atomic>

#include "../../include/bvh_b200.h"
#include "common.cuh"

namespace {

constexpr int64_t kStaticScanTiles = 8192;  // 64 KB of int64 tile sums per GPU

// In host code this name is only a handle of the host-side shadow the runtime registers for the variable, never the
// device address: handing it to a kernel as a pointer would fault (or, on a system where the GPU can reach host
// memory, quietly scribble over host data).  Host code below therefore asks the runtime for the device address.
static __device__ __align__(256) int64_t g_static_tile_sums[kStaticScanTiles];

constexpr int kMaxDevices = 64;
std::atomic<int64_t*> g_tile_sums_address[kMaxDevices];  // per device, filled on the first call made on that device

// The device address of g_static_tile_sums on the CURRENT device.  Looked up once per device (the lookup loads the
// library's module on that device if nothing has yet); a failed lookup is reported and not remembered.  Two threads
// that get here together both store the same address.
cudaError_t static_tile_sums(int64_t** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  int64_t* p = g_tile_sums_address[dev].load(std::memory_order_acquire);
  if (p == nullptr) {
    e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_static_tile_sums);
    if (e != cudaSuccess) return e;
    if (p == nullptr) return cudaErrorInvalidSymbol;
    g_tile_sums_address[dev].store(p, std::memory_order_release);
  }
  *out = p;
  return cudaSuccess;
}

}  // namespace

extern "C" int bvh_scan_counts_static(const int32_t* counts, int64_t q, int64_t* offsets, void* stream) {
  if (q < 0 || !offsets) return BVH_ERR_INVALID_ARGUMENT;
  if (q > 0 && !counts) return BVH_ERR_INVALID_ARGUMENT;
  // the second test keeps the limit honest should the scan's tile size ever change
  if (q > BVH_SCAN_STATIC_MAX_Q || (q > 0 && bvh::scan_scratch_bytes(q) > sizeof(int64_t) * kStaticScanTiles))
    return BVH_ERR_STATIC_LIMIT;
  int64_t* sums = nullptr;
  if (static_tile_sums(&sums) != cudaSuccess) return BVH_ERR_CUDA;
  if (bvh::launch_scan(counts, q, offsets, sums, static_cast<cudaStream_t>(stream)) != cudaSuccess) return BVH_ERR_CUDA;
  return BVH_OK;
}
