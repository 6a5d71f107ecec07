// common.cuh -- shared declarations of the CUDA path (sm_100a only).
// Nothing in this directory is shared with, or included by, oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>

namespace bvh {

constexpr int kSentinel = -1;   // the paper's sentinel node; reading G9
constexpr int kInvalid = -1;    // the paper's "invalid entry value (e.g., -1)" in `store`
constexpr int kNumSMs = 148;    // B200: what sm_count() falls back to when the device cannot be queried; grids are sized from sm_count()

// 32-byte node record, read and written as two float4 (one 32-byte sector per node visit).
//   lo = {min.x, min.y, min.z, bitcast(left_child)}   hi = {max.x, max.y, max.z, bitcast(rope)}
struct __align__(32) Node {
  float4 lo;
  float4 hi;
};

// ---- layout of the caller's `nodes` buffer ----------------------------------------------------------------
//   [0, 64)                          NodesHeader (written by the build; queries read the leaf format there)
//   [64, 64 + 32 (n-1))              internal records I_0 .. I_{n-2} (Karras index), one Node each
//   [leaf_offset_bytes(n), ...)      leaf records L_0 .. L_{n-1} in Morton order:
//        point leaves (bvh_build_points): float4 {x, y, z, bitcast(payload)}          16 bytes
//        box leaves   (bvh_build_boxes) : Node {min.xyz, bitcast(payload)} {max.xyz, 0}  32 bytes
//   payload = original primitive index | kLeafRopeInternal if the leaf's skip-connection is the INTERNAL node
//   i+1 (else it is leaf i+1; the last leaf's is the sentinel): Algorithm 2 needs one bit.
constexpr uint32_t kNodesMagic = 0x42564832u;   // "BVH2"
constexpr int kNodesHeaderBytes = 64;
constexpr int kLeafPoints = 0, kLeafBoxes = 1;
constexpr uint32_t kLeafRopeInternal = 0x80000000u;
constexpr uint32_t kLeafPrimMask = 0x7fffffffu;
struct NodesHeader {
  uint32_t magic;
  int32_t n;
  int32_t leaf_kind;
  int32_t reserved;
  float scene_lo[3];   // = box of the root, bit for bit (D1)
  float scene_hi[3];
  uint32_t pad[6];
};
static_assert(sizeof(NodesHeader) == kNodesHeaderBytes, "nodes header is 64 bytes");
__host__ __device__ inline size_t leaf_offset_bytes(int64_t n) {
  return (size_t)kNodesHeaderBytes + sizeof(Node) * (size_t)(n > 1 ? n - 1 : 0);
}
__host__ __device__ inline size_t leaf_record_bytes(int leaf_kind) { return leaf_kind == kLeafPoints ? 16 : 32; }

// ---- scratch layout of one build (offsets in bytes from the caller's scratch pointer) ---------------
struct ScratchLayout {
  size_t header;        // Header (below)
  size_t hist;          // uint32 [passes][256]   global digit histograms
  size_t status;        // uint32 [passes][tiles][256]  onesweep tile status words
  size_t arrivals;      // uint32 [segments]  children arrived at each window of the bottom-up pass (hierarchy.cu)
  size_t fix_flag;      // uint32 [tie_fixup_tiles]  63-bit codes: tile is on the work list of long runs (tie_fixup.cu)
  size_t zero_bytes;    // header + hist + status + arrivals are contiguous from 0 and zero-initialised per build
  size_t keys[2];       // KeyT [n]   ping-pong; sorted codes end in keys[0]
  size_t vals[2];       // uint32 [n] ping-pong; permutation ends in vals[0]
  size_t seg_items;     // int2 [segments][192]  subtrees handed from one window of the bottom-up pass to its parent
  size_t seg_count;     // int32 [segments]      how many each window handed over
  size_t fix_list;      // uint32 [tie_fixup_tiles]  the work list
  size_t hist2;         // uint32 [8][256], uint32 [8][tiles][256]: histograms and tile status words of the conditional second
  size_t status2;       //   sort of a 63-bit build; NOT zeroed per build, that sort clears them when it runs (it rarely does)
  size_t total;
  int segments;         // windows of all levels of the bottom-up pass (hierarchy.cu)
  int passes;           // 8-bit digits of a code: 4 (30-bit) or 8 (63-bit)
  int slots;            // zeroed histogram / status slots: one per pass (4 for the upper-bit passes of a two-stage sort)
  int tiles;
  int key_bytes;
};

struct Header {
  uint32_t bounds_enc[8];    // [0..2] = ~ord(min.xyz), [3..5] = ord(max.xyz), maximised with atomicMax
  uint32_t tile_counter[16]; // one dynamic tile counter per sort pass (63-bit builds: 4 passes + 8 of the conditional second sort)
  uint32_t sort_fallback;    // raised by tie_long_kernel: a run of equal upper bits did not fit a block; run the second sort
  uint32_t fix_count;        // tiles on the work list of tie_long_kernel
  uint32_t pad[38];
};
static_assert(sizeof(Header) == 256, "header is one 256-byte block");

ScratchLayout scratch_layout(int64_t n, int morton_bits);
int sort_tile_items(int key_bytes);

// ---- order-preserving float <-> uint map (float atomic min/max through atomicMax on uint) ---------
__host__ __device__ inline uint32_t float_to_ordered(float f) {
#ifdef __CUDA_ARCH__
  uint32_t b = __float_as_uint(f);
#else
  union { float f; uint32_t u; } c; c.f = f; uint32_t b = c.u;
#endif
  return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__host__ __device__ inline float ordered_to_float(uint32_t o) {
  uint32_t b = (o & 0x80000000u) ? (o & 0x7fffffffu) : ~o;
#ifdef __CUDA_ARCH__
  return __uint_as_float(b);
#else
  union { float f; uint32_t u; } c; c.u = b; return c.f;
#endif
}

// Scene bounds decoded from the header: {min.xyz, max.xyz}.
__device__ inline void load_scene_bounds(const Header* h, float out[6]) {
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    out[a] = ordered_to_float(~h->bounds_enc[a]);
    out[3 + a] = ordered_to_float(h->bounds_enc[3 + a]);
  }
}

// ---- programmatic dependent launch: the kernels of one build / one query pass run back to back on one stream, each
// depending on the one before.  Launched with this attribute, a kernel is set up on the device while the previous
// one is still running and its blocks start as the previous grid's blocks retire; they block in pdl_wait() until
// the previous grid has completed and its writes are visible.  Every kernel calls pdl_wait() before its first
// access to global memory, so the data flow is that of plain stream order; what is saved is the launch gap
// between kernels (measured: C3 build 742 -> 718 us, C2 280 -> 251 us, n = 65536: 144 -> 116 us).  The previous
// kernel does NOT trigger its dependents early (griddepcontrol.launch_dependents at block start): measured, that
// costs more than it gains on the large configs (C3 765 us), because waiting blocks of the next kernel then hold
// registers and shared memory the tail of the running one needs.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
// Small grids (the launch-bound regime: n up to a few 10^5) do trigger their dependents, right after their own wait:
// the next kernel's blocks then sit resident at their pdl_wait() while this grid runs, and start the moment it has
// completed, instead of being launched then.  A grid that fills the GPU does not (see above).
#ifndef BVH_PDL_TRIGGER_MAX_BLOCKS
#define BVH_PDL_TRIGGER_MAX_BLOCKS 296
#endif
__device__ __forceinline__ void pdl_trigger() {
  if (gridDim.x <= BVH_PDL_TRIGGER_MAX_BLOCKS) asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, Args&&... args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// ---- kernel launchers (each only enqueues on `stream` and returns the first launch error; a caller stops
// enqueueing at the first failure) ---------------------------------------------------------------------------
// K1: scene bounds.  is_box: prim is n*6 floats, else n*3.
cudaError_t launch_scene_bounds(const float* prim, int n, bool is_box, Header* header, cudaStream_t stream);
// K2: Morton codes + the digit histograms of every sort pass.
// passes / shift0: histograms of `passes` 8-bit digits from bit shift0 up.
cudaError_t launch_morton(const float* prim, int n, bool is_box, int morton_bits, const Header* header, void* codes,
                          uint32_t* hist, cudaStream_t stream, int passes, int shift0 = 0);
// K1 + K2 + K3 of a small build (n <= kSmallBuildMax) in one launch by one thread-block cluster (small_build.cu): writes the scene
// bounds into `header`, the sorted codes and the permutation where the one-sweep sort would leave them.  Needs no
// zero-initialised scratch.
#ifndef BVH_SMALL_BUILD_MAX
#define BVH_SMALL_BUILD_MAX 16384
#endif
constexpr int kSmallBuildMax = BVH_SMALL_BUILD_MAX;   // <= 16384: a cluster of 8 blocks x 256 threads x 8 pairs
static_assert(kSmallBuildMax <= 16384, "the pairs of a small build live in one cluster's registers and shared memory");
cudaError_t launch_small_front(const float* prim, int n, bool is_box, int morton_bits, Header* header, void* codes,
                               uint32_t* perm, cudaStream_t stream);
// K3: one-sweep LSD radix sort of (key, index) pairs, `passes` 8-bit digits from the least significant.
// Pass p reads keys[p&1]/vals[p&1] and writes the other buffer; with an even pass count the result is in
// keys[0]/vals[0].  final_vals (optional) receives the last pass's values instead of vals[...].
// hist: [passes][256] digit histograms (already counted); status: [passes][tiles][256] zeroed; tile_counters:
// [passes] zeroed.  pass_events: optional array of cudaEvent_t (as void*), entry p recorded after pass p.
struct SortBuffers {
  void* keys[2];
  uint32_t* vals[2];
  uint32_t* hist;
  uint32_t* status;
  uint32_t* tile_counters;
  uint32_t* final_vals;
};
SortBuffers sort_buffers(void* scratch, const ScratchLayout& L);
// shift0: first bit of pass 0's digit.  slot0: pass p uses histogram, status block and ticket slot0 + p.
cudaError_t launch_sort(const SortBuffers& B, int key_bytes, int passes, int n, cudaStream_t stream, void* const* pass_events,
                        int shift0 = 0, int slot0 = 0);
// The conditional second sort of a 63-bit build as one cooperative launch (radix_sort.cu).
cudaError_t launch_second_sort(const SortBuffers& B, int passes, int n, int slot0, uint32_t* hist, uint32_t* status,
                               const uint32_t* run_if, cudaStream_t stream);
// 63-bit codes sorted by their upper 32 bits: orders every run of equal upper bits by the lower 31 (tie_fixup.cu).
// tile_flag [tie_fixup_tiles(n)] zeroed, tile_list [tie_fixup_tiles(n)], list_count zeroed: the work list of long runs.
cudaError_t launch_tie_fixup(void* keys, uint32_t* vals, int n, uint32_t* tile_flag, uint32_t* tile_list, uint32_t* list_count,
                             uint32_t* fallback, cudaStream_t stream);
int tie_fixup_tiles(int64_t n);
// The query schedule is a locality heuristic (results do not depend on it), so the queries could be sorted by the upper
// 8 * kQueryOrderPasses bits of their 30-bit Morton code only (queries that share those bits stay in input order).
// Measured: three passes save 7-70 us of ordering and cost C3's traversal 2 %; two cost C4 / C5 6 %.  All four it is.
#ifndef BVH_QUERY_ORDER_PASSES
#define BVH_QUERY_ORDER_PASSES 4
#endif
constexpr int kQueryOrderPasses = BVH_QUERY_ORDER_PASSES;
constexpr int kQueryOrderShift = 30 - 8 * kQueryOrderPasses > 0 ? 30 - 8 * kQueryOrderPasses : 0;
// Morton codes (30-bit) of query centres in the frame of the root box + digit histograms: orders queries.
cudaError_t launch_query_morton(const float* queries, int q, int kind, const NodesHeader* frame, uint32_t* codes, uint32_t* hist,
                         cudaStream_t stream);
// K4+K5: leaf gather + modified Apetrei bottom-up pass (Algorithm 4 with boxes).
constexpr int kMaxHierLevels = 8;
cudaError_t launch_hierarchy(const float* prim, bool is_box, const void* sorted_codes, int key_bytes, const uint32_t* perm,
                      void* nodes, int n, const Header* header, int2* seg_items, int* seg_count, uint32_t* arrivals,
                      cudaStream_t stream);
int hierarchy_levels(int n, int segs[kMaxHierLevels]);   // windows per level, level 1 first; returns the level count
int hierarchy_total_segments(int n);
int hierarchy_seg_capacity();
int hierarchy_fan();          // level-1 windows per level-2 window
// NEXT-2 measurement variant (variants.cu): Karras' top-down hierarchy + Algorithm 2 + a separate box pass.
size_t variant_extra_bytes(int64_t n);
int launch_variant_karras(const float* prim, bool is_box, const void* sorted_codes, int key_bytes, const uint32_t* perm,
                          void* nodes, int n, const Header* header, void* extra, cudaStream_t stream);
// ... and the unmodified Algorithm 3 (Apetrei numbering, stored root) followed by a separate skip-connection pass.
int launch_variant_apetrei(const float* prim, bool is_box, const void* sorted_codes, int key_bytes, const uint32_t* perm,
                           void* nodes, int n, const Header* header, void* extra, cudaStream_t stream);
// ... and Algorithm 4 in the same plain form (one thread per leaf, global `store`): byte-identical `nodes`.
int launch_variant_alg4(const float* prim, bool is_box, const void* sorted_codes, int key_bytes, const uint32_t* perm,
                        void* nodes, int n, const Header* header, void* extra, cudaStream_t stream);
int launch_variant_apetrei_export(const void* nodes, void* extra, int n, int32_t* left, int32_t* right, int32_t* rope,
                                  float* aabb, int32_t* root, cudaStream_t stream);
// K6/K8: stackless traversal.  kind 0 = spheres (xyzr), 1 = boxes (minmax), 2 = rays (o.xyz, d.xyz, tmin, tmax).
// mode 0 = count (counts out), 1 = fill (offsets in, out = indices; only_over: only rows with counts[j] > cap),
// 2 = collect (out = rows of cap entries, counts out), 3 = reduce (counts = primitive with the smallest key, keys out;
// spheres and rays), 4 = any hit (counts = 0 / 1).
// order (optional): thread t serves query order[t] (results still land in row order[t]).
cudaError_t launch_traverse(const void* nodes, int n, const float* queries, int64_t q, int kind, int mode,
                            const uint32_t* order, int32_t* counts, const int64_t* offsets, int32_t* out, int64_t cap,
                            bool only_over, float* keys, cudaStream_t stream, int64_t out_limit = 0);
// limit != 0: `indices` holds `limit` entries (< 0: none); rows that would end past it are not copied (fill: out_limit, likewise).
cudaError_t launch_rows_to_csr(const int32_t* rows, int64_t cap, const int32_t* counts, const int64_t* offsets, int64_t q,
                               int32_t* indices, cudaStream_t stream, int64_t limit = 0);
// q <= scan_single_tile_items(): exclusive scan of the counts AND the copy of the rows, one launch.
cudaError_t launch_scan_rows_to_csr_small(const int32_t* rows, int64_t cap, const int32_t* counts, int64_t* offsets, int64_t q,
                                          int32_t* indices, cudaStream_t stream, int64_t limit = 0);
int scan_single_tile_items();
int sm_count();   // multiprocessors of the current device (cached per device)

// One-time set-up that belongs to a (kernel, device) pair -- the opt-in to more than 48 KB of dynamic shared memory, an
// occupancy query -- is remembered per DEVICE, not per process: a process may build on several GPUs, and what
// cudaFuncSetAttribute sets holds only for the device that was current.  A failed set-up is returned and NOT remembered (the
// next call tries again).  Devices beyond kMaxDevices, or an unknown current device, run the set-up on every call.
constexpr int kMaxDevices = 64;
inline int current_device() {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return -1;
  return dev;
}
struct PerDeviceOnce {
  std::atomic<int> value[kMaxDevices];   // 0 = not set up on that device yet; else what the set-up produced (non-zero)
};
// setup(int* value) -> cudaError_t; must leave *value != 0 on success.  Returns the cached / fresh value through *out.
template <typename F>
inline cudaError_t once_per_device(PerDeviceOnce& once, int* out, F&& setup) {
  const int dev = current_device();
  int v = dev >= 0 ? once.value[dev].load(std::memory_order_acquire) : 0;
  if (v == 0) {
    const cudaError_t e = setup(&v);
    if (e != cudaSuccess) return e;
    if (v == 0) return cudaErrorUnknown;
    if (dev >= 0) once.value[dev].store(v, std::memory_order_release);
  }
  if (out) *out = v;
  return cudaSuccess;
}
// K7: exclusive scan of int32 counts into int64 offsets[q+1].
size_t scan_scratch_bytes(int64_t q);
cudaError_t launch_scan(const int32_t* counts, int64_t q, int64_t* offsets, void* scratch, cudaStream_t stream);
// Parity export.
void launch_export(const void* nodes, const void* scratch, const ScratchLayout& L, int n, void* sorted_codes,
                   uint32_t* perm, int32_t* left_child, int32_t* rope, float* aabb, float* scene_bounds,
                   cudaStream_t stream);

}  // namespace bvh
