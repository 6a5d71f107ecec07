// capi.cu -- the C ABI declared in include/bvh_b200.h: argument checks, scratch layout, and the
// sequence of kernel launches of one build / one query pass.  No allocation, no synchronisation.
#include "../../include/bvh_b200.h"
#include "common.cuh"

namespace bvh {

static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

int sm_count() {
  static PerDeviceOnce once;
  int sms = 0;
  const cudaError_t e = once_per_device(once, &sms, [](int* v) {
    int dev = 0;
    cudaError_t err = cudaGetDevice(&dev);
    if (err == cudaSuccess) err = cudaDeviceGetAttribute(v, cudaDevAttrMultiProcessorCount, dev);
    if (err == cudaSuccess && *v <= 0) err = cudaErrorInvalidDevice;
    return err;
  });
  return e == cudaSuccess ? sms : kNumSMs;   // (a failed query is not remembered)
}

#ifndef BVH_TWO_STAGE_SORT
#define BVH_TWO_STAGE_SORT 1
#endif
constexpr bool kTwoStageSort = BVH_TWO_STAGE_SORT != 0;

ScratchLayout scratch_layout(int64_t n, int morton_bits) {
  ScratchLayout L{};
  L.key_bytes = (morton_bits == 30) ? 4 : 8;
  L.passes = (morton_bits == 30) ? 4 : 8;
  // 63-bit codes, two-stage sort: the four upper-bit passes use zeroed slots; the eight slots of the conditional second
  // sort sit past the end (hist2 / status2) and are cleared by that sort itself, only when it runs
  const bool second_sort = morton_bits == 63 && kTwoStageSort;
  L.slots = (morton_bits == 30 || second_sort) ? 4 : 8;
  const int tile = sort_tile_items(L.key_bytes);
  L.tiles = (int)((n + tile - 1) / tile);
  if (L.tiles < 1) L.tiles = 1;
  size_t off = 0;
  L.header = off;
  off += sizeof(Header);
  L.hist = off;
  off += align_up((size_t)L.slots * 256 * sizeof(uint32_t), 256);
  L.status = off;
  off += align_up((size_t)L.slots * L.tiles * 256 * sizeof(uint32_t), 256);
  const size_t nn = (size_t)(n > 0 ? n : 1);
  L.segments = hierarchy_total_segments((int)nn);
  L.arrivals = off;
  off += align_up((size_t)L.segments * sizeof(uint32_t), 256);
  L.fix_flag = off;
  if (morton_bits == 63) off += align_up((size_t)tie_fixup_tiles((int64_t)nn) * sizeof(uint32_t), 256);
  L.zero_bytes = off;
  for (int b = 0; b < 2; ++b) {
    L.keys[b] = off;
    off += align_up(nn * L.key_bytes, 256);
  }
  for (int b = 0; b < 2; ++b) {
    L.vals[b] = off;
    off += align_up(nn * sizeof(uint32_t), 256);
  }
  L.seg_items = off;
  off += align_up((size_t)L.segments * hierarchy_seg_capacity() * sizeof(int2), 256);
  L.seg_count = off;
  off += align_up((size_t)L.segments * sizeof(int32_t), 256);
  L.fix_list = off;
  if (morton_bits == 63) off += align_up((size_t)tie_fixup_tiles((int64_t)nn) * sizeof(uint32_t), 256);
  L.hist2 = L.status2 = off;
  if (second_sort) {
    off += align_up((size_t)8 * 256 * sizeof(uint32_t), 256);
    L.status2 = off;
    off += align_up((size_t)8 * L.tiles * 256 * sizeof(uint32_t), 256);
  }
  L.total = off;
  return L;
}

// ---- parity export ------------------------------------------------------------------------------------
// The canonical arrays of the unified index space (G8) from the internal records and the leaf records.
template <typename KeyT>
__global__ void export_kernel(const char* __restrict__ nodes, const KeyT* __restrict__ keys,
                              const uint32_t* __restrict__ vals, const Header* __restrict__ header, int n,
                              KeyT* sorted_codes, uint32_t* perm, int32_t* left_child, int32_t* rope, float* aabb,
                              float* scene_bounds) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t total = 2 * (int64_t)n - 1;
  const int leaf_base = n - 1;
  if (i < n) {
    if (sorted_codes) sorted_codes[i] = keys[i];
    if (perm) perm[i] = vals[i];
  }
  if (i < total) {
    float lo[3], hi[3];
    int left, rp;
    if (i < leaf_base) {
      const Node* rec = reinterpret_cast<const Node*>(nodes + kNodesHeaderBytes) + i;
      const float4 a = rec->lo, b = rec->hi;
      lo[0] = a.x; lo[1] = a.y; lo[2] = a.z; hi[0] = b.x; hi[1] = b.y; hi[2] = b.z;
      left = __float_as_int(a.w);
      rp = __float_as_int(b.w);
    } else {
      const int li = (int)(i - leaf_base);
      const char* leaves = nodes + leaf_offset_bytes(n);
      uint32_t payload;
      if (reinterpret_cast<const NodesHeader*>(nodes)->leaf_kind == kLeafPoints) {
        const float4 v = reinterpret_cast<const float4*>(leaves)[li];
        lo[0] = hi[0] = v.x; lo[1] = hi[1] = v.y; lo[2] = hi[2] = v.z;
        payload = __float_as_uint(v.w);
      } else {
        const Node* rec = reinterpret_cast<const Node*>(leaves) + li;
        const float4 a = rec->lo, b = rec->hi;
        lo[0] = a.x; lo[1] = a.y; lo[2] = a.z; hi[0] = b.x; hi[1] = b.y; hi[2] = b.z;
        payload = __float_as_uint(a.w);
      }
      left = (int)(payload & kLeafPrimMask);
      rp = (li == n - 1) ? kSentinel : ((payload & kLeafRopeInternal) ? li + 1 : leaf_base + li + 1);
    }
    if (left_child) left_child[i] = left;
    if (rope) rope[i] = rp;
    if (aabb) {
      float* o = aabb + 6 * i;
      o[0] = lo[0]; o[1] = lo[1]; o[2] = lo[2]; o[3] = hi[0]; o[4] = hi[1]; o[5] = hi[2];
    }
  }
  if (i == 0 && scene_bounds) {
    float s[6];
    load_scene_bounds(header, s);
    for (int a = 0; a < 6; ++a) scene_bounds[a] = s[a];
  }
}

void launch_export(const void* nodes_, const void* scratch, const ScratchLayout& L, int n, void* sorted_codes,
                   uint32_t* perm, int32_t* left_child, int32_t* rope, float* aabb, float* scene_bounds,
                   cudaStream_t stream) {
  const char* nodes = static_cast<const char*>(nodes_);
  const char* base = static_cast<const char*>(scratch);
  const Header* header = reinterpret_cast<const Header*>(base + L.header);
  const uint32_t* vals = reinterpret_cast<const uint32_t*>(base + L.vals[0]);
  const int64_t total = 2 * (int64_t)n - 1;
  const unsigned g = (unsigned)((total + 255) / 256);
  if (L.key_bytes == 4)
    export_kernel<uint32_t><<<g, 256, 0, stream>>>(nodes, reinterpret_cast<const uint32_t*>(base + L.keys[0]), vals,
                                                   header, n, (uint32_t*)sorted_codes, perm, left_child, rope, aabb,
                                                   scene_bounds);
  else
    export_kernel<uint64_t><<<g, 256, 0, stream>>>(nodes, reinterpret_cast<const uint64_t*>(base + L.keys[0]), vals,
                                                   header, n, (uint64_t*)sorted_codes, perm, left_child, rope, aabb,
                                                   scene_bounds);
}

__global__ void zero_counts_kernel(int32_t* counts, int64_t q) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < q) counts[i] = 0;
}

static inline bool misaligned(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }

static int check_launch() { return cudaGetLastError() == cudaSuccess ? BVH_OK : BVH_ERR_CUDA; }

static int build(const float* prim, bool is_box, int64_t n, int morton_bits, void* nodes, void* scratch,
                 size_t scratch_bytes, void* stream_, void* const* events = nullptr, int variant = 0) {
  if (n < 0) return BVH_ERR_INVALID_ARGUMENT;
  if (morton_bits != 30 && morton_bits != 63) return BVH_ERR_MORTON_BITS;
  if (n >= ((int64_t)1 << 30)) return BVH_ERR_TOO_LARGE;
  if (n == 0) return BVH_OK;
  if (!prim || !nodes || !scratch) return BVH_ERR_INVALID_ARGUMENT;
  if (misaligned(prim) || misaligned(nodes) || misaligned(scratch)) return BVH_ERR_INVALID_ARGUMENT;
  if ((reinterpret_cast<uintptr_t>(nodes) & 31u) != 0) return BVH_ERR_INVALID_ARGUMENT;
  const ScratchLayout L = scratch_layout(n, morton_bits);
  if (variant < 0 || variant > 3) return BVH_ERR_INVALID_ARGUMENT;
  if (scratch_bytes < L.total + (variant != 0 ? variant_extra_bytes(n) : 0)) return BVH_ERR_SCRATCH;
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  char* base = static_cast<char*>(scratch);
  Header* header = reinterpret_cast<Header*>(base + L.header);
  uint32_t* hist = reinterpret_cast<uint32_t*>(base + L.hist);

  auto mark = [&](int k) {
    if (events && events[k]) cudaEventRecord(static_cast<cudaEvent_t>(events[k]), stream);
  };
  mark(0);
  // A small build: bounds, codes and sort in one launch by one block (small_build.cu); nothing of the scratch needs
  // zeroing then (no histograms, no tile status, and with at most kMergeFan level-1 windows no arrival counter).
  if (variant == 0 && n <= kSmallBuildMax && hierarchy_total_segments((int)n) <= hierarchy_fan() + 1) {
    if (launch_small_front(prim, (int)n, is_box, morton_bits, header, base + L.keys[0],
                           reinterpret_cast<uint32_t*>(base + L.vals[0]), stream) != cudaSuccess)
      return BVH_ERR_CUDA;
    mark(3 + L.passes);    // one launch: only the end of the front is marked (an event per stage would cost more than the stage)
  } else {
    if (cudaMemsetAsync(base, 0, L.zero_bytes, stream) != cudaSuccess) return BVH_ERR_CUDA;
    mark(1);
    if (launch_scene_bounds(prim, (int)n, is_box, header, stream) != cudaSuccess) return BVH_ERR_CUDA;
    mark(2);
    if (morton_bits == 30 || !kTwoStageSort) {
      if (launch_morton(prim, (int)n, is_box, morton_bits, header, base + L.keys[0], hist, stream, L.passes) != cudaSuccess) return BVH_ERR_CUDA;
      mark(3);
      if (launch_sort(sort_buffers(scratch, L), L.key_bytes, L.passes, (int)n, stream, events ? events + 4 : nullptr) != cudaSuccess)
        return BVH_ERR_CUDA;
    } else {
      // 63-bit codes (tie_fixup.cu): four passes over the upper 32 bits, then every run of equal upper bits ordered by the
      // lower 31 in shared memory.  Should a run not fit a block, the fix-up raises header->sort_fallback and eight more
      // passes over all 63 bits redo the order; they are one cooperative launch, enqueued in any case (nothing here may
      // read the flag back), that returns at once while the flag is clear.
      const SortBuffers B = sort_buffers(scratch, L);
      if (launch_morton(prim, (int)n, is_box, morton_bits, header, base + L.keys[0], hist, stream, 4, 31) != cudaSuccess) return BVH_ERR_CUDA;
      mark(3);
      if (launch_sort(B, L.key_bytes, 4, (int)n, stream, events ? events + 4 : nullptr, 31, 0) != cudaSuccess) return BVH_ERR_CUDA;
      if (launch_tie_fixup(base + L.keys[0], B.vals[0], (int)n, reinterpret_cast<uint32_t*>(base + L.fix_flag),
                           reinterpret_cast<uint32_t*>(base + L.fix_list), &header->fix_count, &header->sort_fallback,
                           stream) != cudaSuccess)
        return BVH_ERR_CUDA;
      mark(8);
      if (launch_second_sort(B, 8, (int)n, 4, reinterpret_cast<uint32_t*>(base + L.hist2), reinterpret_cast<uint32_t*>(base + L.status2),
                             &header->sort_fallback, stream) != cudaSuccess) return BVH_ERR_CUDA;
      mark(9);
      mark(10);
      mark(11);
    }
  }
  if (variant == 1) {
    if (launch_variant_karras(prim, is_box, base + L.keys[0], L.key_bytes, reinterpret_cast<const uint32_t*>(base + L.vals[0]),
                              nodes, (int)n, header, base + L.total, stream) != 0)
      return BVH_ERR_CUDA;
    mark(12);
    return check_launch();
  }
  if (variant == 2) {
    if (launch_variant_apetrei(prim, is_box, base + L.keys[0], L.key_bytes, reinterpret_cast<const uint32_t*>(base + L.vals[0]),
                               nodes, (int)n, header, base + L.total, stream) != 0)
      return BVH_ERR_CUDA;
    mark(12);
    return check_launch();
  }
  if (variant == 3) {
    if (launch_variant_alg4(prim, is_box, base + L.keys[0], L.key_bytes, reinterpret_cast<const uint32_t*>(base + L.vals[0]),
                            nodes, (int)n, header, base + L.total, stream) != 0)
      return BVH_ERR_CUDA;
    mark(12);
    return check_launch();
  }
  if (launch_hierarchy(prim, is_box, base + L.keys[0], L.key_bytes, reinterpret_cast<const uint32_t*>(base + L.vals[0]),
                       nodes, (int)n, header, reinterpret_cast<int2*>(base + L.seg_items), reinterpret_cast<int*>(base + L.seg_count),
                       reinterpret_cast<uint32_t*>(base + L.arrivals), stream) != cudaSuccess)
    return BVH_ERR_CUDA;
  mark(12);
  return check_launch();
}

static inline bool misaligned32(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 31u) != 0; }

// mode: kModeCount / kModeFill / kModeCollect of traverse.cu (0 / 1 / 2).  cap: collect: entries per row; fill with
// only_over: rows with counts[j] > cap.  Whether `nodes` holds a finished hierarchy over n primitives is checked on the
// device (NodesHeader), since the library may not synchronise: a stale buffer yields counts of 0 and no stores.
__global__ void fill_reduce_none_kernel(int32_t* index, float* keys, int64_t q) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < q) {
    index[i] = -1;
    keys[i] = __int_as_float(0x7f800000);
  }
}

static int query(const void* nodes, int64_t n, const float* queries, int64_t q, int kind, int mode,
                 const uint32_t* order, int32_t* counts, const int64_t* offsets, int32_t* out, int64_t cap, bool only_over,
                 void* stream_, float* keys = nullptr, int64_t out_limit = 0) {
  if (n < 0 || q < 0) return BVH_ERR_INVALID_ARGUMENT;
  if (n >= ((int64_t)1 << 30)) return BVH_ERR_TOO_LARGE;
  if (kind < 0 || kind > 2) return BVH_ERR_INVALID_ARGUMENT;
  if (q == 0) return BVH_OK;
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  if (mode == 1) {
    if (!offsets || (only_over && !counts)) return BVH_ERR_INVALID_ARGUMENT;
  } else {
    if (!counts) return BVH_ERR_INVALID_ARGUMENT;
  }
  if (mode == 2 && (cap < 8 || cap % 8 != 0 || cap > 0x7fffffff || !out || misaligned32(out))) return BVH_ERR_INVALID_ARGUMENT;
  if (mode == 3 && (!keys || kind == 1)) return BVH_ERR_INVALID_ARGUMENT;
  if (n == 0) {
    if (mode == 3) {
      fill_reduce_none_kernel<<<(unsigned)((q + 255) / 256), 256, 0, stream>>>(counts, keys, q);
      return check_launch();
    }
    if (mode != 1) {
      zero_counts_kernel<<<(unsigned)((q + 255) / 256), 256, 0, stream>>>(counts, q);
      return check_launch();
    }
    return BVH_OK;
  }
  // node records are read with 256-bit loads: 32-byte alignment
  if (!nodes || !queries || misaligned32(nodes) || misaligned(queries)) return BVH_ERR_INVALID_ARGUMENT;
  if (mode == 1 && !out) return BVH_ERR_INVALID_ARGUMENT;  // nnz = 0 callers still pass a valid pointer
  if (launch_traverse(nodes, (int)n, queries, q, kind, mode, order, counts, offsets, out, cap, only_over, keys, stream,
                      out_limit) != cudaSuccess)
    return BVH_ERR_CUDA;
  return BVH_OK;
}

#ifndef BVH_SMALL_ORDER_Q
#define BVH_SMALL_ORDER_Q 8192
#endif
constexpr int64_t kSmallOrderQ = BVH_SMALL_ORDER_Q;

__global__ void iota_kernel(uint32_t* order, int64_t q) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < q) order[i] = (uint32_t)i;
}

// Query order: 30-bit Morton code of each query centre in the frame of the root box, then the same
// one-sweep sort as the build; `order` receives the permutation (query index at each Morton position).
static int query_order(const void* nodes, int64_t n, const float* queries, int64_t q, int kind, uint32_t* order,
                       void* scratch, size_t scratch_bytes, void* stream_) {
  if (n < 0 || q < 0) return BVH_ERR_INVALID_ARGUMENT;
  if (n >= ((int64_t)1 << 30) || q >= ((int64_t)1 << 30)) return BVH_ERR_TOO_LARGE;
  if (q == 0) return BVH_OK;
  if (!order) return BVH_ERR_INVALID_ARGUMENT;
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  // no frame (n = 0), or a batch so small that it is bound by the number of dependent launches and gains nothing from
  // a schedule (the whole hierarchy it touches stays in L2): identity, one launch instead of five
  if (n == 0 || q <= kSmallOrderQ) {
    iota_kernel<<<(unsigned)((q + 255) / 256), 256, 0, stream>>>(order, q);
    return check_launch();
  }
  if (!nodes || !queries || !scratch || misaligned(nodes) || misaligned(queries) || misaligned(scratch))
    return BVH_ERR_INVALID_ARGUMENT;
  const ScratchLayout L = scratch_layout(q, 30);
  if (scratch_bytes < L.total) return BVH_ERR_SCRATCH;
  char* base = static_cast<char*>(scratch);
  if (cudaMemsetAsync(base, 0, L.zero_bytes, stream) != cudaSuccess) return BVH_ERR_CUDA;
  SortBuffers B = sort_buffers(scratch, L);
  if (launch_query_morton(queries, (int)q, kind, static_cast<const NodesHeader*>(nodes), static_cast<uint32_t*>(B.keys[0]),
                          B.hist, stream) != cudaSuccess)
    return BVH_ERR_CUDA;
  B.final_vals = order;
  if (launch_sort(B, 4, kQueryOrderPasses, (int)q, stream, nullptr, kQueryOrderShift, 0) != cudaSuccess) return BVH_ERR_CUDA;
  return check_launch();
}

}  // namespace bvh

extern "C" {

int bvh_version(void) { return 1; }

int bvh_sizes(int64_t n, int morton_bits, size_t* node_bytes, size_t* scratch_bytes) {
  if (n < 0 || !node_bytes || !scratch_bytes) return BVH_ERR_INVALID_ARGUMENT;
  if (morton_bits != 30 && morton_bits != 63) return BVH_ERR_MORTON_BITS;
  if (n >= ((int64_t)1 << 30)) return BVH_ERR_TOO_LARGE;
  // header + internal records + leaf records at their larger (box) size: one size for both leaf formats
  *node_bytes = bvh::leaf_offset_bytes(n) + sizeof(bvh::Node) * (size_t)(n > 0 ? n : 1);
  *scratch_bytes = bvh::scratch_layout(n, morton_bits).total;
  return BVH_OK;
}

int bvh_build_points(const float* xyz, int64_t n, int morton_bits, void* nodes, void* scratch, size_t scratch_bytes,
                     void* stream) {
  return bvh::build(xyz, false, n, morton_bits, nodes, scratch, scratch_bytes, stream);
}

int bvh_build_boxes(const float* minmax, int64_t n, int morton_bits, void* nodes, void* scratch, size_t scratch_bytes,
                    void* stream) {
  return bvh::build(minmax, true, n, morton_bits, nodes, scratch, scratch_bytes, stream);
}

int bvh_build_staged(const float* prim, int prim_is_box, int64_t n, int morton_bits, void* nodes, void* scratch,
                     size_t scratch_bytes, void* stream, void* const* stage_events) {
  return bvh::build(prim, prim_is_box != 0, n, morton_bits, nodes, scratch, scratch_bytes, stream, stage_events);
}

int bvh_variant_sizes(int64_t n, int morton_bits, int variant, size_t* scratch_bytes) {
  if (n < 0 || !scratch_bytes || variant < 1 || variant > 3) return BVH_ERR_INVALID_ARGUMENT;
  if (morton_bits != 30 && morton_bits != 63) return BVH_ERR_MORTON_BITS;
  if (n >= ((int64_t)1 << 30)) return BVH_ERR_TOO_LARGE;
  *scratch_bytes = bvh::scratch_layout(n, morton_bits).total + bvh::variant_extra_bytes(n);
  return BVH_OK;
}

int bvh_build_variant(const float* prim, int prim_is_box, int64_t n, int morton_bits, void* nodes, void* scratch,
                      size_t scratch_bytes, int variant, void* stream, void* const* stage_events) {
  return bvh::build(prim, prim_is_box != 0, n, morton_bits, nodes, scratch, scratch_bytes, stream, stage_events, variant);
}

int bvh_variant_export(const void* nodes, void* scratch, int64_t n, int morton_bits, int variant, int32_t* left,
                       int32_t* right, int32_t* rope, float* aabb, int32_t* root, void* stream) {
  if (n < 0 || variant != 2) return BVH_ERR_INVALID_ARGUMENT;
  if (morton_bits != 30 && morton_bits != 63) return BVH_ERR_MORTON_BITS;
  if (n >= ((int64_t)1 << 30)) return BVH_ERR_TOO_LARGE;
  if (n == 0) return BVH_OK;
  if (!nodes || !scratch) return BVH_ERR_INVALID_ARGUMENT;
  const bvh::ScratchLayout L = bvh::scratch_layout(n, morton_bits);
  if (bvh::launch_variant_apetrei_export(nodes, static_cast<char*>(scratch) + L.total, (int)n, left, right, rope, aabb, root,
                                         static_cast<cudaStream_t>(stream)) != 0)
    return BVH_ERR_CUDA;
  return BVH_OK;
}

int bvh_query_order_sizes(int64_t q, size_t* scratch_bytes) {
  if (q < 0 || !scratch_bytes) return BVH_ERR_INVALID_ARGUMENT;
  if (q >= ((int64_t)1 << 30)) return BVH_ERR_TOO_LARGE;
  *scratch_bytes = bvh::scratch_layout(q, 30).total;
  return BVH_OK;
}

int bvh_query_order_spheres(const void* nodes, int64_t n, const float* xyzr, int64_t q, uint32_t* order, void* scratch,
                            size_t scratch_bytes, void* stream) {
  return bvh::query_order(nodes, n, xyzr, q, 0, order, scratch, scratch_bytes, stream);
}

int bvh_query_order_boxes(const void* nodes, int64_t n, const float* minmax, int64_t q, uint32_t* order, void* scratch,
                          size_t scratch_bytes, void* stream) {
  return bvh::query_order(nodes, n, minmax, q, 1, order, scratch, scratch_bytes, stream);
}

int bvh_query_order_rays(const void* nodes, int64_t n, const float* rays, int64_t q, uint32_t* order, void* scratch,
                         size_t scratch_bytes, void* stream) {
  return bvh::query_order(nodes, n, rays, q, 2, order, scratch, scratch_bytes, stream);
}

int bvh_query_rays_count(const void* nodes, int64_t n, const float* rays, int64_t q, const uint32_t* order,
                         int32_t* counts, void* stream) {
  return bvh::query(nodes, n, rays, q, 2, 0, order, counts, nullptr, nullptr, 0, false, stream);
}

int bvh_query_rays_fill(const void* nodes, int64_t n, const float* rays, int64_t q, const uint32_t* order,
                        const int64_t* offsets, int32_t* indices, void* stream) {
  return bvh::query(nodes, n, rays, q, 2, 1, order, nullptr, offsets, indices, 0, false, stream);
}

int bvh_query_spheres_count(const void* nodes, int64_t n, const float* xyzr, int64_t q, const uint32_t* order,
                            int32_t* counts, void* stream) {
  return bvh::query(nodes, n, xyzr, q, 0, 0, order, counts, nullptr, nullptr, 0, false, stream);
}

int bvh_query_boxes_count(const void* nodes, int64_t n, const float* minmax, int64_t q, const uint32_t* order,
                          int32_t* counts, void* stream) {
  return bvh::query(nodes, n, minmax, q, 1, 0, order, counts, nullptr, nullptr, 0, false, stream);
}

int bvh_scan_sizes(int64_t q, size_t* scratch_bytes) {
  if (q < 0 || !scratch_bytes) return BVH_ERR_INVALID_ARGUMENT;
  *scratch_bytes = bvh::scan_scratch_bytes(q);
  return BVH_OK;
}

int bvh_scan_counts(const int32_t* counts, int64_t q, int64_t* offsets, void* scratch, size_t scratch_bytes,
                    void* stream) {
  if (q < 0 || !offsets) return BVH_ERR_INVALID_ARGUMENT;
  if (q > 0 && (!counts || !scratch)) return BVH_ERR_INVALID_ARGUMENT;
  if (q > 0 && scratch_bytes < bvh::scan_scratch_bytes(q)) return BVH_ERR_SCRATCH;
  if (bvh::launch_scan(counts, q, offsets, scratch, static_cast<cudaStream_t>(stream)) != cudaSuccess) return BVH_ERR_CUDA;
  return BVH_OK;
}

int bvh_query_spheres_fill(const void* nodes, int64_t n, const float* xyzr, int64_t q, const uint32_t* order,
                           const int64_t* offsets, int32_t* indices, void* stream) {
  return bvh::query(nodes, n, xyzr, q, 0, 1, order, nullptr, offsets, indices, 0, false, stream);
}

int bvh_query_boxes_fill(const void* nodes, int64_t n, const float* minmax, int64_t q, const uint32_t* order,
                         const int64_t* offsets, int32_t* indices, void* stream) {
  return bvh::query(nodes, n, minmax, q, 1, 1, order, nullptr, offsets, indices, 0, false, stream);
}

int bvh_query_spheres_nearest(const void* nodes, int64_t n, const float* xyzr, int64_t q, const uint32_t* order,
                              int32_t* index, float* d2, void* stream) {
  return bvh::query(nodes, n, xyzr, q, 0, 3, order, index, nullptr, nullptr, 0, false, stream, d2);
}

int bvh_query_rays_first_hit(const void* nodes, int64_t n, const float* rays, int64_t q, const uint32_t* order,
                             int32_t* index, float* t, void* stream) {
  return bvh::query(nodes, n, rays, q, 2, 3, order, index, nullptr, nullptr, 0, false, stream, t);
}

int bvh_query_any_hit(const void* nodes, int64_t n, const float* queries, int query_kind, int64_t q, const uint32_t* order,
                      int32_t* hit, void* stream) {
  return bvh::query(nodes, n, queries, q, query_kind, 4, order, hit, nullptr, nullptr, 0, false, stream);
}

int bvh_query_collect(const void* nodes, int64_t n, const float* queries, int query_kind, int64_t q, const uint32_t* order,
                      int64_t cap, int32_t* rows, int32_t* counts, void* stream) {
  return bvh::query(nodes, n, queries, q, query_kind, 2, order, counts, nullptr, rows, cap, false, stream);
}

int bvh_rows_to_csr(const int32_t* rows, int64_t cap, const int32_t* counts, const int64_t* offsets, int64_t q,
                    int32_t* indices, void* stream) {
  if (q < 0 || cap < 8 || cap % 8 != 0) return BVH_ERR_INVALID_ARGUMENT;
  if (q == 0) return BVH_OK;
  if (!rows || !counts || !offsets || !indices) return BVH_ERR_INVALID_ARGUMENT;
  if (bvh::launch_rows_to_csr(rows, cap, counts, offsets, q, indices, static_cast<cudaStream_t>(stream)) != cudaSuccess)
    return BVH_ERR_CUDA;
  return BVH_OK;
}

int bvh_query_fill_overflow(const void* nodes, int64_t n, const float* queries, int query_kind, int64_t q,
                            const uint32_t* order, int64_t cap, const int32_t* counts, const int64_t* offsets,
                            int32_t* indices, void* stream) {
  if (cap < 0) return BVH_ERR_INVALID_ARGUMENT;
  return bvh::query(nodes, n, queries, q, query_kind, 1, order, const_cast<int32_t*>(counts), offsets, indices, cap, true, stream);
}

int bvh_query_csr_sizes(int64_t q, size_t* scratch_bytes) {
  if (q < 0 || !scratch_bytes) return BVH_ERR_INVALID_ARGUMENT;
  if (q >= ((int64_t)1 << 30)) return BVH_ERR_TOO_LARGE;
  // the ordering's scratch is dead once `order` is written: the scan reuses its first bytes
  const size_t a = q > bvh::kSmallOrderQ ? bvh::scratch_layout(q, 30).total : 0, b = bvh::scan_scratch_bytes(q);
  *scratch_bytes = a > b ? a : b;
  return BVH_OK;
}

int bvh_query_csr(const void* nodes, int64_t n, const float* queries, int query_kind, int64_t q, int64_t cap,
                  int32_t* rows, uint32_t* order, int32_t* counts, int64_t* offsets, int32_t* indices,
                  int64_t indices_capacity, void* scratch, size_t scratch_bytes, void* stream) {
  if (n < 0 || q < 0 || query_kind < 0 || query_kind > 2 || indices_capacity < 0) return BVH_ERR_INVALID_ARGUMENT;
  if (n >= ((int64_t)1 << 30) || q >= ((int64_t)1 << 30)) return BVH_ERR_TOO_LARGE;
  if (cap < 8 || cap % 8 != 0 || cap > 0x7fffffff) return BVH_ERR_INVALID_ARGUMENT;
  if (!offsets) return BVH_ERR_INVALID_ARGUMENT;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  if (q == 0) return bvh::launch_scan(nullptr, 0, offsets, nullptr, s) == cudaSuccess ? BVH_OK : BVH_ERR_CUDA;
  size_t need = 0;
  bvh_query_csr_sizes(q, &need);
  if (!rows || !counts || !indices || !scratch || bvh::misaligned32(rows) || bvh::misaligned(scratch)) return BVH_ERR_INVALID_ARGUMENT;
  if (scratch_bytes < need) return BVH_ERR_SCRATCH;
  if (n > 0 && (!nodes || !queries || bvh::misaligned32(nodes) || bvh::misaligned(queries))) return BVH_ERR_INVALID_ARGUMENT;
  const int64_t limit = indices_capacity > 0 ? indices_capacity : -1;   // -1: nothing fits (0 means "no limit" inside)
  const uint32_t* ord = nullptr;
  int rc;
  if (n > 0 && q > bvh::kSmallOrderQ) {     // small batches are served in input order (bvh_query_order_* would write the identity)
    if (!order) return BVH_ERR_INVALID_ARGUMENT;
    if ((rc = bvh::query_order(nodes, n, queries, q, query_kind, order, scratch, scratch_bytes, stream)) != BVH_OK) return rc;
    ord = order;
  }
  if ((rc = bvh::query(nodes, n, queries, q, query_kind, 2, ord, counts, nullptr, rows, cap, false, stream)) != BVH_OK) return rc;
  if (q <= bvh::scan_single_tile_items()) {
    if (bvh::launch_scan_rows_to_csr_small(rows, cap, counts, offsets, q, indices, s, limit) != cudaSuccess) return BVH_ERR_CUDA;
  } else {
    if (bvh::launch_scan(counts, q, offsets, scratch, s) != cudaSuccess) return BVH_ERR_CUDA;
    if (bvh::launch_rows_to_csr(rows, cap, counts, offsets, q, indices, s, limit) != cudaSuccess) return BVH_ERR_CUDA;
  }
  if (n == 0) return BVH_OK;
  return bvh::query(nodes, n, queries, q, query_kind, 1, ord, counts, offsets, indices, cap, true, stream, nullptr, limit);
}

int bvh_export(const void* nodes, const void* scratch, int64_t n, int morton_bits, void* sorted_codes, uint32_t* perm,
               int32_t* left_child, int32_t* rope, float* aabb, float* scene_bounds, void* stream) {
  if (n < 0) return BVH_ERR_INVALID_ARGUMENT;
  if (morton_bits != 30 && morton_bits != 63) return BVH_ERR_MORTON_BITS;
  if (n >= ((int64_t)1 << 30)) return BVH_ERR_TOO_LARGE;
  if (n == 0) return BVH_OK;
  if (!nodes || !scratch) return BVH_ERR_INVALID_ARGUMENT;
  const bvh::ScratchLayout L = bvh::scratch_layout(n, morton_bits);
  bvh::launch_export(nodes, scratch, L, (int)n, sorted_codes, perm, left_child, rope,
                     aabb, scene_bounds, static_cast<cudaStream_t>(stream));
  return bvh::check_launch();
}

}  // extern "C"
