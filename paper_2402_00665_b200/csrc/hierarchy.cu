// hierarchy.cu -- K4 + K5: the paper's Algorithm 4, "Modified Apetrei's algorithm
// with skip installation", with the bounding boxes the pseudo-code omits (reading G10), fused with the
// permuted leaf gather.  One thread per leaf climbs towards the root; at every parent the first of
// the two children to arrive stops, the second carries on (ATOMICCAS on `store`),
// so each internal node is written by exactly one thread, which by then knows the node's full range,
// hence its Karras index q, its left child (split = Apetrei index p)
// and its skip-connection (Algorithm 2).
//
// Line references "L#" are the pseudo-code line numbers of Algorithm 4 in the paper.
#include "common.cuh"

namespace bvh {

#ifndef BVH_HIER_THREADS
#define BVH_HIER_THREADS 512
#endif
constexpr int kHierThreads = BVH_HIER_THREADS;  // leaves per block = size of the shared-memory phase

// delta*(i): XOR of adjacent sorted codes; equal codes fall back to the XOR of the
// sorted positions (augmented key, readings G1/G5); +infinity outside [0, n-2].  The
// value is packed so that one unsigned compare orders it (G14): position band < code band < infinity.
template <typename KeyT>
struct Delta;
template <>
struct Delta<uint32_t> {
  using T = uint32_t;
  static constexpr T kInf = 0xFFFFFFFFu;
  __device__ static __forceinline__ T make(uint32_t a, uint32_t b, int i) {
    const uint32_t x = a ^ b;                              // < 2^30
    return x ? (x + 0x40000000u) : (uint32_t)(i ^ (i + 1));  // positions < 2^30
  }
};
template <>
struct Delta<uint64_t> {
  using T = uint64_t;
  static constexpr T kInf = 0xFFFFFFFFFFFFFFFFull;
  __device__ static __forceinline__ T make(uint64_t a, uint64_t b, int i) {
    const uint64_t x = a ^ b;                              // <= 2^63 - 1
    return x ? (x + 0x7FFFFFFFFFFFFFFFull) : (uint64_t)(uint32_t)(i ^ (i + 1));
  }
};

template <typename KeyT>
__device__ __forceinline__ typename Delta<KeyT>::T delta_star(const KeyT* __restrict__ codes, int i, int n) {
  if (i < 0 || i >= n - 1) return Delta<KeyT>::kInf;
  return Delta<KeyT>::make(codes[i], codes[i + 1], i);
}

__device__ __forceinline__ void store_node(Node* nodes, int idx, const float lo[3], const float hi[3], int left, int rope) {
  // one 256-bit store = one full 32-byte sector (STG.E.ENL2.256, sm_100)
  asm volatile("st.global.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(nodes + idx), "f"(lo[0]), "f"(lo[1]), "f"(lo[2]),
               "f"(__int_as_float(left)), "f"(hi[0]), "f"(hi[1]), "f"(hi[2]), "f"(__int_as_float(rope))
               : "memory");
}

// Leaf record i (layout in common.cuh): a point leaf stores the point once.
template <bool IS_BOX>
__device__ __forceinline__ void store_leaf(char* leaves, int i, const float lo[3], const float hi[3], uint32_t payload) {
  if (IS_BOX)
    store_node(reinterpret_cast<Node*>(leaves), i, lo, hi, (int)payload, 0);
  else
    reinterpret_cast<float4*>(leaves)[i] = make_float4(lo[0], lo[1], lo[2], __uint_as_float(payload));
}

// Box of node `idx` of the unified index space, through L2 (written by another block or an earlier kernel).
__device__ __forceinline__ void load_box_cg(const char* nodes, int n, int leaf_kind, int idx, float lo[3], float hi[3]) {
  const int leaf_base = n - 1;
  if (idx >= leaf_base && leaf_kind == kLeafPoints) {
    const float4 v = __ldcg(reinterpret_cast<const float4*>(nodes + leaf_offset_bytes(n)) + (idx - leaf_base));
    lo[0] = hi[0] = v.x; lo[1] = hi[1] = v.y; lo[2] = hi[2] = v.z;
  } else {
    const Node* rec = (idx >= leaf_base) ? reinterpret_cast<const Node*>(nodes + leaf_offset_bytes(n)) + (idx - leaf_base)
                                         : reinterpret_cast<const Node*>(nodes + kNodesHeaderBytes) + idx;
    const float4 a = __ldcg(reinterpret_cast<const float4*>(rec));
    const float4 b = __ldcg(reinterpret_cast<const float4*>(rec) + 1);
    lo[0] = a.x; lo[1] = a.y; lo[2] = a.z; hi[0] = b.x; hi[1] = b.y; hi[2] = b.z;
  }
}

// The pass runs in three phases; the first two inside a block of kHierThreads consecutive leaves [c0, c_last].
//
// Phase 0 (registers, one warp = 32 consecutive leaves).  Algorithm 4's rendezvous at a parent -- "the first
// child to arrive stops, the second carries on" -- is done in lockstep with shuffles instead of ATOMICCAS:
// the node [l, r] that is currently complete is carried by the lane of its leftmost leaf l, with its box in
// registers.  Every round, a carrier that is a LEFT child (delta*(r) < delta*(l-1), L10) looks at the lane of
// leaf r+1; if that lane carries a complete node that is a RIGHT child (its parent's split is then r = the
// Apetrei index p of L11/L16, the same parent), the two have met: the left carrier takes over the union
// (range, delta*, box), computes the parent's Karras index q (L20), left child (L21) and skip-connection
// (L22-26), writes the record, and carries the parent; the right carrier retires.  A child whose sibling is
// not complete yet simply waits for a later round, which is what the first arrival does in the paper.  The
// rounds end when no pair met: what is left are the maximal subtrees inside the warp's 32 leaves, at most
// 2 log2(32) of them, and 31/32 of all merges are done without a single atomic, fence or divergent loop.
//
// Phase 1 (shared memory).  The carriers that are left run Algorithm 4 as written, on a shared-memory copy of
// `store`: the CAS is a shared-memory atomic, the sibling's box a shared-memory read, ordered by
// __threadfence_block().  A thread leaves this phase when (a) it is the first to arrive at a parent (L13 /
// L18: it may be done, or its sibling may be a node that straddles the block boundary and can only arrive
// through global memory), or (b) its parent's split lies on the block boundary.
//
// Phase 2 (global memory), a second kernel.  A thread of kind (a) whose sibling did arrive locally (its
// `store` slot was marked) is done; every other thread that left phase 1 hands its node to a compact queue,
// and the second kernel carries on with Algorithm 4 on the global `store` exactly as the paper states it
// (release fence, ATOMICCAS, acquire fence, sibling box through L2).  Only nodes whose range straddles a
// block boundary are created there: a few per block.
// Any two children of a parent meet in exactly one of the three places (same warp, same block, or global
// memory), so exactly one thread survives each node and the result is the unique hierarchy.
template <typename KeyT, bool IS_BOX>
__global__ void __launch_bounds__(kHierThreads)
hierarchy_local_kernel(const float* __restrict__ prim, const KeyT* __restrict__ codes,
                       const uint32_t* __restrict__ perm, char* nodes_base, int n, const Header* __restrict__ header,
                       int2* __restrict__ queue, uint32_t* __restrict__ queue_count) {
  using D = typename Delta<KeyT>::T;
  constexpr int C = kHierThreads;
  __shared__ uint32_t s_wsum[C / 32];
  __shared__ uint32_t s_qbase;
  __shared__ D s_delta[C + 2];      // s_delta[k] = delta*(c0 - 1 + k)
  __shared__ int s_store[C];        // s_store[p - c0]: -1 empty, >= 0 first arrival's range bound, -2 both arrived
  __shared__ float s_leaf[6][C];    // boxes of leaves that enter phase 1, by local leaf index
  __shared__ float s_int[6][C];     // boxes of internal nodes that enter or are made in phase 1, by local Karras index

  Node* nodes = reinterpret_cast<Node*>(nodes_base + kNodesHeaderBytes);   // internal records, by Karras index
  char* leaves = nodes_base + leaf_offset_bytes(n);
  const int tid = threadIdx.x, lane = tid & 31;
  if (blockIdx.x == 0 && tid == 0) {                          // the hierarchy's header: leaf format and root box
    NodesHeader* h = reinterpret_cast<NodesHeader*>(nodes_base);
    float sb[6];
    load_scene_bounds(header, sb);
    h->magic = kNodesMagic;
    h->n = n;
    h->leaf_kind = IS_BOX ? kLeafBoxes : kLeafPoints;
    h->reserved = 0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      h->scene_lo[a] = sb[a];
      h->scene_hi[a] = sb[3 + a];
    }
  }
  const int c0 = blockIdx.x * C;
  const int c_last = min(c0 + C, n) - 1;
  const int i = c0 + tid;
  const bool valid = i < n;
  const int leaf_base = n - 1;

  // K4: leaf box = box of the primitive sorted to position i (loads issued first: the longest latency)
  float lo[3] = {0.f, 0.f, 0.f}, hi[3] = {0.f, 0.f, 0.f};
  uint32_t orig = 0;
  if (valid) {
    orig = perm[i];
    if (IS_BOX) {
      const float2* p = reinterpret_cast<const float2*>(prim + 6 * (size_t)orig);
      const float2 a = __ldg(p), b = __ldg(p + 1), c = __ldg(p + 2);
      lo[0] = a.x; lo[1] = a.y; lo[2] = b.x; hi[0] = b.y; hi[1] = c.x; hi[2] = c.y;
    } else {
      const float* p = prim + 3 * (size_t)orig;
      lo[0] = hi[0] = __ldg(p);
      lo[1] = hi[1] = __ldg(p + 1);
      lo[2] = hi[2] = __ldg(p + 2);
    }
  }
  s_delta[tid + 1] = delta_star<KeyT>(codes, i, n);
  if (tid == 0) s_delta[0] = delta_star<KeyT>(codes, c0 - 1, n);
  if (tid == C - 1) s_delta[C + 1] = delta_star<KeyT>(codes, c0 + C, n);
  s_store[tid] = kInvalid;                                  // L1
  __syncthreads();

  // L3-4
  int range_left = i, range_right = i;
  const D delta_left0 = s_delta[tid];
  D delta_left = delta_left0, delta_right = s_delta[tid + 1];
  if (valid) {
    // L5-8: leaf skip-connection: L_{i+1} if delta*(i) < delta*(i+1) else I_{i+1} (one bit of the leaf record);
    // the sentinel for the last leaf
    const bool rope_internal = (i != n - 1) && !(delta_right < s_delta[tid + 2]);
    store_leaf<IS_BOX>(leaves, i, lo, hi, orig | (rope_internal ? kLeafRopeInternal : 0u));
  }

  // ---- phase 0: rendezvous inside the warp, in lockstep ----
  bool active = valid && n > 1;                             // G11: a single leaf has no parent
  {
    const int w0 = i - lane;                                // first leaf of this warp
    while (true) {
      const bool is_left = delta_right < delta_left;        // L10
      const int partner = range_right + 1 - w0;             // lane of leaf r+1
      const bool look = active && is_left && partner < 32;
      const int src = look ? partner : lane;
      // what the partner lane carries: its range end (bit 31: it is a complete RIGHT child), delta*(its end), its box
      const uint32_t mine = (uint32_t)range_right | ((active && !is_left) ? 0x80000000u : 0u);
      const uint32_t theirs = __shfl_sync(0xffffffffu, mine, src);
      const D their_delta = __shfl_sync(0xffffffffu, delta_right, src);
      float tlo[3], thi[3];
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        tlo[a] = __shfl_sync(0xffffffffu, lo[a], src);
        thi[a] = __shfl_sync(0xffffffffu, hi[a], src);
      }
      const bool merge = look && (theirs & 0x80000000u);
      const uint32_t met = __ballot_sync(0xffffffffu, merge);
      if (met == 0) break;
      const uint32_t retired = __reduce_or_sync(0xffffffffu, merge ? (1u << partner) : 0u);
      if (merge) {
        const int p = range_right;                                              // L11: Apetrei index = split
        const int left = (range_left == p) ? leaf_base + p : p;                 // L21 (reading G2)
        range_right = (int)(theirs & 0x7fffffffu);                              // L14 (the sibling's range joins)
        delta_right = their_delta;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
          lo[a] = fminf(lo[a], tlo[a]);
          hi[a] = fmaxf(hi[a], thi[a]);
        }
        const int q = (delta_right < delta_left) ? range_right : range_left;    // L20: Karras index
        int rope;
        if (range_right == n - 1)                                               // L22-23
          rope = kSentinel;
        else                                                                    // L25-26
          rope = (delta_right < s_delta[range_right - c0 + 2]) ? leaf_base + range_right + 1 : range_right + 1;
        store_node(nodes, q, lo, hi, left, rope);
        if (q == 0) active = false;                                             // L28: the root; nothing above it
      }
      if ((retired >> lane) & 1u) active = false;
    }
  }

  // ---- phase 1: L9-28 on shared memory for the carriers that are left ----
  bool go_global = false;
  int pending_p = -1;
  if (active) {
    // publish the box of the node this thread carries where its sibling will look for it
    if (range_left == range_right) {
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        s_leaf[a][tid] = lo[a];
        s_leaf[3 + a][tid] = hi[a];
      }
    } else {
      const int q = ((delta_right < delta_left) ? range_right : range_left) - c0;
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        s_int[a][q] = lo[a];
        s_int[3 + a][q] = hi[a];
      }
    }
    __threadfence_block();
    while (true) {
      const bool is_left = delta_right < delta_left;                    // L10
      const int p = is_left ? range_right : range_left - 1;             // L11 / L16: Apetrei index
      const bool interior = is_left ? (range_right < c_last) : (range_left > c0);
      if (!interior) {
        go_global = true;
        break;
      }
      const int other = atomicCAS(&s_store[p - c0], kInvalid, is_left ? range_left : range_right);  // L12 / L17
      if (other == kInvalid) {                                          // L13 / L18: first to arrive here
        pending_p = p;
        break;
      }
      s_store[p - c0] = -2;
      bool sib_leaf;
      int sib;
      if (is_left) {
        range_right = other;
        sib_leaf = (range_right == p + 1);
        sib = p + 1 - c0;
        delta_right = s_delta[range_right - c0 + 1];                    // L14
      } else {
        range_left = other;
        sib_leaf = (range_left == p);
        sib = p - c0;
        delta_left = s_delta[range_left - c0];                          // L19
      }
      __threadfence_block();
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        lo[a] = fminf(lo[a], sib_leaf ? s_leaf[a][sib] : s_int[a][sib]);
        hi[a] = fmaxf(hi[a], sib_leaf ? s_leaf[3 + a][sib] : s_int[3 + a][sib]);
      }
      const int q = (delta_right < delta_left) ? range_right : range_left;   // L20: Karras index
      const int left = (range_left == p) ? leaf_base + p : p;                // L21 (reading G2)
      int rope;
      if (range_right == n - 1)                                              // L22-23
        rope = kSentinel;
      else                                                                   // L25-26
        rope = (delta_right < s_delta[range_right - c0 + 2]) ? leaf_base + range_right + 1 : range_right + 1;
      store_node(nodes, q, lo, hi, left, rope);
      if (q == 0) break;                                                     // L28 (whole tree inside this block)
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        s_int[a][q - c0] = lo[a];
        s_int[3 + a][q - c0] = hi[a];
      }
      __threadfence_block();
    }
  }
  __syncthreads();
  if (pending_p >= 0 && s_store[pending_p - c0] != -2) go_global = true;     // my sibling never came locally

  // The survivors (maximal nodes of the tree inside this block: at most 2 x tree height of them) go to a
  // compact queue; the global phase runs as its own dense kernel instead of keeping this block resident.
  const uint32_t m = __ballot_sync(0xffffffffu, go_global);
  const int warp = tid >> 5;
  if (lane == 0) s_wsum[warp] = __popc(m);
  __syncthreads();
  if (tid == 0) {
    uint32_t total = 0;
    for (int w = 0; w < C / 32; ++w) {
      const uint32_t c = s_wsum[w];
      s_wsum[w] = total;
      total += c;
    }
    s_qbase = total ? atomicAdd(queue_count, total) : 0u;
  }
  __syncthreads();
  if (go_global) queue[s_qbase + s_wsum[warp] + __popc(m & ((1u << lane) - 1u))] = make_int2(range_left, range_right);
}

// Phase 2: Algorithm 4 on global memory for the queued nodes (those whose parent straddles a block boundary).
template <typename KeyT>
__global__ void __launch_bounds__(256)
hierarchy_global_kernel(const KeyT* __restrict__ codes, int* store, char* nodes_base, int n, int leaf_kind,
                        const int2* __restrict__ queue, const uint32_t* __restrict__ queue_count) {
  using D = typename Delta<KeyT>::T;
  Node* nodes = reinterpret_cast<Node*>(nodes_base + kNodesHeaderBytes);
  const int leaf_base = n - 1;
  const uint32_t count = *queue_count;
  for (uint32_t item = blockIdx.x * blockDim.x + threadIdx.x; item < count; item += gridDim.x * blockDim.x) {
    const int2 range = queue[item];
    int range_left = range.x, range_right = range.y;
    D delta_left = delta_star<KeyT>(codes, range_left - 1, n);
    D delta_right = delta_star<KeyT>(codes, range_right, n);
    // the node this item carries: a leaf, or the internal node with that range (Karras index, L20)
    const int carried = (range_left == range_right) ? leaf_base + range_left
                                                    : ((delta_right < delta_left) ? range_right : range_left);
    float lo[3], hi[3];
    load_box_cg(nodes_base, n, leaf_kind, carried, lo, hi);
    bool first_round = true;
    while (true) {
      // the node this thread carries is fully written: publish before arriving (the previous kernel's writes
      // are already visible; a fence is only needed for nodes written in this kernel)
      if (!first_round) __threadfence();
      first_round = false;
      int p, sibling;
      if (delta_right < delta_left) {       // L10: left child of its parent
        p = range_right;                    // L11: Apetrei index
        const int other = atomicCAS(&store[p], kInvalid, range_left);  // L12
        if (other == kInvalid) break;       // L13: first to arrive
        range_right = other;
        sibling = (range_right == p + 1) ? leaf_base + p + 1 : p + 1;  // right child: L_{p+1} or I_{p+1}
        delta_right = delta_star<KeyT>(codes, range_right, n);  // L14
      } else {                              // right child of its parent
        p = range_left - 1;                 // L16
        const int other = atomicCAS(&store[p], kInvalid, range_right);  // L17
        if (other == kInvalid) break;       // L18
        range_left = other;
        sibling = (range_left == p) ? leaf_base + p : p;               // left child: L_p or I_p
        delta_left = delta_star<KeyT>(codes, range_left - 1, n);  // L19
      }
      __threadfence();  // acquire side: the sibling's record was written before its CAS
      float slo[3], shi[3];
      load_box_cg(nodes_base, n, leaf_kind, sibling, slo, shi);
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        lo[a] = fminf(lo[a], slo[a]);
        hi[a] = fmaxf(hi[a], shi[a]);
      }

      const int q = (delta_right < delta_left) ? range_right : range_left;       // L20: Karras index
      const int left = (range_left == p) ? leaf_base + p : p;                    // L21 (reading G2)
      int rope;
      if (range_right == n - 1) {                                                // L22-23
        rope = kSentinel;
      } else {
        const int r = range_right + 1;                                           // L25
        rope = (delta_right < delta_star<KeyT>(codes, r, n)) ? leaf_base + r : r;  // L26
      }
      store_node(nodes, q, lo, hi, left, rope);
      if (q == 0) break;                                                         // L27-28
    }
  }
}

int hierarchy_queue_capacity(int n) {
  const int blocks = (n + kHierThreads - 1) / kHierThreads;
  const int per_block = kHierThreads < 192 ? kHierThreads : 192;  // <= 2 x tree height (93 bits of augmented key)
  return blocks * per_block;
}

void launch_hierarchy(const float* prim, bool is_box, const void* sorted_codes, int key_bytes, const uint32_t* perm,
                      int* store, void* nodes_, int n, const Header* header, int2* queue, uint32_t* queue_count,
                      cudaStream_t stream) {
  char* nodes = static_cast<char*>(nodes_);
  const unsigned g = (unsigned)((n + kHierThreads - 1) / kHierThreads);
  const unsigned g2 = kNumSMs * 4;
  const int kind = is_box ? kLeafBoxes : kLeafPoints;
  if (key_bytes == 4) {
    const uint32_t* c = static_cast<const uint32_t*>(sorted_codes);
    if (is_box)
      hierarchy_local_kernel<uint32_t, true><<<g, kHierThreads, 0, stream>>>(prim, c, perm, nodes, n, header, queue, queue_count);
    else
      hierarchy_local_kernel<uint32_t, false><<<g, kHierThreads, 0, stream>>>(prim, c, perm, nodes, n, header, queue, queue_count);
    hierarchy_global_kernel<uint32_t><<<g2, 256, 0, stream>>>(c, store, nodes, n, kind, queue, queue_count);
  } else {
    const uint64_t* c = static_cast<const uint64_t*>(sorted_codes);
    if (is_box)
      hierarchy_local_kernel<uint64_t, true><<<g, kHierThreads, 0, stream>>>(prim, c, perm, nodes, n, header, queue, queue_count);
    else
      hierarchy_local_kernel<uint64_t, false><<<g, kHierThreads, 0, stream>>>(prim, c, perm, nodes, n, header, queue, queue_count);
    hierarchy_global_kernel<uint64_t><<<g2, 256, 0, stream>>>(c, store, nodes, n, kind, queue, queue_count);
  }
}

}  // namespace bvh
