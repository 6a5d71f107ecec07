// hierarchy.cu -- K4 + K5: the paper's Algorithm 4, "Modified Apetrei's algorithm
// with skip installation", with the bounding boxes the pseudo-code omits (reading G10), fused with the
// permuted leaf gather.  Subtrees climb towards the root; at every parent the first of the two children
// to arrive stops, the second carries on (ATOMICCAS on `store`), so each internal
// node is written by exactly one thread, which by then knows the node's full range, hence its Karras
// index q, its left child (split = Apetrei index p) and its
// skip-connection (Algorithm 2).
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


// ---------------------------------------------------------------------------------------------------------
// Organisation of the pass.  Algorithm 4 lets every leaf climb towards the root; at a parent the first child
// to arrive stops, the second carries on.  Where the two children of a node meet is a free choice -- the
// result is the unique hierarchy either way -- and on a GPU it decides the cost: a rendezvous in global
// memory is a release fence, an ATOMICCAS and an acquire (a few microseconds per tree level), one in shared
// memory a few hundred cycles, one inside a warp a shuffle.  So the tree is built in windows of growing size:
//
//   level 1  hierarchy_local_kernel   one block = a window of kHierThreads consecutive leaves
//            phase 0: rendezvous inside each warp (32 leaves) in lockstep, by shuffles, no atomics;
//            phase 1: the subtrees that are left ("items": at most 2 x tree height of them) are compacted
//                     and run Algorithm 4 as written, one item per lane, on a shared-memory `store`;
//   level 2+ hierarchy_merge_kernel   one block = the windows of kMergeFan blocks of the level below:
//            their left-over items, in leaf order, run the same shared-memory Algorithm 4.
//
// What is left of a window when no more of its items can meet are its maximal complete subtrees, in leaf
// order: at most 2 x (bits of the augmented key) <= 186 of them for ANY window, which bounds the hand-over
// between levels (kSegCap entries per window, no allocation, no atomics).  The last level has one window, the
// whole tree, and ends by creating the root.  A node whose two children lie in different windows of level k
// is created at the first level whose window holds both.  There is no global `store` array any more: the
// array of Algorithm 4 is indexed by the boundary between two adjacent items of the window,
// which is the same thing as the split position p (an item boundary is a leaf boundary), and lives in shared
// memory.
// ---------------------------------------------------------------------------------------------------------
#ifndef BVH_MERGE_FAN
#define BVH_MERGE_FAN 64
#endif
#ifndef BVH_MERGE_MAX_ITEMS
#define BVH_MERGE_MAX_ITEMS 2048
#endif
constexpr int kSegCap = 192;                       // >= 186 = 2 x 93 bits of augmented key
constexpr int kMergeFan = BVH_MERGE_FAN;           // windows of the level below per merge block
constexpr int kMergeThreads = 512;
constexpr int kMergeMaxItems = BVH_MERGE_MAX_ITEMS;  // items a merge block holds in shared memory at once
static_assert(kMergeMaxItems >= 2 * kSegCap, "a pass over windows of kMergeMaxItems items must shrink the list");

// Where delta* comes from while items merge.  Level 1 has delta* of every leaf of its window in shared memory.
template <typename D>
struct DeltaByLeaf {
  const D* s_delta;   // s_delta[k] = delta*(c0 - 1 + k)
  int c0;
  __device__ __forceinline__ D left(int, int range_left) const { return s_delta[range_left - c0]; }       // delta*(l - 1)
  __device__ __forceinline__ D right(int, int range_right) const { return s_delta[range_right - c0 + 1]; }  // delta*(r)
  __device__ __forceinline__ D next(int, int range_right) const { return s_delta[range_right - c0 + 2]; }   // delta*(r + 1)
};
// Higher levels keep, per item k with leaves [l_k, r_k]: bd[k] = delta*(l_k - 1) (the boundary before it) and
// nd[k] = delta*(l_k); entry M describes the leaf after the window.
template <typename D>
struct DeltaByItem {
  const D* bd;
  const D* nd;
  __device__ __forceinline__ D left(int a, int) const { return bd[a]; }
  __device__ __forceinline__ D right(int b, int) const { return bd[b + 1]; }
  __device__ __forceinline__ D next(int b, int) const { return nd[b + 1]; }
};

// Shared-memory state of M items in leaf order (slot k = item k).  A subtree made of items [a, b] is carried
// by one thread and keeps its box in slot a.
struct ItemArrays {
  int* l;        // first leaf of item k
  int* r;        // last leaf of item k
  float* box;    // box[c * stride + k], c = 0..5 (min.xyz, max.xyz)
  int stride;
  int* store;    // Algorithm 4's `store`, one entry per boundary (k | k+1): -1 empty, >= 0 first arrival, -2 both
  int* fin_l;    // where the subtree that started as item e stopped: its leaf range ...
  int* fin_r;
  int* fin_k;    // ... and why: -2 it became the root, -1 its parent straddles the window, k >= 0 it arrived first at boundary k
};

// Algorithm 4, L9-28, for the subtree that starts as item e, on shared memory.
template <typename D, typename DeltaSrc>
__device__ __forceinline__ void climb_from_item(int e, int M, const ItemArrays& A, const DeltaSrc& ds, Node* nodes, int n) {
  const int leaf_base = n - 1;
  int a = e, b = e;                                                   // items covered
  int range_left = A.l[e], range_right = A.r[e];                      // L3 (leaves covered)
  D delta_left = ds.left(a, range_left), delta_right = ds.right(b, range_right);   // L4
  float lo[3], hi[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    lo[c] = A.box[c * A.stride + e];
    hi[c] = A.box[(3 + c) * A.stride + e];
  }
  int fin = -1;
  while (true) {
    const bool is_left = delta_right < delta_left;                    // L10
    if (is_left ? (b >= M - 1) : (a <= 0)) break;                     // the sibling is not in this window
    const int k = is_left ? b : a - 1;                                // L11 / L16: the boundary at the split p
    const int other = atomicCAS(&A.store[k], kInvalid, is_left ? a : b);   // L12 / L17
    if (other == kInvalid) {                                          // L13 / L18: first to arrive
      fin = k;
      break;
    }
    A.store[k] = -2;
    int p, sib;
    if (is_left) {
      p = range_right;                                                // Apetrei index = split
      sib = b + 1;
      b = other;
      range_right = A.r[b];
      delta_right = ds.right(b, range_right);                         // L14
    } else {
      p = range_left - 1;
      sib = other;
      a = other;
      range_left = A.l[a];
      delta_left = ds.left(a, range_left);                            // L19
    }
    __threadfence_block();                                            // the sibling's box was written before its CAS
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      lo[c] = fminf(lo[c], A.box[c * A.stride + sib]);
      hi[c] = fmaxf(hi[c], A.box[(3 + c) * A.stride + sib]);
    }
    const int q = (delta_right < delta_left) ? range_right : range_left;     // L20: Karras index
    const int left = (range_left == p) ? leaf_base + p : p;                  // L21 (reading G2)
    int rope;
    if (range_right == n - 1)                                                // L22-23
      rope = kSentinel;
    else                                                                     // L25-26
      rope = (delta_right < ds.next(b, range_right)) ? leaf_base + range_right + 1 : range_right + 1;
    store_node(nodes, q, lo, hi, left, rope);
    if (q == 0) return;                                                      // L28: the root
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      A.box[c * A.stride + a] = lo[c];
      A.box[(3 + c) * A.stride + a] = hi[c];
    }
    __threadfence_block();
  }
  // recorded under the item the subtree started from: only this thread writes there, and since a subtree
  // contains its first item, the order of the survivors by e is their order by leaf
  A.fin_l[e] = range_left;
  A.fin_r[e] = range_right;
  A.fin_k[e] = fin;
}

// After a barrier: is the subtree that started as item e still without its sibling (a maximal subtree of the window)?
__device__ __forceinline__ bool item_survives(const ItemArrays& A, int e) {
  const int k = A.fin_k[e];
  return k == -1 || (k >= 0 && A.store[k] != -2);
}

// Block-wide compaction: position of this thread's flagged element among the flagged ones, and their number.
// s_wsum: one word per warp (+1).  Two barriers.
__device__ __forceinline__ int block_compact(bool flag, uint32_t* s_wsum, int nwarps, int& total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t m = __ballot_sync(0xffffffffu, flag);
  if (lane == 0) s_wsum[warp] = __popc(m);
  __syncthreads();
  int base = 0, sum = 0;
  for (int w = 0; w < nwarps; ++w) {
    const int c = (int)s_wsum[w];
    if (w < warp) base += c;
    sum += c;
  }
  __syncthreads();
  total = sum;
  return base + __popc(m & ((1u << lane) - 1u));
}

// Level 1.  Phase 0 (registers, one warp = 32 consecutive leaves): the rendezvous at a parent is done in
// lockstep with shuffles instead of ATOMICCAS.  The node [l, r] that is currently complete is carried by the
// lane of its leftmost leaf l, with its box in registers.  Every round, a carrier that is a LEFT child
// (delta*(r) < delta*(l-1), L10) looks at the lane of leaf r+1; if that lane carries a complete node that is a
// RIGHT child (its parent's split is then r = the Apetrei index p of L11/L16, the same parent), the two have
// met: the left carrier takes over the union (range, delta*, box), computes the parent's Karras index q (L20),
// left child (L21) and skip-connection (L22-26), writes the record, and carries the parent; the right carrier
// retires.  A child whose sibling is not complete yet waits for a later round, which is what the first arrival
// does in the paper.  The rounds end when no pair met.  Phase 1: see climb_from_item.
template <typename KeyT, bool IS_BOX>
__global__ void __launch_bounds__(kHierThreads)
hierarchy_local_kernel(const float* __restrict__ prim, const KeyT* __restrict__ codes,
                       const uint32_t* __restrict__ perm, char* nodes_base, int n, const Header* __restrict__ header,
                       int2* __restrict__ seg_items, int* __restrict__ seg_count) {
  using D = typename Delta<KeyT>::T;
  constexpr int C = kHierThreads;
  __shared__ uint32_t s_wsum[C / 32 + 1];
  __shared__ D s_delta[C + 2];      // s_delta[k] = delta*(c0 - 1 + k)
  __shared__ int s_l[C], s_r[C], s_store[C], s_fin_l[C], s_fin_r[C], s_fin_k[C];
  __shared__ float s_box[6 * C];

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
  __syncthreads();

  // L3-4
  int range_left = i, range_right = i;
  D delta_left = s_delta[tid], delta_right = s_delta[tid + 1];
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
      const bool merge = look && (theirs & 0x80000000u);
      const uint32_t met = __ballot_sync(0xffffffffu, merge);
      if (met == 0) break;
      const D their_delta = __shfl_sync(0xffffffffu, delta_right, src);
      float tlo[3], thi[3];
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        tlo[a] = __shfl_sync(0xffffffffu, lo[a], src);
        thi[a] = __shfl_sync(0xffffffffu, hi[a], src);
      }
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

  // ---- phase 1: the subtrees that are left become the items of this window, in leaf order ----
  int M;
  const int slot = block_compact(active, s_wsum, C / 32, M);
  if (active) {
    s_l[slot] = range_left;
    s_r[slot] = range_right;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      s_box[a * C + slot] = lo[a];
      s_box[(3 + a) * C + slot] = hi[a];
    }
  }
  s_store[tid] = kInvalid;                                                    // L1
  s_fin_k[tid] = -2;
  __syncthreads();
  const ItemArrays A{s_l, s_r, s_box, C, s_store, s_fin_l, s_fin_r, s_fin_k};
  if (tid < M) climb_from_item<D>(tid, M, A, DeltaByLeaf<D>{s_delta, c0}, nodes, n);
  __syncthreads();

  // ---- hand over what is left of this window, in leaf order (at most kSegCap subtrees) ----
  const bool surv = tid < M && item_survives(A, tid);
  int total;
  const int pos = block_compact(surv, s_wsum, C / 32, total);
  if (surv) seg_items[(size_t)blockIdx.x * kSegCap + pos] = make_int2(s_fin_l[tid], s_fin_r[tid]);
  if (tid == 0) seg_count[blockIdx.x] = total;
}

// Level 2 and up.  Block g owns the windows [g * kMergeFan, (g + 1) * kMergeFan) of the level below, i.e. one
// contiguous range of leaves; their left-over subtrees, concatenated, are its items.  One pass = load up to
// kMergeMaxItems consecutive items (range, the two delta* next to the item's first leaf, box of the node the
// item stands for, read back through L2), run climb_from_item on them, compact what is left.  Normally the
// whole list fits and the pass writes its <= kSegCap survivors to this block's segment of the next level.  A
// longer list (only degenerate inputs: kMergeFan x 186 worst case) is first shortened by passes over windows of
// kMergeMaxItems items, compacted in place at the start of this block's own input segments -- a pass leaves at
// most 186 items per window, so the list shrinks until it fits.
template <typename KeyT>
__global__ void __launch_bounds__(kMergeThreads)
hierarchy_merge_kernel(const KeyT* __restrict__ codes, char* nodes_base, int n, int leaf_kind, int2* in_items,
                       const int* __restrict__ in_count, int in_segs, int2* __restrict__ out_items,
                       int* __restrict__ out_count) {
  using D = typename Delta<KeyT>::T;
  constexpr int T = kMergeThreads, MAXI = kMergeMaxItems;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  D* s_bd = reinterpret_cast<D*>(smem_raw);               // [MAXI + 1]
  D* s_nd = s_bd + (MAXI + 1);                            // [MAXI + 1]
  float* s_box = reinterpret_cast<float*>(s_nd + (MAXI + 1));   // [6][MAXI]
  int* s_l = reinterpret_cast<int*>(s_box + 6 * MAXI);
  int* s_r = s_l + MAXI;
  int* s_store = s_r + MAXI;
  int* s_fin_l = s_store + MAXI;
  int* s_fin_r = s_fin_l + MAXI;
  int* s_fin_k = s_fin_r + MAXI;
  __shared__ int s_pref[kMergeFan + 1];
  __shared__ uint32_t s_wsum[T / 32 + 1];

  Node* nodes = reinterpret_cast<Node*>(nodes_base + kNodesHeaderBytes);
  const int tid = threadIdx.x;
  const int leaf_base = n - 1;
  const int seg0 = blockIdx.x * kMergeFan;
  const int nseg = min(kMergeFan, in_segs - seg0);
  if (tid == 0) {
    int sum = 0;
    for (int s = 0; s < nseg; ++s) {
      s_pref[s] = sum;
      sum += in_count[seg0 + s];
    }
    for (int s = nseg; s <= kMergeFan; ++s) s_pref[s] = sum;
  }
  __syncthreads();
  int count = s_pref[kMergeFan];
  int2* region = in_items + (size_t)seg0 * kSegCap;       // this block's input segments, contiguous
  bool flat = false;                                      // items compacted at the start of `region`
  const ItemArrays A{s_l, s_r, s_box, MAXI, s_store, s_fin_l, s_fin_r, s_fin_k};

  while (true) {
    const bool last_pass = count <= MAXI;
    int written = 0;                                      // items compacted in place by this pass (uniform)
    for (int w0 = 0; w0 < count || w0 == 0; w0 += MAXI) {
      const int M = min(MAXI, count - w0);
      // ---- load the items [w0, w0 + M) ----
      for (int e = tid; e < M; e += T) {
        const int g = w0 + e;
        int2 it;
        if (flat) {
          it = __ldcg(region + g);
        } else {
          int s = 0;                                      // segment of item g: the last s with s_pref[s] <= g
          for (int step = kMergeFan >> 1; step > 0; step >>= 1)
            if (s + step < kMergeFan && s_pref[s + step] <= g) s += step;
          it = __ldcg(region + (size_t)s * kSegCap + (g - s_pref[s]));
        }
        s_l[e] = it.x;
        s_r[e] = it.y;
        s_bd[e] = delta_star<KeyT>(codes, it.x - 1, n);
        s_nd[e] = delta_star<KeyT>(codes, it.x, n);
        if (e == M - 1) {
          s_bd[M] = delta_star<KeyT>(codes, it.y, n);
          s_nd[M] = delta_star<KeyT>(codes, it.y + 1, n);
        }
        s_store[e] = kInvalid;                            // L1
        s_fin_k[e] = -2;
      }
      __syncthreads();
      for (int e = tid; e < M; e += T) {
        const int l = s_l[e], r = s_r[e];
        // the node the item stands for: a leaf, or the internal node with that range (Karras index, L20)
        const int carried = (l == r) ? leaf_base + l : ((s_bd[e + 1] < s_bd[e]) ? r : l);
        float lo[3], hi[3];
        load_box_cg(nodes_base, n, leaf_kind, carried, lo, hi);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          s_box[c * MAXI + e] = lo[c];
          s_box[(3 + c) * MAXI + e] = hi[c];
        }
      }
      __syncthreads();
      // ---- Algorithm 4 on the window ----
      for (int e = tid; e < M; e += T) climb_from_item<D>(e, M, A, DeltaByItem<D>{s_bd, s_nd}, nodes, n);
      __syncthreads();
      // ---- compact what is left, in leaf order ----
      int2* dst = last_pass ? out_items + (size_t)blockIdx.x * kSegCap : region + written;
      int base = 0;
      for (int e0 = 0; e0 < M; e0 += T) {
        const int e = e0 + tid;
        const bool surv = e < M && item_survives(A, e);
        int total;
        const int pos = block_compact(surv, s_wsum, T / 32, total);
        if (surv) dst[base + pos] = make_int2(s_fin_l[e], s_fin_r[e]);
        base += total;
      }
      written += base;
      __syncthreads();
    }
    if (last_pass) {
      if (tid == 0) out_count[blockIdx.x] = written;
      return;
    }
    __threadfence();
    __syncthreads();
    count = written;
    flat = true;
  }
}

// Windows per level: level 1 has ceil(n / kHierThreads), each further level ceil(previous / kMergeFan), down to 1.
int hierarchy_levels(int n, int segs[kMaxHierLevels]) {
  int levels = 0;
  int s = (n + kHierThreads - 1) / kHierThreads;
  if (s < 1) s = 1;
  segs[levels++] = s;
  while (s > 1 && levels < kMaxHierLevels) {
    s = (s + kMergeFan - 1) / kMergeFan;
    segs[levels++] = s;
  }
  return levels;
}

int hierarchy_total_segments(int n) {
  int segs[kMaxHierLevels];
  const int levels = hierarchy_levels(n, segs);
  int total = 0;
  for (int l = 0; l < levels; ++l) total += segs[l];
  return total;
}

template <typename KeyT>
static void launch_hierarchy_keys(const float* prim, bool is_box, const KeyT* codes, const uint32_t* perm, char* nodes, int n,
                                  const Header* header, int2* seg_items, int* seg_count, cudaStream_t stream) {
  int segs[kMaxHierLevels];
  const int levels = hierarchy_levels(n, segs);
  if (is_box)
    hierarchy_local_kernel<KeyT, true><<<segs[0], kHierThreads, 0, stream>>>(prim, codes, perm, nodes, n, header, seg_items, seg_count);
  else
    hierarchy_local_kernel<KeyT, false><<<segs[0], kHierThreads, 0, stream>>>(prim, codes, perm, nodes, n, header, seg_items, seg_count);
  using D = typename Delta<KeyT>::T;
  const size_t smem = 2 * (kMergeMaxItems + 1) * sizeof(D) + (6 * sizeof(float) + 6 * sizeof(int)) * (size_t)kMergeMaxItems;
  cudaFuncSetAttribute(hierarchy_merge_kernel<KeyT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  const int kind = is_box ? kLeafBoxes : kLeafPoints;
  size_t off = 0;
  for (int l = 1; l < levels; ++l) {
    int2* in_items = seg_items + off * kSegCap;
    int* in_count = seg_count + off;
    off += segs[l - 1];
    hierarchy_merge_kernel<KeyT><<<segs[l], kMergeThreads, smem, stream>>>(codes, nodes, n, kind, in_items, in_count, segs[l - 1],
                                                                          seg_items + off * kSegCap, seg_count + off);
  }
}

void launch_hierarchy(const float* prim, bool is_box, const void* sorted_codes, int key_bytes, const uint32_t* perm,
                      void* nodes, int n, const Header* header, int2* seg_items, int* seg_count, cudaStream_t stream) {
  if (key_bytes == 4)
    launch_hierarchy_keys<uint32_t>(prim, is_box, static_cast<const uint32_t*>(sorted_codes), perm, static_cast<char*>(nodes), n,
                                    header, seg_items, seg_count, stream);
  else
    launch_hierarchy_keys<uint64_t>(prim, is_box, static_cast<const uint64_t*>(sorted_codes), perm, static_cast<char*>(nodes), n,
                                    header, seg_items, seg_count, stream);
}

int hierarchy_seg_capacity() { return kSegCap; }

}  // namespace bvh
