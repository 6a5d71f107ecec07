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
#include "device_helpers.cuh"

namespace bvh {

#ifndef BVH_HIER_WINDOW
#define BVH_HIER_WINDOW 256
#endif
#ifndef BVH_HIER_MINBLOCKS
#define BVH_HIER_MINBLOCKS 12
#endif
#ifndef BVH_HIER_SLOT_TABLE
#define BVH_HIER_SLOT_TABLE 0
#endif
template <bool SMALL>
struct SlotType { using T = uint8_t; };
template <>
struct SlotType<false> { using T = uint16_t; };
#ifndef BVH_HIER_UNROLL_GROUPS
#define BVH_HIER_UNROLL_GROUPS 0
#endif
#ifndef BVH_PHASE0_MAX_ROUNDS
#define BVH_PHASE0_MAX_ROUNDS 3
#endif
constexpr int kPhase0MaxRounds = BVH_PHASE0_MAX_ROUNDS;   // lockstep rounds per group before the rest is left to phase 1 (>= 31: all)
constexpr int kHierThreads = 128;               // threads of a level-1 block
constexpr int kHierWindow = BVH_HIER_WINDOW;    // leaves of a level-1 window (one block); a multiple of kHierThreads
static_assert(kHierWindow % kHierThreads == 0, "a level-1 window is a whole number of 32-leaf groups per warp");

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
//   level 1  hierarchy_local_kernel   one block of kHierThreads threads = a window of kHierWindow consecutive
//            leaves, each warp taking kHierWindow / kHierThreads groups of 32 consecutive leaves in turn
//            phase 0: rendezvous inside each group of 32 leaves in lockstep, by shuffles, no atomics;
//            phase 1: the subtrees that are left ("items": a handful per group) run Algorithm 4 as written,
//                     one item per thread, on a shared-memory `store` -- with four groups per warp the
//                     items of a window keep most of the block's threads busy, where a block of one
//                     thread per leaf left three quarters of its warps waiting at the barrier;
//   level 2+ merge_window              one block = the windows of kMergeFan blocks of the level below:
//            their left-over items, in leaf order, run the same shared-memory Algorithm 4.
//
// Levels 2 and up run in ONE kernel (hierarchy_merge_kernel, one block per level-2 window).  A block that has
// handed over its window counts itself in at its parent window (one atomicAdd per block, after a fence); the
// block that completes the count -- the last of the kMergeFan children to finish -- carries on as the parent
// window, and so on up to the root.  Nobody waits: like the first arrival of Algorithm 4, a
// block that is not the last simply ends.
//
// What is left of a window when no more of its items can meet are its maximal complete subtrees, in leaf
// order: at most 2 x (bits of the augmented key) <= 186 of them for ANY window, which bounds the hand-over
// between levels (kSegCap entries per window, no allocation).  The last level has one window, the whole tree,
// and ends by creating the root.  A node whose two children lie in different windows of level k is created at
// the first level whose window holds both.  There is no global `store` array any more: the array of
// Algorithm 4 is indexed by the boundary between two adjacent items of the window, which is the
// same thing as the split position p (an item boundary is a leaf boundary), and lives in shared memory.
// ---------------------------------------------------------------------------------------------------------
#ifndef BVH_MERGE_FAN
#define BVH_MERGE_FAN 64
#endif
#ifndef BVH_MERGE_MAX_ITEMS
#define BVH_MERGE_MAX_ITEMS 1024
#endif
#ifndef BVH_MERGE_THREADS
#define BVH_MERGE_THREADS 1024
#endif
constexpr int kSegCap = 192;                       // >= 186 = 2 x 93 bits of augmented key
constexpr int kMergeFan = BVH_MERGE_FAN;           // windows of the level below per merge window
#ifndef BVH_MERGE_FAN_MAX
#define BVH_MERGE_FAN_MAX (BVH_MERGE_FAN <= 128 ? 128 : (BVH_MERGE_FAN <= 256 ? 256 : 512))
#endif
constexpr int kMergeFanMax = BVH_MERGE_FAN_MAX;    // a power of two >= kMergeFan: the prefix / search code of merge_window
static_assert((kMergeFanMax & (kMergeFanMax - 1)) == 0 && kMergeFanMax % 32 == 0, "segment prefix: whole lanes, binary search");
static_assert(kMergeFan >= 2 && kMergeFan <= kMergeFanMax, "merge_window handles up to kMergeFanMax child windows");
constexpr int kMergeMaxItems = BVH_MERGE_MAX_ITEMS;  // items a merge window holds in shared memory at once
static_assert(kMergeMaxItems >= 2 * kSegCap, "a pass over windows of kMergeMaxItems items must shrink the list");
constexpr int kMergeThreads = BVH_MERGE_THREADS;
static_assert(kMergeMaxItems % kMergeThreads == 0, "whole items per thread");

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

// Shared-memory state of M items in leaf order.  Item e lives in slot map.slot(e) of the arrays (level 1 leaves the
// items where its warps staged them; the higher levels store them densely).  A subtree made of items [a, b] is
// carried by one thread and keeps its box in the slot of item a.
template <typename RT>
struct ItemArrays {
  RT* l;         // first leaf of the item in this slot, minus `base` (level 1: offsets into the window, 16 bits)
  RT* r;         // last leaf, minus `base`
  int base;
  float2* box;   // box[c * stride + slot] = {min, max} of axis c = 0..2 (one 64-bit shared-memory access per axis)
  int stride;
  int* store;    // Algorithm 4's `store`, one entry per boundary (e | e+1), by item index: -1 empty, >= 0 first arrival, -2 both
};
struct DenseSlots {
  __device__ __forceinline__ int slot(int e) const { return e; }
};
// Level 1: warp w staged its items, in leaf order, from slot w * per_warp on; begin[w] = index of its first item.
struct StagedSlots {
  int b1, b2, b3;      // first item of warps 1, 2, 3 (kHierThreads = 128: four warps)
  int o0, o1, o2, o3;  // slot - item index, per warp
  __device__ __forceinline__ int slot(int e) const {
    return e + (e >= b2 ? (e >= b3 ? o3 : o2) : (e >= b1 ? o1 : o0));
  }
};
// ... looked up in a table the block fills once (one shared-memory load instead of the compare chain, which the climb
// needs up to three times per merge)
template <typename ST>
struct TableSlots {
  const ST* table;
  __device__ __forceinline__ int slot(int e) const { return (int)table[e]; }
};
// Where the subtree that started as one item stopped: its leaf range, and why: fin = -2 it became the root, -1 its
// parent straddles the window, k >= 0 it arrived first at boundary k.
struct ClimbEnd {
  int l, r, fin;
};

// Algorithm 4, L9-28, for the subtree that starts as item e, on shared memory.
template <typename D, typename RT, typename DeltaSrc, typename Slots>
__device__ __forceinline__ ClimbEnd climb_from_item(int e, int M, const ItemArrays<RT>& A, const DeltaSrc& ds, const Slots& map,
                                                    Node* nodes, int n) {
  const int leaf_base = n - 1;
  int a = e, b = e;                                                   // items covered
  const int se = map.slot(e);
  int sa = se;                                                        // slot of item a: where this subtree's box lives
  int range_left = A.base + (int)A.l[se], range_right = A.base + (int)A.r[se];   // L3 (leaves covered)
  D delta_left = ds.left(a, range_left), delta_right = ds.right(b, range_right);   // L4
  float lo[3], hi[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const float2 v = A.box[c * A.stride + se];
    lo[c] = v.x;
    hi[c] = v.y;
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
    int p, ssib;
    if (is_left) {
      p = range_right;                                                // Apetrei index = split
      ssib = map.slot(b + 1);
      b = other;
      range_right = A.base + (int)A.r[map.slot(b)];
      delta_right = ds.right(b, range_right);                         // L14
    } else {
      p = range_left - 1;
      a = other;
      sa = ssib = map.slot(a);
      range_left = A.base + (int)A.l[sa];
      delta_left = ds.left(a, range_left);                            // L19
    }
    __threadfence_block();                                            // the sibling's box was written before its CAS
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const float2 v = A.box[c * A.stride + ssib];
      lo[c] = fminf(lo[c], v.x);
      hi[c] = fmaxf(hi[c], v.y);
    }
    const int q = (delta_right < delta_left) ? range_right : range_left;     // L20: Karras index
    const int left = (range_left == p) ? leaf_base + p : p;                  // L21 (reading G2)
    int rope;
    if (range_right == n - 1)                                                // L22-23
      rope = kSentinel;
    else                                                                     // L25-26
      rope = (delta_right < ds.next(b, range_right)) ? leaf_base + range_right + 1 : range_right + 1;
    store_node(nodes, q, lo, hi, left, rope);
    if (q == 0) return ClimbEnd{range_left, range_right, -2};                // L28: the root
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      A.box[c * A.stride + sa] = make_float2(lo[c], hi[c]);
    }
    __threadfence_block();
  }
  return ClimbEnd{range_left, range_right, fin};
}

// After a barrier: is the subtree that stopped like this still without its sibling (a maximal subtree of the window)?
template <typename RT>
__device__ __forceinline__ bool climb_survives(const ItemArrays<RT>& A, const ClimbEnd& c) {
  return c.fin == -1 || (c.fin >= 0 && A.store[c.fin] != -2);
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

// Shared memory of a level-1 block and of a merge block.
template <typename D>
struct LocalSmem {
  D delta[kHierWindow + 2];      // delta[k] = delta*(c0 - 1 + k)
  int store[kHierWindow];
  float2 box[3 * kHierWindow];
  uint16_t l[kHierWindow], r[kHierWindow];   // offsets from the window's first leaf
};
static_assert(kHierWindow <= 65536, "level-1 item ranges are kept as 16-bit offsets");
template <typename D>
struct MergeSmem {
  D bd[kMergeMaxItems + 1], nd[kMergeMaxItems + 1];
  int l[kMergeMaxItems], r[kMergeMaxItems], store[kMergeMaxItems];
  float2 box[3 * kMergeMaxItems];
  int pref[kMergeFanMax + 1];
};
// Windows of every level (level 1 first) and where each level's hand-over segments and arrival counters start.
struct HierLevels {
  int levels;
  int segs[kMaxHierLevels];      // windows of level l + 1
  int seg_off[kMaxHierLevels];   // first segment of that level in seg_items / seg_count / arrivals
};

// Level 2 and up.  Window g of a level owns the windows [g * kMergeFan, (g + 1) * kMergeFan) of the level below, i.e.
// one contiguous range of leaves; their left-over subtrees, concatenated, are its items.  One pass = load up to
// kMergeMaxItems consecutive items (range, the two delta* next to the item's first leaf, box of the node the
// item stands for, read back through L2), run climb_from_item on them, compact what is left.  Normally the
// whole list fits and the pass writes its <= kSegCap survivors to this window's segment of the next level.  A
// longer list (only degenerate inputs: kMergeFan x 186 worst case) is first shortened by passes over windows of
// kMergeMaxItems items, compacted in place at the start of this window's own input segments -- a pass leaves at
// most 186 items per window, so the list shrinks until it fits.
template <typename KeyT>
__device__ __forceinline__ void merge_window(MergeSmem<typename Delta<KeyT>::T>& S, uint32_t* s_wsum,
                                             const KeyT* __restrict__ codes, char* nodes_base, int n, int leaf_kind,
                                             int window, int2* in_items, const int* in_count, int in_segs,
                                             int2* out_items, int* out_count) {
  using D = typename Delta<KeyT>::T;
  constexpr int T = kMergeThreads, MAXI = kMergeMaxItems, PT = MAXI / T, NW = T / 32;
  Node* nodes = reinterpret_cast<Node*>(nodes_base + kNodesHeaderBytes);
  const int tid = threadIdx.x;
  const int leaf_base = n - 1;
  const int seg0 = window * kMergeFan;
  const int nseg = min(kMergeFan, in_segs - seg0);
  if (tid < 32) {                                         // exclusive prefix of the segment counts, by one warp
    constexpr int PER = kMergeFanMax / 32;
    int c[PER], sum = 0;
#pragma unroll
    for (int u = 0; u < PER; ++u) {
      const int sg = tid * PER + u;
      c[u] = (sg < nseg) ? __ldcg(in_count + seg0 + sg) : 0;
      sum += c[u];
    }
    int incl = sum;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
      const int v = __shfl_up_sync(0xffffffffu, incl, off);
      if (tid >= off) incl += v;
    }
    int run = incl - sum;
#pragma unroll
    for (int u = 0; u < PER; ++u) {
      const int sg = tid * PER + u;
      S.pref[sg] = run;                                   // entries past nseg hold the total
      run += c[u];
    }
    if (tid == 31) S.pref[kMergeFanMax] = incl;
  }
  __syncthreads();
  int count = S.pref[kMergeFanMax];
  int2* region = in_items + (size_t)seg0 * kSegCap;       // this window's input segments, contiguous
  bool flat = false;                                      // items compacted at the start of `region`
  const ItemArrays<int> A{S.l, S.r, 0, S.box, MAXI, S.store};

  while (true) {
    const bool last_pass = count <= MAXI;
    int written = 0;                                      // items compacted in place by this pass (uniform)
    for (int w0 = 0; w0 < count || w0 == 0; w0 += MAXI) {
      const int M = min(MAXI, count - w0);
      // ---- load the items [w0, w0 + M): three rounds of independent loads (items, their delta*, their boxes), each
      // round issued for all of the thread's items before any is consumed ----
      int2 it[PT];
#pragma unroll
      for (int j = 0; j < PT; ++j) {
        const int e = tid + j * T;
        it[j] = make_int2(0, 0);
        if (e < M) {
          const int g = w0 + e;
          if (flat) {
            it[j] = __ldcg(region + g);
          } else {
            int sg = 0;                                   // segment of item g: the last sg with pref[sg] <= g
#pragma unroll
            for (int step = kMergeFanMax / 2; step > 0; step >>= 1)
              if (sg + step < nseg && S.pref[sg + step] <= g) sg += step;
            it[j] = __ldcg(region + (size_t)sg * kSegCap + (g - S.pref[sg]));
          }
        }
      }
      D bd[PT], nd[PT], bdn[PT], ndn[PT];
#pragma unroll
      for (int j = 0; j < PT; ++j) {
        const int e = tid + j * T;
        bd[j] = nd[j] = bdn[j] = ndn[j] = Delta<KeyT>::kInf;
        if (e < M) {
          bd[j] = delta_star<KeyT>(codes, it[j].x - 1, n);
          nd[j] = delta_star<KeyT>(codes, it[j].x, n);
          bdn[j] = delta_star<KeyT>(codes, it[j].y, n);   // = bd of the next item (its first leaf is it.y + 1)
          if (e == M - 1) ndn[j] = delta_star<KeyT>(codes, it[j].y + 1, n);
        }
      }
#pragma unroll
      for (int j = 0; j < PT; ++j) {
        const int e = tid + j * T;
        if (e < M) {
          S.l[e] = it[j].x;
          S.r[e] = it[j].y;
          S.bd[e] = bd[j];
          S.nd[e] = nd[j];
          if (e == M - 1) {
            S.bd[M] = bdn[j];
            S.nd[M] = ndn[j];
          }
          S.store[e] = kInvalid;                          // L1
          // the node the item stands for: a leaf, or the internal node with that range (Karras index, L20)
          const int carried = (it[j].x == it[j].y) ? leaf_base + it[j].x : ((bdn[j] < bd[j]) ? it[j].y : it[j].x);
          float lo[3], hi[3];
          load_box_cg(nodes_base, n, leaf_kind, carried, lo, hi);
#pragma unroll
          for (int c = 0; c < 3; ++c) {
            S.box[c * MAXI + e] = make_float2(lo[c], hi[c]);
          }
        }
      }
      __syncthreads();
      // ---- Algorithm 4 on the window ----
      ClimbEnd end[PT];
#pragma unroll
      for (int j = 0; j < PT; ++j) {
        end[j] = ClimbEnd{0, 0, -2};
        const int e = tid + j * T;
        if (e < M) end[j] = climb_from_item<D>(e, M, A, DeltaByItem<D>{S.bd, S.nd}, DenseSlots{}, nodes, n);
      }
      __syncthreads();
      // ---- compact what is left, in leaf order (a subtree contains the item it started from, so the order of
      // the survivors by starting item is their order by leaf) ----
      int2* dst = last_pass ? out_items : region + written;
      int base = 0;
#pragma unroll
      for (int j = 0; j < PT; ++j) {
        if (j * T >= M && j > 0) break;                   // uniform
        const bool surv = (tid + j * T < M) && climb_survives(A, end[j]);
        int total;
        const int pos = block_compact(surv, s_wsum, NW, total);
        if (surv) dst[base + pos] = make_int2(end[j].l, end[j].r);
        base += total;
      }
      written += base;
      __syncthreads();
    }
    if (last_pass) {
      if (tid == 0) *out_count = written;
      return;
    }
    __threadfence();
    __syncthreads();
    count = written;
    flat = true;
  }
}

// Level 1.  Phase 0 (registers, one group = 32 consecutive leaves, one per lane): the rendezvous at a parent is done
// in lockstep with shuffles instead of ATOMICCAS.  The node [l, r] that is currently complete is carried by the
// lane of its leftmost leaf l, with its box in registers.  Every round, a carrier that is a LEFT child
// (delta*(r) < delta*(l-1), L10) looks at the lane of leaf r+1; if that lane carries a complete node that is a
// RIGHT child (its parent's split is then r = the Apetrei index p of L11/L16, the same parent), the two have
// met: the left carrier takes over the union (range, delta*, box), computes the parent's Karras index q (L20),
// left child (L21) and skip-connection (L22-26), writes the record, and carries the parent; the right carrier
// retires.  A child whose sibling is not complete yet waits for a later round, which is what the first arrival
// does in the paper.  The rounds end when no pair met.  Phase 1: see climb_from_item.  Then the block counts itself
// in at its parent window and, if it is the last child to do so, becomes that window (merge_window), and so on.
template <typename KeyT, bool IS_BOX>
__global__ void __launch_bounds__(kHierThreads, BVH_HIER_MINBLOCKS)
hierarchy_local_kernel(const float* __restrict__ prim, const KeyT* __restrict__ codes, const uint32_t* __restrict__ perm,
                       char* nodes_base, int n, const Header* __restrict__ header, int2* __restrict__ seg_items,
                       int* __restrict__ seg_count) {
  using D = typename Delta<KeyT>::T;
  constexpr int T = kHierThreads, W = kHierWindow, G = W / T, NW = T / 32;
  constexpr int PER_WARP = W / NW;                     // staging slots of a warp = its leaves
  static_assert(NW == 4, "StagedSlots is written for four warps");
  __shared__ LocalSmem<D> smem;
  __shared__ uint32_t s_wsum[NW + 1];
  __shared__ int s_wcount[NW];
  D* const s_delta = smem.delta;
  uint16_t* const s_l = smem.l;
  uint16_t* const s_r = smem.r;
  int* const s_store = smem.store;
  float2* const s_box = smem.box;

  Node* nodes = reinterpret_cast<Node*>(nodes_base + kNodesHeaderBytes);   // internal records, by Karras index
  char* leaves = nodes_base + leaf_offset_bytes(n);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  pdl_wait();
  pdl_trigger();
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
  const int c0 = blockIdx.x * W;
  const int leaf_base = n - 1;
  const int wl0 = c0 + warp * PER_WARP;                        // first leaf of this warp

  // K4: leaf box = box of the primitive sorted to position i.  All loads of the thread's G leaves are issued
  // before anything is consumed: G independent random reads in flight per thread (the gather is what HBM sees).
  uint32_t orig[G];
#pragma unroll
  for (int g = 0; g < G; ++g) {
    const int i = wl0 + g * 32 + lane;
    orig[g] = (i < n) ? __ldcs(perm + i) : 0u;
  }
  // delta* of the warp's own leaves, plus the one before and the one after them: everything phase 0 of this warp reads
  // (the neighbouring warps write the same two values), so the warps need no block barrier before phase 0
#pragma unroll
  for (int g = 0; g < G; ++g) {
    const int k = warp * PER_WARP + g * 32 + lane;             // window slot of this thread's leaf g
    s_delta[k + 1] = delta_star<KeyT>(codes, c0 + k, n);
    s_store[k] = kInvalid;                                     // L1 (read in phase 1, after the barriers below)
  }
  if (lane == 0) s_delta[warp * PER_WARP] = delta_star<KeyT>(codes, wl0 - 1, n);
  if (lane == 1) s_delta[(warp + 1) * PER_WARP + 1] = delta_star<KeyT>(codes, wl0 + PER_WARP, n);
  float plo[G][3], phi[G][IS_BOX ? 3 : 1];
#pragma unroll
  for (int g = 0; g < G; ++g) {
    const int i = wl0 + g * 32 + lane;
    if (IS_BOX) {
      float2 a = make_float2(0.f, 0.f), b = a, c = a;
      if (i < n) {
        const float2* p = reinterpret_cast<const float2*>(prim + 6 * (size_t)orig[g]);
        a = __ldg(p); b = __ldg(p + 1); c = __ldg(p + 2);
      }
      plo[g][0] = a.x; plo[g][1] = a.y; plo[g][2] = b.x; phi[g][0] = b.y; phi[g][1] = c.x; phi[g][2] = c.y;
    } else {
      plo[g][0] = plo[g][1] = plo[g][2] = 0.f;
      if (i < n) {
        const float* p = prim + 3 * (size_t)orig[g];
        plo[g][0] = __ldg(p); plo[g][1] = __ldg(p + 1); plo[g][2] = __ldg(p + 2);
      }
    }
  }
  __syncwarp();

  int wcount = 0;                                              // items this warp has staged (uniform in the warp)
  const uint32_t lt_mask = (1u << lane) - 1u;
#if BVH_HIER_UNROLL_GROUPS
#pragma unroll
#else
#pragma unroll 1
#endif
  for (int g = 0; g < G; ++g) {
    const int w0 = wl0 + g * 32;                               // first leaf of the group
    const int i = w0 + lane;
    const bool valid = i < n;
    const int sd = i - c0;                                     // s_delta[sd] = delta*(i - 1)
    float lo[3], hi[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      // (the selects below are register moves: g is the loop counter of a short unrolled-by-hand switch)
      float l = plo[0][a], h = IS_BOX ? phi[0][a] : plo[0][a];
#pragma unroll
      for (int gg = 1; gg < G; ++gg)
        if (g == gg) {
          l = plo[gg][a];
          h = IS_BOX ? phi[gg][a] : plo[gg][a];
        }
      lo[a] = l;
      hi[a] = h;
    }
    uint32_t og = orig[0];
#pragma unroll
    for (int gg = 1; gg < G; ++gg)
      if (g == gg) og = orig[gg];

    // L3-4
    int range_left = i, range_right = i;
    D delta_left = s_delta[valid ? sd : 0], delta_right = s_delta[valid ? sd + 1 : 0];
    if (valid) {
      // L5-8: leaf skip-connection: L_{i+1} if delta*(i) < delta*(i+1) else I_{i+1} (one bit of the leaf record);
      // the sentinel for the last leaf
      const bool rope_internal = (i != n - 1) && !(delta_right < s_delta[sd + 2]);
      store_leaf<IS_BOX>(leaves, i, lo, hi, og | (rope_internal ? kLeafRopeInternal : 0u));
    }

    // ---- phase 0: rendezvous inside the group, in lockstep ----
    bool active = valid && n > 1;                             // G11: a single leaf has no parent
#pragma unroll
    for (int round = 0; round < kPhase0MaxRounds; ++round) {
      const bool is_left = delta_right < delta_left;          // L10
      const int partner = range_right + 1 - w0;               // lane of leaf r+1
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

    // ---- the subtrees that are left become items of the window: staged by this warp, in leaf order ----
    const uint32_t am = __ballot_sync(0xffffffffu, active);
    if (active) {
      const int slot = warp * PER_WARP + wcount + __popc(am & lt_mask);
      s_l[slot] = (uint16_t)(range_left - c0);
      s_r[slot] = (uint16_t)(range_right - c0);
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        s_box[a * W + slot] = make_float2(lo[a], hi[a]);
      }
    }
    wcount += __popc(am);
  }
  if (lane == 0) s_wcount[warp] = wcount;
  __syncthreads();

  // ---- phase 1: Algorithm 4 over the items of the window ----
  const int c1 = s_wcount[0], c2 = s_wcount[1], c3 = s_wcount[2];
  StagedSlots map;
  map.b1 = c1;
  map.b2 = c1 + c2;
  map.b3 = c1 + c2 + c3;
  map.o0 = 0;
  map.o1 = PER_WARP - map.b1;
  map.o2 = 2 * PER_WARP - map.b2;
  map.o3 = 3 * PER_WARP - map.b3;
  const int M = map.b3 + s_wcount[3];
  const ItemArrays<uint16_t> A{s_l, s_r, c0, s_box, W, s_store};
  ClimbEnd end[G];
#if BVH_HIER_SLOT_TABLE
  using SlotT = typename SlotType<(W <= 256)>::T;
  __shared__ SlotT s_slot[W];
#pragma unroll
  for (int j = 0; j < G; ++j) {
    const int e = tid + j * T;
    if (e < M) s_slot[e] = (SlotT)map.slot(e);
  }
  __syncthreads();
  const TableSlots<SlotT> slots{s_slot};
#else
  const StagedSlots& slots = map;
#endif
#pragma unroll
  for (int j = 0; j < G; ++j) {
    end[j] = ClimbEnd{0, 0, -2};
    const int e = tid + j * T;
    if (e < M) end[j] = climb_from_item<D>(e, M, A, DeltaByLeaf<D>{s_delta, c0}, slots, nodes, n);
  }
  __syncthreads();

  // ---- hand over what is left of this window, in leaf order (at most kSegCap subtrees) ----
  int base = 0;
#pragma unroll
  for (int j = 0; j < G; ++j) {
    if (j * T >= M && j > 0) break;                                             // uniform
    const bool surv = (tid + j * T < M) && climb_survives(A, end[j]);
    int total;
    const int pos = block_compact(surv, s_wsum, NW, total);
    if (surv) seg_items[(size_t)blockIdx.x * kSegCap + base + pos] = make_int2(end[j].l, end[j].r);
    base += total;
  }
  if (tid == 0) seg_count[blockIdx.x] = base;

}

// Levels 2 and up: block b starts as window b of level 2 and climbs while it is the last child to arrive.
template <typename KeyT>
__global__ void __launch_bounds__(kMergeThreads)
hierarchy_merge_kernel(const KeyT* __restrict__ codes, char* nodes_base, int n, int leaf_kind, int2* seg_items,
                       int* seg_count, uint32_t* arrivals, const HierLevels lv) {
  using D = typename Delta<KeyT>::T;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  MergeSmem<D>& S = *reinterpret_cast<MergeSmem<D>*>(smem_raw);
  __shared__ uint32_t s_wsum[kMergeThreads / 32 + 1];
  __shared__ int s_last;
  const int tid = threadIdx.x;
  pdl_wait();
  pdl_trigger();
  int window = blockIdx.x;
  for (int level = 1; level < lv.levels; ++level) {     // array index of the level this block is a window of
    merge_window<KeyT>(S, s_wsum, codes, nodes_base, n, leaf_kind, window,
                       seg_items + (size_t)lv.seg_off[level - 1] * kSegCap, seg_count + lv.seg_off[level - 1],
                       lv.segs[level - 1], seg_items + ((size_t)lv.seg_off[level] + window) * kSegCap,
                       seg_count + lv.seg_off[level] + window);
    if (level + 1 == lv.levels) return;                 // that was the whole tree
    __threadfence();                                    // hand-over and node records before the arrival
    __syncthreads();
    const int parent = window / kMergeFan;
    if (tid == 0) {
      const int children = min(kMergeFan, lv.segs[level] - parent * kMergeFan);
      const uint32_t before = atomicAdd(arrivals + lv.seg_off[level + 1] + parent, 1u);
      s_last = (before == (uint32_t)(children - 1));
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();                                    // the other children's hand-over, written before their arrival
    window = parent;
  }
}

// Windows per level: level 1 has ceil(n / kHierWindow), each further level ceil(previous / kMergeFan), down to 1.
int hierarchy_levels(int n, int segs[kMaxHierLevels]) {
  int levels = 0;
  int s = (n + kHierWindow - 1) / kHierWindow;
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
static cudaError_t launch_hierarchy_keys(const float* prim, bool is_box, const KeyT* codes, const uint32_t* perm, char* nodes,
                                         int n, const Header* header, int2* seg_items, int* seg_count, uint32_t* arrivals,
                                         cudaStream_t stream) {
  HierLevels lv{};
  lv.levels = hierarchy_levels(n, lv.segs);
  int off = 0;
  for (int l = 0; l < lv.levels; ++l) {
    lv.seg_off[l] = off;
    off += lv.segs[l];
  }
  cudaError_t e;
  if (is_box)
    e = launch_pdl(hierarchy_local_kernel<KeyT, true>, dim3(lv.segs[0]), dim3(kHierThreads), 0, stream, prim, codes, perm, nodes,
                   n, header, seg_items, seg_count);
  else
    e = launch_pdl(hierarchy_local_kernel<KeyT, false>, dim3(lv.segs[0]), dim3(kHierThreads), 0, stream, prim, codes, perm, nodes,
                   n, header, seg_items, seg_count);
  if (e != cudaSuccess || lv.levels <= 1) return e;
  using D = typename Delta<KeyT>::T;
  const size_t smem = sizeof(MergeSmem<D>);
  // the opt-in to more than 48 KB of dynamic shared memory holds for the device that was current: once per device
  static PerDeviceOnce once;   // (one per KeyT instantiation)
  const cudaError_t attr = once_per_device(once, nullptr, [&](int* done) {
    *done = 1;
    return cudaFuncSetAttribute(hierarchy_merge_kernel<KeyT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  });
  if (attr != cudaSuccess) return attr;
  return launch_pdl(hierarchy_merge_kernel<KeyT>, dim3(lv.segs[1]), dim3(kMergeThreads), smem, stream, codes, nodes, n,
                    is_box ? kLeafBoxes : kLeafPoints, seg_items, seg_count, arrivals, lv);
}

cudaError_t launch_hierarchy(const float* prim, bool is_box, const void* sorted_codes, int key_bytes, const uint32_t* perm,
                             void* nodes, int n, const Header* header, int2* seg_items, int* seg_count, uint32_t* arrivals,
                             cudaStream_t stream) {
  if (key_bytes == 4)
    return launch_hierarchy_keys<uint32_t>(prim, is_box, static_cast<const uint32_t*>(sorted_codes), perm,
                                           static_cast<char*>(nodes), n, header, seg_items, seg_count, arrivals, stream);
  return launch_hierarchy_keys<uint64_t>(prim, is_box, static_cast<const uint64_t*>(sorted_codes), perm,
                                         static_cast<char*>(nodes), n, header, seg_items, seg_count, arrivals, stream);
}

int hierarchy_seg_capacity() { return kSegCap; }
int hierarchy_fan() { return kMergeFan; }

}  // namespace bvh
