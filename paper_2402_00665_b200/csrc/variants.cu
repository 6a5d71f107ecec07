// variants.cu -- NEXT-2: the construction the paper compares itself with, built to MEASURE the
// paper's claim on B200, not as a product path.  The paper says the bottom-up merge is "a faster algorithm" than
// Karras' per-node search and that Karras needs "a separate bottom-up pass for boxes"
// (PAPER.md:93); it gives no number.  bvh_build_variant(variant = 1) replaces the last step of the build (K4+K5,
// hierarchy.cu) by exactly that:
//   1. karras_leaf_kernel      leaf records (permuted gather) and leaf skip-connections (Alg. 4 L5-8, same as K4);
//   2. karras_topdown_kernel   one thread per internal node i: range by the direction / doubling / binary search on
//                              the common-prefix length delta(i, j) of the augmented keys, split by binary search
//                              (Karras 2012 as the paper restates it), children at the split
//                              (gamma, gamma + 1), skip-connection by Algorithm 2 from the
//                              node's own range, parent pointers of both children;
//   3. karras_box_kernel       boxes bottom-up: every leaf walks up; at a parent the first child to arrive stops
//                              (atomic counter in global memory), the second reads both children's boxes through
//                              L2, writes the parent's record and carries on.
// Bounds, Morton codes, sort, node layout and leaf format are the product's, so the resulting `nodes` buffer must be
// byte-identical to the one Algorithm 4 produces (tests/test_gpu_parity.py::test_variant_karras_topdown).
#include "../../include/bvh_b200.h"
#include "common.cuh"

namespace bvh {

// Common-prefix length of the augmented keys (code, sorted position) i and j; -1 outside [0, n-1].
template <typename KeyT>
__device__ __forceinline__ int prefix_len(const KeyT* __restrict__ codes, int n, KeyT ci, int i, int j) {
  if (j < 0 || j >= n) return -1;
  const KeyT cj = codes[j];
  if (sizeof(KeyT) == 4) {
    const uint64_t x = ((uint64_t)(uint32_t)(ci ^ cj) << 32) | (uint32_t)(i ^ j);
    return __clzll((long long)x);
  } else {
    const uint64_t x = (uint64_t)(ci ^ cj);
    return x ? __clzll((long long)x) : 64 + __clz(i ^ j);
  }
}

struct VariantScratch {
  int32_t* parent;   // [2n-1] parent of every node of the unified index space
  uint32_t* flags;   // [n-1]   variant 1: children arrived at each internal node (zeroed); variant 2: Algorithm 3's `store`
  int32_t* left;     // [n-1]   left child, by Karras index (variant 1)
  int32_t* right;    // [n-1]   right child (variant 1: Karras index; variant 2: Apetrei index)
  int32_t* rope;     // [n-1]   skip-connection, by Karras index (variant 1)
  int32_t* leaf_rope;  // [n]   variant 2: skip-connection of every leaf (an Apetrei index does not fit the leaf record's one bit)
};
static inline size_t align256(size_t x) { return (x + 255) / 256 * 256; }
size_t variant_extra_bytes(int64_t n) {
  const size_t nn = (size_t)(n > 0 ? n : 1);
  return align256(4 * (2 * nn)) + 5 * align256(4 * nn);
}
static VariantScratch variant_scratch(char* base, int64_t n) {
  const size_t nn = (size_t)(n > 0 ? n : 1);
  VariantScratch v;
  v.parent = reinterpret_cast<int32_t*>(base);
  base += align256(4 * (2 * nn));
  v.flags = reinterpret_cast<uint32_t*>(base);
  base += align256(4 * nn);
  v.left = reinterpret_cast<int32_t*>(base);
  base += align256(4 * nn);
  v.right = reinterpret_cast<int32_t*>(base);
  base += align256(4 * nn);
  v.rope = reinterpret_cast<int32_t*>(base);
  base += align256(4 * nn);
  v.leaf_rope = reinterpret_cast<int32_t*>(base);
  return v;
}

template <typename KeyT, bool IS_BOX>
__global__ void __launch_bounds__(256)
karras_leaf_kernel(const float* __restrict__ prim, const KeyT* __restrict__ codes, const uint32_t* __restrict__ perm,
                   char* nodes_base, int n, const Header* __restrict__ header) {
  pdl_wait();
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0) {
    NodesHeader* h = reinterpret_cast<NodesHeader*>(nodes_base);
    float sb[6];
    load_scene_bounds(header, sb);
    h->magic = kNodesMagic;
    h->n = n;
    h->leaf_kind = IS_BOX ? kLeafBoxes : kLeafPoints;
    h->reserved = 0;
    for (int a = 0; a < 3; ++a) {
      h->scene_lo[a] = sb[a];
      h->scene_hi[a] = sb[3 + a];
    }
  }
  if (i >= n) return;
  const uint32_t o = perm[i];
  const KeyT ci = codes[i];
  // leaf skip-connection (Algorithm 2 for a leaf): leaf i+1 if keys i, i+1 share a longer prefix than i+1, i+2
  const bool rope_internal = (i != n - 1) && !(prefix_len(codes, n, ci, i, i + 1) > prefix_len(codes, n, codes[i + 1], i + 1, i + 2));
  const uint32_t payload = o | (rope_internal ? kLeafRopeInternal : 0u);
  char* leaves = nodes_base + leaf_offset_bytes(n);
  if (IS_BOX) {
    const float2* p = reinterpret_cast<const float2*>(prim + 6 * (size_t)o);
    const float2 a = __ldg(p), b = __ldg(p + 1), c = __ldg(p + 2);
    float4* rec = reinterpret_cast<float4*>(leaves + 32 * (size_t)i);
    rec[0] = make_float4(a.x, a.y, b.x, __uint_as_float(payload));
    rec[1] = make_float4(b.y, c.x, c.y, 0.0f);
  } else {
    const float* p = prim + 3 * (size_t)o;
    reinterpret_cast<float4*>(leaves)[i] = make_float4(__ldg(p), __ldg(p + 1), __ldg(p + 2), __uint_as_float(payload));
  }
}

template <typename KeyT>
__global__ void __launch_bounds__(256)
karras_topdown_kernel(const KeyT* __restrict__ codes, int n, VariantScratch v) {
  pdl_wait();
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n - 1) return;
  const int leaf_base = n - 1;
  const KeyT ci = codes[i];
  auto delta = [&](int j) { return prefix_len(codes, n, ci, i, j); };
  // direction of the range and the prefix every key of the range shares beyond its neighbour on the other side
  const int d = (delta(i + 1) - delta(i - 1)) < 0 ? -1 : 1;
  const int dmin = delta(i - d);
  int lmax = 2;
  while (delta(i + lmax * d) > dmin) lmax <<= 1;            // upper bound of the range length
  int l = 0;
  for (int t = lmax >> 1; t >= 1; t >>= 1)
    if (delta(i + (l + t) * d) > dmin) l += t;               // the other end, by binary search
  const int j = i + l * d;
  const int dnode = delta(j);
  int s = 0;                                                 // split: the last key that shares more than dnode with key i
  for (int t = (l + 1) >> 1;; t = (t + 1) >> 1) {
    if (delta(i + (s + t) * d) > dnode) s += t;
    if (t == 1) break;
  }
  const int gamma = i + s * d + min(d, 0);
  const int first = min(i, j), last = max(i, j);
  const int left = (first == gamma) ? leaf_base + gamma : gamma;          // children at gamma, gamma + 1
  const int right = (last == gamma + 1) ? leaf_base + gamma + 1 : gamma + 1;
  // Algorithm 2: the skip-connection is the node whose range starts at last + 1
  int rope = kSentinel;
  if (last != n - 1) {
    const int r = last + 1;
    const KeyT cr = codes[r];
    rope = (prefix_len(codes, n, cr, r, r - 1) > prefix_len(codes, n, cr, r, r + 1)) ? leaf_base + r : r;
  }
  v.left[i] = left;
  v.right[i] = right;
  v.rope[i] = rope;
  v.parent[left] = i;
  v.parent[right] = i;
  if (i == 0) v.parent[0] = kSentinel;
}

__device__ __forceinline__ void load_box_any(const char* nodes, int n, int leaf_kind, int idx, float lo[3], float hi[3]) {
  const int leaf_base = n - 1;
  if (idx >= leaf_base && leaf_kind == kLeafPoints) {
    const float4 p = __ldcg(reinterpret_cast<const float4*>(nodes + leaf_offset_bytes(n)) + (idx - leaf_base));
    lo[0] = hi[0] = p.x; lo[1] = hi[1] = p.y; lo[2] = hi[2] = p.z;
  } else {
    const Node* rec = (idx >= leaf_base) ? reinterpret_cast<const Node*>(nodes + leaf_offset_bytes(n)) + (idx - leaf_base)
                                         : reinterpret_cast<const Node*>(nodes + kNodesHeaderBytes) + idx;
    const float4 a = __ldcg(reinterpret_cast<const float4*>(rec));
    const float4 b = __ldcg(reinterpret_cast<const float4*>(rec) + 1);
    lo[0] = a.x; lo[1] = a.y; lo[2] = a.z; hi[0] = b.x; hi[1] = b.y; hi[2] = b.z;
  }
}

// Boxes, bottom-up (the "separate bottom-up pass" of PAPER.md:93).
__global__ void __launch_bounds__(256) karras_box_kernel(char* nodes_base, int n, int leaf_kind, VariantScratch v) {
  pdl_wait();
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n || n < 2) return;
  const int leaf_base = n - 1;
  Node* internal = reinterpret_cast<Node*>(nodes_base + kNodesHeaderBytes);
  int node = leaf_base + i;
  while (true) {
    const int p = v.parent[node];
    if (p < 0) return;                                       // the root is done
    __threadfence();                                         // this child's record before its arrival
    if (atomicAdd(&v.flags[p], 1u) == 0u) return;            // first child to arrive stops
    __threadfence();
    const int left = v.left[p], rc = v.right[p];
    float lo[3], hi[3], lo2[3], hi2[3];
    load_box_any(nodes_base, n, leaf_kind, left, lo, hi);
    load_box_any(nodes_base, n, leaf_kind, rc, lo2, hi2);
    for (int a = 0; a < 3; ++a) {
      lo[a] = fminf(lo[a], lo2[a]);
      hi[a] = fmaxf(hi[a], hi2[a]);
    }
    Node rec;
    rec.lo = make_float4(lo[0], lo[1], lo[2], __int_as_float(left));
    rec.hi = make_float4(hi[0], hi[1], hi[2], __int_as_float(v.rope[p]));
    internal[p] = rec;
    node = p;
  }
}

template <typename KeyT>
static cudaError_t launch_variant_keys(const float* prim, bool is_box, const KeyT* codes, const uint32_t* perm, char* nodes, int n,
                                       const Header* header, VariantScratch v, cudaStream_t stream) {
  const unsigned gl = (unsigned)((n + 255) / 256);
  cudaError_t e;
  if (is_box)
    e = launch_pdl(karras_leaf_kernel<KeyT, true>, dim3(gl), dim3(256), 0, stream, prim, codes, perm, nodes, n, header);
  else
    e = launch_pdl(karras_leaf_kernel<KeyT, false>, dim3(gl), dim3(256), 0, stream, prim, codes, perm, nodes, n, header);
  if (e != cudaSuccess || n < 2) return e;
  e = launch_pdl(karras_topdown_kernel<KeyT>, dim3((unsigned)((n - 1 + 255) / 256)), dim3(256), 0, stream, codes, n, v);
  if (e != cudaSuccess) return e;
  return launch_pdl(karras_box_kernel, dim3(gl), dim3(256), 0, stream, nodes, n, is_box ? kLeafBoxes : kLeafPoints, v);
}

// ---------------------------------------------------------------------------------------------------------------------
// variant 2: the UNMODIFIED Algorithm 3, followed by what the paper's modification removes: "an
// extra tree traversal pass" that installs the skip-connections.  Internal nodes are numbered by
// their split position p, both children write themselves into the parent before the ATOMICCAS on
// `store` (L7-8, L13-14), the first arrival stops, the second merges the boxes (G10: the sibling's box is read back
// through L2 after a fence) and carries on; the node whose range is [0, n-1] is the root and its index is stored in
// the header.  The records are the product's {min, left | max, rope}, indexed by Apetrei index; the
// right child, which the product never stores (Karras numbering: it is left + 1), goes to the variant's scratch, as
// do the leaves' skip-connections.  The product's traversal relies on Karras numbering (the skip target's index is
// the first leaf after the subtree), so this hierarchy is not handed to it: its header carries another magic.
constexpr uint32_t kNodesMagicApetrei = 0x42564133u;   // "BVA3"

template <typename KeyT>
__global__ void __launch_bounds__(256)
apetrei_kernel(const KeyT* __restrict__ codes, char* nodes_base, int n, int leaf_kind, VariantScratch v) {
  pdl_wait();
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n || n < 2) return;
  const int leaf_base = n - 1;
  Node* internal = reinterpret_cast<Node*>(nodes_base + kNodesHeaderBytes);
  int* store = reinterpret_cast<int*>(v.flags);
  auto dstar = [&](int a) { return (a < 0 || a >= n - 1) ? -1 : prefix_len(codes, n, codes[a], a, a + 1); };   // larger = more similar
  int cur = leaf_base + i;                                   // the node this thread has just completed
  int range_left = i, range_right = i;                       // L3-4
  int sim_left = dstar(i - 1), sim_right = dstar(i);         // delta*(l-1), delta*(r) as prefix lengths: delta_right < delta_left <=> sim_right > sim_left
  float lo[3], hi[3];
  load_box_any(nodes_base, n, leaf_kind, cur, lo, hi);
  while (true) {
    const bool is_left = sim_right > sim_left;               // L5
    const int p = is_left ? range_right : range_left - 1;    // L6 / L12: Apetrei index = split
    if (is_left)
      reinterpret_cast<int*>(internal + p)[3] = cur;         // L7: I_p.left
    else
      v.right[p] = cur;                                      // L13: I_p.right
    v.parent[cur] = p;                                       // (for the skip-connection pass)
    __threadfence();                                         // this child's record and pointer before its arrival
    const int other = atomicCAS(store + p, kInvalid, is_left ? range_left : range_right);   // L8 / L14
    if (other == kInvalid) return;                           // L9 / L15: first to arrive
    __threadfence();
    int sib;
    if (is_left) {
      range_right = other;
      sim_right = dstar(range_right);                        // L10
      sib = __ldcg(v.right + p);
    } else {
      range_left = other;
      sim_left = dstar(range_left - 1);                      // L16
      sib = __ldcg(reinterpret_cast<const int*>(internal + p) + 3);
    }
    float lo2[3], hi2[3];
    load_box_any(nodes_base, n, leaf_kind, sib, lo2, hi2);
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      lo[a] = fminf(lo[a], lo2[a]);
      hi[a] = fmaxf(hi[a], hi2[a]);
    }
    Node rec;
    rec.lo = make_float4(lo[0], lo[1], lo[2], __int_as_float(is_left ? cur : sib));
    rec.hi = make_float4(hi[0], hi[1], hi[2], __int_as_float(kSentinel));   // the skip-connection comes with the next pass
    internal[p] = rec;
    cur = p;                                                 // L18
    if (range_left == 0 && range_right == n - 1) {           // L19: the root; "its index now needs to be stored"
      reinterpret_cast<NodesHeader*>(nodes_base)->reserved = p;
      v.parent[p] = kSentinel;
      return;
    }
  }
}

// The extra pass: the skip-connection of a node is the right child of the nearest ancestor (itself
// included) that is a left child's parent ... i.e. walk up while the node is a right child; the sibling of the first
// left child on the way is the target; the right-most path ends at the sentinel.
__global__ void __launch_bounds__(256) apetrei_rope_kernel(char* nodes_base, int n, VariantScratch v) {
  pdl_wait();
  const int x = blockIdx.x * blockDim.x + threadIdx.x;
  if (x == 0) reinterpret_cast<NodesHeader*>(nodes_base)->magic = kNodesMagicApetrei;
  if (x >= 2 * n - 1) return;
  const int leaf_base = n - 1;
  const Node* internal = reinterpret_cast<const Node*>(nodes_base + kNodesHeaderBytes);
  int rope = kSentinel;
  if (n >= 2) {
    int c = x;
    while (true) {
      const int p = v.parent[c];
      if (p < 0) break;
      if (reinterpret_cast<const int*>(internal + p)[3] == c) {   // c is the left child of p
        rope = v.right[p];
        break;
      }
      c = p;
    }
  }
  if (x < leaf_base)
    reinterpret_cast<int*>(const_cast<Node*>(internal) + x)[7] = rope;
  else
    v.leaf_rope[x - leaf_base] = rope;
}

template <typename KeyT>
static cudaError_t launch_apetrei_keys(const float* prim, bool is_box, const KeyT* codes, const uint32_t* perm, char* nodes, int n,
                                       const Header* header, VariantScratch v, cudaStream_t stream) {
  const unsigned gl = (unsigned)((n + 255) / 256);
  cudaError_t e;
  if (is_box)
    e = launch_pdl(karras_leaf_kernel<KeyT, true>, dim3(gl), dim3(256), 0, stream, prim, codes, perm, nodes, n, header);
  else
    e = launch_pdl(karras_leaf_kernel<KeyT, false>, dim3(gl), dim3(256), 0, stream, prim, codes, perm, nodes, n, header);
  if (e != cudaSuccess) return e;
  e = launch_pdl(apetrei_kernel<KeyT>, dim3(gl), dim3(256), 0, stream, codes, nodes, n, is_box ? kLeafBoxes : kLeafPoints, v);
  if (e != cudaSuccess) return e;
  return launch_pdl(apetrei_rope_kernel, dim3((unsigned)((2 * (int64_t)n - 1 + 255) / 256)), dim3(256), 0, stream, nodes, n, v);
}

// ---------------------------------------------------------------------------------------------------------------------
// variant 3: Algorithm 4 AS THE PAPER WRITES IT, in the same plain form as variant 2: one thread per
// leaf, `store` in global memory initialised to the invalid value (L1), ATOMICCAS (L12 / L17), the first thread to arrive
// at a parent stops (L13 / L18), the second extends its range by the sibling's (L14 / L19), numbers the parent with its
// Karras index q (L20: the right end of the range if the parent is itself a left child, else the left end), writes the
// left child (L21, reading G2: L_p if the left range is the single leaf p, else I_p) and the skip-connection (L22-26:
// sentinel on the right-most path, else leaf or internal node r = range_right + 1 by comparing delta*(range_right) with
// delta*(r)), and -- G10 -- the union of its own box with the sibling's, read back through L2 after a fence.  No shared
// memory, no windows, no lock-step rounds: against variant 2 (Algorithm 3 + the extra skip-connection pass) this isolates
// what the paper's MODIFICATION saves; against the product (hierarchy.cu) it shows what the windowed organisation adds.
// The sibling needs no pointer exchange: with Karras numbering its index follows from the ranges (the left child of split
// p is L_p / I_p, the right child L_{p+1} / I_{p+1}).  `nodes` comes out byte-identical to the product's.
template <typename KeyT>
__global__ void __launch_bounds__(256)
alg4_plain_kernel(const KeyT* __restrict__ codes, char* nodes_base, int n, int leaf_kind, VariantScratch v) {
  pdl_wait();
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n || n < 2) return;
  const int leaf_base = n - 1;
  Node* internal = reinterpret_cast<Node*>(nodes_base + kNodesHeaderBytes);
  int* store = reinterpret_cast<int*>(v.flags);
  auto sim = [&](int a) { return (a < 0 || a >= n - 1) ? -1 : prefix_len(codes, n, codes[a], a, a + 1); };   // larger = smaller delta*
  int range_left = i, range_right = i;                       // L2
  int sim_left = sim(i - 1), sim_right = sim(i);             // L3-4 (the leaf's own skip-connection, L5-8: karras_leaf_kernel)
  float lo[3], hi[3];
  load_box_any(nodes_base, n, leaf_kind, leaf_base + i, lo, hi);
  while (true) {
    const bool is_left = sim_right > sim_left;               // L10: delta_right < delta_left
    const int p = is_left ? range_right : range_left - 1;    // L11 / L16: the split of the parent
    __threadfence();                                         // this node's record before its arrival
    const int other = atomicCAS(store + p, kInvalid, is_left ? range_left : range_right);   // L12 / L17
    if (other == kInvalid) return;                           // L13 / L18
    __threadfence();
    int sib;
    if (is_left) {
      range_right = other;                                   // L14
      sim_right = sim(range_right);
      sib = (range_right == p + 1) ? leaf_base + p + 1 : p + 1;
    } else {
      range_left = other;                                    // L19
      sim_left = sim(range_left - 1);
      sib = (range_left == p) ? leaf_base + p : p;
    }
    const int q = (sim_right > sim_left) ? range_right : range_left;            // L20
    const int left = (range_left == p) ? leaf_base + p : p;                     // L21
    int rope = kSentinel;                                                       // L22-23
    if (range_right != n - 1) {
      const int r = range_right + 1;                                            // L25
      rope = (sim_right > sim(r)) ? leaf_base + r : r;                          // L26: delta*(range_right) < delta*(r) -> leaf
    }
    float lo2[3], hi2[3];
    load_box_any(nodes_base, n, leaf_kind, sib, lo2, hi2);
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      lo[a] = fminf(lo[a], lo2[a]);
      hi[a] = fmaxf(hi[a], hi2[a]);
    }
    Node rec;
    rec.lo = make_float4(lo[0], lo[1], lo[2], __int_as_float(left));
    rec.hi = make_float4(hi[0], hi[1], hi[2], __int_as_float(rope));
    internal[q] = rec;
    if (q == 0) return;                                      // L28: the root
  }
}

template <typename KeyT>
static cudaError_t launch_alg4_keys(const float* prim, bool is_box, const KeyT* codes, const uint32_t* perm, char* nodes, int n,
                                    const Header* header, VariantScratch v, cudaStream_t stream) {
  const unsigned gl = (unsigned)((n + 255) / 256);
  cudaError_t e;
  if (is_box)
    e = launch_pdl(karras_leaf_kernel<KeyT, true>, dim3(gl), dim3(256), 0, stream, prim, codes, perm, nodes, n, header);
  else
    e = launch_pdl(karras_leaf_kernel<KeyT, false>, dim3(gl), dim3(256), 0, stream, prim, codes, perm, nodes, n, header);
  if (e != cudaSuccess) return e;
  return launch_pdl(alg4_plain_kernel<KeyT>, dim3(gl), dim3(256), 0, stream, codes, nodes, n, is_box ? kLeafBoxes : kLeafPoints, v);
}

int launch_variant_alg4(const float* prim, bool is_box, const void* sorted_codes, int key_bytes, const uint32_t* perm,
                        void* nodes, int n, const Header* header, void* extra, cudaStream_t stream) {
  VariantScratch v = variant_scratch(static_cast<char*>(extra), n);
  if (n >= 2 && cudaMemsetAsync(v.flags, 0xFF, sizeof(uint32_t) * (size_t)(n - 1), stream) != cudaSuccess) return -1;   // store <- invalid (L1)
  cudaError_t e;
  if (key_bytes == 4)
    e = launch_alg4_keys<uint32_t>(prim, is_box, static_cast<const uint32_t*>(sorted_codes), perm, static_cast<char*>(nodes), n,
                                   header, v, stream);
  else
    e = launch_alg4_keys<uint64_t>(prim, is_box, static_cast<const uint64_t*>(sorted_codes), perm, static_cast<char*>(nodes), n,
                                   header, v, stream);
  return e == cudaSuccess ? 0 : -1;
}

// variant 2 export: the arrays of the Apetrei-numbered hierarchy in the unified index space (internal I_p -> p).
__global__ void apetrei_export_kernel(const char* __restrict__ nodes, VariantScratch v, int n, int32_t* left, int32_t* right,
                                      int32_t* rope, float* aabb, int32_t* root) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int leaf_base = n - 1;
  const NodesHeader* h = reinterpret_cast<const NodesHeader*>(nodes);
  if (i == 0 && root) *root = n >= 2 ? h->reserved : 0;
  if (i >= 2 * (int64_t)n - 1) return;
  float lo[3], hi[3];
  if (i < leaf_base) {
    const Node* rec = reinterpret_cast<const Node*>(nodes + kNodesHeaderBytes) + i;
    const float4 a = rec->lo, b = rec->hi;
    lo[0] = a.x; lo[1] = a.y; lo[2] = a.z; hi[0] = b.x; hi[1] = b.y; hi[2] = b.z;
    if (left) left[i] = __float_as_int(a.w);
    if (right) right[i] = v.right[i];
    if (rope) rope[i] = __float_as_int(b.w);
  } else {
    const int li = (int)(i - leaf_base);
    const char* leaves = nodes + leaf_offset_bytes(n);
    if (h->leaf_kind == kLeafPoints) {
      const float4 p = reinterpret_cast<const float4*>(leaves)[li];
      lo[0] = hi[0] = p.x; lo[1] = hi[1] = p.y; lo[2] = hi[2] = p.z;
    } else {
      const Node* rec = reinterpret_cast<const Node*>(leaves) + li;
      const float4 a = rec->lo, b = rec->hi;
      lo[0] = a.x; lo[1] = a.y; lo[2] = a.z; hi[0] = b.x; hi[1] = b.y; hi[2] = b.z;
    }
    if (rope) rope[i] = v.leaf_rope[li];
  }
  if (aabb) {
    float* o = aabb + 6 * i;
    o[0] = lo[0]; o[1] = lo[1]; o[2] = lo[2]; o[3] = hi[0]; o[4] = hi[1]; o[5] = hi[2];
  }
}

int launch_variant_apetrei_export(const void* nodes, void* extra, int n, int32_t* left, int32_t* right, int32_t* rope,
                                  float* aabb, int32_t* root, cudaStream_t stream) {
  VariantScratch v = variant_scratch(static_cast<char*>(extra), n);
  const int64_t total = 2 * (int64_t)n - 1;
  apetrei_export_kernel<<<(unsigned)((total + 255) / 256), 256, 0, stream>>>(static_cast<const char*>(nodes), v, n, left, right,
                                                                            rope, aabb, root);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

int launch_variant_apetrei(const float* prim, bool is_box, const void* sorted_codes, int key_bytes, const uint32_t* perm,
                           void* nodes, int n, const Header* header, void* extra, cudaStream_t stream) {
  VariantScratch v = variant_scratch(static_cast<char*>(extra), n);
  if (n >= 2 && cudaMemsetAsync(v.flags, 0xFF, sizeof(uint32_t) * (size_t)(n - 1), stream) != cudaSuccess) return -1;   // store <- invalid (L1)
  cudaError_t e;
  if (key_bytes == 4)
    e = launch_apetrei_keys<uint32_t>(prim, is_box, static_cast<const uint32_t*>(sorted_codes), perm, static_cast<char*>(nodes),
                                      n, header, v, stream);
  else
    e = launch_apetrei_keys<uint64_t>(prim, is_box, static_cast<const uint64_t*>(sorted_codes), perm, static_cast<char*>(nodes),
                                      n, header, v, stream);
  return e == cudaSuccess ? 0 : -1;
}

// The last step of the build, Karras-style.  extra: variant_extra_bytes(n) of scratch after the product's layout.
int launch_variant_karras(const float* prim, bool is_box, const void* sorted_codes, int key_bytes, const uint32_t* perm,
                          void* nodes, int n, const Header* header, void* extra, cudaStream_t stream) {
  VariantScratch v = variant_scratch(static_cast<char*>(extra), n);
  if (n >= 2 && cudaMemsetAsync(v.flags, 0, sizeof(uint32_t) * (size_t)(n - 1), stream) != cudaSuccess) return -1;
  cudaError_t e;
  if (key_bytes == 4)
    e = launch_variant_keys<uint32_t>(prim, is_box, static_cast<const uint32_t*>(sorted_codes), perm, static_cast<char*>(nodes), n,
                                      header, v, stream);
  else
    e = launch_variant_keys<uint64_t>(prim, is_box, static_cast<const uint64_t*>(sorted_codes), perm, static_cast<char*>(nodes), n,
                                      header, v, stream);
  return e == cudaSuccess ? 0 : -1;
}

}  // namespace bvh
