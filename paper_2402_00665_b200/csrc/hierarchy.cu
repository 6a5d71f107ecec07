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

constexpr int kHierThreads = 256;

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

__device__ __forceinline__ void store_node(Node* nodes, int idx, float lo0, float lo1, float lo2, float hi0, float hi1,
                                           float hi2, int left, int rope) {
  float4* p = reinterpret_cast<float4*>(nodes + idx);
  p[0] = make_float4(lo0, lo1, lo2, __int_as_float(left));
  p[1] = make_float4(hi0, hi1, hi2, __int_as_float(rope));
}

template <typename KeyT, bool IS_BOX>
__global__ void __launch_bounds__(kHierThreads)
hierarchy_kernel(const float* __restrict__ prim, const KeyT* __restrict__ codes, const uint32_t* __restrict__ perm,
                 int* store, Node* nodes, int n) {
  using D = typename Delta<KeyT>::T;
  const int i0 = blockIdx.x * kHierThreads + threadIdx.x;
  if (i0 >= n) return;
  const int leaf_base = n - 1;
  int i = i0;

  // L3-4
  int range_left = i, range_right = i;
  D delta_left = delta_star<KeyT>(codes, i - 1, n);
  D delta_right = delta_star<KeyT>(codes, i, n);

  // leaf box = box of the primitive sorted to position i (K4)
  const uint32_t orig = perm[i];
  float lo[3], hi[3];
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
  // L5-8: leaf skip-connection
  int rope;
  if (i == n - 1)
    rope = kSentinel;
  else
    rope = (delta_right < delta_star<KeyT>(codes, i + 1, n)) ? leaf_base + i + 1 : i + 1;
  store_node(nodes, leaf_base + i, lo[0], lo[1], lo[2], hi[0], hi[1], hi[2], (int)orig, rope);
  if (n == 1) return;  // G11

  // L9-28
  do {
    // the node this thread carries (leaf or internal `i`) is fully written: publish before arriving
    __threadfence();
    int p, sibling;
    if (delta_right < delta_left) {       // L10: left child of its parent
      p = range_right;                    // L11: Apetrei index
      const int other = atomicCAS(&store[p], kInvalid, range_left);  // L12
      if (other == kInvalid) return;      // L13: first to arrive
      range_right = other;
      sibling = (range_right == p + 1) ? leaf_base + p + 1 : p + 1;  // right child: L_{p+1} or I_{p+1}
      delta_right = delta_star<KeyT>(codes, range_right, n);  // L14
    } else {                              // right child of its parent
      p = range_left - 1;                 // L16
      const int other = atomicCAS(&store[p], kInvalid, range_right);  // L17
      if (other == kInvalid) return;      // L18
      range_left = other;
      sibling = (range_left == p) ? leaf_base + p : p;               // left child: L_p or I_p
      delta_left = delta_star<KeyT>(codes, range_left - 1, n);  // L19
    }
    __threadfence();  // acquire side: the sibling's record was written before its CAS
    const float4 slo = __ldcg(reinterpret_cast<const float4*>(nodes + sibling));
    const float4 shi = __ldcg(reinterpret_cast<const float4*>(nodes + sibling) + 1);
    lo[0] = fminf(lo[0], slo.x); lo[1] = fminf(lo[1], slo.y); lo[2] = fminf(lo[2], slo.z);
    hi[0] = fmaxf(hi[0], shi.x); hi[1] = fmaxf(hi[1], shi.y); hi[2] = fmaxf(hi[2], shi.z);

    const int q = (delta_right < delta_left) ? range_right : range_left;       // L20: Karras index
    const int left = (range_left == p) ? leaf_base + p : p;                    // L21 (reading G2)
    if (range_right == n - 1) {                                                // L22-23
      rope = kSentinel;
    } else {
      const int r = range_right + 1;                                           // L25
      rope = (delta_right < delta_star<KeyT>(codes, r, n)) ? leaf_base + r : r;  // L26
    }
    store_node(nodes, q, lo[0], lo[1], lo[2], hi[0], hi[1], hi[2], left, rope);
    i = q;                                                                     // L27
  } while (i != 0);                                                            // L28
}

void launch_hierarchy(const float* prim, bool is_box, const void* sorted_codes, int key_bytes, const uint32_t* perm,
                      int* store, Node* nodes, int n, cudaStream_t stream) {
  const unsigned g = (unsigned)((n + kHierThreads - 1) / kHierThreads);
  if (key_bytes == 4) {
    const uint32_t* c = static_cast<const uint32_t*>(sorted_codes);
    if (is_box)
      hierarchy_kernel<uint32_t, true><<<g, kHierThreads, 0, stream>>>(prim, c, perm, store, nodes, n);
    else
      hierarchy_kernel<uint32_t, false><<<g, kHierThreads, 0, stream>>>(prim, c, perm, store, nodes, n);
  } else {
    const uint64_t* c = static_cast<const uint64_t*>(sorted_codes);
    if (is_box)
      hierarchy_kernel<uint64_t, true><<<g, kHierThreads, 0, stream>>>(prim, c, perm, store, nodes, n);
    else
      hierarchy_kernel<uint64_t, false><<<g, kHierThreads, 0, stream>>>(prim, c, perm, store, nodes, n);
  }
}

}  // namespace bvh
