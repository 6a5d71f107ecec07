// traverse.cu -- K6 / K8: the paper's Algorithm 1 (reading G3), stackless traversal
// with skip-connections for a predicate query, one thread per query.  The count pass (K6) counts the
// leaves that satisfy the predicate; the fill pass (K8) repeats the walk and stores the original
// primitive index of each such leaf at offsets[query] + k ("Store the result", Alg. 1 L5).
//
// A node is one 32-byte record = one sector: two 128-bit loads through the read-only path.
// Predicates (D8): sphere {c, r} -- squared distance from c to the box, fp32 round-to-nearest with
// explicit intrinsics (no FMA contraction): d = max(max(lo - c, c - hi), 0) per axis,
// d2 = (dx*dx + dy*dy) + dz*dz, hit iff d2 <= r*r.  Box -- closed-interval overlap on each axis.
#include "common.cuh"

namespace bvh {

constexpr int kTravThreads = 128;

struct SphereQuery {
  float cx, cy, cz, r2;
  __device__ __forceinline__ void load(const float* __restrict__ q, int64_t j) {
    const float4 v = __ldg(reinterpret_cast<const float4*>(q) + j);
    cx = v.x; cy = v.y; cz = v.z;
    r2 = __fmul_rn(v.w, v.w);
  }
  __device__ __forceinline__ bool hit(const float4& lo, const float4& hi) const {
    const float dx = fmaxf(fmaxf(__fsub_rn(lo.x, cx), __fsub_rn(cx, hi.x)), 0.0f);
    const float dy = fmaxf(fmaxf(__fsub_rn(lo.y, cy), __fsub_rn(cy, hi.y)), 0.0f);
    const float dz = fmaxf(fmaxf(__fsub_rn(lo.z, cz), __fsub_rn(cz, hi.z)), 0.0f);
    const float d2 = __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
    return d2 <= r2;
  }
};

struct BoxQuery {
  float lo[3], hi[3];
  __device__ __forceinline__ void load(const float* __restrict__ q, int64_t j) {
    const float2* p = reinterpret_cast<const float2*>(q + 6 * j);
    const float2 a = __ldg(p), b = __ldg(p + 1), c = __ldg(p + 2);
    lo[0] = a.x; lo[1] = a.y; lo[2] = b.x; hi[0] = b.y; hi[1] = c.x; hi[2] = c.y;
  }
  __device__ __forceinline__ bool hit(const float4& nlo, const float4& nhi) const {
    return lo[0] <= nhi.x && nlo.x <= hi[0] && lo[1] <= nhi.y && nlo.y <= hi[1] && lo[2] <= nhi.z && nlo.z <= hi[2];
  }
};

template <typename Query, bool FILL>
__global__ void __launch_bounds__(kTravThreads)
traverse_kernel(const Node* __restrict__ nodes, int n, const float* __restrict__ queries, int64_t q,
                const uint32_t* __restrict__ order, int32_t* __restrict__ counts, const int64_t* __restrict__ offsets,
                int32_t* __restrict__ indices) {
  const int64_t t = (int64_t)blockIdx.x * kTravThreads + threadIdx.x;
  if (t >= q) return;
  // Neighbouring threads serve queries that are neighbours on the Morton curve when `order` is given: they
  // walk nearly the same nodes, which is what keeps the node reads in L1/L2 (PAPER.md:15-17 data divergence).
  const int64_t j = order ? (int64_t)order[t] : t;
  Query query;
  query.load(queries, j);
  const int leaf_base = n - 1;
  int32_t* out = nullptr;
  if (FILL) out = indices + offsets[j];
  int count = 0;
  int node = 0;                                              // L1: start from the root
  do {                                                       // L2
    const float4* p = reinterpret_cast<const float4*>(nodes + node);
    const float4 lo = __ldg(p);
    const float4 hi = __ldg(p + 1);
    const bool hit = query.hit(lo, hi);                      // L3
    const bool leaf = node >= leaf_base;
    if (hit && leaf) {                                       // L4-5
      if (FILL) out[count] = __float_as_int(lo.w);
      ++count;
    }
    node = (hit && !leaf) ? __float_as_int(lo.w)             // L8: N_left
                          : __float_as_int(hi.w);            // L6 / L10: N_skip
  } while (node != kSentinel);                               // L11
  if (!FILL) counts[j] = count;
}

void launch_traverse(const Node* nodes, int n, const float* queries, int64_t q, int kind, bool fill,
                     const uint32_t* order, int32_t* counts, const int64_t* offsets, int32_t* indices,
                     cudaStream_t stream) {
  const unsigned g = (unsigned)((q + kTravThreads - 1) / kTravThreads);
  if (kind == 0) {
    if (fill)
      traverse_kernel<SphereQuery, true><<<g, kTravThreads, 0, stream>>>(nodes, n, queries, q, order, counts, offsets, indices);
    else
      traverse_kernel<SphereQuery, false><<<g, kTravThreads, 0, stream>>>(nodes, n, queries, q, order, counts, offsets, indices);
  } else {
    if (fill)
      traverse_kernel<BoxQuery, true><<<g, kTravThreads, 0, stream>>>(nodes, n, queries, q, order, counts, offsets, indices);
    else
      traverse_kernel<BoxQuery, false><<<g, kTravThreads, 0, stream>>>(nodes, n, queries, q, order, counts, offsets, indices);
  }
}

}  // namespace bvh
