// traverse.cu -- K6 / K8: the paper's Algorithm 1 (reading G3), stackless traversal
// with skip-connections for a predicate query, one thread per query.  The count pass (K6) counts the
// leaves that satisfy the predicate; the fill pass (K8) repeats the walk and stores the original
// primitive index of each such leaf at offsets[query] + k ("Store the result", Alg. 1 L5).
//
// B200 specifics
//  * A node is one 32-byte record = one sector, fetched with ONE 256-bit load (LDG.E.ENL2.256, new on
//    sm_100): one L1 wavefront per lane and visit instead of two 128-bit halves of the same sector.
//  * Scheduling.  The grid is persistent: 148 SMs x kTravCtasPerSm CTAs, and CTA b works on query chunk
//    ((k*148 + b%148) * R + b/148) at its step k.  Blocks b, b+148, b+296, ... are co-resident on one SM,
//    so at any time an SM's 2048 threads serve 2048 consecutive positions of the (Morton-ordered) query
//    list: their node reads overlap and stay in that SM's L1 (data divergence).  The
//    mapping of blocks to SMs is only a locality assumption; any mapping gives the same results.
//  * Fill output.  Hits of a row are staged in a per-thread 8-slot shared-memory ring indexed by the
//    global output position, and an aligned group of 8 leaves as one 256-bit store = one full sector
//    (no partial-sector writes, 8x fewer store requests than 4-byte stores to 32 different rows per warp).
//
// Predicates (D8): sphere {c, r} -- squared distance from c to the box, fp32 round-to-nearest with
// explicit intrinsics (no FMA contraction): d = max(max(lo - c, c - hi), 0) per axis,
// d2 = (dx*dx + dy*dy) + dz*dz, hit iff d2 <= r*r.  Box -- closed-interval overlap on each axis.
#include "common.cuh"

namespace bvh {

#ifndef BVH_TRAV_CTAS
#define BVH_TRAV_CTAS 8
#endif
#ifndef BVH_SCAN_LEAVES
#define BVH_SCAN_LEAVES 32
#endif
constexpr int kTravThreads = 128;
constexpr int kTravCtasPerSm = BVH_TRAV_CTAS;  // 8 x 128 threads: 64 registers per thread for the leaf-scan batch

struct NodeRec {
  float lox, loy, loz;
  int left;
  float hix, hiy, hiz;
  int rope;
};

__device__ __forceinline__ NodeRec load_node(const Node* __restrict__ nodes, int idx) {
  NodeRec r;
  float l, p;
  asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=f"(r.lox), "=f"(r.loy), "=f"(r.loz), "=f"(l), "=f"(r.hix), "=f"(r.hiy), "=f"(r.hiz), "=f"(p)
               : "l"(nodes + idx));
  r.left = __float_as_int(l);
  r.rope = __float_as_int(p);
  return r;
}

struct SphereQuery {
  float cx, cy, cz, r2;
  __device__ __forceinline__ void load(const float* __restrict__ q, int64_t j) {
    const float4 v = __ldg(reinterpret_cast<const float4*>(q) + j);
    cx = v.x; cy = v.y; cz = v.z;
    r2 = __fmul_rn(v.w, v.w);
  }
  __device__ __forceinline__ bool hit(const NodeRec& n) const {
    const float dx = fmaxf(fmaxf(__fsub_rn(n.lox, cx), __fsub_rn(cx, n.hix)), 0.0f);
    const float dy = fmaxf(fmaxf(__fsub_rn(n.loy, cy), __fsub_rn(cy, n.hiy)), 0.0f);
    const float dz = fmaxf(fmaxf(__fsub_rn(n.loz, cz), __fsub_rn(cz, n.hiz)), 0.0f);
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
  __device__ __forceinline__ bool hit(const NodeRec& n) const {
    return lo[0] <= n.hix && n.lox <= hi[0] && lo[1] <= n.hiy && n.loy <= hi[1] && lo[2] <= n.hiz && n.loz <= hi[2];
  }
};

// Output side of the fill pass for one thread: ring of 8 slots per thread in shared memory.
template <bool FILL>
struct Emitter {
  int (*ring)[kTravThreads];
  int32_t* indices;
  int64_t base;
  int count;
  bool vec_store;
  __device__ __forceinline__ void emit(int value) {
    if (FILL) {
      const int64_t gi = base + count;                       // global output position of this hit
      ring[gi & 7][threadIdx.x] = value;
      if (((gi + 1) & 7) == 0) {                             // an aligned group of 8 positions is complete
        const int64_t g0 = gi - 7;
        if (g0 >= base && vec_store) {
          asm volatile("st.global.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(indices + g0),
                       "r"(ring[0][threadIdx.x]), "r"(ring[1][threadIdx.x]), "r"(ring[2][threadIdx.x]),
                       "r"(ring[3][threadIdx.x]), "r"(ring[4][threadIdx.x]), "r"(ring[5][threadIdx.x]),
                       "r"(ring[6][threadIdx.x]), "r"(ring[7][threadIdx.x])
                       : "memory");
        } else {                                             // head of a row that starts inside the group
          for (int64_t g = (g0 > base ? g0 : base); g <= gi; ++g) indices[g] = ring[g & 7][threadIdx.x];
        }
      }
    }
    ++count;
  }
  __device__ __forceinline__ void finish() {                 // tail of the row: the incomplete last group
    if (FILL) {
      const int64_t end = base + count;
      int64_t g = end & ~(int64_t)7;
      if (g < base) g = base;
      for (; g < end; ++g) indices[g] = ring[g & 7][threadIdx.x];
    }
  }
};

// Leaf-range shortcut.  In Karras ordering the leaves below a node are the consecutive leaf records
// [first, last], and the walk knows both bounds for free: the node a skip-connection leads to starts right
// after the subtree it skips (Algorithm 2: N_skip is node range_right + 1), so
// last + 1 = index of N_skip, and `first` is inherited on the way down (a left child starts where its
// parent starts).  When a node that satisfies the predicate covers at most kScanLeaves leaves, its leaves are
// tested directly from their consecutive records (independent, contiguous 256-bit loads: 4 leaves per 128-byte
// line) instead of walking the small subtree node by node.  Every leaf of the subtree is still tested, in the
// same ascending order, so the result and its order are those of Algorithm 1.
constexpr int kScanLeaves = BVH_SCAN_LEAVES;
#ifndef BVH_SCAN_BATCH
#define BVH_SCAN_BATCH 2
#endif
constexpr int kScanBatch = BVH_SCAN_BATCH;

template <typename Query, bool FILL>
__global__ void __launch_bounds__(kTravThreads, kTravCtasPerSm)
traverse_kernel(const Node* __restrict__ nodes, int n, const float* __restrict__ queries, int64_t q,
                const uint32_t* __restrict__ order, int32_t* __restrict__ counts, const int64_t* __restrict__ offsets,
                int32_t* __restrict__ indices, int64_t num_chunks, int ctas_per_sm, bool vec_store) {
  __shared__ int s_ring[FILL ? 8 : 1][kTravThreads];
  const int leaf_base = n - 1;
  const int64_t sm_slot = blockIdx.x % kNumSMs;
  const int64_t r = blockIdx.x / kNumSMs;
  for (int64_t k = 0;; ++k) {
    const int64_t chunk = (k * kNumSMs + sm_slot) * ctas_per_sm + r;
    if (chunk >= num_chunks) break;
    const int64_t t = chunk * kTravThreads + threadIdx.x;
    if (t >= q) continue;
    const int64_t j = order ? (int64_t)order[t] : t;
    Query query;
    query.load(queries, j);
    Emitter<FILL> out{s_ring, indices, FILL ? offsets[j] : 0, 0, vec_store};
    int node = 0;                                            // L1: start from the root
    int first = 0;                                           // first leaf below `node`
    int scan_i = 0, scan_end = 0;                            // pending leaf-range scan [scan_i, scan_end)
    // One loop for both activities, so that the lanes of a warp stay converged: every trip loads kScanBatch
    // records (tree step: the node and nothing else; scan step: the next kScanBatch consecutive leaves).
    do {                                                     // L2
      const bool scanning = scan_i < scan_end;
      NodeRec rec[kScanBatch];
      rec[0] = load_node(nodes, scanning ? leaf_base + scan_i : node);
#pragma unroll
      for (int u = 1; u < kScanBatch; ++u)
        if (scanning && scan_i + u < scan_end) rec[u] = load_node(nodes, leaf_base + scan_i + u);
      const bool hit0 = query.hit(rec[0]);                   // L3
      if (scanning) {
        if (hit0) out.emit(rec[0].left);                     // L4-5 on the leaves of the range, in order
#pragma unroll
        for (int u = 1; u < kScanBatch; ++u)
          if (scan_i + u < scan_end && query.hit(rec[u])) out.emit(rec[u].left);
        scan_i += kScanBatch;
      } else {
        const int rope = rec[0].rope;
        // first leaf after this subtree = index of the skip target (leaf or internal alike); n after the last one
        const int next_first = rope < 0 ? n : (rope >= leaf_base ? rope - leaf_base : rope);
        int next = rope;                                     // L6 / L10: N_skip
        if (hit0) {
          if (node >= leaf_base) {                           // L4-5
            out.emit(rec[0].left);
          } else if (next_first - first <= kScanLeaves) {    // small subtree: test its leaves directly
            scan_i = first;
            scan_end = next_first;
          } else {
            next = rec[0].left;                              // L8: N_left (same first leaf)
          }
        }
        if (next == rope) first = next_first;
        node = next;
      }
    } while (node != kSentinel || scan_i < scan_end);        // L11
    out.finish();
    if (!FILL) counts[j] = out.count;
  }
}

void launch_traverse(const Node* nodes, int n, const float* queries, int64_t q, int kind, bool fill,
                     const uint32_t* order, int32_t* counts, const int64_t* offsets, int32_t* indices,
                     cudaStream_t stream) {
  const int64_t num_chunks = (q + kTravThreads - 1) / kTravThreads;
  // persistent grid: up to 148 x 16 CTAs; fewer CTAs per SM when there is not enough work to fill them
  int ctas_per_sm = (int)((num_chunks + kNumSMs - 1) / kNumSMs);
  if (ctas_per_sm > kTravCtasPerSm) ctas_per_sm = kTravCtasPerSm;
  if (ctas_per_sm < 1) ctas_per_sm = 1;
  const unsigned g = (unsigned)(kNumSMs * ctas_per_sm);
  const bool vec = (reinterpret_cast<uintptr_t>(indices) & 31u) == 0;
  if (kind == 0) {
    if (fill)
      traverse_kernel<SphereQuery, true><<<g, kTravThreads, 0, stream>>>(nodes, n, queries, q, order, counts, offsets,
                                                                        indices, num_chunks, ctas_per_sm, vec);
    else
      traverse_kernel<SphereQuery, false><<<g, kTravThreads, 0, stream>>>(nodes, n, queries, q, order, counts, offsets,
                                                                         indices, num_chunks, ctas_per_sm, vec);
  } else {
    if (fill)
      traverse_kernel<BoxQuery, true><<<g, kTravThreads, 0, stream>>>(nodes, n, queries, q, order, counts, offsets,
                                                                     indices, num_chunks, ctas_per_sm, vec);
    else
      traverse_kernel<BoxQuery, false><<<g, kTravThreads, 0, stream>>>(nodes, n, queries, q, order, counts, offsets,
                                                                      indices, num_chunks, ctas_per_sm, vec);
  }
}

}  // namespace bvh
