// traverse.cu -- K6 / K8: the paper's Algorithm 1 (reading G3), stackless traversal
// with skip-connections for a predicate query.  The count pass (K6) counts the leaves that satisfy
// the predicate; the fill pass (K8) repeats the walk and stores the original primitive index of each
// such leaf at offsets[query] + k ("Store the result", Alg. 1 L5).
//
// Work split inside a warp (32 queries, neighbours on the Morton curve when `order` is given):
//  * WALK, one lane per query.  Each lane follows Algorithm 1 over the internal nodes: one 32-byte record =
//    one sector = ONE 256-bit load (LDG.E.ENL2.256, new on sm_100) per visit; hit -> left child, miss ->
//    skip-connection.  No stack, no per-thread memory.
//  * SCAN, the whole warp per leaf range.  In Karras ordering the leaves below a node are the consecutive
//    leaf records [first, last], and the walk knows both bounds for free: the node a skip-connection leads to
//    starts right after the subtree it skips (Algorithm 2: N_skip is node range_right + 1),
//    and `first` is inherited on the way down (a left child starts where its parent starts).  When a node that
//    satisfies the predicate covers at most kScanLeaves leaves, the lane does not walk that small subtree
//    node by node: it posts the range, and the warp tests those leaves together, lane l taking leaf
//    first + l -- one coalesced load of consecutive leaf records instead of 32 scattered ones, no
//    divergence, and in the fill pass the hits of the row leave as one contiguous run of stores
//    (warp-cooperative CSR output; ballot + popc give each hit its slot).  Every leaf of the subtree is
//    still tested, in ascending order, so the result and its order are those of Algorithm 1.
//  * Scheduling.  The grid is persistent: 148 SMs x CTAs per SM, and CTA b works on query chunk
//    ((k*148 + b%148) * R + b/148) at its step k, so that at any time the threads of an SM serve consecutive
//    positions of the (Morton-ordered) query list: their node reads overlap and stay in that SM's L1
//    (data divergence).  The block-to-SM mapping is only a locality assumption.
//
// Predicates (D8): sphere {c, r} -- squared distance from c to the box, fp32 round-to-nearest with
// explicit intrinsics (no FMA contraction): d = max(max(lo - c, c - hi), 0) per axis,
// d2 = (dx*dx + dy*dy) + dz*dz, hit iff d2 <= r*r.  Box -- closed-interval overlap on each axis.
// A point leaf stores the point once; with lo = hi = p the sphere formula reduces exactly to
// d = |p - c| (lo - c and c - hi are exact negatives of each other under round-to-nearest) and the box
// test to min <= p <= max, which is what the point-leaf tests below compute.
#include "common.cuh"

namespace bvh {

#ifndef BVH_TRAV_CTAS
#define BVH_TRAV_CTAS 8
#endif
#ifndef BVH_SCAN_LEAVES
#define BVH_SCAN_LEAVES 128
#endif
constexpr int kTravThreads = 128;
constexpr int kTravCtasPerSm = BVH_TRAV_CTAS;
constexpr int kScanLeaves = BVH_SCAN_LEAVES;

struct NodeRec {
  float lox, loy, loz;
  int left;
  float hix, hiy, hiz;
  int rope;
};

__device__ __forceinline__ NodeRec load_rec(const Node* __restrict__ p) {
  NodeRec r;
  float l, q;
  asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=f"(r.lox), "=f"(r.loy), "=f"(r.loz), "=f"(l), "=f"(r.hix), "=f"(r.hiy), "=f"(r.hiz), "=f"(q)
               : "l"(p));
  r.left = __float_as_int(l);
  r.rope = __float_as_int(q);
  return r;
}

struct SphereQuery {
  static constexpr int kWords = 4;
  static constexpr int kCtasPerSm = kTravCtasPerSm;
  float cx, cy, cz, r2;
  __device__ __forceinline__ void load(const float* __restrict__ q, int64_t j) {
    const float4 v = __ldg(reinterpret_cast<const float4*>(q) + j);
    cx = v.x; cy = v.y; cz = v.z;
    r2 = __fmul_rn(v.w, v.w);
  }
  // one slot of kSlotWords floats per thread in shared memory: how the warp reads the query of the lane it scans for
  static constexpr int kSlotWords = 4;
  __device__ __forceinline__ void to_shared(float* slot) const {
    *reinterpret_cast<float4*>(slot) = make_float4(cx, cy, cz, r2);
  }
  __device__ __forceinline__ void from_shared(const float* slot) {
    const float4 v = *reinterpret_cast<const float4*>(slot);     // one broadcast LDS.128
    cx = v.x; cy = v.y; cz = v.z; r2 = v.w;
  }
  __device__ __forceinline__ bool hit_box(float lox, float loy, float loz, float hix, float hiy, float hiz) const {
    const float dx = fmaxf(fmaxf(__fsub_rn(lox, cx), __fsub_rn(cx, hix)), 0.0f);
    const float dy = fmaxf(fmaxf(__fsub_rn(loy, cy), __fsub_rn(cy, hiy)), 0.0f);
    const float dz = fmaxf(fmaxf(__fsub_rn(loz, cz), __fsub_rn(cz, hiz)), 0.0f);
    const float d2 = __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
    return d2 <= r2;
  }
  __device__ __forceinline__ bool hit_point(float x, float y, float z) const {
    const float dx = fabsf(__fsub_rn(x, cx)), dy = fabsf(__fsub_rn(y, cy)), dz = fabsf(__fsub_rn(z, cz));
    const float d2 = __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
    return d2 <= r2;
  }
};

struct BoxQuery {
  static constexpr int kWords = 6;
  static constexpr int kCtasPerSm = kTravCtasPerSm;
  float lo[3], hi[3];
  __device__ __forceinline__ void load(const float* __restrict__ q, int64_t j) {
    const float2* p = reinterpret_cast<const float2*>(q + 6 * j);
    const float2 a = __ldg(p), b = __ldg(p + 1), c = __ldg(p + 2);
    lo[0] = a.x; lo[1] = a.y; lo[2] = b.x; hi[0] = b.y; hi[1] = c.x; hi[2] = c.y;
  }
  static constexpr int kSlotWords = 8;
  __device__ __forceinline__ void to_shared(float* slot) const {
    reinterpret_cast<float4*>(slot)[0] = make_float4(lo[0], lo[1], lo[2], hi[0]);
    reinterpret_cast<float2*>(slot)[2] = make_float2(hi[1], hi[2]);
  }
  __device__ __forceinline__ void from_shared(const float* slot) {
    const float4 a = reinterpret_cast<const float4*>(slot)[0];
    const float2 b = reinterpret_cast<const float2*>(slot)[2];
    lo[0] = a.x; lo[1] = a.y; lo[2] = a.z; hi[0] = a.w; hi[1] = b.x; hi[2] = b.y;
  }
  __device__ __forceinline__ bool hit_box(float lox, float loy, float loz, float hix, float hiy, float hiz) const {
    return lo[0] <= hix && lox <= hi[0] && lo[1] <= hiy && loy <= hi[1] && lo[2] <= hiz && loz <= hi[2];
  }
  __device__ __forceinline__ bool hit_point(float x, float y, float z) const {
    return lo[0] <= x && x <= hi[0] && lo[1] <= y && y <= hi[1] && lo[2] <= z && z <= hi[2];
  }
};

// Ray {o.xyz, d.xyz, tmin, tmax} (NEXT-1; "a ray intersects"): D9 of DESIGN.md, the slab test.  Per axis
// with d != 0: inv = 1 / d, t1 = (lo - o) * inv, t2 = (hi - o) * inv clip [tmin, tmax] to [min(t1,t2), max(t1,t2)];
// per axis with d == 0: lo <= o <= hi.  Hit iff the clipped interval is not empty.  1 / d is computed once per ray
// (the same IEEE division the oracle does per test); an axis with d == 0 keeps inv = 0 and is tested by bounds.
#ifndef BVH_TRAV_CTAS_RAYS
#define BVH_TRAV_CTAS_RAYS 6
#endif
struct RayQuery {
  static constexpr int kWords = 8;
  static constexpr int kCtasPerSm = BVH_TRAV_CTAS_RAYS;   // the ray state does not fit the 64 registers of 8 CTAs per SM
  float o[3], inv[3], tmin, tmax;
  uint32_t par;        // bit a: d[a] == 0
  __device__ __forceinline__ void load(const float* __restrict__ q, int64_t j) {
    const float4 a = __ldg(reinterpret_cast<const float4*>(q) + 2 * j);
    const float4 b = __ldg(reinterpret_cast<const float4*>(q) + 2 * j + 1);
    o[0] = a.x; o[1] = a.y; o[2] = a.z;
    const float d[3] = {a.w, b.x, b.y};
    tmin = b.z; tmax = b.w;
    par = 0;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      if (d[k] == 0.0f) {
        par |= 1u << k;
        inv[k] = 0.0f;
      } else {
        inv[k] = __fdiv_rn(1.0f, d[k]);
      }
    }
  }
  static constexpr int kSlotWords = 12;
  __device__ __forceinline__ void to_shared(float* slot) const {
    reinterpret_cast<float4*>(slot)[0] = make_float4(o[0], o[1], o[2], tmin);
    reinterpret_cast<float4*>(slot)[1] = make_float4(inv[0], inv[1], inv[2], tmax);
    reinterpret_cast<uint32_t*>(slot)[8] = par;
  }
  __device__ __forceinline__ void from_shared(const float* slot) {
    const float4 a = reinterpret_cast<const float4*>(slot)[0];
    const float4 b = reinterpret_cast<const float4*>(slot)[1];
    o[0] = a.x; o[1] = a.y; o[2] = a.z; tmin = a.w;
    inv[0] = b.x; inv[1] = b.y; inv[2] = b.z; tmax = b.w;
    par = reinterpret_cast<const uint32_t*>(slot)[8];
  }
  __device__ __forceinline__ bool hit_box(float lox, float loy, float loz, float hix, float hiy, float hiz) const {
    const float lo[3] = {lox, loy, loz}, hi[3] = {hix, hiy, hiz};
    float tn = tmin, tf = tmax;
    bool ok = true;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      const float t1 = __fmul_rn(__fsub_rn(lo[k], o[k]), inv[k]);
      const float t2 = __fmul_rn(__fsub_rn(hi[k], o[k]), inv[k]);
      if ((par >> k) & 1u) {
        ok = ok && (lo[k] <= o[k]) && (o[k] <= hi[k]);
      } else {
        tn = fmaxf(tn, fminf(t1, t2));
        tf = fminf(tf, fmaxf(t1, t2));
      }
    }
    return ok && (tn <= tf);
  }
  __device__ __forceinline__ bool hit_point(float x, float y, float z) const { return hit_box(x, y, z, x, y, z); }
};

// One leaf record: loaded first (so that several loads can be in flight), tested later.
template <bool POINT_LEAF>
struct LeafRec;
template <>
struct LeafRec<true> {
  float4 v;
  __device__ __forceinline__ void load(const char* __restrict__ leaves, int i) {
    v = __ldg(reinterpret_cast<const float4*>(leaves) + i);
  }
  __device__ __forceinline__ uint32_t payload() const { return __float_as_uint(v.w); }
  template <typename Query>
  __device__ __forceinline__ bool hit(const Query& q) const { return q.hit_point(v.x, v.y, v.z); }
};
template <>
struct LeafRec<false> {
  NodeRec r;
  __device__ __forceinline__ void load(const char* __restrict__ leaves, int i) {
    r = load_rec(reinterpret_cast<const Node*>(leaves) + i);
  }
  __device__ __forceinline__ uint32_t payload() const { return (uint32_t)r.left; }
  template <typename Query>
  __device__ __forceinline__ bool hit(const Query& q) const { return q.hit_box(r.lox, r.loy, r.loz, r.hix, r.hiy, r.hiz); }
};

#ifndef BVH_SCAN_UNROLL
#define BVH_SCAN_UNROLL 4
#endif

template <typename Query, bool FILL, bool POINT_LEAF>
__device__ __forceinline__ void traverse_body(const char* __restrict__ nodes, int n, const float* __restrict__ queries,
                                              int64_t q, const uint32_t* __restrict__ order, int32_t* __restrict__ counts,
                                              const int64_t* __restrict__ offsets, int32_t* __restrict__ indices,
                                              int64_t num_chunks, int ctas_per_sm) {
  constexpr int U = POINT_LEAF ? BVH_SCAN_UNROLL : (BVH_SCAN_UNROLL > 2 ? 2 : BVH_SCAN_UNROLL);   // leaf loads in flight per lane
  // what a lane posts for the warp to read: its query, the leaf range to scan, (fill) where its row starts
  __shared__ __align__(16) float s_query[kTravThreads * Query::kSlotWords];
  __shared__ int2 s_range[kTravThreads];
  __shared__ int64_t s_row[FILL ? kTravThreads : 1];
  const Node* __restrict__ internal = reinterpret_cast<const Node*>(nodes + kNodesHeaderBytes);
  const char* __restrict__ leaves = nodes + leaf_offset_bytes(n);
  const int leaf_base = n - 1;
  const int lane = threadIdx.x & 31;
  const int warp_first = threadIdx.x - lane;               // slot of lane 0 of this warp
  const uint32_t lt_mask = (1u << lane) - 1u;
  const int64_t sm_slot = blockIdx.x % kNumSMs;
  const int64_t r = blockIdx.x / kNumSMs;
  for (int64_t k = 0;; ++k) {
    const int64_t chunk = (k * kNumSMs + sm_slot) * ctas_per_sm + r;
    if (chunk >= num_chunks) break;
    const int64_t t = chunk * kTravThreads + threadIdx.x;
    const bool have = t < q;
    const int64_t j = have ? (order ? (int64_t)order[t] : t) : 0;
    Query query;
    query.load(queries, j);
    __syncwarp();                                            // the previous chunk's scans are over
    query.to_shared(s_query + threadIdx.x * Query::kSlotWords);
    if (FILL) s_row[threadIdx.x] = have ? offsets[j] : 0;    // this query's CSR row
    __syncwarp();
    int32_t* const row = FILL ? indices + s_row[FILL ? threadIdx.x : 0] : nullptr;
    int count = 0;
    int node = have ? 0 : kSentinel;                         // L1: start from the root
    int first = 0;                                           // first leaf below `node`
    bool post = false;                                       // this lane posted a leaf range in the last round
    while (true) {                                           // L2 ... L11 for the 32 queries of the warp
      const bool walking = node != kSentinel;
      uint32_t posted = __ballot_sync(0xffffffffu, post);
      if (!__any_sync(0xffffffffu, walking) && posted == 0) break;
      post = false;
      // ---- WALK, first half: fetch this lane's node; the record is consumed after the SCAN below, which runs while
      // the load is in flight ----
      const bool at_internal = walking && node < leaf_base;
      NodeRec rec;
      if (at_internal) rec = load_rec(internal + node);
      // ---- SCAN: the warp tests every range posted in the previous round, 32 consecutive leaves per step ----------
      while (posted) {
        const int o = __ffs(posted) - 1;
        posted &= posted - 1;
        Query oq;
        oq.from_shared(s_query + (warp_first + o) * Query::kSlotWords);
        const int2 range = s_range[warp_first + o];
        const int end = range.y;
        int ocount = 0;                                    // count: this lane's hits; fill: the row's running length
        int32_t* orow = nullptr;
        if (FILL) {
          ocount = __shfl_sync(0xffffffffu, count, o);
          orow = indices + s_row[warp_first + o];
        }
        for (int c = range.x + lane; c < end + lane; c += 32 * U) {   // c - lane is warp-uniform
          LeafRec<POINT_LEAF> leaf[U];
#pragma unroll
          for (int u = 0; u < U; ++u)
            if (c + 32 * u < end) leaf[u].load(leaves, c + 32 * u);
#pragma unroll
          for (int u = 0; u < U; ++u) {
            const bool inside = c + 32 * u < end;
            const bool sat = leaf[u].hit(oq);              // evaluated on every lane (no branch); masked below
            const bool hit = inside & sat;                 // L3-5 on leaf c + 32u
            if (FILL) {
              const uint32_t m = __ballot_sync(0xffffffffu, hit);
              if (hit) orow[ocount + __popc(m & lt_mask)] = (int)(leaf[u].payload() & kLeafPrimMask);
              ocount += __popc(m);
            } else {
              ocount += hit ? 1 : 0;
            }
          }
        }
        if (FILL) {
          if (lane == o) count = ocount;
        } else {
          const int total = __reduce_add_sync(0xffffffffu, ocount);   // one REDUX per range instead of a ballot per step
          if (lane == o) count += total;
        }
      }
      // ---- WALK, second half: one step of Algorithm 1 per lane ---------------------------------------------------
      if (walking) {
        if (!at_internal) {                                  // a single leaf (reached as a child or through a rope)
          const int i = node - leaf_base;
          LeafRec<POINT_LEAF> leaf;
          leaf.load(leaves, i);
          const uint32_t payload = leaf.payload();
          if (leaf.hit(query)) {                             // L3-5
            if (FILL) row[count] = (int)(payload & kLeafPrimMask);
            ++count;
          }
          // L6: N_skip of leaf i (Algorithm 2): leaf i+1 or internal node i+1, one bit in the record
          node = (i == n - 1) ? kSentinel : ((payload & kLeafRopeInternal) ? i + 1 : leaf_base + i + 1);
          first = i + 1;
        } else {
          const int rope = rec.rope;
          // first leaf after this subtree = index of the skip target (leaf or internal alike); n after the last one
          const int next_first = rope < 0 ? n : (rope >= leaf_base ? rope - leaf_base : rope);
          int next = rope;                                   // L10: N_skip
          if (query.hit_box(rec.lox, rec.loy, rec.loz, rec.hix, rec.hiy, rec.hiz)) {   // L3
            if (next_first - first <= kScanLeaves) {         // small subtree: post its leaves, continue after it
              s_range[threadIdx.x] = make_int2(first, next_first);
              post = true;
            } else {
              next = rec.left;                               // L8: N_left (same first leaf)
            }
          }
          if (next == rope) first = next_first;
          node = next;
        }
      }
      __syncwarp();                                          // posted ranges are visible to the warp
    }
    if (!FILL && have) counts[j] = count;
  }
}

// The leaf format (point or box records) is a property of the hierarchy, recorded in its header by the build;
// the kernel reads it there (one uniform branch), so the query entry points need no extra argument.
template <typename Query, bool FILL>
__global__ void __launch_bounds__(kTravThreads, Query::kCtasPerSm)
traverse_kernel(const char* __restrict__ nodes, int n, const float* __restrict__ queries, int64_t q,
                const uint32_t* __restrict__ order, int32_t* __restrict__ counts, const int64_t* __restrict__ offsets,
                int32_t* __restrict__ indices, int64_t num_chunks, int ctas_per_sm) {
  if (reinterpret_cast<const NodesHeader*>(nodes)->leaf_kind == kLeafPoints)
    traverse_body<Query, FILL, true>(nodes, n, queries, q, order, counts, offsets, indices, num_chunks, ctas_per_sm);
  else
    traverse_body<Query, FILL, false>(nodes, n, queries, q, order, counts, offsets, indices, num_chunks, ctas_per_sm);
}

template <typename Query>
static void launch_traverse_kind(const char* nodes, int n, const float* queries, int64_t q, bool fill,
                                 const uint32_t* order, int32_t* counts, const int64_t* offsets, int32_t* indices,
                                 cudaStream_t stream) {
  const int64_t num_chunks = (q + kTravThreads - 1) / kTravThreads;
  // persistent grid: up to 148 x Query::kCtasPerSm CTAs; fewer CTAs per SM when there is not enough work to fill them
  int ctas_per_sm = (int)((num_chunks + kNumSMs - 1) / kNumSMs);
  if (ctas_per_sm > Query::kCtasPerSm) ctas_per_sm = Query::kCtasPerSm;
  if (ctas_per_sm < 1) ctas_per_sm = 1;
  const unsigned g = (unsigned)(kNumSMs * ctas_per_sm);
  if (fill)
    traverse_kernel<Query, true><<<g, kTravThreads, 0, stream>>>(nodes, n, queries, q, order, counts, offsets, indices,
                                                                num_chunks, ctas_per_sm);
  else
    traverse_kernel<Query, false><<<g, kTravThreads, 0, stream>>>(nodes, n, queries, q, order, counts, offsets, indices,
                                                                 num_chunks, ctas_per_sm);
}

void launch_traverse(const void* nodes, int n, const float* queries, int64_t q, int kind, bool fill,
                     const uint32_t* order, int32_t* counts, const int64_t* offsets, int32_t* indices,
                     cudaStream_t stream) {
  const char* base = static_cast<const char*>(nodes);
  if (kind == 0)
    launch_traverse_kind<SphereQuery>(base, n, queries, q, fill, order, counts, offsets, indices, stream);
  else if (kind == 1)
    launch_traverse_kind<BoxQuery>(base, n, queries, q, fill, order, counts, offsets, indices, stream);
  else
    launch_traverse_kind<RayQuery>(base, n, queries, q, fill, order, counts, offsets, indices, stream);
}

}  // namespace bvh
