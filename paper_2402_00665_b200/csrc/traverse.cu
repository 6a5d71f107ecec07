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
//    satisfies the predicate covers at most SCAN leaves (96; 64 / 128 in two cases: kScanLeaves below), the lane does not walk that small subtree
//    node by node: it posts the range, and the warp tests those leaves together, lane l taking leaf
//    first + l -- one coalesced load of consecutive leaf records instead of 32 scattered ones, no
//    divergence, and in the fill pass the hits of the row leave as one contiguous run of stores
//    (warp-cooperative CSR output; ballot + popc give each hit its slot).  Every leaf of the subtree is
//    still tested, in ascending order, so the result and its order are those of Algorithm 1.
//  * Scheduling.  One block per chunk of kTravThreads consecutive positions of the (Morton-ordered) query list; the
//    hardware hands the chunks out in order as blocks retire, so the blocks that run at the same time serve
//    neighbouring queries -- their node reads overlap in L1 / L2 (data divergence) -- and expensive
//    chunks do not hold up a static share of the list.  A batch too small to fill the GPU is spread: one query per
//    2^s lanes (launch_traverse_kind).
//
// Predicates (D8): sphere {c, r} -- squared distance from c to the box, fp32 round-to-nearest with
// explicit intrinsics (no FMA contraction): d = max(max(lo - c, c - hi), 0) per axis,
// d2 = (dx*dx + dy*dy) + dz*dz, hit iff d2 <= r*r.  Box -- closed-interval overlap on each axis.
// A point leaf stores the point once; with lo = hi = p the sphere formula reduces exactly to
// d = |p - c| (lo - c and c - hi are exact negatives of each other under round-to-nearest) and the box
// test to min <= p <= max, which is what the point-leaf tests below compute.
#include "common.cuh"

namespace bvh {

#ifndef BVH_TRAV_THREADS
#define BVH_TRAV_THREADS 128
#endif
#ifndef BVH_TRAV_WARPS_PER_SM
#define BVH_TRAV_WARPS_PER_SM 32
#endif
#ifndef BVH_SCAN_LEAVES
#define BVH_SCAN_LEAVES 96
#endif
#ifndef BVH_SCAN_LEAVES_SPARSE
#define BVH_SCAN_LEAVES_SPARSE 64
#endif
constexpr int kTravThreads = BVH_TRAV_THREADS;         // queries of a block (one per thread)
static_assert(kTravThreads % 32 == 0 && kTravThreads >= 32 && kTravThreads <= 1024, "whole warps");
constexpr int kTravCtasPerSm = BVH_TRAV_WARPS_PER_SM * 32 / kTravThreads;   // resident blocks asked of the register allocator
// Largest subtree (in leaves) whose leaves the warp scans instead of walking it; the scan loop is unrolled to take such
// a range in ONE iteration (threshold / 32 loads in flight per lane).  Measured on B200 (profiles/r02_experiments.md):
// 96 for batches with long rows (C3: 591 hits per query), 64 where rows are short (C2, C4, C5: 3 to 31 hits per
// query: fewer leaves tested in vain per hit) -- which the single-pass call knows from its row capacity.
constexpr int kScanLeaves = BVH_SCAN_LEAVES;
constexpr int kScanLeavesSparse = BVH_SCAN_LEAVES_SPARSE;
constexpr int kScanLeavesSpread = 128;                 // small batches, one query per warp: scanning is cheap, walking is latency
constexpr int kSparseRowCap = 64;                      // collect with rows of at most this many entries: the sparse threshold
static_assert(kScanLeaves % 32 == 0 && kScanLeavesSparse % 32 == 0 && kScanLeavesSparse <= kScanLeaves, "whole warp steps");

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
  static constexpr bool kHasKey = true;                    // D10: candidates are ranked by their distance
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
  // The whole box lies inside the sphere, in the arithmetic of D8: with f = max(c - lo, hi - c) per axis (the farthest
  // the box reaches from the centre), F2 = (fx*fx + fy*fy) + fz*fz <= r*r.  Then every box B inside this one satisfies
  // the predicate: per axis its distance term max(max(B.lo - c, c - B.hi), 0) <= f because B.lo <= hi, B.hi >= lo and
  // round-to-nearest subtraction is monotone (and f >= 0 since lo <= hi); squaring non-negatives and rounded addition
  // are monotone too, so d2(B) <= F2 <= r*r -- the argument SURVEY.md 8(c) D8 uses for "a hit leaf has hit ancestors".
  // D10 (nearest within the radius): the key of a candidate is its D8 distance; a found candidate shrinks the radius
  // to its distance (closed comparisons keep candidates at the same distance in play for the index tie rule).
  __device__ __forceinline__ bool cand_box(float lox, float loy, float loz, float hix, float hiy, float hiz, float& key) const {
    const float dx = fmaxf(fmaxf(__fsub_rn(lox, cx), __fsub_rn(cx, hix)), 0.0f);
    const float dy = fmaxf(fmaxf(__fsub_rn(loy, cy), __fsub_rn(cy, hiy)), 0.0f);
    const float dz = fmaxf(fmaxf(__fsub_rn(loz, cz), __fsub_rn(cz, hiz)), 0.0f);
    key = __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
    return key <= r2;
  }
  __device__ __forceinline__ bool cand_point(float x, float y, float z, float& key) const {
    const float dx = fabsf(__fsub_rn(x, cx)), dy = fabsf(__fsub_rn(y, cy)), dz = fabsf(__fsub_rn(z, cz));
    key = __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
    return key <= r2;
  }
  __device__ __forceinline__ void shrink(float key) { r2 = key; }
  __device__ __forceinline__ float extent() const { return 2.0f * sqrtf(r2); }   // only gates the shortcut: any value is safe
  __device__ __forceinline__ bool contains_box(float lox, float loy, float loz, float hix, float hiy, float hiz) const {
    const float fx = fmaxf(__fsub_rn(cx, lox), __fsub_rn(hix, cx));
    const float fy = fmaxf(__fsub_rn(cy, loy), __fsub_rn(hiy, cy));
    const float fz = fmaxf(__fsub_rn(cz, loz), __fsub_rn(hiz, cz));
    const float f2 = __fadd_rn(__fadd_rn(__fmul_rn(fx, fx), __fmul_rn(fy, fy)), __fmul_rn(fz, fz));
    return f2 <= r2;
  }
};

struct BoxQuery {
  static constexpr bool kHasKey = false;                   // overlap has no ranking: count / fill / any only
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
  // The node's box lies inside the query box: every box B inside the node (B.lo <= B.hi) then overlaps the query on
  // every axis (query.lo <= node.lo <= B.lo <= B.hi and B.lo <= B.hi <= node.hi <= query.hi).  Comparisons only.
  __device__ __forceinline__ float extent() const { return fminf(fminf(hi[0] - lo[0], hi[1] - lo[1]), hi[2] - lo[2]); }
  __device__ __forceinline__ bool contains_box(float lox, float loy, float loz, float hix, float hiy, float hiz) const {
    return lo[0] <= lox && hix <= hi[0] && lo[1] <= loy && hiy <= hi[1] && lo[2] <= loz && hiz <= hi[2];
  }
};

// Ray {o.xyz, d.xyz, tmin, tmax} (NEXT-1; "a ray intersects"): D9 of DESIGN.md, the slab test.  Per axis
// with d != 0: inv = 1 / d, t1 = (lo - o) * inv, t2 = (hi - o) * inv clip [tmin, tmax] to [min(t1,t2), max(t1,t2)];
// per axis with d == 0: lo <= o <= hi.  Hit iff the clipped interval is not empty.  1 / d is computed once per ray
// (the same IEEE division the oracle does per test); an axis with d == 0 keeps inv = 0 and is tested by bounds.
#ifndef BVH_TRAV_WARPS_PER_SM_RAYS
#define BVH_TRAV_WARPS_PER_SM_RAYS 24
#endif
struct RayQuery {
  static constexpr bool kHasKey = true;                    // D11: candidates are ranked by where the ray enters them
  static constexpr int kWords = 8;
  static constexpr int kCtasPerSm = BVH_TRAV_WARPS_PER_SM_RAYS * 32 / kTravThreads;   // the ray state does not fit 64 registers
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
    float key;
    return cand_box(lox, loy, loz, hix, hiy, hiz, key);
  }
  // D11 (first hit): the key of a candidate is where the clipped interval starts; a found candidate shortens the
  // segment to end there (tmax is only the start value of the interval's end, so the entry parameters of the boxes
  // still in play do not change, and boxes entered at the same parameter stay in play for the index tie rule).
  __device__ __forceinline__ void shrink(float key) { tmax = key; }
  __device__ __forceinline__ bool cand_point(float x, float y, float z, float& key) const { return cand_box(x, y, z, x, y, z, key); }
  __device__ __forceinline__ bool cand_box(float lox, float loy, float loz, float hix, float hiy, float hiz, float& key) const {
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
    key = tn;
    return ok && (tn <= tf);
  }
  __device__ __forceinline__ bool hit_point(float x, float y, float z) const { return hit_box(x, y, z, x, y, z); }
  // a segment does not contain a box
  __device__ __forceinline__ float extent() const { return 0.0f; }
  __device__ __forceinline__ bool contains_box(float, float, float, float, float, float) const { return false; }
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
  template <typename Query>
  __device__ __forceinline__ bool cand(const Query& q, float& key) const { return q.cand_point(v.x, v.y, v.z, key); }
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
  template <typename Query>
  __device__ __forceinline__ bool cand(const Query& q, float& key) const { return q.cand_box(r.lox, r.loy, r.loz, r.hix, r.hiy, r.hiz, key); }
};

#ifndef BVH_TRAV_LOAD_AFTER_SCAN
#define BVH_TRAV_LOAD_AFTER_SCAN 0
#endif
#ifndef BVH_SCAN_SKIP_EMPTY
#define BVH_SCAN_SKIP_EMPTY 0
#endif

// What a pass does with a leaf that satisfies the predicate (Alg. 1 L5, "Store the result or perform an operation"):
//   kModeCount    count it (K6);
//   kModeFill     store its primitive at offsets[query] + k (K8);
//   kModeCollect  single-pass variant: store it in the query's own slice of `cap` entries of a
//                 caller-provided buffer (rows + query * cap; hits past cap are dropped) AND count it, so that one
//                 traversal yields counts and, for every row that fits, its content.
//   kModeReduce   "perform an operation" (NEXT-1): keep the candidate with the smallest key -- its D8 distance for sphere
//                 queries (D10, nearest within the radius), the parameter at which the ray enters its box for rays (D11,
//                 first hit) -- smallest primitive index among equal keys; the query shrinks as candidates are found.
//   kModeAny      "any hit": 1 if some leaf satisfies the predicate, found or not; the walk stops at the first one.
enum { kModeCount = 0, kModeFill = 1, kModeCollect = 2, kModeReduce = 3, kModeAny = 4 };

struct TraverseArgs {
  const char* nodes;
  int n;
  const float* queries;
  int64_t q;
  const uint32_t* order;     // optional: thread t serves query order[t]
  int32_t* counts;           // count, collect: out.  fill with only_over: in.  reduce: primitive index out; any: flag out
  float* keys;               // reduce: key of that primitive (d2 / t_enter), +infinity if none
  const int64_t* offsets;    // fill
  int32_t* out;              // fill: indices; collect: rows
  int64_t cap;               // collect: entries per row.  fill with only_over: only rows with counts[j] > cap are filled
  int only_over;
  int64_t out_limit;         // fill: entries `out` can hold; rows that would end past it are not written (0: no limit, < 0: nothing fits)
  int spread_log2;           // small batches: only every 2^spread_log2-th thread carries a query (see launch_traverse_kind)
};

// Row output of the fill / collect passes.  The hits of a row arrive a few at a time (one scan step of 32 leaves gives
// ~8 on C3), at whatever alignment the row has: stored as they come, almost every 32-byte sector of the result would
// be written in two or three pieces, and a sector that reaches L2 in pieces costs a DRAM read to complete it (round 1:
// 1.78 x the algorithmic DRAM traffic).  So hits are staged: each query keeps the tail of its row that does not fill a
// sector yet (< 8 entries) in shared memory; the hits of a posted range are appended to it in a per-warp buffer, and
// the warp writes out what is complete up to the last 32-byte boundary of the global address, as consecutive lanes =
// whole sectors, and keeps the rest.  Only the first and last sector of a row can be partial.
#ifndef BVH_FILL_STAGE
#define BVH_FILL_STAGE 0
#endif
constexpr int kFillStage = BVH_FILL_STAGE;        // 0: store hits as they come; 1: per posted range, coalesced; 2: whole sectors
#ifndef BVH_CONTAINMENT
#define BVH_CONTAINMENT 1
#endif
#ifndef BVH_CONTAIN_MIN_LEAVES
#define BVH_CONTAIN_MIN_LEAVES 1024
#endif
// Containment shortcut of the COUNT pass: a subtree whose box lies inside the query is counted (one addition) without
// walking or testing it.  The test costs ~15 instructions per visited node that satisfies the predicate, and a warp
// executes them whenever any of its 32 lanes stands at such a node, i.e. in almost every round.  On the benchmark
// configs the queries are much smaller than the scene (C3: 1.5 % of the tested leaves lie in contained nodes, counted
// on the oracle's tree) and the test is a net loss when applied to every node: C3 count 4.29 -> 4.79 ms with the test
// on every node, 4.66 ms on all subtrees of more than kScanLeaves leaves, 4.44 ms on subtrees of more than 1024.  So
// it is (a) applied to subtrees of more than kContainMinLeaves leaves only, where a success skips a lot, and (b)
// skipped by warps whose queries are all too small to contain such a subtree (try_contain below): C3 4.28 ms.  Even
// for large queries the gain is modest (2^20 uniform points, r = 0.2, 28 000 hits per query: count 6.43 -> 5.81 ms),
// because in a radix tree over Morton codes the big nodes that a sphere overlaps are rarely inside it.  The store
// passes must write every hit anyway (a contained subtree saves them only the tests) and the extra loop costs them
// 3 % on C3, so they do not use it.
constexpr bool kContainment = BVH_CONTAINMENT != 0;
constexpr int kContainMinLeaves = BVH_CONTAIN_MIN_LEAVES;
constexpr int kStageInts = 8;                      // one sector
constexpr int kScanLeavesMax = kScanLeaves > kScanLeavesSpread ? kScanLeaves : kScanLeavesSpread;
constexpr int kRangeBufInts = kScanLeavesMax + kStageInts;

__device__ __forceinline__ void store_sector(int32_t* p, const int* v) {   // 32-byte aligned: one full sector
  asm volatile("st.global.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]),
               "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7])
               : "memory");
}

// Shared memory of a block: what a lane posts for the warp to read (its query, the leaf range to scan, where its row
// starts) and the staging of the row output.
template <typename Query, bool STORE>
struct TravSmem {
  __align__(16) float query[kTravThreads * Query::kSlotWords];
  int2 range[kTravThreads];
  int32_t* row[STORE ? kTravThreads : 1];
  __align__(32) int stage[STORE ? kTravThreads * kStageInts : 8];
  int buf[STORE ? (kTravThreads / 32) * kRangeBufInts : 1];
};

__host__ __device__ constexpr bool mode_stores(int mode) { return mode == kModeFill || mode == kModeCollect; }

template <typename Query, int MODE, bool POINT_LEAF, bool SPREAD, int SCAN>
__device__ __forceinline__ void traverse_body(const TraverseArgs& A, TravSmem<Query, mode_stores(MODE)>& S) {
  constexpr bool STORE = mode_stores(MODE);
  constexpr bool REDUCE = MODE == kModeReduce, ANY = MODE == kModeAny;
  constexpr int U = POINT_LEAF ? SCAN / 32 : (SCAN / 32 > 2 ? 2 : SCAN / 32);   // leaf loads in flight per lane
  float* const s_query = S.query;
  int2* const s_range = S.range;
  int32_t** const s_row = S.row;
  int* const s_stage = S.stage;
  int* const s_buf = S.buf;
  const char* __restrict__ nodes = A.nodes;
  const int n = A.n;
  const float* __restrict__ queries = A.queries;
  const uint32_t* __restrict__ order = A.order;
  const Node* __restrict__ internal = reinterpret_cast<const Node*>(nodes + kNodesHeaderBytes);
  const char* __restrict__ leaves = nodes + leaf_offset_bytes(n);
  const int leaf_base = n - 1;
  const int lane = threadIdx.x & 31;
  const int warp_first = threadIdx.x - lane;               // slot of lane 0 of this warp
  const uint32_t lt_mask = (1u << lane) - 1u;
  int* const buf = s_buf + (STORE ? (threadIdx.x >> 5) * kRangeBufInts : 0);
  const int cap = (MODE == kModeCollect) ? (int)A.cap : 0x7fffffff;   // row positions >= cap are not stored
  float contain_extent = 0.0f;
  if (kContainment) {
    const NodesHeader* h = reinterpret_cast<const NodesHeader*>(nodes);
    const float e = fmaxf(fmaxf(h->scene_hi[0] - h->scene_lo[0], h->scene_hi[1] - h->scene_lo[1]), h->scene_hi[2] - h->scene_lo[2]);
    contain_extent = e * cbrtf((float)kContainMinLeaves / (float)n);   // side of a cube holding that share of a uniform scene
  }
  {
    // One block per chunk of kTravThreads consecutive positions of the (Morton-ordered) query list.  The hardware's block
    // scheduler hands the chunks out in order as blocks retire, which balances queries of very different cost (C3: 100
    // to 2800 hits) and keeps the chunks that run at the same time neighbours on the curve.  Round 1 ran a persistent
    // grid with a static, SM-local assignment of chunks instead: 26-35 % slower on C3 (4.26 / 6.42 ms count / fill
    // against 3.3 / 4.4), because blocks whose chunks were expensive finished long after the others.
    const int64_t thread = (int64_t)blockIdx.x * kTravThreads + threadIdx.x;
    const int spread_log2 = SPREAD ? A.spread_log2 : 0;      // (a separate instantiation: the large-batch kernel is untouched)
    const int64_t t = thread >> spread_log2;                 // position in the query list
    bool have = t < A.q && (thread & ((1 << spread_log2) - 1)) == 0;
    const int64_t j = have ? (order ? (int64_t)order[t] : t) : 0;
    if (MODE == kModeFill && A.only_over) have = have && (int64_t)A.counts[j] > A.cap;
    if (MODE == kModeFill && A.out_limit != 0) have = have && A.offsets[j + 1] <= A.out_limit;
    Query query;
    query.load(queries, have ? j : 0);                       // (the overflow pass serves few rows: no gather for the others)
    __syncwarp();                                            // the previous chunk's scans are over
    query.to_shared(s_query + threadIdx.x * Query::kSlotWords);
    int32_t* row = nullptr;
    if (STORE) {
      row = (MODE == kModeFill) ? A.out + (have ? A.offsets[j] : 0) : A.out + j * A.cap;   // this query's row
      s_row[threadIdx.x] = row;
    }
    __syncwarp();
    const int align = STORE ? (int)((reinterpret_cast<uintptr_t>(row) >> 2) & (kStageInts - 1)) : 0;
    // The containment test is only worth its instructions for queries that can contain a subtree of kContainMinLeaves
    // leaves at all; warps whose 32 queries are all smaller than the typical box of such a subtree skip it (a
    // heuristic gate: it changes which nodes are tested for containment, never a result).
    const bool try_contain = kContainment && MODE == kModeCount && __any_sync(0xffffffffu, have && query.extent() >= contain_extent);
    float best_key = __int_as_float(0x7f800000);             // reduce: key and primitive of the best candidate so far
    int best_idx = -1;
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
#if !BVH_TRAV_LOAD_AFTER_SCAN
      if (at_internal) rec = load_rec(internal + node);
#else
      if (at_internal) asm volatile("prefetch.global.L1 [%0];" ::"l"(internal + node));
#endif
      // ---- SCAN: the warp tests every range posted in the previous round, 32 consecutive leaves per step ----------
      while (posted) {
        const int o = __ffs(posted) - 1;
        posted &= posted - 1;
        Query oq;
        oq.from_shared(s_query + (warp_first + o) * Query::kSlotWords);
        const int2 range = s_range[warp_first + o];
        const int end = range.y;
        if constexpr (REDUCE) {
          // the best candidate of the range: smallest key, then smallest primitive index (two warp reductions per step)
          uint32_t rk = 0xFFFFFFFFu;                       // order-preserving image of the key; all ones: none
          int ri = 0x7fffffff;
          for (int c = range.x + lane; c < end + lane; c += 32) {
            LeafRec<POINT_LEAF> leaf;
            float key = 0.0f;
            bool hit = false;
            if (c < end) {
              leaf.load(leaves, c);
              hit = leaf.cand(oq, key);
            }
            const uint32_t kb = hit ? float_to_ordered(key) : 0xFFFFFFFFu;
            const uint32_t kmin = __reduce_min_sync(0xffffffffu, kb);
            if (kmin != 0xFFFFFFFFu && kmin <= rk) {       // warp-uniform
              const int ci = (hit && kb == kmin) ? (int)(leaf.payload() & kLeafPrimMask) : 0x7fffffff;
              const int imin = __reduce_min_sync(0xffffffffu, ci);
              if (kmin < rk || imin < ri) {
                rk = kmin;
                ri = imin;
              }
            }
          }
          if (lane == o && rk != 0xFFFFFFFFu) {
            const float k = ordered_to_float(rk);
            if (best_idx < 0 || k < best_key || (k == best_key && ri < best_idx)) {
              best_key = k;
              best_idx = ri;
              query.shrink(k);
              query.to_shared(s_query + threadIdx.x * Query::kSlotWords);
            }
          }
          __syncwarp();
          continue;
        }
        if constexpr (ANY) {
          bool found = false;
          for (int c = range.x + lane; c < end + lane && !found; c += 32) {
            LeafRec<POINT_LEAF> leaf;
            bool hit = false;
            if (c < end) {
              leaf.load(leaves, c);
              hit = leaf.hit(oq);
            }
            found = __any_sync(0xffffffffu, hit);
          }
          if (lane == o && found) {
            count = 1;
            node = kSentinel;                              // nothing more to learn for this query
          }
          continue;
        }
        int ocount = 0;                                    // count: this lane's hits; store: entries in `buf`
        int32_t* orow = nullptr;
        int p0 = 0, oalign = 0;
        if (STORE) {
          const int oc = __shfl_sync(0xffffffffu, count, o);
          orow = s_row[warp_first + o];
          if (kFillStage == 2) {
            // the row's staged tail comes first in the range buffer
            oalign = __shfl_sync(0xffffffffu, align, o);
            const int carry = min(oc, (oalign + oc) & (kStageInts - 1));
            p0 = oc - carry;                               // row position of buf[0]: sector-aligned, or the row's start
            if (lane < carry) buf[lane] = s_stage[(warp_first + o) * kStageInts + lane];
            ocount = carry;
          } else {
            p0 = oc;
          }
        }
        for (int c = range.x + lane; c < end + lane; c += 32 * U) {   // c - lane is warp-uniform
          LeafRec<POINT_LEAF> leaf[U];
#pragma unroll
          for (int u = 0; u < U; ++u)
            if (c + 32 * u < end) leaf[u].load(leaves, c + 32 * u);
#pragma unroll
          for (int u = 0; u < U; ++u) {
#if BVH_SCAN_SKIP_EMPTY
            if (u > 0 && c - lane + 32 * u >= end) break;   // (warp-uniform) no leaf of the range is left for this step
#endif
            const bool inside = c + 32 * u < end;
            const bool sat = leaf[u].hit(oq);              // evaluated on every lane (no branch); masked below
            const bool hit = inside & sat;                 // L3-5 on leaf c + 32u
            if (STORE) {
              const uint32_t m = __ballot_sync(0xffffffffu, hit);
              const int at = ocount + __popc(m & lt_mask);
              if (kFillStage == 0) {
                // (fill: the row is exactly as long as its hits; collect: positions past the capacity are dropped)
                if (hit && (MODE == kModeFill || p0 + at < cap)) orow[p0 + at] = (int)(leaf[u].payload() & kLeafPrimMask);
              } else {
                if (hit) buf[at] = (int)(leaf[u].payload() & kLeafPrimMask);
              }
              ocount += __popc(m);
            } else {
              ocount += hit ? 1 : 0;
            }
          }
        }
        if (STORE) {
          if (kFillStage == 2) {
            __syncwarp();
            // write out up to the last sector boundary of the global address; keep the rest staged
            const int rem = (oalign + p0 + ocount) & (kStageInts - 1);
            const int flush = ocount - rem > 0 ? ocount - rem : 0;
            for (int e = lane; e < flush; e += 32)
              if (p0 + e < cap) orow[p0 + e] = buf[e];
            if (lane < ocount - flush) s_stage[(warp_first + o) * kStageInts + lane] = buf[flush + lane];
            __syncwarp();
          } else if (kFillStage == 1) {
            __syncwarp();
            for (int e = lane; e < ocount; e += 32)
              if (p0 + e < cap) orow[p0 + e] = buf[e];
            __syncwarp();
          }
          if (lane == o) count = p0 + ocount;
        } else {
          const int total = __reduce_add_sync(0xffffffffu, ocount);   // one REDUX per range instead of a ballot per step
          if (lane == o) count += total;
        }
      }
      // ---- WALK, second half: one step of Algorithm 1 per lane ---------------------------------------------------
#if BVH_TRAV_LOAD_AFTER_SCAN
      if (at_internal) rec = load_rec(internal + node);
#endif
      if (walking && !(ANY && count != 0)) {               // (any hit: a lane whose scan just found one is done)
        if (!at_internal) {                                  // a single leaf (reached as a child or through a rope)
          const int i = node - leaf_base;
          LeafRec<POINT_LEAF> leaf;
          leaf.load(leaves, i);
          const uint32_t payload = leaf.payload();
          if constexpr (REDUCE) {
            float key;
            if (leaf.cand(query, key)) {                     // L3-5, "perform an operation"
              const int pi = (int)(payload & kLeafPrimMask);
              if (best_idx < 0 || key < best_key || (key == best_key && pi < best_idx)) {
                best_key = key;
                best_idx = pi;
                query.shrink(key);
                query.to_shared(s_query + threadIdx.x * Query::kSlotWords);
              }
            }
          } else if (leaf.hit(query)) {                      // L3-5
            if (STORE && kFillStage != 2) {
              if (count < cap) row[count] = (int)(payload & kLeafPrimMask);
            } else if (STORE) {
              int* st = s_stage + threadIdx.x * kStageInts;
              const int carry = min(count, (align + count) & (kStageInts - 1));
              st[carry] = (int)(payload & kLeafPrimMask);
              if (((align + count + 1) & (kStageInts - 1)) == 0) {   // the sector is complete
                const int p = count - carry;
                if (carry + 1 == kStageInts) {
                  if (p < cap) store_sector(row + p, st);    // (cap is a multiple of 8: a sector is inside or outside)
                } else {
                  for (int e = 0; e <= carry; ++e)
                    if (p + e < cap) row[p + e] = st[e];
                }
              }
            }
            ++count;
          }
          // L6: N_skip of leaf i (Algorithm 2): leaf i+1 or internal node i+1, one bit in the record
          node = (i == n - 1) ? kSentinel : ((payload & kLeafRopeInternal) ? i + 1 : leaf_base + i + 1);
          if (ANY && count) node = kSentinel;
          first = i + 1;
        } else {
          const int rope = rec.rope;
          // first leaf after this subtree = index of the skip target (leaf or internal alike); n after the last one
          const int next_first = rope < 0 ? n : (rope >= leaf_base ? rope - leaf_base : rope);
          int next = rope;                                   // L10: N_skip
          if (query.hit_box(rec.lox, rec.loy, rec.loz, rec.hix, rec.hiy, rec.hiz)) {   // L3
            if (next_first - first <= SCAN) {                // small subtree: post its leaves, continue after it
              s_range[threadIdx.x] = make_int2(first, next_first);
              post = true;
            } else if (try_contain && next_first - first > kContainMinLeaves &&
                       query.contains_box(rec.lox, rec.loy, rec.loz, rec.hix, rec.hiy, rec.hiz)) {
              // a large subtree that lies inside the query: all its leaves are results; nothing below is walked or tested
              count += next_first - first;
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
    if (STORE && kFillStage == 2) {                          // what is still staged: the row's last, partial sector
      const int carry = min(count, (align + count) & (kStageInts - 1));
      const int* st = s_stage + threadIdx.x * kStageInts;
      for (int e = 0; e < carry; ++e)
        if (count - carry + e < cap) row[count - carry + e] = st[e];
    }
    if constexpr (REDUCE) {
      if (have) {
        A.counts[j] = best_idx;
        A.keys[j] = best_key;
      }
    } else if (MODE != kModeFill && have) {
      A.counts[j] = count;
    }
  }
}

// The leaf format (point or box records) is a property of the hierarchy, recorded in its header by the build;
// the kernel reads it there (one uniform branch), so the query entry points need no extra argument.  The same
// header tells whether `nodes` holds a finished hierarchy over n primitives at all: if not (never built, built for
// another n, overwritten), nothing is traversed -- counts come out as 0, nothing is stored -- instead of following
// garbage indices.
template <typename Query, int MODE, bool SPREAD, int SCAN = kScanLeaves>
__global__ void __launch_bounds__(kTravThreads, Query::kCtasPerSm) traverse_kernel(const TraverseArgs A) {
  if (SPREAD) {      // small batches are launched with programmatic stream serialisation
    pdl_wait();      // the previous kernel of the stream has completed
    pdl_trigger();
  }
  const NodesHeader* h = reinterpret_cast<const NodesHeader*>(A.nodes);
  if (h->magic != kNodesMagic || h->n != A.n) {
    if (MODE != kModeFill)
      for (int64_t t = (int64_t)blockIdx.x * kTravThreads + threadIdx.x; t < A.q; t += (int64_t)gridDim.x * kTravThreads) {
        A.counts[t] = (MODE == kModeReduce) ? -1 : 0;
        if (MODE == kModeReduce) A.keys[t] = __int_as_float(0x7f800000);
      }
    return;
  }
  __shared__ TravSmem<Query, mode_stores(MODE)> S;
  if (h->leaf_kind == kLeafPoints)
    traverse_body<Query, MODE, true, SPREAD, SCAN>(A, S);
  else
    traverse_body<Query, MODE, false, SPREAD, SCAN>(A, S);
}

// Small batches.  With one query per lane a warp serves its 32 queries' leaf scans one after the other, each a chain of
// dependent loads; a batch of a few thousand queries is then a few hundred warps that each run for a long time on a
// mostly empty GPU (C1: 4096 queries = 128 warps, 58 us).  When the batch cannot fill the GPU's warp slots anyway, the
// queries are spread out -- only every 2^s-th lane carries one -- so that up to 32 times as many warps share the same
// scans (C1: ... us).  Results and their order do not depend on which lane serves a query.
#ifndef BVH_TRAV_SPREAD_THREADS_PER_SM
#define BVH_TRAV_SPREAD_THREADS_PER_SM 1024
#endif
template <typename Query>
static cudaError_t launch_traverse_kind(TraverseArgs A, int mode, cudaStream_t stream) {
  A.spread_log2 = 0;
  const int64_t spread_threads = (int64_t)sm_count() * BVH_TRAV_SPREAD_THREADS_PER_SM;
  while (A.spread_log2 < 5 && (A.q << (A.spread_log2 + 1)) <= spread_threads) ++A.spread_log2;
  const int64_t chunks = ((A.q << A.spread_log2) + kTravThreads - 1) / kTravThreads;
  if (chunks > 0x7fffffff) return cudaErrorInvalidValue;
  const dim3 g((unsigned)chunks), b(kTravThreads);
  if (A.spread_log2 > 0) {
    // small batch: bound by the latency of its dependent launches -> programmatic dependent launch
    if (mode == kModeCount) return launch_pdl(traverse_kernel<Query, kModeCount, true, kScanLeavesSpread>, g, b, 0, stream, A);
    if (mode == kModeFill) return launch_pdl(traverse_kernel<Query, kModeFill, true, kScanLeavesSpread>, g, b, 0, stream, A);
    if (mode == kModeCollect) return launch_pdl(traverse_kernel<Query, kModeCollect, true, kScanLeavesSpread>, g, b, 0, stream, A);
    if (mode == kModeAny) return launch_pdl(traverse_kernel<Query, kModeAny, true, kScanLeavesSpread>, g, b, 0, stream, A);
    if constexpr (Query::kHasKey) return launch_pdl(traverse_kernel<Query, kModeReduce, true, kScanLeavesSpread>, g, b, 0, stream, A);
    return cudaErrorInvalidValue;
  }
  // a batch that fills the GPU: plain stream order (measured on C3: with the attribute the one-call query is 1.5 % slower)
  if (mode == kModeCount)
    traverse_kernel<Query, kModeCount, false><<<g, b, 0, stream>>>(A);
  else if (mode == kModeFill)
    traverse_kernel<Query, kModeFill, false><<<g, b, 0, stream>>>(A);
  else if (mode == kModeCollect && A.cap <= kSparseRowCap)
    traverse_kernel<Query, kModeCollect, false, kScanLeavesSparse><<<g, b, 0, stream>>>(A);
  else if (mode == kModeCollect)
    traverse_kernel<Query, kModeCollect, false><<<g, b, 0, stream>>>(A);
  else if (mode == kModeAny)
    traverse_kernel<Query, kModeAny, false><<<g, b, 0, stream>>>(A);
  else if constexpr (Query::kHasKey)
    traverse_kernel<Query, kModeReduce, false><<<g, b, 0, stream>>>(A);
  else
    return cudaErrorInvalidValue;
  return cudaGetLastError();
}

cudaError_t launch_traverse(const void* nodes, int n, const float* queries, int64_t q, int kind, int mode,
                            const uint32_t* order, int32_t* counts, const int64_t* offsets, int32_t* out, int64_t cap,
                            bool only_over, float* keys, cudaStream_t stream, int64_t out_limit) {
  TraverseArgs A{};
  A.out_limit = out_limit;
  A.keys = keys;
  A.nodes = static_cast<const char*>(nodes);
  A.n = n;
  A.queries = queries;
  A.q = q;
  A.order = order;
  A.counts = counts;
  A.offsets = offsets;
  A.out = out;
  A.cap = cap;
  A.only_over = only_over ? 1 : 0;
  if (kind == 0) return launch_traverse_kind<SphereQuery>(A, mode, stream);
  if (kind == 1) return launch_traverse_kind<BoxQuery>(A, mode, stream);
  return launch_traverse_kind<RayQuery>(A, mode, stream);
}

// rows -> CSR (single-pass variant): row j of `rows` (cap entries, counts[j] of them valid if counts[j] <= cap) is copied
// to indices[offsets[j] ...).  Rows that did not fit (counts[j] > cap) are skipped: the fill pass restricted to them
// (only_over) writes those.  One group of G lanes per row.  limit != 0: rows that would end past `limit` entries of
// `indices` are skipped too (the caller sized `indices` before it knew nnz, and reads offsets[q] afterwards).
template <int G>
__device__ __forceinline__ void copy_row(const int32_t* __restrict__ src, int32_t* __restrict__ dst, int c, int gl) {
  int e = gl;
  for (; e + 3 * G < c; e += 4 * G) {                     // four loads in flight per lane
    const int v0 = __ldcs(src + e), v1 = __ldcs(src + e + G), v2 = __ldcs(src + e + 2 * G), v3 = __ldcs(src + e + 3 * G);
    dst[e] = v0;
    dst[e + G] = v1;
    dst[e + 2 * G] = v2;
    dst[e + 3 * G] = v3;
  }
  for (; e < c; e += G) dst[e] = __ldcs(src + e);
}

// The same copy by a whole warp with 128-bit accesses (rows of 128 entries and more: C3's rows_to_csr moves 4.7 GB, a fifth
// of the query).  `src`, a row of `rows`, is 32-byte aligned; dst = indices + offsets[j] is aligned to 4 bytes only.  The
// DESTINATION is cut at its 16-byte boundaries: with dst = D + a (D aligned, a in 0..3) the aligned vector m holds
// D[4m .. 4m+3] = src[4m-a .. 4m-a+3], i.e. the last a entries of source vector m-1 and the first 4-a of source vector m.
// Every lane loads source vector m (aligned), takes vector m-1 from the lane below it by shuffle, and stores one aligned
// vector; the up to three entries before the first and after the last whole vector go as 4-byte copies.  Four vectors per
// lane are in flight per round (2 KB per warp; the 4-byte version had 512 B).  Loads stay inside the row: for a whole
// destination vector 4m <= c+a-4 < cap, and cap is a multiple of 8.  All loop bounds are warp-uniform (shuffles inside).
__device__ __forceinline__ int4 shifted_vector(const int4& prev, const int4& cur, int a) {
  if (a == 1) return make_int4(prev.w, cur.x, cur.y, cur.z);
  if (a == 2) return make_int4(prev.z, prev.w, cur.x, cur.y);
  if (a == 3) return make_int4(prev.y, prev.z, prev.w, cur.x);
  return cur;
}
__device__ __forceinline__ void copy_row_wide(const int32_t* __restrict__ src, int32_t* __restrict__ dst, int c, int lane) {
  constexpr int U = 4;
  const int a = (int)((reinterpret_cast<uintptr_t>(dst) >> 2) & 3);
  const int head = min(c, (4 - a) & 3);                    // src[0, head) lie before the first aligned vector
  const int m0 = a ? 1 : 0, m_end = (c + a) >> 2;          // whole destination vectors: m0 <= m < m_end
  if (lane < head) dst[lane] = __ldcs(src + lane);
  const int4* __restrict__ s4 = reinterpret_cast<const int4*>(src);
  int4* __restrict__ d4 = reinterpret_cast<int4*>(dst - a);
  for (int mb = m0; mb < m_end; mb += 32 * U) {
    int4 cur[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int m = mb + 32 * u + lane;
      cur[u] = m < m_end ? __ldcs(s4 + m) : make_int4(0, 0, 0, 0);
    }
    int4 below = make_int4(0, 0, 0, 0);                    // lane 0 of the first vector: source vector mb - 1
    if (a != 0 && lane == 0) below = __ldcs(s4 + mb - 1);
#pragma unroll
    for (int u = 0; u < U; ++u) {
      int4 prev;
      prev.y = __shfl_up_sync(0xffffffffu, cur[u].y, 1);
      prev.z = __shfl_up_sync(0xffffffffu, cur[u].z, 1);
      prev.w = __shfl_up_sync(0xffffffffu, cur[u].w, 1);
      prev.x = 0;
      if (lane == 0) prev = below;
      below.y = __shfl_sync(0xffffffffu, cur[u].y, 31);    // lane 0 of the next vector continues after lane 31 of this one
      below.z = __shfl_sync(0xffffffffu, cur[u].z, 31);
      below.w = __shfl_sync(0xffffffffu, cur[u].w, 31);
      const int m = mb + 32 * u + lane;
      if (m < m_end) d4[m] = shifted_vector(prev, cur[u], a);
    }
  }
  const int t = max(head, 4 * m_end - a) + lane;           // fewer than four entries after the last whole vector
  if (t < c) dst[t] = __ldcs(src + t);
}

template <int G>
__global__ void __launch_bounds__(256) rows_to_csr_kernel(const int32_t* __restrict__ rows, int64_t cap,
                                                          const int32_t* __restrict__ counts,
                                                          const int64_t* __restrict__ offsets, int64_t q,
                                                          int32_t* __restrict__ indices, int64_t limit) {
  pdl_wait();
  pdl_trigger();
  const int64_t group = ((int64_t)blockIdx.x * 256 + threadIdx.x) / G;
  const int64_t groups = (int64_t)gridDim.x * 256 / G;
  const int gl = threadIdx.x % G;
  for (int64_t j = group; j < q; j += groups) {
    const int c = counts[j];
    if (c <= 0 || c > cap) continue;
    const int64_t off = offsets[j];
    if (limit != 0 && off + c > limit) continue;
    if (G == 32)
      copy_row_wide(rows + j * cap, indices + off, c, gl);
    else
      copy_row<G>(rows + j * cap, indices + off, c, gl);
  }
}

cudaError_t launch_rows_to_csr(const int32_t* rows, int64_t cap, const int32_t* counts, const int64_t* offsets, int64_t q,
                               int32_t* indices, cudaStream_t stream, int64_t limit) {
  const int sms = sm_count();
  if (cap >= 128) {
    int64_t blocks = (q * 32 + 255) / 256;
    if (blocks > (int64_t)sms * 16) blocks = (int64_t)sms * 16;
    return launch_pdl(rows_to_csr_kernel<32>, dim3((unsigned)blocks), dim3(256), 0, stream, rows, cap, counts, offsets, q, indices, limit);
  }
  int64_t blocks = (q * 8 + 255) / 256;
  if (blocks > (int64_t)sms * 16) blocks = (int64_t)sms * 16;
  return launch_pdl(rows_to_csr_kernel<8>, dim3((unsigned)blocks), dim3(256), 0, stream, rows, cap, counts, offsets, q, indices, limit);
}

// Small batches (q <= kSmallScan): the exclusive scan of the counts and the copy of the rows in ONE launch.  Every block
// scans all q counts by itself (a few microseconds of redundant work that saves a dependent launch) and keeps the
// offsets in shared memory; block 0 also writes them out.  Then one group of 8 lanes per row, as above.
constexpr int kSmallScan = 4096;
int scan_single_tile_items() { return kSmallScan; }
__global__ void __launch_bounds__(256) scan_rows_to_csr_small_kernel(const int32_t* __restrict__ rows, int64_t cap,
                                                                     const int32_t* __restrict__ counts,
                                                                     int64_t* __restrict__ offsets, int q,
                                                                     int32_t* __restrict__ indices, int64_t limit) {
  constexpr int ITEMS = kSmallScan / 256, G = 8;
  __shared__ int64_t s_off[kSmallScan];
  __shared__ int64_t s_warp[8];
  pdl_wait();
  pdl_trigger();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int base = threadIdx.x * ITEMS;                     // blocked arrangement
  int c[ITEMS];
  int64_t v = 0;
#pragma unroll
  for (int k = 0; k < ITEMS; ++k) {
    c[k] = (base + k < q) ? counts[base + k] : 0;
    v += c[k];
  }
  int64_t incl = v;
#pragma unroll
  for (int off = 1; off < 32; off <<= 1) {
    const int64_t a = __shfl_up_sync(0xffffffffu, incl, off);
    if (lane >= off) incl += a;
  }
  if (lane == 31) s_warp[warp] = incl;
  __syncthreads();
  int64_t run = incl - v, total = 0;
#pragma unroll
  for (int w = 0; w < 8; ++w) {
    const int64_t sw = s_warp[w];
    if (w < warp) run += sw;
    total += sw;
  }
#pragma unroll
  for (int k = 0; k < ITEMS; ++k) {
    if (base + k < q) {
      s_off[base + k] = run;
      if (blockIdx.x == 0) offsets[base + k] = run;
    }
    run += c[k];
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) offsets[q] = total;
  __syncthreads();
  const int gl = threadIdx.x % G;
  for (int j = (blockIdx.x * 256 + threadIdx.x) / G; j < q; j += gridDim.x * 256 / G) {
    const int cj = counts[j];
    if (cj <= 0 || cj > cap) continue;
    const int64_t off = s_off[j];
    if (limit != 0 && off + cj > limit) continue;
    copy_row<G>(rows + (int64_t)j * cap, indices + off, cj, gl);
  }
}

cudaError_t launch_scan_rows_to_csr_small(const int32_t* rows, int64_t cap, const int32_t* counts, int64_t* offsets, int64_t q,
                                          int32_t* indices, cudaStream_t stream, int64_t limit) {
  if (q > kSmallScan) return cudaErrorInvalidValue;
  const unsigned blocks = (unsigned)((q * 8 + 255) / 256);
  return launch_pdl(scan_rows_to_csr_small_kernel, dim3(blocks), dim3(256), 0, stream, rows, cap, counts, offsets, (int)q, indices, limit);
}

}  // namespace bvh
