// oracle/bvh_oracle.cpp
//
// TEST INFRASTRUCTURE ONLY.  A plain, serial, slow CPU statement of what the hot path computes,
// written from /root/reference/PAPER.md ("Revising Apetrei's bounding volume hierarchy construction
// algorithm to allow stackless traversal") and the readings D1-D8 / G1-G21 listed in DESIGN.md.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load
// this file.  It shares no code, header, table or helper with the CUDA path under
// paper_2402_00665_b200/csrc/, and neither includes the other.
//
// Build:  g++ -O2 -std=c++17 -ffp-contract=off -fPIC -shared   (no -ffast-math, no -march flags)
// All floating point is fp32, round-to-nearest, one operation per statement (no contraction), the
// precision BASELINE.json `north_star` fixes.
//
// What each function follows (PAPER.md line numbers):
//   oracle_scene_bounds   D1  union of primitive boxes (frame for step 1)
//   oracle_morton         D2  "calculate Morton indices"; formula is DESIGN.md's reading
//   oracle_sort           D3  "sort Morton indices", stable = index tie-break
//   oracle_hierarchy      D5  Karras' top-down split search, Karras numbering
//   oracle_ropes          D6  skip-connection by its definition: explicit stack walk
//   oracle_ropes_alg2     P2  Algorithm 2 closed form -- second derivation
//   oracle_boxes          D7  step 4 "compute the bounding boxes of the internal nodes"
//   oracle_query_*_tree   D8  range search with a STACK on {left,right}
//   oracle_query_*_brute  D8  the plain definition: test every primitive
//   oracle_nearest_*      D10 "perform an operation" (Alg. 1 L5): nearest primitive within the radius
//   oracle_first_hit_*    D11 the same for rays: the primitive a ray enters first
//   oracle_apetrei        Algorithm 3 run serially: Apetrei's node numbering (index = split)
//   oracle_ropes_from / oracle_boxes_from   D6 / D7 on a hierarchy whose root is not node 0
//
// Parity pins (tests/test_oracle_*.py): P1 worked example reconstructed from PAPER.md:120/166,
// P2 Algorithm 2, P3 invariants, P4 closed forms, P5 brute force, P6 numpy stable sort, P7 Morton
// corners and exact-grid codes, and a test-side transliteration of Algorithm 4.  No function here
// is "parity unpinned".

#include <algorithm>
#include <cstdint>
#include <cstring>
#include <numeric>
#include <utility>
#include <vector>

namespace {

constexpr int32_t SENTINEL = -1;  // the paper's black diamond; G9

struct Box {
  float lo[3];
  float hi[3];
};

// Primitive i as a box.  Points are degenerate boxes (min = max = point).
inline Box prim_box(const float* prim, int64_t i, int is_box) {
  Box b;
  if (is_box) {
    for (int a = 0; a < 3; ++a) {
      b.lo[a] = prim[6 * i + a];
      b.hi[a] = prim[6 * i + 3 + a];
    }
  } else {
    for (int a = 0; a < 3; ++a) {
      b.lo[a] = prim[3 * i + a];
      b.hi[a] = prim[3 * i + a];
    }
  }
  return b;
}

inline float fmin2(float a, float b) { return (b < a) ? b : a; }
inline float fmax2(float a, float b) { return (b > a) ? b : a; }

// Augmented key k'_i = (code_i, i) (reading G5).  Bit numbering: bits 32..95 are the
// code, bits 0..31 the sorted position.
inline int aug_bit(uint64_t code, uint32_t idx, int bit) {
  if (bit >= 32) return (int)((code >> (bit - 32)) & 1u);
  return (int)((idx >> bit) & 1u);
}

// Highest bit at which k'_f and k'_l differ (f != l so they differ somewhere).
inline int highest_differing_bit(uint64_t cf, uint32_t f, uint64_t cl, uint32_t l) {
  const uint64_t xc = cf ^ cl;
  if (xc != 0) return 32 + (63 - __builtin_clzll(xc));  // position of the top set bit of the code XOR
  const uint32_t xi = f ^ l;
  if (xi != 0) return 31 - __builtin_clz(xi);
  return -1;
}

// D8 squared distance from a point to a box, exact association fixed in DESIGN.md.
inline float sphere_d2(const float c[3], const float lo[3], const float hi[3]) {
  float s[3];
  for (int a = 0; a < 3; ++a) {
    float u = lo[a] - c[a];
    float v = c[a] - hi[a];
    float d = fmax2(fmax2(u, v), 0.0f);
    s[a] = d * d;
  }
  float d2 = s[0] + s[1];
  d2 = d2 + s[2];
  return d2;
}

// D8 sphere-vs-box.
inline bool sphere_hits_box(const float c[3], float r, const float lo[3], const float hi[3]) {
  float d2 = sphere_d2(c, lo, hi);
  float r2 = r * r;
  return d2 <= r2;
}

// D8 box-vs-box, closed comparisons (G12).
inline bool box_hits_box(const float qlo[3], const float qhi[3], const float lo[3], const float hi[3]) {
  for (int a = 0; a < 3; ++a) {
    if (!(qlo[a] <= hi[a])) return false;
    if (!(lo[a] <= qhi[a])) return false;
  }
  return true;
}

// D9 ray-vs-box (NEXT-1; "all triangles ... that a ray intersects").  Ray {o.xyz, d.xyz, tmin, tmax}:
// the points o + t d, tmin <= t <= tmax.  Slab test, fp32 round-to-nearest, one operation per step:
// per axis with d != 0: inv = 1 / d, t1 = (lo - o) * inv, t2 = (hi - o) * inv, the ray's interval is clipped to
// [min(t1,t2), max(t1,t2)]; per axis with d == 0 the ray never leaves the slab or never enters it: lo <= o <= hi
// (closed, G12).  Hit iff the clipped interval is not empty (tn <= tf: touching counts).
inline bool ray_enters_box(const float ray[8], const float lo[3], const float hi[3], float* t_enter);
inline bool ray_hits_box(const float ray[8], const float lo[3], const float hi[3]) {
  float t;
  return ray_enters_box(ray, lo, hi, &t);
}
// ... and where the clipped interval starts (D11: the parameter at which the ray is inside all three slabs for the
// first time, never less than tmin).
inline bool ray_enters_box(const float ray[8], const float lo[3], const float hi[3], float* t_enter) {
  float tn = ray[6], tf = ray[7];
  for (int a = 0; a < 3; ++a) {
    const float o = ray[a], d = ray[3 + a];
    if (d == 0.0f) {
      if (!(lo[a] <= o && o <= hi[a])) return false;
    } else {
      const float inv = 1.0f / d;
      float t1 = lo[a] - o;
      t1 = t1 * inv;
      float t2 = hi[a] - o;
      t2 = t2 * inv;
      const float tmin_a = t1 < t2 ? t1 : t2;
      const float tmax_a = t1 < t2 ? t2 : t1;
      tn = fmax2(tn, tmin_a);
      tf = tf < tmax_a ? tf : tmax_a;
    }
  }
  *t_enter = tn;
  return tn <= tf;
}

inline bool query_hits_box(int kind, const float* queries, int64_t j, const float lo[3], const float hi[3]) {
  if (kind == 0) return sphere_hits_box(queries + 4 * j, queries[4 * j + 3], lo, hi);
  if (kind == 1) return box_hits_box(queries + 6 * j, queries + 6 * j + 3, lo, hi);
  return ray_hits_box(queries + 8 * j, lo, hi);
}

struct CsrResult {
  std::vector<int64_t> offsets;
  std::vector<int32_t> indices;
};

}  // namespace

extern "C" {

// D1.  out6 = {lo.x, lo.y, lo.z, hi.x, hi.y, hi.z}.  n >= 1.
void oracle_scene_bounds(const float* prim, int64_t n, int is_box, float* out6) {
  Box s = prim_box(prim, 0, is_box);
  for (int64_t i = 1; i < n; ++i) {
    Box b = prim_box(prim, i, is_box);
    for (int a = 0; a < 3; ++a) {
      s.lo[a] = fmin2(s.lo[a], b.lo[a]);
      s.hi[a] = fmax2(s.hi[a], b.hi[a]);
    }
  }
  for (int a = 0; a < 3; ++a) {
    out6[a] = s.lo[a];
    out6[3 + a] = s.hi[a];
  }
}

// D2.  bits = 30 (10 per axis) or 63 (21 per axis).  x is the most significant axis: bit k of
// cell_x -> code bit 3k+2, cell_y -> 3k+1, cell_z -> 3k.  Interleave is a bit-by-bit loop.
void oracle_morton(const float* prim, int64_t n, int is_box, const float* scene6, int bits,
                   uint64_t* codes) {
  const int b = bits / 3;
  const float scale = (float)((uint32_t)1 << b);  // 2^b, exact
  const uint32_t cell_max = ((uint32_t)1 << b) - 1u;
  for (int64_t i = 0; i < n; ++i) {
    Box p = prim_box(prim, i, is_box);
    uint32_t cell[3];
    for (int a = 0; a < 3; ++a) {
      float sum = p.lo[a] + p.hi[a];
      float c = sum * 0.5f;
      float e = scene6[3 + a] - scene6[a];
      float t = 0.0f;
      if (e > 0.0f) {
        float num = c - scene6[a];
        t = num / e;
      }
      float scaled = t * scale;
      uint32_t q = (uint32_t)scaled;  // truncation
      cell[a] = (q < cell_max) ? q : cell_max;
    }
    uint64_t code = 0;
    for (int k = 0; k < b; ++k) {
      code |= (uint64_t)((cell[0] >> k) & 1u) << (3 * k + 2);
      code |= (uint64_t)((cell[1] >> k) & 1u) << (3 * k + 1);
      code |= (uint64_t)((cell[2] >> k) & 1u) << (3 * k + 0);
    }
    codes[i] = code;
  }
}

// D3.  perm[i] = original index at sorted position i; equal codes keep ascending original index.
void oracle_sort(const uint64_t* codes, int64_t n, uint64_t* sorted, uint32_t* perm) {
  std::vector<uint32_t> idx((size_t)n);
  std::iota(idx.begin(), idx.end(), 0u);
  std::stable_sort(idx.begin(), idx.end(),
                   [codes](uint32_t a, uint32_t b) { return codes[a] < codes[b]; });
  for (int64_t i = 0; i < n; ++i) {
    perm[i] = idx[(size_t)i];
    sorted[i] = codes[idx[(size_t)i]];
  }
}

// D5.  Karras' construction over the augmented keys (sorted[i], i).
// Unified node index (G8): internal I_k -> k, leaf L_i -> (n-1)+i.  Outputs, all of length n-1:
// left[k], right[k] (unified child indices), first[k], last[k] (range covered by I_k).
// n >= 2 (n = 1 has no internal node).
void oracle_hierarchy(const uint64_t* sorted, int64_t n, int32_t* left, int32_t* right,
                      int32_t* first, int32_t* last) {
  struct Item {
    int32_t f, l, idx;
  };
  std::vector<Item> stack;
  stack.push_back({0, (int32_t)(n - 1), 0});  // "The root node is assigned index 0" PAPER.md:101
  const int32_t leaf_base = (int32_t)(n - 1);
  while (!stack.empty()) {
    Item it = stack.back();
    stack.pop_back();
    const int32_t f = it.f, l = it.l;
    // "partitions its keys according to the highest differing bit in its range" PAPER.md:99
    const int B = highest_differing_bit(sorted[f], (uint32_t)f, sorted[l], (uint32_t)l);
    // gamma = last position in [f, l) whose key has bit B clear.  Keys in [f,l] agree above B and
    // are sorted, so "bit B clear" holds on a prefix of the range: binary search for its end.
    int32_t a = f, b = l;  // invariant: bit clear at a, bit set at b
    while (b - a > 1) {
      int32_t m = a + (b - a) / 2;
      if (aug_bit(sorted[m], (uint32_t)m, B) == 0)
        a = m;
      else
        b = m;
    }
    const int32_t gamma = a;
    first[it.idx] = f;
    last[it.idx] = l;
    // "The children of an internal node with a split gamma are assigned indices gamma and gamma+1
    //  in either the internal node array or the leaf node array" PAPER.md:101
    if (f == gamma) {
      left[it.idx] = leaf_base + gamma;
    } else {
      left[it.idx] = gamma;
      stack.push_back({f, gamma, gamma});
    }
    if (gamma + 1 == l) {
      right[it.idx] = leaf_base + gamma + 1;
    } else {
      right[it.idx] = gamma + 1;
      stack.push_back({gamma + 1, l, gamma + 1});
    }
  }
}

// D6.  "each skip-connection points to the right child of the last internal node that a given node
// is in the left subtree of ... the nodes on the right-most path (including the root node) ... all
// point to the sentinel".  Pre-order walk carrying that right child down.
// rope has 2n-1 entries (unified index).  Works for n = 1 (single leaf = node 0).
void oracle_ropes_from(const int32_t* left, const int32_t* right, int64_t n, int32_t root, int32_t* rope);
void oracle_ropes(const int32_t* left, const int32_t* right, int64_t n, int32_t* rope) {
  oracle_ropes_from(left, right, n, 0, rope);   // Karras numbering: "The root node is assigned index 0" PAPER.md:101
}
// The same walk from a root that is not node 0 (Apetrei numbering: "the root node is no longer guaranteed to be I_0,
// and its index now needs to be stored in the hierarchy").
void oracle_ropes_from(const int32_t* left, const int32_t* right, int64_t n, int32_t root, int32_t* rope) {
  const int32_t leaf_base = (int32_t)(n - 1);
  std::vector<std::pair<int32_t, int32_t>> stack;
  stack.push_back({n >= 2 ? root : 0, SENTINEL});
  while (!stack.empty()) {
    auto [node, r] = stack.back();
    stack.pop_back();
    rope[node] = r;
    if (node < leaf_base) {
      stack.push_back({right[node], r});           // right subtree inherits the rope
      stack.push_back({left[node], right[node]});  // left subtree escapes to the right child
    }
  }
}

// P2.  Algorithm 2 with delta* read as the XOR magnitude of adjacent augmented
// keys (G1): larger = less similar.  Comparing two XOR values of adjacent sorted pairs is done here
// through their highest set bit (position in the 96-bit augmented key), an independent route from
// the CUDA path's packed integer compare.
void oracle_ropes_alg2(const uint64_t* sorted, const int32_t* first, const int32_t* last, int64_t n,
                       int32_t* rope) {
  (void)first;
  const int32_t leaf_base = (int32_t)(n - 1);
  auto dstar = [&](int64_t i) -> int {  // highest differing bit of k'_i, k'_{i+1}; 1000 = +inf
    if (i < 0 || i >= n - 1) return 1000;
    return highest_differing_bit(sorted[i], (uint32_t)i, sorted[i + 1], (uint32_t)(i + 1));
  };
  auto skip_for_right_bound = [&](int32_t e) -> int32_t {
    if (e == n - 1) return SENTINEL;                        // Alg. 2 L1-2
    const int32_t r = e + 1;                                // L4
    if (dstar(r - 1) < dstar(r)) return leaf_base + r;      // L5-6  L_r
    return r;                                               // L8    I_r
  };
  for (int32_t k = 0; k < n - 1; ++k) rope[k] = skip_for_right_bound(last[k]);
  for (int32_t i = 0; i < n; ++i) rope[leaf_base + i] = skip_for_right_bound(i);
}

// D7.  aabb[node][6] = {lo.xyz, hi.xyz}.  Leaf (n-1)+i = box of primitive perm[i]; internal =
// component-wise min / max of its two children, post-order.
void oracle_boxes_from(const float* prim, int is_box, const uint32_t* perm, const int32_t* left,
                       const int32_t* right, int64_t n, int32_t root, float* aabb);
void oracle_boxes(const float* prim, int is_box, const uint32_t* perm, const int32_t* left,
                  const int32_t* right, int64_t n, float* aabb) {
  oracle_boxes_from(prim, is_box, perm, left, right, n, 0, aabb);
}
void oracle_boxes_from(const float* prim, int is_box, const uint32_t* perm, const int32_t* left,
                       const int32_t* right, int64_t n, int32_t root, float* aabb) {
  const int32_t leaf_base = (int32_t)(n - 1);
  for (int64_t i = 0; i < n; ++i) {
    Box b = prim_box(prim, perm[i], is_box);
    for (int a = 0; a < 3; ++a) {
      aabb[6 * (leaf_base + i) + a] = b.lo[a];
      aabb[6 * (leaf_base + i) + 3 + a] = b.hi[a];
    }
  }
  if (n < 2) return;
  std::vector<std::pair<int32_t, int>> stack;  // (node, children_done)
  stack.push_back({root, 0});
  while (!stack.empty()) {
    auto [node, done] = stack.back();
    stack.pop_back();
    if (!done) {
      stack.push_back({node, 1});
      if (right[node] < leaf_base) stack.push_back({right[node], 0});
      if (left[node] < leaf_base) stack.push_back({left[node], 0});
    } else {
      const float* L = aabb + 6 * (int64_t)left[node];
      const float* R = aabb + 6 * (int64_t)right[node];
      float* O = aabb + 6 * (int64_t)node;
      for (int a = 0; a < 3; ++a) {
        O[a] = fmin2(L[a], R[a]);
        O[3 + a] = fmax2(L[3 + a], R[3 + a]);
      }
    }
  }
}

// Whole build, D1-D7.  Output arrays: sorted[n], perm[n], left_child[2n-1] (leaf entries = perm,
// the leaf payload convention of the boundary), rope[2n-1], aabb[2n-1][6], scene6[6];
// right_child[n-1] is oracle-private and optional (may be null).
void oracle_build(const float* prim, int64_t n, int is_box, int bits, uint64_t* sorted,
                  uint32_t* perm, int32_t* left_child, int32_t* rope, float* aabb, float* scene6,
                  int32_t* right_child) {
  if (n <= 0) return;
  oracle_scene_bounds(prim, n, is_box, scene6);
  std::vector<uint64_t> codes((size_t)n);
  oracle_morton(prim, n, is_box, scene6, bits, codes.data());
  oracle_sort(codes.data(), n, sorted, perm);
  std::vector<int32_t> left((size_t)std::max<int64_t>(n - 1, 0)), right(left.size()),
      first(left.size()), last(left.size());
  if (n >= 2) oracle_hierarchy(sorted, n, left.data(), right.data(), first.data(), last.data());
  oracle_ropes(left.data(), right.data(), n, rope);
  oracle_boxes(prim, is_box, perm, left.data(), right.data(), n, aabb);
  for (int64_t k = 0; k < n - 1; ++k) left_child[k] = left[(size_t)k];
  for (int64_t i = 0; i < n; ++i) left_child[(n - 1) + i] = (int32_t)perm[i];
  if (right_child)
    for (int64_t k = 0; k < n - 1; ++k) right_child[k] = right[(size_t)k];
}

// ---- D8 queries ---------------------------------------------------------------------------------
// Tree versions walk the oracle's own {left, right} tree with an explicit stack (the
// technique the paper replaces) and report original primitive indices (leaf payload) in the order
// found.  They return a handle; read it with oracle_result_*.

static void* query_tree(int kind, const float* aabb, const int32_t* left_child,
                        const int32_t* right_child, int64_t n, const float* queries, int64_t q) {
  auto* res = new CsrResult();
  res->offsets.assign((size_t)q + 1, 0);
  const int32_t leaf_base = (int32_t)(n - 1);
  std::vector<int32_t> stack;
  for (int64_t j = 0; j < q; ++j) {
    if (n > 0) {
      stack.clear();
      stack.push_back(0);
      while (!stack.empty()) {
        int32_t node = stack.back();
        stack.pop_back();
        const float* b = aabb + 6 * (int64_t)node;
        const bool hit = query_hits_box(kind, queries, j, b, b + 3);
        if (!hit) continue;
        if (node >= leaf_base) {
          res->indices.push_back(left_child[node]);
        } else {
          stack.push_back(right_child[node]);
          stack.push_back(left_child[node]);
        }
      }
    }
    res->offsets[(size_t)j + 1] = (int64_t)res->indices.size();
  }
  return res;
}

void* oracle_query_spheres_tree(const float* aabb, const int32_t* left_child,
                                const int32_t* right_child, int64_t n, const float* xyzr, int64_t q) {
  return query_tree(0, aabb, left_child, right_child, n, xyzr, q);
}

void* oracle_query_boxes_tree(const float* aabb, const int32_t* left_child,
                              const int32_t* right_child, int64_t n, const float* minmax, int64_t q) {
  return query_tree(1, aabb, left_child, right_child, n, minmax, q);
}

void* oracle_query_rays_tree(const float* aabb, const int32_t* left_child, const int32_t* right_child,
                             int64_t n, const float* rays, int64_t q) {
  return query_tree(2, aabb, left_child, right_child, n, rays, q);
}

// Brute force: the plain definition of range search: every primitive is tested.
// Reports original primitive indices in ascending order.
static void* query_brute(int kind, const float* prim, int64_t n, int is_box, const float* queries,
                         int64_t q) {
  auto* res = new CsrResult();
  res->offsets.assign((size_t)q + 1, 0);
  for (int64_t j = 0; j < q; ++j) {
    for (int64_t i = 0; i < n; ++i) {
      Box b = prim_box(prim, i, is_box);
      if (query_hits_box(kind, queries, j, b.lo, b.hi)) res->indices.push_back((int32_t)i);
    }
    res->offsets[(size_t)j + 1] = (int64_t)res->indices.size();
  }
  return res;
}

void* oracle_query_spheres_brute(const float* prim, int64_t n, int is_box, const float* xyzr,
                                 int64_t q) {
  return query_brute(0, prim, n, is_box, xyzr, q);
}

void* oracle_query_boxes_brute(const float* prim, int64_t n, int is_box, const float* minmax,
                               int64_t q) {
  return query_brute(1, prim, n, is_box, minmax, q);
}

void* oracle_query_rays_brute(const float* prim, int64_t n, int is_box, const float* rays, int64_t q) {
  return query_brute(2, prim, n, is_box, rays, q);
}

// ---- D10 / D11: "Store the result or perform an operation" (Alg. 1 L5) -----------------------------------
// An operation at the leaf instead of a stored row.  Both are defined over the SAME candidate set as the range search
// (the primitives whose box satisfies the predicate), so they are reductions of a CSR row, made unique by a tie rule.
//
// D10 nearest within the radius (sphere queries): among the primitives with d2 <= r*r (D8), the one with the smallest
// d2; equal d2: the smallest original index.  idx[j] = that primitive or -1; d2[j] = its d2 or +infinity.
// D11 first hit (ray queries): among the primitives whose box the ray hits (D9), the one the ray enters first
// (smallest t_enter, the start of the clipped interval); equal t_enter: the smallest original index.
// idx[j] = that primitive or -1; t[j] = its t_enter or +infinity.  "Any hit" is idx[j] >= 0.
static inline float pos_inf() {
  const uint32_t b = 0x7f800000u;
  float f;
  std::memcpy(&f, &b, 4);
  return f;
}

static inline bool candidate(int kind, const float* queries, int64_t j, const float lo[3], const float hi[3], float* key) {
  if (kind == 0) {
    const float* s = queries + 4 * j;
    *key = sphere_d2(s, lo, hi);
    float r2 = s[3] * s[3];
    return *key <= r2;
  }
  return ray_enters_box(queries + 8 * j, lo, hi, key);
}

// Brute force: the plain definition (every primitive is a candidate test).  kind 0 = spheres (D10), 2 = rays (D11).
static void reduce_brute(int kind, const float* prim, int64_t n, int is_box, const float* queries, int64_t q,
                         int32_t* idx, float* key_out) {
  for (int64_t j = 0; j < q; ++j) {
    int32_t best = -1;
    float best_key = pos_inf();
    for (int64_t i = 0; i < n; ++i) {      // ascending original index: a strict "<" keeps the smallest index on ties
      Box b = prim_box(prim, i, is_box);
      float key;
      if (candidate(kind, queries, j, b.lo, b.hi, &key) && (best < 0 || key < best_key)) {
        best = (int32_t)i;
        best_key = key;
      }
    }
    idx[j] = best;
    key_out[j] = best_key;
  }
}

// The same over the oracle's own tree (stack on {left, right}; no pruning beyond the predicate itself, so it visits
// exactly the leaves the range search reports).
static void reduce_tree(int kind, const float* aabb, const int32_t* left_child, const int32_t* right_child, int64_t n,
                        const float* queries, int64_t q, int32_t* idx, float* key_out) {
  const int32_t leaf_base = (int32_t)(n - 1);
  std::vector<int32_t> stack;
  for (int64_t j = 0; j < q; ++j) {
    int32_t best = -1;
    float best_key = pos_inf();
    if (n > 0) {
      stack.clear();
      stack.push_back(0);
      while (!stack.empty()) {
        int32_t node = stack.back();
        stack.pop_back();
        const float* b = aabb + 6 * (int64_t)node;
        float key;
        if (!candidate(kind, queries, j, b, b + 3, &key)) continue;
        if (node >= leaf_base) {
          const int32_t prim_index = left_child[node];
          if (best < 0 || key < best_key || (key == best_key && prim_index < best)) {
            best = prim_index;
            best_key = key;
          }
        } else {
          stack.push_back(right_child[node]);
          stack.push_back(left_child[node]);
        }
      }
    }
    idx[j] = best;
    key_out[j] = best_key;
  }
}

void oracle_nearest_spheres_brute(const float* prim, int64_t n, int is_box, const float* xyzr, int64_t q, int32_t* idx,
                                  float* d2) {
  reduce_brute(0, prim, n, is_box, xyzr, q, idx, d2);
}
void oracle_nearest_spheres_tree(const float* aabb, const int32_t* left_child, const int32_t* right_child, int64_t n,
                                 const float* xyzr, int64_t q, int32_t* idx, float* d2) {
  reduce_tree(0, aabb, left_child, right_child, n, xyzr, q, idx, d2);
}
void oracle_first_hit_rays_brute(const float* prim, int64_t n, int is_box, const float* rays, int64_t q, int32_t* idx,
                                 float* t) {
  reduce_brute(2, prim, n, is_box, rays, q, idx, t);
}
void oracle_first_hit_rays_tree(const float* aabb, const int32_t* left_child, const int32_t* right_child, int64_t n,
                                const float* rays, int64_t q, int32_t* idx, float* t) {
  reduce_tree(2, aabb, left_child, right_child, n, rays, q, idx, t);
}

// ---- Algorithm 3, "Apetrei's algorithm", run serially --------------------------------------------
// The leaf "threads" run one after the other; a thread that finds store[p] empty (ATOMICCAS returned the invalid
// value) stops, the second one to arrive carries on.  Internal nodes are numbered by their split
// position p ("indexed using the split positions gamma"), both children write themselves into the parent
// (L7, L13), and the root -- the node whose range is [0, n-1] -- is wherever the last merge happened: its index is
// returned in *root.  delta* is the XOR magnitude of adjacent augmented keys (G1), compared through its
// highest set bit; +infinity outside [0, n-2].  Unified child indices: I_p -> p, L_i -> (n-1)+i.  n >= 2.
void oracle_apetrei(const uint64_t* sorted, int64_t n, int32_t* left, int32_t* right, int32_t* root) {
  const int32_t leaf_base = (int32_t)(n - 1);
  auto dstar = [&](int64_t i) -> int {
    if (i < 0 || i >= n - 1) return 1000;
    return highest_differing_bit(sorted[i], (uint32_t)i, sorted[i + 1], (uint32_t)(i + 1));
  };
  std::vector<int32_t> store((size_t)(n - 1), -1);                                    // L1
  *root = -1;
  for (int32_t leaf = 0; leaf < n; ++leaf) {                                          // L2
    int32_t i = leaf;                                                                 // index of the current node
    int32_t range_left = leaf, range_right = leaf;                                    // L3-4
    int dl = dstar(range_left - 1), dr = dstar(range_right);
    while (true) {
      const bool is_leaf = range_left == range_right;
      int32_t p;
      if (dr < dl) {                                                                  // L5: left child of its parent
        p = range_right;                                                              // L6: Apetrei index
        left[p] = is_leaf ? leaf_base + i : i;                                        // L7
        const int32_t old = store[p];                                                 // L8: ATOMICCAS
        if (old == -1) {
          store[p] = range_left;
          break;                                                                      // L9
        }
        range_right = old;
        dr = dstar(range_right);                                                      // L10
      } else {                                                                        // L12: right child of its parent
        p = range_left - 1;
        right[p] = is_leaf ? leaf_base + i : i;                                       // L13
        const int32_t old = store[p];                                                 // L14
        if (old == -1) {
          store[p] = range_right;
          break;                                                                      // L15
        }
        range_left = old;
        dl = dstar(range_left - 1);                                                   // L16
      }
      i = p;                                                                          // L18
      if (range_left == 0 && range_right == n - 1) {                                  // L19: the range is everything
        *root = p;
        break;
      }
    }
  }
}

int64_t oracle_result_nnz(void* h) { return (int64_t) static_cast<CsrResult*>(h)->indices.size(); }

void oracle_result_copy(void* h, int64_t* offsets, int32_t* indices) {
  auto* r = static_cast<CsrResult*>(h);
  std::memcpy(offsets, r->offsets.data(), r->offsets.size() * sizeof(int64_t));
  if (!r->indices.empty())
    std::memcpy(indices, r->indices.data(), r->indices.size() * sizeof(int32_t));
}

void oracle_result_free(void* h) { delete static_cast<CsrResult*>(h); }

// Algorithm 1 (reading G3) run with an always-true predicate on a
// {left_child, rope} hierarchy: writes the visit order (unified indices) and returns its length,
// or -1 if more than max_visits nodes are visited (a cycle).  Used to check P3 on any hierarchy.
int64_t oracle_walk_all(const int32_t* left_child, const int32_t* rope, int64_t n, int32_t* order,
                        int64_t max_visits) {
  if (n <= 0) return 0;
  const int32_t leaf_base = (int32_t)(n - 1);
  int64_t k = 0;
  int32_t node = 0;
  do {
    if (k >= max_visits) return -1;
    order[k++] = node;
    node = (node >= leaf_base) ? rope[node] : left_child[node];
  } while (node != SENTINEL);
  return k;
}

}  // extern "C"
