/* bvh_b200.h -- C ABI of libbvh_b200.so: linear-BVH construction with skip-connections in a single
 * bottom-up pass, and stackless range queries, on one NVIDIA B200 (sm_100a).
 *
 * Method: "Revising Apetrei's bounding volume hierarchy construction algorithm to allow stackless
 * traversal" (arXiv 2402.00665).  "PAPER.md:N" cites line N of the paper's text; "G#"/"D#" cite the
 * readings and definitions listed in DESIGN.md where the paper is silent or garbled.
 *
 * Conventions for EVERY entry point
 *  - All data pointers are DEVICE pointers (cudaMalloc / torch CUDA memory), 16-byte aligned (`nodes`
 *    and the `rows` of bvh_query_collect: 32-byte aligned), owned by the caller.  The only host
 *    pointers are the `size_t*` outputs of the *_sizes functions.
 *  - The library never allocates, frees or synchronises; it holds no global state and is re-entrant
 *    across streams (one documented exception: bvh_scan_counts_static keeps its scratch inside the library).  Every call only enqueues work on `stream` (a cudaStream_t passed as void*;
 *    NULL = the legacy default stream) and returns.
 *  - `scratch` of a build must stay alive until that build's stream work is complete; it also
 *    holds the sorted codes and permutation that bvh_export reads.  `nodes` must stay alive until
 *    the last query that uses it is complete.
 *  - Return value: BVH_OK (0) or a negative BVH_ERR_* code.  Nothing is enqueued when an argument
 *    check fails.  Asynchronous kernel faults surface at the caller's next synchronisation.
 *  - Inputs must not contain NaN; radii must be >= 0; boxes must have min <= max.  Not checked.
 *
 * Node addressing (G8).  A hierarchy over n primitives has n leaves and n-1 internal nodes
 * in ONE index space of 2n-1 nodes: internal node I_k -> k (k in [0, n-2], Karras
 * numbering: siblings at consecutive indices, root = 0), leaf L_i -> (n-1)+i where
 * i is the position in Morton order.  The sentinel is -1.  For n = 1 the single
 * leaf is node 0.  `nodes` is an opaque buffer of bvh_sizes' node_bytes: a 64-byte header, the n-1 internal
 * records { float min[3]; int32 left_child;  float max[3]; int32 rope; } by Karras index, then the n leaf records
 * in Morton order (16 bytes {x, y, z, payload} after bvh_build_points, 32 bytes after bvh_build_boxes; the
 * payload is the ORIGINAL index of the primitive plus one bit that tells whether the leaf's skip-connection is
 * the leaf or the internal node i+1, Algorithm 2).  bvh_export turns it into the canonical arrays of the
 * unified index space: left_child (PAPER.md:46 N_left; for a leaf: the primitive), rope (N_skip), boxes.
 */
#ifndef BVH_B200_H
#define BVH_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define BVH_OK 0
#define BVH_ERR_INVALID_ARGUMENT (-1) /* null pointer, negative count, misaligned pointer            */
#define BVH_ERR_MORTON_BITS (-2)      /* morton_bits is not 30 or 63                                   */
#define BVH_ERR_TOO_LARGE (-3)        /* n >= 2^30 (node indices and sort counters are 32-bit)         */
#define BVH_ERR_SCRATCH (-4)          /* scratch_bytes smaller than bvh_sizes / bvh_scan_sizes report  */
#define BVH_ERR_CUDA (-5)             /* a kernel launch failed (cudaGetLastError)                     */
#define BVH_ERR_STATIC_LIMIT (-6)     /* bvh_scan_counts_static: q > BVH_SCAN_STATIC_MAX_Q             */

/* Library version, for the binding's sanity check. */
int bvh_version(void);

/* Bytes the caller must provide for a hierarchy over n primitives: node_bytes = 64 + 32*(n-1) + 32*n (one
 * size for both leaf formats), scratch_bytes = codes + permutation ping-pong buffers, radix-sort histograms
 * and tile status words, the hand-over segments and arrival counters of the bottom-up pass (the `store`
 * array of Algorithm 4, lives in shared memory) and the scene bounds.  Host call. */
int bvh_sizes(int64_t n, int morton_bits, size_t* node_bytes, size_t* scratch_bytes);

/* Build (PAPER.md:83-93 with steps 3-4 replaced by Algorithm 4).
 *   1. scene bounds (D1)  2. Morton index of each primitive's centroid, 10 or 21 bits per axis (D2,
 *   PAPER.md:85)  3. stable LSD radix sort of (code, index) (ties by index)
 *   4. one bottom-up pass from the leaves that merges ranges through ATOMICCAS on `store`, numbers
 *   each parent with its Karras index q, writes its left child and
 *   skip-connection (Alg. 4 L21-26, Algorithm 2) and the union of its children's boxes (G10).
 * How step 3 is organised does not change its result (the stable order by (code, index) is unique): 30-bit codes take
 * four one-sweep passes; 63-bit codes four passes over the upper 32 bits, then every run of equal upper bits is
 * ordered by the lower 31 (a conditional eight-pass sort behind a device flag covers runs too long for a block); for
 * n <= 16384 steps 1-3 are one launch of a thread-block cluster.  The sorted codes and the permutation are left in
 * `scratch` for bvh_export.
 * xyz: n*3 floats (points; a point is the box min = max = point).  minmax: n*6 floats
 * {min.xyz, max.xyz}.  n = 0 is valid and enqueues nothing.  Output: `nodes` (node_bytes). */
int bvh_build_points(const float* xyz, int64_t n, int morton_bits, void* nodes, void* scratch,
                     size_t scratch_bytes, void* stream);
int bvh_build_boxes(const float* minmax, int64_t n, int morton_bits, void* nodes, void* scratch,
                    size_t scratch_bytes, void* stream);

/* The same build with stage boundaries marked for measurement: after stage k the library records
 * stage_events[k] (a cudaEvent_t created by the caller, passed as void*) on `stream` -- recording is
 * asynchronous, nothing is created or synchronised.  NULL entries are skipped.  Stages:
 *   [0] start  [1] scratch initialised  [2] scene bounds  [3] Morton codes + digit histograms
 *   [4+p] sort pass p (30-bit: p < 4.  63-bit: [4..7] the four passes over the upper bits, [8] the tie fix-up,
 *   [9..11] recorded together after the kernels of the conditional second sort)  [12] bottom-up pass (Algorithm 4)
 * A small build (n <= 16384) runs bounds, Morton codes and the whole sort as ONE launch and initialises no scratch: only
 * [0], the event of the last sort pass ([7] or [11]) and [12] are recorded then.
 * stage_events must hold BVH_NUM_STAGE_EVENTS entries.  prim_is_box: 0 = xyz points, 1 = minmax boxes. */
#define BVH_NUM_STAGE_EVENTS 13
int bvh_build_staged(const float* prim, int prim_is_box, int64_t n, int morton_bits, void* nodes, void* scratch,
                     size_t scratch_bytes, void* stream, void* const* stage_events);

/* Query scheduling (optional; "data divergence").  Computes a Morton order of the queries
 * in the frame of the hierarchy's root box: order[t] = index of the query at position t along the curve
 * (30-bit code of the sphere centre / box centroid, clamped into the frame; same kernels as the build's
 * steps 1-2).  Passing `order` to the count and fill calls makes thread t serve query order[t], so that
 * neighbouring threads walk nearly the same nodes.  Results are unaffected: row j of the CSR still
 * belongs to query j.  order: uint32[q].  bvh_query_order_sizes is a host call.
 * A batch of q <= 8192 queries (or n = 0: no frame) gets the IDENTITY order, order[t] = t, in one launch: so small a
 * batch is bound by the number of dependent launches, and the part of the hierarchy it touches stays in L2 whatever the
 * schedule.  `nodes`, the queries and `scratch` are not read then (they may be NULL); `order` is still written in full.
 * queries and scratch must be 16-byte aligned (the codes are computed with 128-bit loads). */
int bvh_query_order_sizes(int64_t q, size_t* scratch_bytes);
int bvh_query_order_spheres(const void* nodes, int64_t n, const float* xyzr, int64_t q, uint32_t* order,
                            void* scratch, size_t scratch_bytes, void* stream);
int bvh_query_order_boxes(const void* nodes, int64_t n, const float* minmax, int64_t q, uint32_t* order,
                          void* scratch, size_t scratch_bytes, void* stream);

/* Range search by Algorithm 1: stackless traversal over
 * {left_child, rope}.  Count pass: counts[j] = number of primitives whose box satisfies query j.
 * Sphere query {x,y,z,r}: squared distance from the centre to the box <= r*r, fp32 round-to-nearest,
 * association of D8.  Box query {min.xyz,max.xyz}: closed-interval overlap on every axis (G12).
 * order: NULL (thread t serves query t) or a permutation of [0,q) from bvh_query_order_*.
 * q = 0 or n = 0: counts (if q > 0) are set to 0.  `nodes` must hold a finished build over exactly n
 * primitives; the library cannot synchronise to check that on the host, so the query kernels check the
 * header the build wrote (magic, n) on the device: a buffer that fails the check yields counts of 0 and no
 * stores instead of a walk over garbage indices. */
int bvh_query_spheres_count(const void* nodes, int64_t n, const float* xyzr, int64_t q, const uint32_t* order,
                            int32_t* counts, void* stream);
int bvh_query_boxes_count(const void* nodes, int64_t n, const float* minmax, int64_t q, const uint32_t* order,
                          int32_t* counts, void* stream);

/* Exclusive prefix sum of counts into 64-bit CSR offsets: offsets[0] = 0, offsets[q] = nnz (G21).
 * bvh_scan_sizes is a host call giving the scratch the scan needs. */
int bvh_scan_sizes(int64_t q, size_t* scratch_bytes);
int bvh_scan_counts(const int32_t* counts, int64_t q, int64_t* offsets, void* scratch,
                    size_t scratch_bytes, void* stream);

/* bvh_scan_counts for a caller that cannot supply `scratch`.  bvh_scan_counts needs a little working memory (one
 * int64 per tile of 4096 counts) and, like the rest of this library, expects the caller to bring it.  That does not
 * work for code that is not allowed to allocate when it runs: a component that starts after the application has handed
 * all device memory to its own pool, a callback inside a framework that forbids allocator calls (cudaMalloc
 * synchronises the whole device, and fails while a stream of the process is being captured), a latency-critical loop
 * that must not wait on the allocator's lock.  This entry point takes no scratch: the tile sums go to a fixed 64 KB
 * array that is part of the library's device image.  It calls no cudaMalloc / cudaFree and no library routine that
 * allocates, and produces the same `offsets`, bit for bit, as bvh_scan_counts.
 *   Limit     q <= BVH_SCAN_STATIC_MAX_Q (2^25 counts = what 64 KB of tile sums cover).  A larger q returns
 *             BVH_ERR_STATIC_LIMIT and enqueues nothing; use bvh_scan_counts with your own scratch for it.
 *   Cost      the 64 KB are resident on every GPU that loads the library, until the process exits, used or not.
 *   Sharing   this is the one place where the library keeps state: one array per GPU, used by every call on that GPU.
 *             Calls that can overlap on the GPU (two streams with no event between them, two host threads) race on
 *             it and spoil each other's offsets; serialise them (one stream per device is enough).  Calls on different
 *             GPUs do not interfere.  The array keeps the previous call's tile sums; nothing in it has to start at
 *             zero, since each scan first writes every entry it later reads.
 *   Set-up    the first call on a device looks up the array's address on that device (and loads the library's kernels
 *             there if nothing has yet); later calls only enqueue.  Make that first call at start-up, on the device and
 *             before any stream capture begins.  The device that is current at the call must be the one that owns
 *             `counts`, `offsets` and `stream`.
 * counts, offsets, q, stream and the q = 0 behaviour (offsets[0] = 0) are as for bvh_scan_counts. */
#define BVH_SCAN_STATIC_MAX_Q ((int64_t)8192 * 4096)
int bvh_scan_counts_static(const int32_t* counts, int64_t q, int64_t* offsets, void* stream);

/* Fill pass: the same traversal again; row j of the CSR, indices[offsets[j] .. offsets[j+1]), gets
 * the ORIGINAL indices of the primitives hit, in traversal order (ascending Morton position; PAPER.md:56
 * "Store the result").  The caller reads offsets[q] to size `indices` (the one device->host sync
 * of the path, and it is the caller's). */
int bvh_query_spheres_fill(const void* nodes, int64_t n, const float* xyzr, int64_t q, const uint32_t* order,
                           const int64_t* offsets, int32_t* indices, void* stream);
int bvh_query_boxes_fill(const void* nodes, int64_t n, const float* minmax, int64_t q, const uint32_t* order,
                         const int64_t* offsets, int32_t* indices, void* stream);

/* Single-pass variant of count-then-fill (Alg. 1 L5 "Store the result";
 * the traversal is the expensive, divergent part, so it should run once).  The caller guesses a row
 * capacity `cap` (entries per query: from an estimate, or from the counts of the previous batch) and provides
 * rows = int32[q * cap], 32-byte aligned; cap is a multiple of 8, >= 8.
 *   bvh_query_collect        ONE traversal: counts[j] = number of hits of query j (exact, whatever cap is), and the
 *                            first min(counts[j], cap) hits of query j, in traversal order, in rows[j*cap ...).
 *                            query_kind: 0 spheres {x,y,z,r}, 1 boxes {min,max}, 2 rays (8 floats); predicates,
 *                            `order` and the n = 0 / q = 0 behaviour as in the count calls.
 *   bvh_scan_counts          (as before) counts -> offsets; the caller reads offsets[q] to size `indices`.
 *   bvh_rows_to_csr          copies every row that fitted (counts[j] <= cap) to indices[offsets[j] ...).
 *   bvh_query_fill_overflow  the fill traversal for the rows that did not fit (counts[j] > cap) only; a no-op walk
 *                            when there are none.
 * After the three calls `offsets` / `indices` are byte-identical to what count -> scan -> fill produce. */
int bvh_query_collect(const void* nodes, int64_t n, const float* queries, int query_kind, int64_t q,
                      const uint32_t* order, int64_t cap, int32_t* rows, int32_t* counts, void* stream);
int bvh_rows_to_csr(const int32_t* rows, int64_t cap, const int32_t* counts, const int64_t* offsets, int64_t q,
                    int32_t* indices, void* stream);
int bvh_query_fill_overflow(const void* nodes, int64_t n, const float* queries, int query_kind, int64_t q,
                            const uint32_t* order, int64_t cap, const int32_t* counts, const int64_t* offsets,
                            int32_t* indices, void* stream);

/* The whole single-pass query as ONE call (the sequence above, enqueued back to back with programmatic dependent
 * launch, so that a small batch is not bound by the host's call overhead): query order (batches of more than 8192
 * queries; smaller ones are served in input order), bvh_query_collect, scan, rows -> CSR, overflow rows.
 *   rows     int32[q * cap], 32-byte aligned, cap a multiple of 8 (the caller's guess of a row capacity, as above)
 *   order    uint32[q] (written; may be NULL when q <= 8192)      counts  int32[q] (written)
 *   offsets  int64[q + 1] (written; offsets[q] = nnz)
 *   indices  int32[indices_capacity]: the caller sizes it BEFORE nnz is known.  No row is written past the capacity: a
 *            row that would end beyond it is skipped.  The caller reads offsets[q] after its own synchronisation; if
 *            nnz <= indices_capacity the CSR is complete and byte-identical to count -> scan -> fill, otherwise it
 *            provides a larger buffer and calls bvh_rows_to_csr + bvh_query_fill_overflow (counts, offsets, order and
 *            rows are all valid).
 *   scratch  bvh_query_csr_sizes(q) bytes, 16-byte aligned.
 * n = 0: offsets all 0.  q = 0: offsets[0] = 0. */
int bvh_query_csr_sizes(int64_t q, size_t* scratch_bytes);
int bvh_query_csr(const void* nodes, int64_t n, const float* queries, int query_kind, int64_t q, int64_t cap,
                  int32_t* rows, uint32_t* order, int32_t* counts, int64_t* offsets, int32_t* indices,
                  int64_t indices_capacity, void* scratch, size_t scratch_bytes, void* stream);

/* NEXT-1: ray queries, "all [primitives] that a ray intersects", through the same
 * Algorithm 1 kernel with a third predicate.  A ray is 8 floats {origin.xyz, direction.xyz, tmin, tmax}: the points
 * o + t d with tmin <= t <= tmax (a segment; tmax may be large).  Predicate D9: slab test in fp32
 * round-to-nearest; per axis with d != 0, inv = 1/d, t1 = (min - o) * inv, t2 = (max - o) * inv clip the interval;
 * per axis with d == 0 the test is min <= o <= max; hit iff the clipped interval is not empty (touching counts).
 * Direction components must be 0 or normal numbers whose reciprocal is finite; not checked.  rays: q*8 floats,
 * 16-byte aligned.  Same count -> bvh_scan_counts -> fill protocol, same CSR, same `order` semantics (rays are
 * ordered by the Morton code of their origin clamped into the root box). */
int bvh_query_order_rays(const void* nodes, int64_t n, const float* rays, int64_t q, uint32_t* order, void* scratch,
                         size_t scratch_bytes, void* stream);
int bvh_query_rays_count(const void* nodes, int64_t n, const float* rays, int64_t q, const uint32_t* order,
                         int32_t* counts, void* stream);
int bvh_query_rays_fill(const void* nodes, int64_t n, const float* rays, int64_t q, const uint32_t* order,
                        const int64_t* offsets, int32_t* indices, void* stream);

/* NEXT-1, second half: "Store the result or perform an operation" (Algorithm 1 L5).  Operations that
 * replace the stored row; same kernel, same walk, no CSR, one call.  Each is a reduction over the set of primitives the
 * range search would report, made unique by a tie rule on the ORIGINAL primitive index.
 *   bvh_query_spheres_nearest (D10)  index[j] = the primitive with the smallest squared distance d2 (the D8 arithmetic)
 *       among those with d2 <= r*r; equal d2: the smallest index; -1 if there is none.  d2[j] = that distance, +infinity
 *       if none.  The radius shrinks to the best distance found so far, so the walk prunes as it goes.
 *   bvh_query_rays_first_hit (D11)   index[j] = the primitive whose box the ray enters first: smallest t_enter, the
 *       start of the clipped interval of D9 (never less than tmin; a ray that starts inside a box enters it at tmin);
 *       equal t_enter: the smallest index; -1 if none.  t[j] = that parameter, +infinity if none.
 *   bvh_query_any_hit                hit[j] = 1 if some primitive satisfies the predicate of query j, else 0
 *       (query_kind 0 spheres, 1 boxes, 2 rays); the walk of a query stops at its first hit.
 * index, hit: int32[q]; d2, t: float[q]; `order` and the n = 0 / q = 0 behaviour as in the count calls (n = 0:
 * index = -1, keys = +infinity, hit = 0). */
int bvh_query_spheres_nearest(const void* nodes, int64_t n, const float* xyzr, int64_t q, const uint32_t* order,
                              int32_t* index, float* d2, void* stream);
int bvh_query_rays_first_hit(const void* nodes, int64_t n, const float* rays, int64_t q, const uint32_t* order,
                             int32_t* index, float* t, void* stream);
int bvh_query_any_hit(const void* nodes, int64_t n, const float* queries, int query_kind, int64_t q,
                      const uint32_t* order, int32_t* hit, void* stream);

/* NEXT-2: MEASUREMENT variants of the build, not product paths.  They replace the last step (the single
 * bottom-up pass of Algorithm 4) by what the paper compares itself with; bounds, Morton codes, sort and the record
 * layout are unchanged.  (variant = 3 below is the paper's own algorithm in unoptimised form, for the same purpose.)
 *   variant = 1  Karras' top-down construction, one thread per internal node searching its range and split on the
 *                common-prefix length of the augmented keys, skip-connections by Algorithm 2
 *                (PAPER.md:105-116), and a separate bottom-up pass for the boxes with atomic arrival counters in global
 *                memory.  `nodes` comes out byte-identical to bvh_build_points / bvh_build_boxes.
 *   variant = 2  the unmodified Algorithm 3: bottom-up with ATOMICCAS on a global `store`, internal
 *                nodes numbered by their split position (Apetrei numbering), root index stored, followed by
 *                "an extra tree traversal pass" for the skip-connections.  The hierarchy is the same
 *                tree with other node indices; it is NOT traversable by bvh_query_* (which rely on Karras numbering;
 *                the buffer is marked and the query kernels refuse it) and is read back with bvh_variant_export:
 *                left, right: int32[n-1] by Apetrei index (unified child indices: internal p -> p, leaf i -> n-1+i);
 *                rope: int32[2n-1]; aabb: float[2n-1][6]; root: int32[1].  Any output may be NULL.
 *   variant = 3  Algorithm 4 exactly as the paper writes it, in the plain form of variant 2: one
 *                thread per leaf, `store` in global memory, ATOMICCAS, the second arrival numbers the parent (L20), writes
 *                left child and skip-connection (L21-26) and the union of the two boxes, the sibling's read back through L2.
 *                `nodes` comes out byte-identical to bvh_build_points / bvh_build_boxes.  Against variant 2 it measures what
 *                the paper's modification saves; against the product, what the windowed organisation of hierarchy.cu adds.
 * scratch must hold bvh_variant_sizes bytes (the product's scratch plus parent / child / counter arrays).  stage_events
 * as in bvh_build_staged (may be NULL); event [12] closes the replaced step.  bvh_variant_sizes is a host call. */
int bvh_variant_sizes(int64_t n, int morton_bits, int variant, size_t* scratch_bytes);
int bvh_build_variant(const float* prim, int prim_is_box, int64_t n, int morton_bits, void* nodes, void* scratch,
                      size_t scratch_bytes, int variant, void* stream, void* const* stage_events);
int bvh_variant_export(const void* nodes, void* scratch, int64_t n, int morton_bits, int variant, int32_t* left,
                       int32_t* right, int32_t* rope, float* aabb, int32_t* root, void* stream);

/* Parity export: the canonical arrays of a finished build, for bit-exact comparison.
 * sorted_codes: uint32[n] when morton_bits = 30, uint64[n] when 63.  perm: uint32[n], original
 * index at each Morton position.  left_child, rope: int32[2n-1].  aabb: float[2n-1][6]
 * {min.xyz,max.xyz}.  scene_bounds: float[6].  Any output pointer may be NULL to skip it.
 * `scratch` is the one the build used, untouched since. */
int bvh_export(const void* nodes, const void* scratch, int64_t n, int morton_bits, void* sorted_codes,
               uint32_t* perm, int32_t* left_child, int32_t* rope, float* aabb, float* scene_bounds,
               void* stream);

#ifdef __cplusplus
}
#endif
#endif /* BVH_B200_H */
