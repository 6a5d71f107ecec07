// bounds_morton.cu -- K1 scene bounds (D1) and K2 Morton encoding (D2) fused with the
// digit histograms the one-sweep sort needs.  Both are single streaming passes over the input.
#include "common.cuh"
#include "device_helpers.cuh"

namespace bvh {

// ---------------------------------------------------------------------------------------------------
// K1.  The input is read as a flat float array with 128-bit loads, a warp covering 96 consecutive
// float4 (1536 B) per step with lane-contiguous addresses.  The role of a scalar (which axis; for
// boxes also min or max) is periodic in the flat index with period 3 (points) or 6 (boxes) floats, and
// 96 float4 = 384 floats is a multiple of both, so each (load slot j, component c) of a lane always
// sees the same role: 12 running mins and 12 running maxes per thread, sorted into axes once at the
// end.  Then warp shuffles, one shared-memory step per block, and one atomicMax per block and bound
// on the order-preserving uint image of the float (min is kept as ~ord so that everything is a max
// and the zero-initialised header is the identity).
// ---------------------------------------------------------------------------------------------------
constexpr int kBoundsThreads = 256;

__device__ __forceinline__ void fold_role(int role, bool is_box, float mn, float mx, float lo[3], float hi[3]) {
  // role: flat index modulo 6.  points: axis = role % 3, both bounds.  boxes: role < 3 -> min of axis role,
  // else max of axis role - 3.
  const int axis = role % 3;
  const bool use_min = !is_box || role < 3;
  const bool use_max = !is_box || role >= 3;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    if (axis == a) {
      if (use_min) lo[a] = fminf(lo[a], mn);
      if (use_max) hi[a] = fmaxf(hi[a], mx);
    }
  }
}

__global__ void __launch_bounds__(kBoundsThreads) scene_bounds_kernel(const float* __restrict__ prim, int64_t nfloats,
                                                                      bool is_box, Header* __restrict__ header) {
  pdl_wait();
  pdl_trigger();
  const float inf = __int_as_float(0x7f800000);
  // (load slot j, component c) of a lane sees the scalar with flat index 4 * (32 j + lane) + c of the chunk, whose role is
  // that index modulo 6 = (2 j + c + 4 lane) mod 6: the twelve (j, c) fall into six classes k = (2 j + c) mod 6 of two
  // members each, whatever the lane.  Six running mins and six maxes per thread.
  float mn[6], mx[6];
#pragma unroll
  for (int k = 0; k < 6; ++k) {
    mn[k] = inf;
    mx[k] = -inf;
  }
  const int lane = threadIdx.x & 31;
  const int64_t warp_global = ((int64_t)blockIdx.x * kBoundsThreads + threadIdx.x) >> 5;
  const int64_t num_warps = ((int64_t)gridDim.x * kBoundsThreads) >> 5;
  const int64_t nvec = nfloats >> 2;          // whole float4s
  const int64_t nchunks = nvec / 96;          // whole 96-float4 chunks
  const float4* __restrict__ v = reinterpret_cast<const float4*>(prim);
  auto fold = [&](const float4 (&x)[3]) {
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      const float f[4] = {x[j].x, x[j].y, x[j].z, x[j].w};
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        const int k = (2 * j + c) % 6;
        mn[k] = fminf(mn[k], f[c]);
        mx[k] = fmaxf(mx[k], f[c]);
      }
    }
  };
  int64_t ch = warp_global;
  for (; ch + num_warps < nchunks; ch += 2 * num_warps) {   // two chunks per turn: six 128-bit loads in flight per lane
    const float4* p = v + ch * 96 + lane;
    const float4* p2 = v + (ch + num_warps) * 96 + lane;
    float4 x[3], y[3];
#pragma unroll
    for (int j = 0; j < 3; ++j) x[j] = __ldcs(p + j * 32);   // streaming: read exactly once
#pragma unroll
    for (int j = 0; j < 3; ++j) y[j] = __ldcs(p2 + j * 32);
    fold(x);
    fold(y);
  }
  for (; ch < nchunks; ch += num_warps) {
    const float4* p = v + ch * 96 + lane;
    float4 x[3];
#pragma unroll
    for (int j = 0; j < 3; ++j) x[j] = __ldcs(p + j * 32);
    fold(x);
  }
  float lo[3] = {inf, inf, inf}, hi[3] = {-inf, -inf, -inf};
#pragma unroll
  for (int k = 0; k < 6; ++k) fold_role((k + 4 * lane) % 6, is_box, mn[k], mx[k], lo, hi);
  // tail: scalars after the last whole chunk
  const int64_t tail0 = nchunks * 96 * 4;
  for (int64_t e = tail0 + (int64_t)blockIdx.x * kBoundsThreads + threadIdx.x; e < nfloats;
       e += (int64_t)gridDim.x * kBoundsThreads) {
    const float f = prim[e];
    fold_role((int)(e % 6), is_box, f, f, lo, hi);
  }
  // warp reduce
#pragma unroll
  for (int a = 0; a < 3; ++a) {
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
      lo[a] = fminf(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], off));
      hi[a] = fmaxf(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], off));
    }
  }
  __shared__ float s[kBoundsThreads / 32][6];
  const int warp = threadIdx.x >> 5;
  if (lane == 0) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      s[warp][a] = lo[a];
      s[warp][3 + a] = hi[a];
    }
  }
  __syncthreads();
  if (threadIdx.x < 6) {
    float r = s[0][threadIdx.x];
    for (int w = 1; w < kBoundsThreads / 32; ++w)
      r = (threadIdx.x < 3) ? fminf(r, s[w][threadIdx.x]) : fmaxf(r, s[w][threadIdx.x]);
    // canonical zero: -0.0 and +0.0 compare equal for fminf/fmaxf; inputs carry no -0.0 (G19)
    const uint32_t o = float_to_ordered(r);
    atomicMax(&header->bounds_enc[threadIdx.x], threadIdx.x < 3 ? ~o : o);
  }
}

cudaError_t launch_scene_bounds(const float* prim, int n, bool is_box, Header* header, cudaStream_t stream) {
  const int64_t nfloats = (int64_t)n * (is_box ? 6 : 3);
  const int64_t chunks = nfloats / (96 * 4);
  int64_t blocks = (chunks + (kBoundsThreads / 32) - 1) / (kBoundsThreads / 32);
  const int64_t cap = (int64_t)sm_count() * 8;
  if (blocks > cap) blocks = cap;
  if (blocks < 1) blocks = 1;
  return launch_pdl(scene_bounds_kernel, dim3((unsigned)blocks), dim3(kBoundsThreads), 0, stream, prim, nfloats, is_box, header);
}

// ---------------------------------------------------------------------------------------------------
// K2.  One thread per group of four points / two boxes (one query in the query-ordering variants).  D2: centroid c = (min + max) * 0.5, t = (c - lo) / (hi - lo) (0 when
// the extent is 0), cell = min(trunc(t * 2^b), 2^b - 1), all fp32 round-to-nearest with explicit
// intrinsics so that nvcc cannot contract them.  Bits are spread with magic-number masks; x is the
// most significant axis of each triple.  The same pass accumulates the 256-bin histogram of every
// 8-bit digit of the code in shared memory and flushes it with one global atomic per non-empty bin
// and block: the sort then needs no histogram pass of its own.
// ---------------------------------------------------------------------------------------------------
constexpr int kMortonThreads = 256;

// PRIM_FLOATS: 3 = points, 6 = boxes {min,max}, 4 = sphere queries {x,y,z,r} (centre only; used to order queries),
// 8 = ray queries {o.xyz, d.xyz, tmin, tmax} (origin only; used to order queries).
// FROM_ROOT: the frame is the root box of a finished hierarchy (kept in its NodesHeader) instead of the build header.
template <typename KeyT, int PASSES, int PRIM_FLOATS, bool FROM_ROOT>
__global__ void __launch_bounds__(kMortonThreads) morton_kernel(const float* __restrict__ prim, int n,
                                                                const Header* __restrict__ header,
                                                                const NodesHeader* __restrict__ root,
                                                                KeyT* __restrict__ codes, uint32_t* __restrict__ hist,
                                                                int shift0) {
  // shift0: the histograms are those of the PASSES 8-bit digits from bit shift0 up (63-bit codes are sorted by their
  // upper 32 bits first: tie_fixup.cu).
  __shared__ uint32_t s_hist[PASSES * 256];
  for (int i = threadIdx.x; i < PASSES * 256; i += kMortonThreads) s_hist[i] = 0;
  pdl_wait();
  pdl_trigger();
  float scene[6];
  if (FROM_ROOT) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      scene[a] = root->scene_lo[a];
      scene[3 + a] = root->scene_hi[a];
    }
  } else {
    load_scene_bounds(header, scene);
  }
  __syncthreads();
  constexpr int B = (sizeof(KeyT) == 4) ? 10 : 21;
  const float scale = (float)(1u << B);
  const uint32_t cell_max = (1u << B) - 1u;
  // code of one primitive (D2) + its digits into the block's histograms
  auto encode = [&](float lo[3], float hi[3]) -> KeyT {
    uint32_t cell[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      if (FROM_ROOT) {  // queries may lie outside the frame: clamp the centroid into it (ordering heuristic only)
        const float c = __fmul_rn(__fadd_rn(lo[a], hi[a]), 0.5f);
        lo[a] = hi[a] = fminf(fmaxf(c, scene[a]), scene[3 + a]);
      }
      cell[a] = quantise(lo[a], hi[a], scene[a], scene[3 + a], scale, cell_max);
    }
    const KeyT code = morton_code<KeyT>(cell);
#pragma unroll
    for (int p = 0; p < PASSES; ++p) atomicAdd(&s_hist[p * 256 + (int)((code >> (shift0 + 8 * p)) & 0xFF)], 1u);
    return code;
  };
  const int64_t tid0 = (int64_t)blockIdx.x * kMortonThreads + threadIdx.x, stride = (int64_t)gridDim.x * kMortonThreads;
  int64_t done = 0;                                       // primitives [0, done) are covered by the vector loop
  if (PRIM_FLOATS == 3 || PRIM_FLOATS == 6) {
    // 12 consecutive floats = three 128-bit loads per thread = four points or two boxes: a quarter of the load
    // instructions of one scalar load per coordinate, and 48 bytes in flight per thread instead of 12 (the kernel
    // waits on its loads, not on its arithmetic).  The codes leave as one or two 128-bit stores.  Box QUERIES (FROM_ROOT
    // with six floats) come this way too.  The 128-bit accesses need `prim` and `codes` 16-byte aligned: the build and
    // query_order (capi.cu) refuse a misaligned pointer, and the scratch layout keeps `codes` on a 256-byte boundary.
    constexpr int PG = (PRIM_FLOATS == 3) ? 4 : 2;        // primitives per group
    const int64_t groups = n / PG;
    const float4* __restrict__ v = reinterpret_cast<const float4*>(prim);
    for (int64_t g = tid0; g < groups; g += stride) {
      const float4 x0 = __ldcs(v + 3 * g), x1 = __ldcs(v + 3 * g + 1), x2 = __ldcs(v + 3 * g + 2);
      const float f[12] = {x0.x, x0.y, x0.z, x0.w, x1.x, x1.y, x1.z, x1.w, x2.x, x2.y, x2.z, x2.w};
      KeyT c[PG];
#pragma unroll
      for (int k = 0; k < PG; ++k) {
        float lo[3], hi[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
          lo[a] = f[(PRIM_FLOATS == 3 ? 3 : 6) * k + a];
          hi[a] = f[(PRIM_FLOATS == 3 ? 3 : 6) * k + (PRIM_FLOATS == 3 ? 0 : 3) + a];
        }
        c[k] = encode(lo, hi);
      }
      if (sizeof(KeyT) == 4) {
        if (PG == 4)
          reinterpret_cast<uint4*>(codes)[g] = make_uint4((uint32_t)c[0], (uint32_t)c[1], (uint32_t)c[2], (uint32_t)c[PG - 1]);
        else
          reinterpret_cast<uint2*>(codes)[g] = make_uint2((uint32_t)c[0], (uint32_t)c[1]);
      } else {
#pragma unroll
        for (int k = 0; k < PG; k += 2)
          reinterpret_cast<ulonglong2*>(codes)[(PG / 2) * g + k / 2] = make_ulonglong2((unsigned long long)c[k], (unsigned long long)c[k + 1]);
      }
    }
    done = groups * PG;
  }
  for (int64_t i = done + tid0; i < n; i += stride) {     // the last n % PG primitives; every sphere and ray query (4 / 8 floats)
    float lo[3], hi[3];
    if (PRIM_FLOATS == 6) {
      const float* p = prim + 6 * i;
      lo[0] = p[0]; lo[1] = p[1]; lo[2] = p[2]; hi[0] = p[3]; hi[1] = p[4]; hi[2] = p[5];
    } else if (PRIM_FLOATS == 4 || PRIM_FLOATS == 8) {
      const float4 q4 = __ldg(reinterpret_cast<const float4*>(prim) + (PRIM_FLOATS / 4) * i);
      lo[0] = hi[0] = q4.x; lo[1] = hi[1] = q4.y; lo[2] = hi[2] = q4.z;
    } else {
      const float* p = prim + 3 * i;
      lo[0] = hi[0] = p[0];
      lo[1] = hi[1] = p[1];
      lo[2] = hi[2] = p[2];
    }
    codes[i] = encode(lo, hi);
  }
  __syncthreads();
  for (int i = threadIdx.x; i < PASSES * 256; i += kMortonThreads) {
    const uint32_t c = s_hist[i];
    if (c) atomicAdd(&hist[i], c);
  }
}

static unsigned morton_grid(int n, int per_thread = 1) {
  const int64_t units = ((int64_t)n + per_thread - 1) / per_thread;
  int64_t blocks = (units + kMortonThreads - 1) / kMortonThreads;
  const int64_t cap = (int64_t)sm_count() * 8;
  if (blocks > cap) blocks = cap;
  if (blocks < 1) blocks = 1;
  return (unsigned)blocks;
}

cudaError_t launch_morton(const float* prim, int n, bool is_box, int morton_bits, const Header* header, void* codes,
                          uint32_t* hist, cudaStream_t stream, int passes, int shift0) {
  const unsigned g = morton_grid(n, is_box ? 2 : 4);
  const dim3 G(g), T(kMortonThreads);
  const NodesHeader* none = nullptr;
  if (morton_bits == 30) {
    if (is_box) return launch_pdl(morton_kernel<uint32_t, 4, 6, false>, G, T, 0, stream, prim, n, header, none, (uint32_t*)codes, hist, shift0);
    return launch_pdl(morton_kernel<uint32_t, 4, 3, false>, G, T, 0, stream, prim, n, header, none, (uint32_t*)codes, hist, shift0);
  }
  if (passes == 4) {   // 63-bit codes sorted by their upper 32 bits first (tie_fixup.cu)
    if (is_box) return launch_pdl(morton_kernel<uint64_t, 4, 6, false>, G, T, 0, stream, prim, n, header, none, (uint64_t*)codes, hist, shift0);
    return launch_pdl(morton_kernel<uint64_t, 4, 3, false>, G, T, 0, stream, prim, n, header, none, (uint64_t*)codes, hist, shift0);
  }
  if (is_box) return launch_pdl(morton_kernel<uint64_t, 8, 6, false>, G, T, 0, stream, prim, n, header, none, (uint64_t*)codes, hist, shift0);
  return launch_pdl(morton_kernel<uint64_t, 8, 3, false>, G, T, 0, stream, prim, n, header, none, (uint64_t*)codes, hist, shift0);
}

cudaError_t launch_query_morton(const float* queries, int q, int kind, const NodesHeader* root, uint32_t* codes, uint32_t* hist,
                                cudaStream_t stream) {
  // histograms of the kQueryOrderPasses digits from bit kQueryOrderShift up: the schedule only sorts by those
  const unsigned g = morton_grid(q);
  constexpr int P = kQueryOrderPasses, S = kQueryOrderShift;
  if (kind == 0)
    return launch_pdl(morton_kernel<uint32_t, P, 4, true>, dim3(g), dim3(kMortonThreads), 0, stream, queries, q, nullptr, root, codes, hist, S);
  else if (kind == 2)
    return launch_pdl(morton_kernel<uint32_t, P, 8, true>, dim3(g), dim3(kMortonThreads), 0, stream, queries, q, nullptr, root, codes, hist, S);
  else
    return launch_pdl(morton_kernel<uint32_t, P, 6, true>, dim3(g), dim3(kMortonThreads), 0, stream, queries, q, nullptr, root, codes, hist, S);
}

}  // namespace bvh
