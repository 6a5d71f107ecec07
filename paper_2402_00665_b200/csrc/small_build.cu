// small_build.cu -- K1 + K2 + K3 of a SMALL build in one launch: scene bounds (D1), Morton codes (D2) and the sort of
// (code, index) pairs for n <= kSmallBuildMax primitives, by ONE thread-block cluster whose blocks
// exchange through distributed shared memory.
//
// Below a few 10^4 primitives the pipeline of memset, bounds, Morton and 4 (30-bit) or 8 (63-bit) one-sweep passes is a
// chain of dependent launches that each run for 4-10 us on one or two SMs (C1, 4096 primitives: 4.4 + 4.1 + 7.7 + 8.8 +
// 8.8 + 10.5 us of the 54 us build; 63-bit codes: eleven launches).  Here the whole front of the build is one kernel: a
// cluster of up to 8 blocks of 256 threads, block r owning the positions [r * PER, (r + 1) * PER) of the sequence.
// Min/max per block and an all-to-all of six floats; the codes computed into registers; then an LSD radix sort whose
// passes never leave the cluster -- the same stable ranking as the one-sweep tile (one ballot per digit bit + per-warp
// counters; position order = (block, warp, item, lane)), a scan over (digit, block, warp) instead of the look-back
// (every block sends its 256 digit totals to every other block), and the exchange as remote shared-memory stores
// into the block that owns the destination.  Two cluster barriers per pass.  No global histograms, no tile status, no
// zero-initialised scratch: the build's memset goes too.  The arithmetic of D1 / D2 is the shared device code of
// bounds_morton.cu (quantise, morton_code), bit for bit; the sort is stable, so equal codes keep ascending original
// index (readings G5/G6).
#include <cooperative_groups.h>

#include "common.cuh"
#include "device_helpers.cuh"

namespace bvh {

namespace cg = cooperative_groups;

constexpr int kSmallThreads = 256;
constexpr int kSmallWarps = kSmallThreads / 32;
constexpr int kSmallMaxCluster = 8;               // the portable cluster size

template <typename KeyT, int IT>
struct SmallSmem {
  KeyT key[kSmallThreads * IT];
  uint32_t val[kSmallThreads * IT];
  uint32_t cnt[kSmallWarps][256];                 // per-warp digit counters, then each (warp, digit)'s first position
  uint32_t ctot[kSmallMaxCluster][256];           // digit totals of every block of the cluster (each block has a copy)
  uint32_t wsum[kSmallWarps];
  float red[kSmallWarps][6];
  float cred[kSmallMaxCluster][6];                // bounds of every block of the cluster
};

template <typename KeyT, bool IS_BOX, int IT>
__global__ void __launch_bounds__(kSmallThreads)
small_front_kernel(const float* __restrict__ prim, int n, Header* __restrict__ header, KeyT* __restrict__ codes_out,
                   uint32_t* __restrict__ perm_out) {
  __shared__ SmallSmem<KeyT, IT> S;
  cg::cluster_group cluster = cg::this_cluster();
  const int crank = (int)cluster.block_rank(), csize = (int)cluster.num_blocks();
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  constexpr int PF = IS_BOX ? 6 : 3;
  constexpr int PASSES = sizeof(KeyT) == 4 ? 4 : 8;
  constexpr int PER = kSmallThreads * IT;         // positions a block owns
  const int block_first = crank * PER;
  const int warp_off = block_first + warp * 32 * IT + lane;   // item j of this lane is position warp_off + 32 j
  pdl_wait();
  pdl_trigger();

  // ---- D1: scene bounds; D2 needs them, so the primitives stay in registers meanwhile ------------------------------
  const float inf = __int_as_float(0x7f800000);
  float plo[IT][3], phi[IT][IS_BOX ? 3 : 1];
  float lo[3] = {inf, inf, inf}, hi[3] = {-inf, -inf, -inf};
#pragma unroll
  for (int j = 0; j < IT; ++j) {
    const int i = warp_off + j * 32;
    if (i < n) {
      const float* p = prim + (size_t)PF * i;
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        plo[j][a] = p[a];
        if (IS_BOX) phi[j][a] = p[3 + a];
        lo[a] = fminf(lo[a], plo[j][a]);
        hi[a] = fmaxf(hi[a], IS_BOX ? phi[j][a] : plo[j][a]);
      }
    }
  }
#pragma unroll
  for (int a = 0; a < 3; ++a) {
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
      lo[a] = fminf(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], off));
      hi[a] = fmaxf(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], off));
    }
  }
  if (lane == 0) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      S.red[warp][a] = lo[a];
      S.red[warp][3 + a] = hi[a];
    }
  }
  __syncthreads();
  if (tid < 6 * csize) {                           // thread (c, k): this block's bound k goes to block c
    const int c = tid / 6, k = tid % 6;
    float r = S.red[0][k];
    for (int w = 1; w < kSmallWarps; ++w) r = (k < 3) ? fminf(r, S.red[w][k]) : fmaxf(r, S.red[w][k]);
    cluster.map_shared_rank(&S.cred[0][0], c)[crank * 6 + k] = r;
  }
  cluster.sync();
  float scene[6];
#pragma unroll
  for (int k = 0; k < 6; ++k) {
    float r = S.cred[0][k];
    for (int c = 1; c < csize; ++c) r = (k < 3) ? fminf(r, S.cred[c][k]) : fmaxf(r, S.cred[c][k]);
    // through the image the large build keeps (atomicMax on ordered uints): the hierarchy kernels and bvh_export decode it
    const uint32_t o = float_to_ordered(r);
    if (crank == 0 && tid == 0) header->bounds_enc[k] = k < 3 ? ~o : o;
    scene[k] = ordered_to_float(o);
  }

  // ---- D2: Morton codes ----------------------------------------------------------------------------------------
  constexpr int B = (sizeof(KeyT) == 4) ? 10 : 21;
  const float scale = (float)(1u << B);
  const uint32_t cell_max = (1u << B) - 1u;
  KeyT key[IT];
  uint32_t val[IT];
#pragma unroll
  for (int j = 0; j < IT; ++j) {
    const int i = warp_off + j * 32;
    key[j] = 0;
    val[j] = (uint32_t)i;
    if (i < n) {
      uint32_t cell[3];
#pragma unroll
      for (int a = 0; a < 3; ++a)
        cell[a] = quantise(plo[j][a], IS_BOX ? phi[j][a] : plo[j][a], scene[a], scene[3 + a], scale, cell_max);
      key[j] = morton_code<KeyT>(cell);
    }
  }

  // ---- K3: LSD radix sort, 8 bits per pass, every pass inside the cluster ----------------------------------------
  const uint32_t lt_mask = (1u << lane) - 1u;
#pragma unroll 1
  for (int pass = 0; pass < PASSES; ++pass) {
    const int shift = 8 * pass;
#pragma unroll
    for (int u = 0; u < kSmallWarps; ++u) S.cnt[u][tid] = 0;
    __syncthreads();
    uint32_t rank[IT];
#pragma unroll
    for (int j = 0; j < IT; ++j) {
      const uint32_t d = (uint32_t)(key[j] >> shift) & 0xFFu;
      const bool valid = (warp_off + j * 32) < n;
      uint32_t peers = match_digit<false>(d, __ballot_sync(0xffffffffu, valid));
      if (!valid) peers = 0;
      const uint32_t below = __popc(peers & lt_mask);
      const uint32_t pre = S.cnt[warp][d];
      __syncwarp();
      if (below == 0 && peers) S.cnt[warp][d] = pre + __popc(peers);
      __syncwarp();
      rank[j] = pre + below;
    }
    __syncthreads();
    // thread d owns digit d: exclusive scan over this block's warps, the block's total to every block of the cluster
    uint32_t mine = 0;
#pragma unroll
    for (int w = 0; w < kSmallWarps; ++w) {
      const uint32_t c = S.cnt[w][tid];
      S.cnt[w][tid] = mine;
      mine += c;
    }
    for (int c = 0; c < csize; ++c) cluster.map_shared_rank(&S.ctot[0][0], c)[crank * 256 + tid] = mine;
    cluster.sync();
    uint32_t base = 0, total = 0;                  // pairs with digit d in the blocks before this one / in all blocks
    for (int c = 0; c < csize; ++c) {
      const uint32_t t = S.ctot[c][tid];
      if (c < crank) base += t;
      total += t;
    }
    uint32_t incl = total;                         // exclusive scan of the totals over the digits
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
      const uint32_t v = __shfl_up_sync(0xffffffffu, incl, off);
      if (lane >= off) incl += v;
    }
    if (lane == 31) S.wsum[warp] = incl;
    __syncthreads();
#pragma unroll
    for (int w = 0; w < kSmallWarps; ++w)
      if (w < warp) base += S.wsum[w];
    base += incl - total;
#pragma unroll
    for (int w = 0; w < kSmallWarps; ++w) S.cnt[w][tid] += base;
    __syncthreads();
    // exchange: position -> the block that owns it
#pragma unroll
    for (int j = 0; j < IT; ++j) {
      if ((warp_off + j * 32) < n) {
        const uint32_t d = (uint32_t)(key[j] >> shift) & 0xFFu;
        const uint32_t pos = S.cnt[warp][d] + rank[j];
        const uint32_t owner = pos / PER, slot = pos % PER;
        cluster.map_shared_rank(&S.key[0], owner)[slot] = key[j];
        cluster.map_shared_rank(&S.val[0], owner)[slot] = val[j];
      }
    }
    cluster.sync();
    if (pass + 1 < PASSES) {
#pragma unroll
      for (int j = 0; j < IT; ++j) {
        const int i = warp_off + j * 32;
        if (i < n) {
          key[j] = S.key[i - block_first];
          val[j] = S.val[i - block_first];
        }
      }
    }
  }

  // ---- sorted codes and permutation, where the one-sweep sort leaves them ----------------------------------
  for (int s = tid; s < PER && block_first + s < n; s += kSmallThreads) {
    codes_out[block_first + s] = S.key[s];
    perm_out[block_first + s] = S.val[s];
  }
}

template <typename KeyT, bool IS_BOX, int IT>
static cudaError_t launch_small_it(const float* prim, int n, Header* header, KeyT* codes, uint32_t* perm, cudaStream_t stream) {
  constexpr int PER = kSmallThreads * IT;
  int csize = 1;
  while (csize * PER < n) csize <<= 1;
  if (csize > kSmallMaxCluster) return cudaErrorInvalidValue;
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(csize);
  cfg.blockDim = dim3(kSmallThreads);
  cfg.dynamicSmemBytes = 0;
  cfg.stream = stream;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  attr[1].id = cudaLaunchAttributeClusterDimension;
  attr[1].val.clusterDim.x = csize;
  attr[1].val.clusterDim.y = 1;
  attr[1].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 2;
  return cudaLaunchKernelEx(&cfg, small_front_kernel<KeyT, IS_BOX, IT>, prim, n, header, codes, perm);
}

template <typename KeyT, bool IS_BOX>
static cudaError_t launch_small_keys(const float* prim, int n, Header* header, void* codes, uint32_t* perm, cudaStream_t stream) {
  // as many blocks as the cluster may have, as few pairs per thread as that allows: the ranking of a thread's pairs is
  // a serial chain, and a pass is bound by latency, not by issue slots
  if (n <= kSmallThreads * 1 * kSmallMaxCluster)
    return launch_small_it<KeyT, IS_BOX, 1>(prim, n, header, static_cast<KeyT*>(codes), perm, stream);
  if (n <= kSmallThreads * 2 * kSmallMaxCluster)
    return launch_small_it<KeyT, IS_BOX, 2>(prim, n, header, static_cast<KeyT*>(codes), perm, stream);
  if (n <= kSmallThreads * 4 * kSmallMaxCluster)
    return launch_small_it<KeyT, IS_BOX, 4>(prim, n, header, static_cast<KeyT*>(codes), perm, stream);
  return launch_small_it<KeyT, IS_BOX, 8>(prim, n, header, static_cast<KeyT*>(codes), perm, stream);
}

cudaError_t launch_small_front(const float* prim, int n, bool is_box, int morton_bits, Header* header, void* codes,
                               uint32_t* perm, cudaStream_t stream) {
  if (n > kSmallThreads * 8 * kSmallMaxCluster) return cudaErrorInvalidValue;
  if (morton_bits == 30)
    return is_box ? launch_small_keys<uint32_t, true>(prim, n, header, codes, perm, stream)
                  : launch_small_keys<uint32_t, false>(prim, n, header, codes, perm, stream);
  return is_box ? launch_small_keys<uint64_t, true>(prim, n, header, codes, perm, stream)
                : launch_small_keys<uint64_t, false>(prim, n, header, codes, perm, stream);
}

}  // namespace bvh
