// radix_sort.cu -- K3: in-house one-sweep LSD radix sort of (Morton code, index) pairs (
// stable, so equal codes keep ascending original index: PAPER.md:172 / reading G6).
//
// One kernel per 8-bit digit.  Each pass reads every pair once and writes it once: a tile's position
// in the output is known inside the pass through a chained scan with decoupled look-back over
// per-tile digit counts, so there is no separate scan or per-pass histogram kernel (the global digit
// histograms come from the Morton kernel).  Tiles take their id from an atomic ticket, so a tile
// only ever waits on tiles that are already running: forward progress without co-residency
// assumptions.
//
// Inside a tile: warp w owns a contiguous run of 32*ITEMS pairs, item j of lane l at offset j*32+l
// (coalesced loads; tile order = (warp, item, lane)).  Ranks come from one ballot per digit bit plus a
// per-warp 256-bin counter array in shared memory, which keeps the order of equal digits = stability.
// Keys and values are then permuted through shared memory into tile-sorted order and written out in
// runs of equal digit, i.e. coalesced.  On B200 this kernel is bound by instruction issue, not by HBM
// (profiles/): the code below is written to keep the per-pair instruction count down -- full tiles take
// a path without bounds predicates, positions are 32-bit, values are loaded after the ranking so that
// fewer registers are live (4 CTAs of 256 threads per SM).
#include <cooperative_groups.h>

#include "common.cuh"
#include "device_helpers.cuh"

namespace bvh {

#ifndef BVH_SORT_THREADS
#define BVH_SORT_THREADS 256
#endif
#ifndef BVH_EARLY_PUBLISH
#define BVH_EARLY_PUBLISH 1
#endif
constexpr int kSortThreads = BVH_SORT_THREADS;   // >= 256: thread d < 256 owns digit d
constexpr bool kEarlyPublish = BVH_EARLY_PUBLISH != 0;
constexpr int kSortWarps = kSortThreads / 32;
constexpr uint32_t kFlagPartial = 1u << 30;
constexpr uint32_t kFlagInclusive = 2u << 30;
constexpr uint32_t kValueMask = (1u << 30) - 1u;

template <typename KeyT>
struct SortCfg {
#ifndef BVH_SORT_ITEMS32
#define BVH_SORT_ITEMS32 16
#endif
#ifndef BVH_SORT_ITEMS64
#define BVH_SORT_ITEMS64 12
#endif
  static constexpr int ITEMS = (sizeof(KeyT) == 4) ? BVH_SORT_ITEMS32 : BVH_SORT_ITEMS64;
  static constexpr int TILE = kSortThreads * ITEMS;
};

int sort_tile_items(int key_bytes) { return key_bytes == 4 ? SortCfg<uint32_t>::TILE : SortCfg<uint64_t>::TILE; }

// Tile status words are single 32-bit values (flag + count in one word), so relaxed GPU-scope accesses
// are all the protocol needs: a reader either sees the whole word or the zero it was initialised with.
__device__ __forceinline__ uint32_t ld_status(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_status(uint32_t* p, uint32_t v) {
  asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

#ifndef BVH_LOOKBACK_BATCH
#define BVH_LOOKBACK_BATCH 4
#endif
constexpr int kLookbackBatch = BVH_LOOKBACK_BATCH;
// Independent ranking chains per warp.  Ranking item j reads and bumps the warp's running count of its digit in shared
// memory, so consecutive items form one dependent chain of shared-memory round trips.  With C chains the warp's items
// are split into C consecutive runs (tile order is (warp, item, lane), so run c precedes run c + 1), each ranked against
// its own counter array, C items per step: the chains overlap, and the runs are put back in order by the scan over
// (warp, chain) below.
#ifndef BVH_SORT_CHAINS
#define BVH_SORT_CHAINS 1
#endif
constexpr int kSortChains = BVH_SORT_CHAINS;

template <typename KeyT>
struct SortSmem {
  uint32_t warp_hist[kSortWarps][kSortChains][256];
  uint32_t tile_excl[256];     // first tile-sorted position of each digit
  uint32_t digit_base[256];    // global position of tile-sorted position 0 of each digit (mod 2^32; n < 2^30)
  uint32_t tile_hist[256];     // early publish: digit counts of the tile, by shared-memory atomics
  uint32_t scan[2][8];
  uint32_t tile;
  KeyT keys[SortCfg<KeyT>::TILE];
  uint32_t vals[SortCfg<KeyT>::TILE];
};

template <typename KeyT, bool IOTA, bool FULL, bool TOP>
__device__ __forceinline__ void sort_tile(SortSmem<KeyT>& s, const KeyT* __restrict__ keys_in, KeyT* __restrict__ keys_out,
                                          const uint32_t* __restrict__ vals_in, uint32_t* __restrict__ vals_out,
                                          const uint32_t* __restrict__ hist, uint32_t* status, uint32_t tile,
                                          uint32_t tile_base, int valid_in_tile, int shift) {
  constexpr int ITEMS = SortCfg<KeyT>::ITEMS;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int warp_off = warp * 32 * ITEMS + lane;
  const bool owner = tid < 256;                       // thread d owns digit d
  uint32_t* my_status = status + (size_t)tile * 256 + tid;

  // ---- load keys (coalesced; warp-contiguous runs) ------------------------------------------------------
  KeyT key[ITEMS];
#pragma unroll
  for (int j = 0; j < ITEMS; ++j) {
    const int t = warp_off + j * 32;
    key[j] = (FULL || t < valid_in_tile) ? keys_in[tile_base + t] : (KeyT)0;
  }

  // ---- early publish: the tile's digit counts, long before the (expensive) ranking is done -----------------
  // A later tile that looks back never has to spin on this tile's ranking; it only walks over published counts.
  uint32_t tile_count = 0;
  if (kEarlyPublish) {
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) {
      const uint32_t d = (uint32_t)(key[j] >> shift) & 0xFFu;
      const bool valid = FULL || (warp_off + j * 32) < valid_in_tile;
      // a warp whose 32 keys share the digit (constant high digits, coincident points) adds once
      int all_same;
      __match_all_sync(0xffffffffu, valid ? d : 0x100u, &all_same);
      if (all_same) {
        if (lane == 0 && valid) atomicAdd(&s.tile_hist[d], 32u);
      } else if (valid) {
        atomicAdd(&s.tile_hist[d], 1u);
      }
    }
    __syncthreads();
    if (owner) {
      tile_count = s.tile_hist[tid];
      st_status(my_status, (tile == 0 ? kFlagInclusive : kFlagPartial) | tile_count);
    }
  }

  // ---- rank within the warp, in tile order ---------------------------------------------------------------
  uint32_t rank2[ITEMS / 2];                          // two 16-bit ranks per register (a rank is < TILE <= 65536)
  static_assert(ITEMS % 2 == 0 && SortCfg<KeyT>::TILE <= 65536, "packed ranks");
  const uint32_t lt_mask = (1u << lane) - 1u;
  constexpr int CH = kSortChains, RUN = ITEMS / CH;   // RUN consecutive items per chain
  static_assert(ITEMS % CH == 0, "whole runs per chain");
  uint32_t(*my_hist)[256] = s.warp_hist[warp];
#pragma unroll
  for (int u = 0; u < ITEMS / 2; ++u) rank2[u] = 0;
#pragma unroll
  for (int jj = 0; jj < RUN; ++jj) {
    uint32_t d[CH], peers[CH], below[CH], pre[CH];
#pragma unroll
    for (int c = 0; c < CH; ++c) {
      const int j = c * RUN + jj;
      d[c] = (uint32_t)(key[j] >> shift) & 0xFFu;
      if (FULL) {
        peers[c] = match_digit<TOP>(d[c], 0xffffffffu);
      } else {
        const bool valid = (warp_off + j * 32) < valid_in_tile;
        peers[c] = match_digit<TOP>(d[c], __ballot_sync(0xffffffffu, valid));
        if (!valid) peers[c] = 0;
      }
    }
    // every peer reads the warp's running count of its digit (a broadcast), the lowest peer then bumps it
#pragma unroll
    for (int c = 0; c < CH; ++c) {
      below[c] = __popc(peers[c] & lt_mask);
      pre[c] = my_hist[c][d[c]];
    }
    __syncwarp();
#pragma unroll
    for (int c = 0; c < CH; ++c)
      if (below[c] == 0 && (FULL || peers[c])) my_hist[c][d[c]] = pre[c] + __popc(peers[c]);
    __syncwarp();
#pragma unroll
    for (int c = 0; c < CH; ++c) {
      const int j = c * RUN + jj;
      rank2[j / 2] |= (pre[c] + below[c]) << ((j & 1) ? 16 : 0);
    }
  }

  // values are only needed for the scatter: issue their loads now, they land during the look-back
  uint32_t val[ITEMS];
#pragma unroll
  for (int j = 0; j < ITEMS; ++j) {
    const int t = warp_off + j * 32;
    if (IOTA)
      val[j] = tile_base + t;
    else
      val[j] = (FULL || t < valid_in_tile) ? vals_in[tile_base + t] : 0u;
  }
  __syncthreads();

  // ---- per digit (thread d owns digit d): exclusive scan over warps, publish tile count, look back -------
  uint32_t tile_excl = 0, glob_excl = 0, g = 0;
  if (owner) {
    uint32_t sum = 0;
#pragma unroll
    for (int w = 0; w < kSortWarps; ++w) {
#pragma unroll
      for (int ch = 0; ch < kSortChains; ++ch) {
        const uint32_t c = s.warp_hist[w][ch][tid];
        s.warp_hist[w][ch][tid] = sum;
        sum += c;
      }
    }
    if (!kEarlyPublish) {
      tile_count = sum;
      st_status(my_status, (tile == 0 ? kFlagInclusive : kFlagPartial) | tile_count);
    }
    // exclusive scan of tile_count over digits (tile-sorted layout) and of the global histogram over digits
    g = hist[tid];
    uint32_t incl_t = tile_count, incl_g = g;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
      const uint32_t a = __shfl_up_sync(0xffffffffu, incl_t, off);
      const uint32_t b = __shfl_up_sync(0xffffffffu, incl_g, off);
      if (lane >= off) {
        incl_t += a;
        incl_g += b;
      }
    }
    if (lane == 31) {
      s.scan[0][warp] = incl_t;
      s.scan[1][warp] = incl_g;
    }
    tile_excl = incl_t - tile_count;
    glob_excl = incl_g - g;
  }
  __syncthreads();
  if (owner) {
#pragma unroll
    for (int w = 0; w < 8; ++w) {
      if (w < warp) {
        tile_excl += s.scan[0][w];
        glob_excl += s.scan[1][w];
      }
    }

    // decoupled look-back over the previous tiles' counts of this digit.  Tiles start faster than one status
    // word can be fetched (about 20 tiles per L2 round trip on C3) and not in perfect order, so the chain to the
    // nearest tile that already knows its inclusive prefix is several tiles long: the words of kLookbackBatch
    // predecessors are fetched at once and consumed in order.  A word that is not published yet (flag 0) is
    // polled alone, with a pause, so that waiting tiles do not flood the L2 slice that holds it.
    uint32_t excl = 0;
    if (tile > 0) {
      int64_t t = (int64_t)tile - 1;
      bool done = false;
      while (!done) {
        uint32_t sw[kLookbackBatch];
#pragma unroll
        for (int u = 0; u < kLookbackBatch; ++u)
          sw[u] = (t - u >= 0) ? ld_status(status + (size_t)(t - u) * 256 + tid) : kFlagInclusive;
        int used = 0;
#pragma unroll
        for (int u = 0; u < kLookbackBatch; ++u) {
          const uint32_t flag = sw[u] & ~kValueMask;
          if (!done && used == u && flag != 0) {
            excl += sw[u] & kValueMask;
            done = (flag == kFlagInclusive);
            used = u + 1;
          }
        }
        t -= used;
        if (!done && used < kLookbackBatch) {   // tile t is running but has not published: wait for that one word
          uint32_t w;
          while (((w = ld_status(status + (size_t)t * 256 + tid)) & ~kValueMask) == 0) __nanosleep(64);
          excl += w & kValueMask;
          done = ((w & ~kValueMask) == kFlagInclusive);
          --t;
        }
      }
      st_status(my_status, kFlagInclusive | (excl + tile_count));
    }
    s.tile_excl[tid] = tile_excl;
    s.digit_base[tid] = glob_excl + excl - tile_excl;
  }
  __syncthreads();

  // ---- permute through shared memory into tile-sorted order -----------------------------------------------
#pragma unroll
  for (int j = 0; j < ITEMS; ++j) {
    if (FULL || (warp_off + j * 32) < valid_in_tile) {
      const uint32_t d = (uint32_t)(key[j] >> shift) & 0xFFu;
      const uint32_t pos = s.tile_excl[d] + my_hist[j / RUN][d] + ((j & 1) ? (rank2[j / 2] >> 16) : (rank2[j / 2] & 0xFFFFu));
      s.keys[pos] = key[j];
      s.vals[pos] = val[j];
    }
  }
  __syncthreads();

  // ---- write out: consecutive tile-sorted positions of one digit are consecutive in global memory -------
#pragma unroll
  for (int j = 0; j < ITEMS; ++j) {
    const int pos = tid + j * kSortThreads;
    if (FULL || pos < valid_in_tile) {
      const KeyT k = s.keys[pos];
      const uint32_t d = (uint32_t)(k >> shift) & 0xFFu;
      const uint32_t dst = s.digit_base[d] + (uint32_t)pos;
      keys_out[dst] = k;
      vals_out[dst] = s.vals[pos];
    }
  }
}

#ifndef BVH_SORT_MINBLOCKS
#define BVH_SORT_MINBLOCKS 4
#endif
template <typename KeyT, bool IOTA, bool TOP>
__global__ void __launch_bounds__(kSortThreads, BVH_SORT_MINBLOCKS)
onesweep_pass_kernel(const KeyT* __restrict__ keys_in, KeyT* __restrict__ keys_out, const uint32_t* __restrict__ vals_in,
                     uint32_t* __restrict__ vals_out, const uint32_t* __restrict__ hist, uint32_t* status,
                     uint32_t* tile_counter, int n, int shift) {
  constexpr int TILE = SortCfg<KeyT>::TILE;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  SortSmem<KeyT>& s = *reinterpret_cast<SortSmem<KeyT>*>(smem_raw);

  const int tid = threadIdx.x;
  for (int i = tid; i < kSortWarps * kSortChains * 256; i += kSortThreads) (&s.warp_hist[0][0][0])[i] = 0;
  if (tid < 256) s.tile_hist[tid] = 0;
  pdl_wait();
  pdl_trigger();
  if (tid == 0) s.tile = atomicAdd(tile_counter, 1u);
  __syncthreads();
  const uint32_t tile = s.tile;
  const uint32_t tile_base = tile * (uint32_t)TILE;
  const int valid_in_tile = min(TILE, n - (int)tile_base);
  if (valid_in_tile == TILE)
    sort_tile<KeyT, IOTA, true, TOP>(s, keys_in, keys_out, vals_in, vals_out, hist, status, tile, tile_base, TILE, shift);
  else
    sort_tile<KeyT, IOTA, false, TOP>(s, keys_in, keys_out, vals_in, vals_out, hist, status, tile, tile_base, valid_in_tile,
                                      shift);
}

template <typename KeyT>
static cudaError_t sort_all(const SortBuffers& B, int n, int passes, cudaStream_t stream, void* const* pass_events, int shift0,
                            int slot0) {
  const int tiles = (n + SortCfg<KeyT>::TILE - 1) / SortCfg<KeyT>::TILE;
  KeyT* keys[2] = {static_cast<KeyT*>(B.keys[0]), static_cast<KeyT*>(B.keys[1])};
  const size_t smem = sizeof(SortSmem<KeyT>);
  // the opt-in to more than 48 KB of dynamic shared memory holds for the device that was current: once per device
  static PerDeviceOnce once;
  const cudaError_t attr = once_per_device(once, nullptr, [&](int* done) {
    cudaError_t e = cudaFuncSetAttribute(onesweep_pass_kernel<KeyT, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(onesweep_pass_kernel<KeyT, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(onesweep_pass_kernel<KeyT, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    *done = 1;
    return e;
  });
  if (attr != cudaSuccess) return attr;
  for (int p = 0; p < passes; ++p) {
    const int in = p & 1, out = in ^ 1, slot = slot0 + p;     // slot: which histogram / status block / ticket this pass uses
    uint32_t* st = B.status + (size_t)slot * tiles * 256;
    uint32_t* vout = (p == passes - 1 && B.final_vals) ? B.final_vals : B.vals[out];
    const int shift = shift0 + 8 * p;
    const uint32_t* vin = B.vals[in];
    const uint32_t* none = nullptr;
    cudaError_t e;
    if (p == 0)
      e = launch_pdl(onesweep_pass_kernel<KeyT, true, false>, dim3(tiles), dim3(kSortThreads), smem, stream,
                 keys[in], keys[out], none, vout, B.hist + slot * 256, st, B.tile_counters + slot, n, shift);
    else if (p == passes - 1 && sizeof(KeyT) == 4)   // (64-bit codes: the top digit of neighbouring keys is rarely shared; ballots)
      e = launch_pdl(onesweep_pass_kernel<KeyT, false, true>, dim3(tiles), dim3(kSortThreads), smem, stream,
                 keys[in], keys[out], vin, vout, B.hist + slot * 256, st, B.tile_counters + slot, n, shift);
    else
      e = launch_pdl(onesweep_pass_kernel<KeyT, false, false>, dim3(tiles), dim3(kSortThreads), smem, stream,
                 keys[in], keys[out], vin, vout, B.hist + slot * 256, st, B.tile_counters + slot, n, shift);
    if (e != cudaSuccess) return e;
    if (pass_events && pass_events[p]) cudaEventRecord(static_cast<cudaEvent_t>(pass_events[p]), stream);
  }
  return cudaSuccess;
}

// The conditional second sort of a 63-bit build (tie_fixup.cu) as ONE cooperative launch: nothing unless *run_if != 0
// (the usual case costs one launch instead of nine); else the digit histograms of the codes as they stand, then the
// eight passes, a grid-wide barrier after each.  It starts from the codes and indices the four upper-bit passes left
// in keys[0] / vals[0]: equal codes are in ascending original index there (those passes are stable), and eight more
// stable passes over all 63 bits keep them so -- the order of the plain eight-pass sort.
template <typename KeyT>
__global__ void __launch_bounds__(kSortThreads, BVH_SORT_MINBLOCKS)
second_sort_kernel(KeyT* keys0, KeyT* keys1, uint32_t* vals0, uint32_t* vals1, uint32_t* hist, uint32_t* status,
                   uint32_t* tile_counters, int n, int passes, const uint32_t* __restrict__ run_if) {
  constexpr int TILE = SortCfg<KeyT>::TILE;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  SortSmem<KeyT>& s = *reinterpret_cast<SortSmem<KeyT>*>(smem_raw);
  pdl_wait();
  if (*run_if == 0) return;
  namespace cg = cooperative_groups;
  cg::grid_group grid = cg::this_grid();
  const int tid = threadIdx.x;
  const uint32_t tiles = (uint32_t)((n + TILE - 1) / TILE);
  // ---- this sort's histograms and tile status words lie outside the part of the scratch a build zeroes (they would be
  // two thirds of that memset for a sort that almost never runs): cleared here, by the sort that needs them ----
  {
    const size_t stride = (size_t)gridDim.x * kSortThreads, first = (size_t)blockIdx.x * kSortThreads + tid;
    for (size_t i = first; i < (size_t)passes * 256; i += stride) hist[i] = 0;
    for (size_t i = first; i < (size_t)passes * tiles * 256; i += stride) status[i] = 0;
    grid.sync();
  }
  // ---- digit histograms of all passes (shared-memory atomics, one global atomic per bin and block) ----
  uint32_t* s_hist = reinterpret_cast<uint32_t*>(smem_raw);          // passes * 256 words <= 8 KB: aliases the sort's shared memory
  for (int i = tid; i < passes * 256; i += kSortThreads) s_hist[i] = 0;
  __syncthreads();
  for (int64_t i = (int64_t)blockIdx.x * kSortThreads + tid; i < n; i += (int64_t)gridDim.x * kSortThreads) {
    const KeyT k = keys0[i];
    for (int p = 0; p < passes; ++p) atomicAdd(&s_hist[p * 256 + (int)((k >> (8 * p)) & 0xFF)], 1u);
  }
  __syncthreads();
  for (int i = tid; i < passes * 256; i += kSortThreads)
    if (s_hist[i]) atomicAdd(&hist[i], s_hist[i]);
  grid.sync();
  // ---- the passes ----
  for (int p = 0; p < passes; ++p) {
    const KeyT* kin = (p & 1) ? keys1 : keys0;
    KeyT* kout = (p & 1) ? keys0 : keys1;
    const uint32_t* vin = (p & 1) ? vals1 : vals0;
    uint32_t* vout = (p & 1) ? vals0 : vals1;
    uint32_t* st = status + (size_t)p * tiles * 256;
    while (true) {
      __syncthreads();
      for (int i = tid; i < kSortWarps * kSortChains * 256; i += kSortThreads) (&s.warp_hist[0][0][0])[i] = 0;
      if (tid < 256) s.tile_hist[tid] = 0;
      if (tid == 0) s.tile = atomicAdd(tile_counters + p, 1u);
      __syncthreads();
      const uint32_t tile = s.tile;
      if (tile >= tiles) break;
      const uint32_t tile_base = tile * (uint32_t)TILE;
      const int valid_in_tile = min(TILE, n - (int)tile_base);
      if (valid_in_tile == TILE)
        sort_tile<KeyT, false, true, false>(s, kin, kout, vin, vout, hist + p * 256, st, tile, tile_base, TILE, 8 * p);
      else
        sort_tile<KeyT, false, false, false>(s, kin, kout, vin, vout, hist + p * 256, st, tile, tile_base, valid_in_tile, 8 * p);
    }
    grid.sync();
  }
}

// hist [passes][256] / status [passes][tiles][256]: this sort's own, in any state (the kernel clears them); tile counters:
// those of slot `slot0` on, zeroed by the build; passes must be even (the result returns to keys[0]).
cudaError_t launch_second_sort(const SortBuffers& B, int passes, int n, int slot0, uint32_t* hist, uint32_t* status,
                               const uint32_t* run_if, cudaStream_t stream) {
  using KeyT = uint64_t;
  const size_t smem = sizeof(SortSmem<KeyT>);
  // shared-memory opt-in and occupancy of the kernel on the CURRENT device: once per device
  static PerDeviceOnce once;
  int blocks_per_sm = 0;
  const cudaError_t attr = once_per_device(once, &blocks_per_sm, [&](int* per_sm) {
    cudaError_t e = cudaFuncSetAttribute(second_sort_kernel<KeyT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(per_sm, second_sort_kernel<KeyT>, kSortThreads, smem);
    if (e == cudaSuccess && *per_sm < 1) e = cudaErrorInvalidValue;
    return e;
  });
  if (attr != cudaSuccess) return attr;
  if (passes & 1) return cudaErrorInvalidValue;
  const int tiles = (n + SortCfg<KeyT>::TILE - 1) / SortCfg<KeyT>::TILE;
  int blocks = blocks_per_sm * sm_count();                    // all co-resident: the grid-wide barrier needs that
  if (blocks > tiles) blocks = tiles;
  cudaLaunchConfig_t cfg{};
  cfg.blockDim = dim3(kSortThreads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeCooperative;
  at[0].val.cooperative = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  // The occupancy query counts the whole device; the context may own less of it (an MPS active-thread percentage, a green
  // context, SM partitioning), and then the runtime refuses the grid as too large for a cooperative launch.  The kernel
  // draws its tiles from a ticket counter and works with ANY number of co-resident blocks, so the refused launch is
  // repeated with half the grid until it is accepted: a build must not fail over a sort that almost never runs.
  cudaError_t e = cudaErrorCooperativeLaunchTooLarge;
  for (; blocks >= 1 && e == cudaErrorCooperativeLaunchTooLarge; blocks = blocks > 1 ? blocks / 2 : 0) {
    cfg.gridDim = dim3(blocks);
    e = cudaLaunchKernelEx(&cfg, second_sort_kernel<KeyT>, static_cast<KeyT*>(B.keys[0]), static_cast<KeyT*>(B.keys[1]), B.vals[0],
                           B.vals[1], hist, status, B.tile_counters + slot0, n, passes, run_if);
    if (e == cudaErrorCooperativeLaunchTooLarge) (void)cudaGetLastError();   // not sticky: clear it before the next attempt
  }
  return e;
}

SortBuffers sort_buffers(void* scratch, const ScratchLayout& L) {
  char* base = static_cast<char*>(scratch);
  SortBuffers B{};
  B.keys[0] = base + L.keys[0];
  B.keys[1] = base + L.keys[1];
  B.vals[0] = reinterpret_cast<uint32_t*>(base + L.vals[0]);
  B.vals[1] = reinterpret_cast<uint32_t*>(base + L.vals[1]);
  B.hist = reinterpret_cast<uint32_t*>(base + L.hist);
  B.status = reinterpret_cast<uint32_t*>(base + L.status);
  B.tile_counters = reinterpret_cast<Header*>(base + L.header)->tile_counter;
  B.final_vals = nullptr;
  return B;
}

cudaError_t launch_sort(const SortBuffers& B, int key_bytes, int passes, int n, cudaStream_t stream, void* const* pass_events,
                        int shift0, int slot0) {
  if (key_bytes == 4) return sort_all<uint32_t>(B, n, passes, stream, pass_events, shift0, slot0);
  return sort_all<uint64_t>(B, n, passes, stream, pass_events, shift0, slot0);
}

}  // namespace bvh
