// tie_fixup.cu -- second half of the sort of 63-bit Morton codes (K3).
//
// An LSD radix sort of 63-bit codes is eight 8-bit passes, and on B200 the passes are what a 63-bit build spends most
// of its time in (C4: 345 of 626 us, C5: 1.22 of 2.02 ms).  Almost all of that work orders primitives that the upper
// half of the code has already separated: 2^32 cells for 10^6 .. 10^7 primitives.  So the pairs are first sorted by the
// UPPER 32 bits only (bits 31..62: four stable passes), which leaves every group of primitives that share those bits
// contiguous and in ascending original index, and this kernel then sorts each such group ("run") by its lower 31 bits,
// stably -- the order an LSD sort of all 63 bits gives (readings G5/G6).  Runs are short unless the input is
// degenerate, so the fix-up is a streaming read of the codes plus a little work in shared memory.
//
// Two kernels.  tie_short_kernel streams over the codes, a tile of kFixTile positions per block in shared memory: every
// pair of a run of 2 .. kFixSerial pairs finds its rank in the run by (lower bits, position) and moves there; a longer
// run puts the tile it starts in on a work list.  tie_long_kernel takes the listed tiles: one block
// loads the runs that START in the tile (the last of them may reach into the next tile) into shared memory and
// orders the long ones by a bitonic network over (lower bits, original index), the whole block per run.  A run that
// reaches more than a tile past the tile it starts in does not fit: the block then raises `fallback`, and eight more
// stable passes over all 63 bits (second_sort_kernel in radix_sort.cu: ONE cooperative launch, enqueued in any case
// because nothing may read the flag back, that returns at once while the flag is clear) redo the order -- correct for
// every input, slower only for those with thousands of primitives inside one of 2^32 cells.
#include "common.cuh"

namespace bvh {

constexpr int kFixThreads = 256;
constexpr int kFixTile = 2048;                 // positions per block
constexpr int kFixCap = 2 * kFixTile;          // pairs a block may have to hold: its tile and a run reaching into the next
constexpr int kFixSerial = 32;                 // longest run ordered by one thread
constexpr int kFixHighShift = 31;              // runs = equal bits 31..62

struct FixSmem {
  unsigned long long key[kFixCap];
  unsigned long long comp[kFixCap];            // bitonic workspace: (lower bits << 32) | original index
  uint32_t val[kFixCap];
  int long_start[kFixCap / kFixSerial + 1], long_len[kFixCap / kFixSerial + 1];
  int n_long;
  int found;
  int any;
};

__device__ __forceinline__ uint32_t high_word(unsigned long long k) { return (uint32_t)(k >> kFixHighShift); }

// Smallest run start in [from, from + kFixTile] (a position i with i == 0, i == n, or other upper bits than i - 1), or -1.
// Block-uniform: every thread returns the same value and passes the same barriers.
__device__ __forceinline__ int first_run_start(const unsigned long long* __restrict__ keys, int n, int from, int* s_found) {
  if (from >= n) return n;
  if (from == 0) return 0;
  for (int base = from; base <= from + kFixTile; base += kFixThreads) {
    const int i = base + (int)threadIdx.x;
    const bool start = i <= from + kFixTile && (i >= n || high_word(keys[i]) != high_word(keys[i - 1]));
    if (__syncthreads_or(start)) {
      if (threadIdx.x == 0) *s_found = 0x7fffffff;
      __syncthreads();
      if (start) atomicMin(s_found, i);
      __syncthreads();
      const int r = *s_found;
      __syncthreads();
      return r;
    }
  }
  return -1;
}

// Short runs, and the work list of the long ones.  The block's tile of codes (with a halo: the position before it and
// the kFixSerial + 1 after it) is staged in shared memory; every pair of a run that STARTS in the tile finds its own
// place: its rank among the pairs of its run, by (lower bits, position) -- a stable order -- counted in shared memory.
// The pairs that are part of a run are first listed, with their indices, in shared memory; then every listed pair that
// has to move stores its code and index at its new position.  Pairs outside runs (almost all of them) cost three
// shared-memory reads.  A run of more than
// kFixSerial pairs is left alone and its tile goes on the work list.
__global__ void __launch_bounds__(kFixThreads) tie_short_kernel(unsigned long long* __restrict__ keys, uint32_t* __restrict__ vals,
                                                                int n, uint32_t* __restrict__ tile_flag,
                                                                uint32_t* __restrict__ tile_list, uint32_t* __restrict__ list_count) {
  constexpr int HALO = kFixSerial + 1;
  constexpr int PER = (kFixTile + HALO + kFixThreads - 1) / kFixThreads;
  __shared__ unsigned long long s_key[1 + kFixTile + HALO];    // s_key[1 + e] = keys[tile0 + e]
  pdl_wait();
  pdl_trigger();
  const int tile0 = blockIdx.x * kFixTile;
  const int avail = min(n - tile0, kFixTile + HALO);           // positions of [tile0, ...) that exist and are staged
  for (int e = (int)threadIdx.x - 1; e < avail; e += kFixThreads)
    if (tile0 + e >= 0) s_key[1 + e] = keys[tile0 + e];
  __syncthreads();
  // the pairs that are part of a run of two or more (few): their positions go on a list in shared memory ...
  __shared__ int s_tied[kFixTile + HALO];
  __shared__ uint32_t s_val[kFixTile + HALO];                  // ... with their indices, read before anything is stored
  __shared__ int s_count;
  if (threadIdx.x == 0) s_count = 0;
  __syncthreads();
  for (int u = 0; u < PER; ++u) {
    const int e = u * kFixThreads + (int)threadIdx.x;
    if (e >= avail) break;
    const uint32_t h = high_word(s_key[1 + e]);
    const bool tied_prev = tile0 + e > 0 && high_word(s_key[e]) == h;
    const bool tied_next = e + 1 < avail && high_word(s_key[2 + e]) == h;
    if (tied_prev || tied_next) {
      const int w = atomicAdd(&s_count, 1);
      s_tied[w] = e;
      s_val[w] = vals[tile0 + e];
    }
  }
  __syncthreads();
  // ... and are then handled kFixThreads at a time, all lanes busy
  const int count = s_count;
  for (int w = threadIdx.x; w < count; w += kFixThreads) {
    const int e = s_tied[w];
    const unsigned long long k = s_key[1 + e];
    const uint32_t h = high_word(k);
    int s = e;                                                 // first position of the run (-1: it starts before the tile)
    while (s >= 0 && e - s <= kFixSerial && (tile0 + s > 0 && high_word(s_key[s]) == h)) --s;
    if (s < 0 || s >= kFixTile || e - s > kFixSerial) continue;   // another tile's run, or a long one (its start reports it)
    int f = e + 1;                                             // one past the last position of the run
    while (f < avail && f - s <= kFixSerial && high_word(s_key[1 + f]) == h) ++f;
    if (f - s > kFixSerial) {                                  // long: its tile goes on the list, once
      if (e == s && atomicExch(&tile_flag[blockIdx.x], 1u) == 0u) tile_list[atomicAdd(list_count, 1u)] = blockIdx.x;
      continue;
    }
    int rank = 0;
    for (int g = s; g < f; ++g) {
      const unsigned long long kg = s_key[1 + g];
      rank += (kg < k || (kg == k && g < e)) ? 1 : 0;
    }
    if (s + rank != e) {                                       // codes come from shared memory, indices were read above:
      keys[tile0 + s + rank] = k;                              // nothing that is stored here is read again by this kernel
      vals[tile0 + s + rank] = s_val[w];
    }
  }
}

// Long runs: the listed tiles, one block per tile at a time.
__global__ void __launch_bounds__(kFixThreads) tie_long_kernel(unsigned long long* __restrict__ keys, uint32_t* __restrict__ vals,
                                                               int n, const uint32_t* __restrict__ tile_list,
                                                               const uint32_t* __restrict__ list_count,
                                                               uint32_t* __restrict__ fallback) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  FixSmem& S = *reinterpret_cast<FixSmem*>(smem_raw);
  pdl_wait();
  pdl_trigger();
  const int tid = threadIdx.x;
  const uint32_t listed = *list_count;
  for (uint32_t w = blockIdx.x; w < listed; w += gridDim.x) {
  __syncthreads();                                                 // the previous tile's shared memory is no longer read
  const int tile0 = (int)tile_list[w] * kFixTile;
  const int begin = first_run_start(keys, n, tile0, &S.found);
  if (begin < 0 || begin >= min(n, tile0 + kFixTile)) continue;   // no run starts in this tile
  int end = first_run_start(keys, n, tile0 + kFixTile, &S.found);
  if (end < 0) {                                                   // the last run of this tile is longer than a tile
    if (tid == 0) atomicExch(fallback, 1u);
    continue;
  }
  const int m = end - begin;                                       // <= kFixCap
  if (tid == 0) {
    S.any = 0;
    S.n_long = 0;
  }
  __syncthreads();
  bool tie = false;
  for (int e = tid; e < m; e += kFixThreads) {
    const unsigned long long k = keys[begin + e];
    S.key[e] = k;
    if (e > 0) tie = tie || high_word(k) == high_word(keys[begin + e - 1]);
  }
  if (__syncthreads_or(tie) == 0) continue;                        // every run is a single pair: nothing to do
  for (int e = tid; e < m; e += kFixThreads) S.val[e] = vals[begin + e];
  __syncthreads();
  // ---- one thread per run: length, already in order?, short runs by stable insertion ----
  for (int e = tid; e < m; e += kFixThreads) {
    const uint32_t h = high_word(S.key[e]);
    if ((e > 0 && high_word(S.key[e - 1]) == h) || e + 1 >= m || high_word(S.key[e + 1]) != h) continue;   // not the start of a run of >= 2
    int len = 2;
    while (e + len < m && high_word(S.key[e + len]) == h) ++len;
    bool sorted = true;
    for (int u = 1; u < len && sorted; ++u) sorted = S.key[e + u - 1] <= S.key[e + u];     // equal codes: indices already ascend
    if (sorted) continue;
    if (len <= kFixSerial) {
      for (int u = 1; u < len; ++u) {
        const unsigned long long k = S.key[e + u];
        const uint32_t v = S.val[e + u];
        int w = u;
        while (w > 0 && S.key[e + w - 1] > k) {                   // strict: equal codes keep their order (stable)
          S.key[e + w] = S.key[e + w - 1];
          S.val[e + w] = S.val[e + w - 1];
          --w;
        }
        S.key[e + w] = k;
        S.val[e + w] = v;
      }
    } else {
      const int slot = atomicAdd(&S.n_long, 1);
      S.long_start[slot] = e;
      S.long_len[slot] = len;
    }
  }
  __syncthreads();
  // ---- long runs: the whole block, bitonic network over (lower 31 bits, original index): distinct, so any order of
  // the network's equal-key choices cannot arise ----
  const int n_long = S.n_long;
  for (int r = 0; r < n_long; ++r) {
    const int e0 = S.long_start[r], len = S.long_len[r];
    int p2 = 64;
    while (p2 < len) p2 <<= 1;
    const unsigned long long hi = (unsigned long long)high_word(S.key[e0]) << kFixHighShift;
    for (int u = tid; u < p2; u += kFixThreads)
      S.comp[u] = u < len ? (((S.key[e0 + u] & 0x7fffffffull) << 32) | S.val[e0 + u]) : ~0ull;
    __syncthreads();
    for (int k = 2; k <= p2; k <<= 1) {
      for (int j = k >> 1; j > 0; j >>= 1) {
        for (int t = tid; t < (p2 >> 1); t += kFixThreads) {
          const int i = ((t & ~(j - 1)) << 1) | (t & (j - 1));
          const int l = i | j;
          const bool up = (i & k) == 0;
          const unsigned long long a = S.comp[i], b = S.comp[l];
          if ((a > b) == up) {
            S.comp[i] = b;
            S.comp[l] = a;
          }
        }
        __syncthreads();
      }
    }
    for (int u = tid; u < len; u += kFixThreads) {
      const unsigned long long c = S.comp[u];
      S.key[e0 + u] = hi | (c >> 32);
      S.val[e0 + u] = (uint32_t)c;
    }
    __syncthreads();
  }
  for (int e = tid; e < m; e += kFixThreads) {
    keys[begin + e] = S.key[e];
    vals[begin + e] = S.val[e];
  }
  }
}

int tie_fixup_tiles(int64_t n) { return (int)((n + kFixTile - 1) / kFixTile); }

cudaError_t launch_tie_fixup(void* keys, uint32_t* vals, int n, uint32_t* tile_flag, uint32_t* tile_list, uint32_t* list_count,
                             uint32_t* fallback, cudaStream_t stream) {
  const size_t smem = sizeof(FixSmem);
  // the opt-in to more than 48 KB of dynamic shared memory holds for the device that was current: once per device
  static PerDeviceOnce once;
  const cudaError_t attr = once_per_device(once, nullptr, [&](int* done) {
    *done = 1;
    return cudaFuncSetAttribute(tie_long_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  });
  if (attr != cudaSuccess) return attr;
  unsigned long long* k = static_cast<unsigned long long*>(keys);
  const int tiles = tie_fixup_tiles(n);
  cudaError_t e = launch_pdl(tie_short_kernel, dim3(tiles), dim3(kFixThreads), 0, stream, k, vals, n, tile_flag, tile_list, list_count);
  if (e != cudaSuccess) return e;
  const int blocks = tiles < 2 * sm_count() ? tiles : 2 * sm_count();
  return launch_pdl(tie_long_kernel, dim3(blocks), dim3(kFixThreads), smem, stream, k, vals, n,
                    static_cast<const uint32_t*>(tile_list), static_cast<const uint32_t*>(list_count), fallback);
}

}  // namespace bvh
