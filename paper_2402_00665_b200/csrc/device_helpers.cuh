// device_helpers.cuh -- small __device__ helpers shared by the kernels of the CUDA path (hierarchy.cu, bounds_morton.cu,
// radix_sort.cu).  Nothing here is shared with, or included by, oracle/.
#pragma once

#include "common.cuh"

namespace bvh {

// delta*(i): XOR of adjacent sorted codes; equal codes fall back to the XOR of the
// sorted positions (augmented key, readings G1/G5); +infinity outside [0, n-2].  The
// value is packed so that one unsigned compare orders it (G14): position band < code band < infinity.
template <typename KeyT>
struct Delta;
template <>
struct Delta<uint32_t> {
  using T = uint32_t;
  static constexpr T kInf = 0xFFFFFFFFu;
  __device__ static __forceinline__ T make(uint32_t a, uint32_t b, int i) {
    const uint32_t x = a ^ b;                              // < 2^30
    return x ? (x + 0x40000000u) : (uint32_t)(i ^ (i + 1));  // codes and positions < 2^30 (capi.cu rejects n >= 2^30)
  }
};
// 64-bit codes: the value kept is the INDEX of the highest differing bit, not the XOR itself.  Every comparison
// Algorithm 4 makes is between delta*(l-1) and delta*(r) of a node's range [l, r], or between delta*(r) and
// delta*(r+1) (L8, L26); in both cases the two XORs cannot share their highest set bit (sorted keys: a key cannot
// have that bit both set, as the upper key of one pair, and clear, as the lower key of the other, under the
// same prefix), so the order of the XORs is the order of their highest bits -- Karras' common-prefix length
// (PAPER.md:97).  One 32-bit word instead of two: half the shuffles and shared memory of the 63-bit build.
template <>
struct Delta<uint64_t> {
  using T = uint32_t;
  static constexpr T kInf = 0xFFFFFFFFu;
  __device__ static __forceinline__ T make(uint64_t a, uint64_t b, int i) {
    const uint64_t x = a ^ b;                              // <= 2^63 - 1
    return x ? (0x40000000u + (uint32_t)(63 - __clzll((long long)x))) : (uint32_t)(i ^ (i + 1));
  }
};

template <typename KeyT>
__device__ __forceinline__ typename Delta<KeyT>::T delta_star(const KeyT* __restrict__ codes, int i, int n) {
  if (i < 0 || i >= n - 1) return Delta<KeyT>::kInf;
  return Delta<KeyT>::make(codes[i], codes[i + 1], i);
}

__device__ __forceinline__ void store_node(Node* nodes, int idx, const float lo[3], const float hi[3], int left, int rope) {
  // one 256-bit store = one full 32-byte sector (STG.E.ENL2.256, sm_100)
  asm volatile("st.global.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(nodes + idx), "f"(lo[0]), "f"(lo[1]), "f"(lo[2]),
               "f"(__int_as_float(left)), "f"(hi[0]), "f"(hi[1]), "f"(hi[2]), "f"(__int_as_float(rope))
               : "memory");
}

// Leaf record i (layout in common.cuh): a point leaf stores the point once.
template <bool IS_BOX>
__device__ __forceinline__ void store_leaf(char* leaves, int i, const float lo[3], const float hi[3], uint32_t payload) {
  if (IS_BOX)
    store_node(reinterpret_cast<Node*>(leaves), i, lo, hi, (int)payload, 0);
  else
    reinterpret_cast<float4*>(leaves)[i] = make_float4(lo[0], lo[1], lo[2], __uint_as_float(payload));
}

// ---- D2: Morton quantisation and bit spreading (bounds_morton.cu) ---------------------------------------
__device__ __forceinline__ uint32_t spread10(uint32_t x) {
  x = (x | (x << 16)) & 0x030000FFu;
  x = (x | (x << 8)) & 0x0300F00Fu;
  x = (x | (x << 4)) & 0x030C30C3u;
  x = (x | (x << 2)) & 0x09249249u;
  return x;
}
__device__ __forceinline__ uint64_t spread21(uint32_t v) {
  uint64_t x = v & 0x1fffffu;
  x = (x | (x << 32)) & 0x001f00000000ffffull;
  x = (x | (x << 16)) & 0x001f0000ff0000ffull;
  x = (x | (x << 8)) & 0x100f00f00f00f00full;
  x = (x | (x << 4)) & 0x10c30c30c30c30c3ull;
  x = (x | (x << 2)) & 0x1249249249249249ull;
  return x;
}

__device__ __forceinline__ uint32_t quantise(float lo, float hi, float slo, float shi, float scale, uint32_t cell_max) {
  const float c = __fmul_rn(__fadd_rn(lo, hi), 0.5f);
  const float e = __fsub_rn(shi, slo);
  float t = 0.0f;
  if (e > 0.0f) t = __fdiv_rn(__fsub_rn(c, slo), e);
  const uint32_t q = __float2uint_rz(__fmul_rn(t, scale));
  return min(q, cell_max);
}

template <typename KeyT>
__device__ __forceinline__ KeyT morton_code(const uint32_t cell[3]) {
  if (sizeof(KeyT) == 4) return (KeyT)((spread10(cell[0]) << 2) | (spread10(cell[1]) << 1) | spread10(cell[2]));
  return (KeyT)((spread21(cell[0]) << 2) | (spread21(cell[1]) << 1) | spread21(cell[2]));
}

// ---- radix ranking (radix_sort.cu) --------------------------------------------------------------------------
// Lanes of the warp whose digit equals this lane's: AND over the 8 digit bits of (ballot of the bit) or its
// complement.  `peers` enters as the mask of participating lanes.  MATCH_ANY: one MATCH.ANY instruction instead;
// its cost grows with the number of distinct digits in the warp, so it only pays for the most significant
// digit (few distinct values among 32 keys that are neighbours in the input; measured on C3: 59 vs 68 us for
// that pass, but 105 vs 75 us for the least significant one).
template <bool MATCH_ANY>
__device__ __forceinline__ uint32_t match_digit(uint32_t d, uint32_t peers) {
  if (MATCH_ANY) {
    peers &= __match_any_sync(0xffffffffu, d);
  } else {
#pragma unroll
    for (int b = 0; b < 8; ++b) {
      // four SASS instructions per bit: bit test -> predicate, VOTE, and one predicated LOP3 per polarity
      asm volatile(
          "{\n\t"
          ".reg .pred p;\n\t"
          ".reg .b32 t, bal;\n\t"
          "and.b32 t, %1, %2;\n\t"
          "setp.ne.u32 p, t, 0;\n\t"
          "vote.sync.ballot.b32 bal, p, 0xffffffff;\n\t"
          "@p and.b32 %0, %0, bal;\n\t"
          "@!p not.b32 bal, bal;\n\t"
          "@!p and.b32 %0, %0, bal;\n\t"
          "}"
          : "+r"(peers)
          : "r"(d), "r"(1u << b));
    }
  }
  return peers;
}

}  // namespace bvh
