// Philox4x32-10 keyed by (event, seed), counter (id_lo, id_hi, step, block)  -- SURVEY.md §8(c) R1-R3
// (PAPER.md:55 asks for a portable counter-based RNG usable from scalar-argument physics functions).
#pragma once
#include "types.cuh"

namespace adept {

struct Philox4 { uint32_t w0, w1, w2, w3; };

// Inlined: the ten rounds are integer work that the scheduler interleaves with the fp64 chains around
// them (measured 1.3 % of a config-2 pass over a call).
__device__ __forceinline__ Philox4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                 uint32_t k0, uint32_t k1) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t h0 = __umulhi(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
    const uint32_t h1 = __umulhi(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
    const uint32_t n0 = h1 ^ c1 ^ k0, n2 = h0 ^ c3 ^ k1;
    c0 = n0; c1 = l1; c2 = n2; c3 = l0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  return Philox4{c0, c1, c2, c3};
}

// R2: 53-bit mantissa from two words, U = (m + 0.5) 2^-53
__device__ __forceinline__ double to_uniform(uint32_t hi, uint32_t lo) {
  const unsigned long long m = (static_cast<unsigned long long>(hi >> 5) << 26) + (lo >> 6);
  return (__ull2double_rn(m) + 0.5) * 0x1.0p-53;
}

// The random stream of one (event, track, step): uniforms are addressed by slot number n
// (block n>>1, words (w0,w1) for even n, (w2,w3) for odd n); a block is generated once and cached.
struct Stream {
  uint32_t k0, k1, c0, c1, c2;
  uint32_t cached_block;
  Philox4 w;
  uint32_t next;  // sequential cursor for the samplers (U8..)

  __device__ __forceinline__ void init(uint32_t event, uint32_t seed, uint64_t id, uint32_t step) {
    k0 = event; k1 = seed;
    c0 = static_cast<uint32_t>(id); c1 = static_cast<uint32_t>(id >> 32); c2 = step;
    cached_block = 0xFFFFFFF0u;  // never a sampler block
    next = 8;
  }
  __device__ __forceinline__ double uniform(uint32_t n) {
    const uint32_t b = n >> 1;
    if (b != cached_block) { w = philox4x32_10(c0, c1, c2, b, k0, k1); cached_block = b; }
    return (n & 1u) ? to_uniform(w.w2, w.w3) : to_uniform(w.w0, w.w1);
  }
  __device__ __forceinline__ double draw() { return uniform(next++); }
  // R3: child track id = (w0 | w1<<32) of block 0xFFFFFFFF - child_index
  __device__ __forceinline__ uint64_t child_id(uint32_t child) const {
    const Philox4 v = philox4x32_10(c0, c1, c2, 0xFFFFFFFFu - child, k0, k1);
    return static_cast<uint64_t>(v.w0) | (static_cast<uint64_t>(v.w1) << 32);
  }
};

}  // namespace adept
