/* ORACLE -- TEST INFRASTRUCTURE ONLY (see oracle.h).
 *
 * R1-R3 of SURVEY.md §8(c): Philox4x32-10 (the published counter-based generator; PAPER.md:55
 * only says "a portable RNG", BASELINE.json:north_star fixes Philox keyed by (event, track, step)).
 * Pinned by tests/test_oracle_rng.py: known-answer vectors, an exact-rational recomputation of the
 * uniform mapping, and equidistribution moments.
 */
#include "internal.h"

extern "C" void orc_philox(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    const uint64_t p0 = static_cast<uint64_t>(M0) * c0;
    const uint64_t p1 = static_cast<uint64_t>(M1) * c2;
    const uint32_t n0 = static_cast<uint32_t>(p1 >> 32) ^ c1 ^ k0;
    const uint32_t n1 = static_cast<uint32_t>(p1);
    const uint32_t n2 = static_cast<uint32_t>(p0 >> 32) ^ c3 ^ k1;
    const uint32_t n3 = static_cast<uint32_t>(p0);
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += W0; k1 += W1;  /* key bumped after the round: round 1 uses the raw key */
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* R2: uniform n of the step: block n>>1, words (w0,w1) if n even else (w2,w3);
   U = (((hi>>5)<<26) + (lo>>6) + 0.5) * 2^-53 */
extern "C" double orc_uniform(uint32_t event, uint32_t seed, uint64_t id, uint32_t step, uint32_t n) {
  const uint32_t ctr[4] = {static_cast<uint32_t>(id), static_cast<uint32_t>(id >> 32), step, n >> 1};
  const uint32_t key[2] = {event, seed};
  uint32_t w[4];
  orc_philox(ctr, key, w);
  const uint32_t hi = (n & 1u) ? w[2] : w[0];
  const uint32_t lo = (n & 1u) ? w[3] : w[1];
  const uint64_t mant = (static_cast<uint64_t>(hi >> 5) << 26) + (lo >> 6);
  return (static_cast<double>(mant) + 0.5) * 0x1.0p-53;
}

/* R3: child track id = (w0 | w1<<32) of the parent's block 0xFFFFFFFF - child_index */
extern "C" uint64_t orc_child_id(uint32_t event, uint32_t seed, uint64_t id, uint32_t step, uint32_t child) {
  const uint32_t ctr[4] = {static_cast<uint32_t>(id), static_cast<uint32_t>(id >> 32), step, 0xFFFFFFFFu - child};
  const uint32_t key[2] = {event, seed};
  uint32_t w[4];
  orc_philox(ctr, key, w);
  return static_cast<uint64_t>(w[0]) | (static_cast<uint64_t>(w[1]) << 32);
}
