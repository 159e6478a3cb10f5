// ORACLE (test infrastructure).  Philox4x32-10 counter-based generator and the
// per-superphoton stream layout (O5, reading G11; north_star "counter-based
// RNG keyed per superphoton (Philox)").  The paper itself uses cuRAND XORWOW
// (PAPER.md:186); only uniformity on [0,1) is required by Eqs. 7-9 and PAPER.md:176.
//
// Pin: three known-answer vectors (tests/golden/philox_kat.txt), chi^2 uniformity.
#include "oracle.hpp"

namespace orc {

void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  const uint64_t M0 = 0xD2511F53ull, M1 = 0xCD9E8D57ull;
  const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; round++) {
    uint64_t p0 = M0 * (uint64_t)c0;
    uint64_t p1 = M1 * (uint64_t)c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0;
    uint32_t n1 = lo1;
    uint32_t n2 = hi0 ^ c3 ^ k1;
    uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += W0; k1 += W1;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

static inline double to_unit(uint32_t hi, uint32_t lo) {
  uint64_t v = ((uint64_t)hi << 32) | (uint64_t)lo;
  return (double)(v >> 11) * (1.0 / 9007199254740992.0);  // 2^-53
}

void uniform_pair(uint64_t seed, uint32_t tag, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t n,
                  double* u0, double* u1) {
  uint32_t ctr[4] = {c0, c1, c2, n};
  uint32_t key[2] = {(uint32_t)(seed & 0xffffffffu) ^ tag, (uint32_t)(seed >> 32)};
  uint32_t o[4];
  philox4x32_10(ctr, key, o);
  *u0 = to_unit(o[0], o[1]);
  *u1 = to_unit(o[2], o[3]);
}

Stream::Stream(uint64_t seed, uint32_t tag, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t n0,
               uint32_t key1_xor) {
  ctr[0] = c0; ctr[1] = c1; ctr[2] = c2; ctr[3] = n0;
  key[0] = (uint32_t)(seed & 0xffffffffu) ^ tag;
  key[1] = (uint32_t)(seed >> 32) ^ key1_xor;
  have = 0;
}

double Stream::next() {
  if (have == 0) {
    uint32_t o[4];
    philox4x32_10(ctr, key, o);
    ctr[3] += 1;
    buf[0] = to_unit(o[0], o[1]);
    buf[1] = to_unit(o[2], o[3]);
    have = 2;
  }
  double u = buf[2 - have];
  have--;
  return u;
}

// child id = first 96 bits of philox(ctr = (parent id, j), key = seed ^ TAG_SPAWN)
PhotonId child_id(uint64_t seed, PhotonId parent, uint32_t j) {
  uint32_t ctr[4] = {parent.i0, parent.i1, parent.i2, j};
  uint32_t key[2] = {(uint32_t)(seed & 0xffffffffu) ^ (uint32_t)TAG_SPAWN, (uint32_t)(seed >> 32)};
  uint32_t o[4];
  philox4x32_10(ctr, key, o);
  PhotonId c = {o[0], o[1], o[2]};
  return c;
}

}  // namespace orc
