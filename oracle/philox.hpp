// TEST INFRASTRUCTURE — CPU oracle for arXiv 2605.08916 ("Diffusion Restore").
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// leg may use anything under oracle/. It shares no code with the CUDA path.
//
// Philox4x32-10 counter-based generator (Salmon et al. 2011), the generator the paper
// names for its per-chain `rng` field.  Stream keying is the DESIGN.md
// reading Q14: key = (seed_lo, seed_hi), counter = (chain, iteration, slot,
// purpose | epoch << 8).  Pin: tests/test_oracle_rng.py compares this function word
// for word with ATen's independent at::Philox4_32 (torch/include/ATen/core/
// PhiloxRNGEngine.h), compiled on the spot.
#pragma once
#include <cmath>
#include <cstdint>

namespace orc {

inline void philox4x32_10(const uint32_t key[2], const uint32_t ctr[4], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    if (round > 0) {  // key schedule: Weyl sequence, bumped between rounds
      k0 += 0x9E3779B9u;
      k1 += 0xBB67AE85u;
    }
    const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
    const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    const uint32_t n1 = (uint32_t)p1;
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    const uint32_t n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Purposes of a block (Q14).
enum Purpose : uint32_t {
  REGEN_U = 0,  // slot j -> uniforms for PSS dims 4j..4j+3 of a regenerated / initial state
  PROP_N = 1,   // slot j -> two Box-Muller pairs -> normals for dims 4j..4j+3
  DECIDE = 2,   // w0 = u_large, w1 = u_accept, w2 = u_hold, w3 = u_kill
  LARGE_U = 3   // slot j -> uniforms for dims 4j..4j+3 of a large-step proposal
};

inline void stream_block(uint64_t seed, uint32_t chain, uint32_t iteration, uint32_t slot,
                         uint32_t purpose, uint32_t epoch, uint32_t out[4]) {
  const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  const uint32_t ctr[4] = {chain, iteration, slot, purpose | (epoch << 8)};
  philox4x32_10(key, ctr, out);
}

// u in [0,1): top 24 bits.  u in (0,1]: the same plus one ulp of 2^-24; used under every log.
template <class Real> inline Real u01_co(uint32_t w) { return Real(w >> 8) * Real(1.0 / 16777216.0); }
template <class Real> inline Real u01_oc(uint32_t w) { return Real((w >> 8) + 1u) * Real(1.0 / 16777216.0); }

// Box-Muller: (wa, wb) -> two independent N(0,1).  xi ~ N(0, I_2) of Alg. 4 line 3.
template <class Real> inline void box_muller(uint32_t wa, uint32_t wb, Real& z0, Real& z1) {
  const Real ua = u01_oc<Real>(wa);
  const Real ub = u01_co<Real>(wb);
  const Real r = std::sqrt(Real(-2) * std::log(ua));
  const Real phi = Real(6.283185307179586476925286766559) * ub;
  z0 = r * std::cos(phi);
  z1 = r * std::sin(phi);
}

}  // namespace orc
