// oracle/rng.hpp -- counter-based random streams of the oracle.  TEST INFRASTRUCTURE ONLY.
//
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, "Parallel random numbers: as easy as 1, 2, 3", SC'11)
// restated from its published definition; replaces the "pseudo-random number generator library"
// of PAPER.md:65 (fn. 2) and :142.  Stream layout: DESIGN.md section 4 (north_star: "streams keyed
// by (seed, object, iteration, draw)").  Shares nothing with the CUDA tree.
#pragma once
#include <cmath>
#include <cstdint>

namespace oracle {

struct Words { uint32_t w[4]; };

// One Philox4x32 bijection with 10 rounds.  Round: (hi0,lo0) = M0*c0, (hi1,lo1) = M1*c2 as
// 32x32->64 products; c <- (hi1^c1^k0, lo1, hi0^c3^k1, lo0); key bumped by (W0,W1) between rounds.
inline Words philox4x32_10(const uint32_t ctr[4], const uint32_t key[2]) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    if (round > 0) { k0 += W0; k1 += W1; }
    const uint64_t p0 = (uint64_t)M0 * (uint64_t)c0;
    const uint64_t p1 = (uint64_t)M1 * (uint64_t)c2;
    const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    const uint32_t n0 = hi1 ^ c1 ^ k0;
    const uint32_t n1 = lo1;
    const uint32_t n2 = hi0 ^ c3 ^ k1;
    const uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
  }
  Words r; r.w[0] = c0; r.w[1] = c1; r.w[2] = c2; r.w[3] = c3;
  return r;
}

// key = (seed low word, seed high word);
// counter = (object bits 0..31, kind<<24 | object bits 32..55, iteration t, draw index d).
inline Words stream_words(uint64_t seed, int kind, uint64_t obj, uint32_t t, uint32_t d) {
  uint32_t key[2] = { (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32) };
  uint32_t ctr[4] = { (uint32_t)(obj & 0xffffffffu),
                      ((uint32_t)kind << 24) | (uint32_t)((obj >> 32) & 0xffffffu), t, d };
  return philox4x32_10(ctr, key);
}

// 52 random bits + 1/2, scaled by 2^-52: a dyadic rational in [2^-53, 1-2^-53], exact in fp64.
inline double u01_f64(uint32_t wa, uint32_t wb) {
  const uint64_t k = ((uint64_t)(wa >> 6) << 26) | (uint64_t)(wb >> 6);
  return ((double)k + 0.5) * 0x1.0p-52;
}
// 32 random bits + 1/2, scaled by 2^-32: a dyadic rational in [2^-33, 1-2^-33], exact in fp64.
inline double u01_32(uint32_t w) {
  return ((double)w + 0.5) * 0x1.0p-32;
}
// 23 random bits + 1/2, scaled by 2^-23: exact in fp32, never 0 or 1.
inline float u01_f32(uint32_t w) {
  return ((float)(w >> 9) + 0.5f) * 0x1.0p-23f;
}

// fp64 draws.  Draw d = 0: the accept uniform from words (w0,w1).  Draw d = 1+k: the Box-Muller pair
// (z_{2k}, z_{2k+1}) with u1 from (w0,w1), u2 from (w2,w3):
//   z_{2k} = sqrt(-2 ln u1) cos(2 pi u2),  z_{2k+1} = sqrt(-2 ln u1) sin(2 pi u2).
inline double accept_uniform_f64(uint64_t seed, int kind, uint64_t obj, uint32_t t) {
  const Words r = stream_words(seed, kind, obj, t, 0u);
  return u01_f64(r.w[0], r.w[1]);
}
inline void normals_f64(uint64_t seed, int kind, uint64_t obj, uint32_t t, int n, double* z) {
  const double two_pi = 6.283185307179586476925286766559;
  for (int k = 0; 2 * k < n; ++k) {
    const Words r = stream_words(seed, kind, obj, t, (uint32_t)(1 + k));
    const double u1 = u01_f64(r.w[0], r.w[1]);
    const double u2 = u01_f64(r.w[2], r.w[3]);
    const double rad = std::sqrt(-2.0 * std::log(u1));
    z[2 * k] = rad * std::cos(two_pi * u2);
    if (2 * k + 1 < n) z[2 * k + 1] = rad * std::sin(two_pi * u2);
  }
}

// fp32 draws (plate streams of the fp32-state configuration; p <= 2): ONE call, draw d = 0:
// w0 -> u1, w1 -> u2 (Box-Muller pair z0, z1), w2 -> accept uniform, w3 unused.
inline void draws_f32(uint64_t seed, int kind, uint64_t obj, uint32_t t, float z[2], float* u) {
  const float two_pi = 6.283185307179586476925286766559f;
  const Words r = stream_words(seed, kind, obj, t, 0u);
  const float u1 = u01_f32(r.w[0]);
  const float u2 = u01_f32(r.w[1]);
  const float rad = std::sqrt(-2.0f * std::log(u1));
  z[0] = rad * std::cos(two_pi * u2);
  z[1] = rad * std::sin(two_pi * u2);
  *u = u01_f32(r.w[2]);
}

// ---- plate-level draws of object i at iteration t --------------------------------
// Objects are taken in PAIRS m = i >> 1, h = i & 1, so that one Philox call and one Box-Muller evaluation
// serve two objects (both branches of Box-Muller are independent N(0,1) variates; nothing is discarded).
//   fp64  p = 1: ONE call per pair, draw 0 of PAIR m, every word a 32-bit uniform u = (w + 1/2) 2^-32 (exact in fp64, in
//                [2^-33, 1 - 2^-33]): w0 -> u1 (radius sqrt(-2 ln u1)), w1 -> u2 (angle), z = radius cos(2 pi u2) for
//                h = 0, radius sin(2 pi u2) for h = 1; accept uniform from w2 (h = 0) / w3 (h = 1).  (The proposal stays
//                symmetric -- all a Metropolis step needs -- with its radius capped at sqrt(66 ln 2) = 6.76.)
//         p >= 2: accept uniform (52 bits): draw 0 of PAIR m -- words (w0,w1) for h = 0, (w2,w3) for h = 1;
//                normals: per OBJECT, draws 1+k of object i exactly as normals_f64.
//   fp32  p = 1: ONE call per pair, draw 0 of PAIR m: w0 -> u1, w1 -> u2, z = cos / sin branch for h = 0 / 1,
//                accept uniform from w2 (h = 0) / w3 (h = 1).
//         p = 2: per OBJECT as draws_f32.
inline void plate_draws_f64(uint64_t seed, uint64_t i, uint32_t t, int p, double* z, double* u) {
  const double two_pi = 6.283185307179586476925286766559;
  const uint64_t m = i >> 1;
  const int h = (int)(i & 1);
  const Words a = stream_words(seed, 0 /* PLATE */, m, t, 0u);
  if (p == 1) {
    const double u1 = u01_32(a.w[0]);
    const double u2 = u01_32(a.w[1]);
    const double rad = std::sqrt(-2.0 * std::log(u1));
    z[0] = h ? rad * std::sin(two_pi * u2) : rad * std::cos(two_pi * u2);
    *u = u01_32(h ? a.w[3] : a.w[2]);
  } else {
    *u = h ? u01_f64(a.w[2], a.w[3]) : u01_f64(a.w[0], a.w[1]);
    normals_f64(seed, 0, i, t, p, z);
  }
}
inline void plate_draws_f32(uint64_t seed, uint64_t i, uint32_t t, int p, float* z, float* u) {
  if (p != 1) { draws_f32(seed, 0, i, t, z, u); return; }
  const float two_pi = 6.283185307179586476925286766559f;
  const uint64_t m = i >> 1;
  const int h = (int)(i & 1);
  const Words r = stream_words(seed, 0, m, t, 0u);
  const float u1 = u01_f32(r.w[0]);
  const float u2 = u01_f32(r.w[1]);
  const float rad = std::sqrt(-2.0f * std::log(u1));
  z[0] = h ? rad * std::sin(two_pi * u2) : rad * std::cos(two_pi * u2);
  *u = u01_f32(h ? r.w[3] : r.w[2]);
}

}  // namespace oracle
