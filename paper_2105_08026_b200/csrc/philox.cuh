// philox.cuh -- counter-based Philox4x32-10 streams of the CUDA path (host + device).
//
// Replaces the PRNG library of the paper (PAPER.md:65 fn. 2, :142) with streams keyed by
// (seed, object, iteration, draw) so any thread can produce any variate with no RNG state in HBM
// (DESIGN.md section 4).  Shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#define HM_HD __host__ __device__ __forceinline__

namespace hm {

enum : int { KIND_PLATE = 0, KIND_THETA = 1 };

struct U4 { uint32_t x, y, z, w; };

HM_HD uint32_t mulhi32(uint32_t a, uint32_t b) {
#ifdef __CUDA_ARCH__
  return __umulhi(a, b);
#else
  return (uint32_t)(((uint64_t)a * (uint64_t)b) >> 32);
#endif
}

// 10 rounds of the Philox-4x32 S-P network; the key schedule is a Weyl sequence.  (Writing the two products of a
// round as one 64-bit multiply each -- IMAD.WIDE -- measured 5 % SLOWER than separate high and low halves.)
HM_HD U4 philox4x32_10(U4 c, uint32_t k0, uint32_t k1) {
  constexpr uint32_t PM0 = 0xD2511F53u, PM1 = 0xCD9E8D57u, PW0 = 0x9E3779B9u, PW1 = 0xBB67AE85u;
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t h0 = mulhi32(PM0, c.x), l0 = PM0 * c.x;
    const uint32_t h1 = mulhi32(PM1, c.z), l1 = PM1 * c.z;
    c = U4{h1 ^ c.y ^ k0, l1, h0 ^ c.w ^ k1, l0};
    k0 += PW0; k1 += PW1;
  }
  return c;
}

// The key schedule (a Weyl sequence of the seed) is the same for every call: the sweep takes the 10 round keys ready-made
// from the kernel parameters (constant bank operands of the XORs) instead of bumping the key twice per round and call --
// 20 integer adds less per Philox call, about 6 % of the instructions of the fp32 kernel.  Same words bit for bit.
struct RoundKeys { uint32_t k0[10], k1[10]; };
HM_HD RoundKeys make_round_keys(uint64_t seed) {
  RoundKeys rk;
  uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
  for (int r = 0; r < 10; ++r) { rk.k0[r] = k0; rk.k1[r] = k1; k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
  return rk;
}
HM_HD U4 philox4x32_10(U4 c, const RoundKeys& rk) {
  constexpr uint32_t PM0 = 0xD2511F53u, PM1 = 0xCD9E8D57u;
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t h0 = mulhi32(PM0, c.x), l0 = PM0 * c.x;
    const uint32_t h1 = mulhi32(PM1, c.z), l1 = PM1 * c.z;
    c = U4{h1 ^ c.y ^ rk.k0[r], l1, h0 ^ c.w ^ rk.k1[r], l0};
  }
  return c;
}
HM_HD U4 stream(const RoundKeys& rk, int kind, uint64_t obj, uint32_t t, uint32_t d) {
  U4 c{(uint32_t)obj, ((uint32_t)kind << 24) | ((uint32_t)(obj >> 32) & 0xffffffu), t, d};
  return philox4x32_10(c, rk);
}

// counter = (object lo, kind<<24 | object bits 32..55, iteration, draw); key = seed words
HM_HD U4 stream(uint64_t seed, int kind, uint64_t obj, uint32_t t, uint32_t d) {
  U4 c{(uint32_t)obj, ((uint32_t)kind << 24) | ((uint32_t)(obj >> 32) & 0xffffffu), t, d};
  return philox4x32_10(c, (uint32_t)seed, (uint32_t)(seed >> 32));
}

// (52 random bits k + 1/2) * 2^-52: exact, in [2^-53, 1 - 2^-53].  k = (a >> 6) * 2^26 + (b >> 6) is dropped into
// the mantissa of a double in [1, 2) and (1 - 2^-53) is subtracted: both steps exact, no int -> fp conversion.
HM_HD double u01(uint32_t a, uint32_t b) {
  const uint32_t hi = 0x3FF00000u | (a >> 12), lo = ((a >> 6) << 26) | (b >> 6);
#ifdef __CUDA_ARCH__
  const double d = __hiloint2double((int)hi, (int)lo);
#else
  const uint64_t bits = ((uint64_t)hi << 32) | lo;
  double d;
  __builtin_memcpy(&d, &bits, sizeof d);
#endif
  return d - 0x1.fffffffffffffp-1;
}
// (32 random bits w + 1/2) * 2^-32: exact, in [2^-33, 1 - 2^-33].  w is dropped into the top of the mantissa of a double in
// [1, 2) and (1 - 2^-33) is subtracted: both steps exact, no int -> fp conversion.
HM_HD double u01_32(uint32_t w) {
  const uint32_t hi = 0x3FF00000u | (w >> 12), lo = w << 20;
#ifdef __CUDA_ARCH__
  const double d = __hiloint2double((int)hi, (int)lo);
#else
  const uint64_t bits = ((uint64_t)hi << 32) | lo;
  double d;
  __builtin_memcpy(&d, &bits, sizeof d);
#endif
  return d - 0x1.ffffffffp-1;
}
// (23 random bits k + 1/2) * 2^-23: exact in fp32; k goes into the mantissa of a float in [1, 2), then 1 - 2^-24 is
// subtracted (both steps exact, no int -> fp conversion)
HM_HD float u01f(uint32_t a) {
  const uint32_t bits = 0x3f800000u | (a >> 9);
#ifdef __CUDA_ARCH__
  return __uint_as_float(bits) - 0x1.fffffep-1f;
#else
  float f;
  __builtin_memcpy(&f, &bits, sizeof f);
  return f - 0x1.fffffep-1f;
#endif
}

// Box-Muller pair from one Philox call (fp64): u1 from (x,y), u2 from (z,w).
// Returns radius and the unit vector (cos, sin)(2 pi u2): z = rad * (c, s) and z/|z| = (c, s).
HM_HD void box_muller(const U4& r, double* rad, double* c, double* s) {
  const double u1 = u01(r.x, r.y), u2 = u01(r.z, r.w);
  *rad = sqrt(-2.0 * log(u1));
#ifdef __CUDA_ARCH__
  sincospi(2.0 * u2, s, c);
#else
  sincos(6.283185307179586476925286766559 * u2, s, c);
#endif
}

// n fp64 standard normals of stream (seed, kind, obj, t): pair k comes from draw d = 1 + k
HM_HD void normals(uint64_t seed, int kind, uint64_t obj, uint32_t t, int n, double* z) {
  for (int k = 0; 2 * k < n; ++k) {
    double rad, c, s;
    box_muller(stream(seed, kind, obj, t, 1u + (uint32_t)k), &rad, &c, &s);
    z[2 * k] = rad * c;
    if (2 * k + 1 < n) z[2 * k + 1] = rad * s;
  }
}

}  // namespace hm
