// fastmath.cuh -- fp64 exp / log / sqrt specialised to the arguments the sweep feeds them (host + device).
//
// The ncu source page of the on-chip kernel (profiles/r01b) attributes 42 % of all executed instructions to four
// libm calls per object-update: log + sqrt of the Box-Muller radius (99 instructions), two exp (97), cospi (50).
// The CUDA libm versions pay for argument ranges that cannot occur here (denormals, infinities, huge arguments).
// These versions keep 1-2 ulp accuracy (exp <= 1.5, log <= 2, sqrt <= 1) on the ranges below with about half the
// instructions:
//   hm_exp_fast(x)   any finite x (clamped to [-708, 709]); x = -inf gives exp(-708) ~ 3e-308, NOT 0 (callers that
//                    need exp(-inf) = 0 select it themselves)
//   hm_log_pos(x)    positive normal numbers only (the Box-Muller uniforms u in [2^-53, 1); 1 + alpha^2 of the prior)
//   hm_sqrt_fast(w)  w > 0 normal
// tests/test_fastmath_host.py measures their error against mpmath on the host build of this very header.
#pragma once
#include <cmath>
#include <cstdint>
#include <cstring>
#include <cuda_runtime.h>

#ifndef HM_HD
#define HM_HD __host__ __device__ __forceinline__
#endif

namespace hm {

HM_HD double hm_bits2d(uint64_t b) {
#ifdef __CUDA_ARCH__
  return __longlong_as_double((long long)b);
#else
  double d; std::memcpy(&d, &b, sizeof d); return d;
#endif
}
HM_HD uint64_t hm_d2bits(double d) {
#ifdef __CUDA_ARCH__
  return (uint64_t)__double_as_longlong(d);
#else
  uint64_t b; std::memcpy(&b, &d, sizeof b); return b;
#endif
}
HM_HD double hm_fma(double a, double b, double c) {
#ifdef __CUDA_ARCH__
  return __fma_rn(a, b, c);
#else
  return std::fma(a, b, c);
#endif
}

// Seeds with about 20 good bits (one MUFU each on the device: the instruction works on the upper 32-bit word of its
// argument and returns a result whose lower word is zero).  The host build imitates the WORST such seed -- the exact value
// with its lower word cleared -- so that the host pins cover what the device may return; tests/test_gpu_fastmath.py
// holds the device build itself to the same pins.  One Newton step takes 2^-20 to 2^-40, and every user below ends with a
// correction step that squares the residual once more (2^-80): a second Newton step would buy nothing.
HM_HD double hm_rcp_seed(double a) {
#ifdef __CUDA_ARCH__
  double r; asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(a)); return r;
#else
  return hm_bits2d(hm_d2bits(1.0 / a) & 0xffffffff00000000ull);
#endif
}
HM_HD double hm_rsqrt_seed(double a) {
#ifdef __CUDA_ARCH__
  double r; asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(a)); return r;
#else
  return hm_bits2d(hm_d2bits(1.0 / std::sqrt(a)) & 0xffffffff00000000ull);
#endif
}

// e^x = 2^k T[j] e^r with n = 64 k + j = round(64 x / ln2), r = x - n ln2/64 (Cody-Waite, two pieces, |r| <= ln2/128),
// T[j] = 2^(j/64) from a 64-entry (hi, lo) table (1 KB, stays in L1) and e^r - 1 by its degree-6 Taylor polynomial
// (truncation 3e-20).  The result is scaled by 2^k through the exponent field (normal for x in [-708, 709]).
// Half the polynomial of a table-free version, and -- what matters more here -- half the fp64 immediates.
#include "exp_table.inc"
#include "log_coeffs.inc"
struct hm_d2 { double hi, lo; };
#ifdef __CUDACC__
__device__ const hm_d2 hm_exp2_tab_dev[64] = {HM_EXP2_TABLE};
#endif
// Where the polynomial coefficients of exp / log come from on the device.  As literals they reach the fp64 pipe through
// uniform registers, two UMOV per coefficient and use (44 of the 425 warp-instructions per 32 updates of the C2 kernel);
// from the constant bank one LDCU.128 brings two of them (sm_100a's DFMA takes a register or a uniform register, never a
// c[bank][offset] operand: probed).  Fewer issue slots, but a constant-cache latency in front of the dependent chain, so
// which is faster depends on the kernel: measured -2 to -3.5 % on the streaming p = 2 kernel (C3), -1.9 % on C1
// (k_resident<M1, SEL_SWEEP>), -0.6 % on C0, +0.3 % on C2, +1.3 % on C6, noise on C5 -- so a translation unit opts in with
// HM_CONST_BANK_COEFFS (inst_binormal2d.cu and inst_thinned_schechter1d_selsweep.cu do).
#if defined(__CUDACC__) && defined(HM_CONST_BANK_COEFFS)
__constant__ double hm_kc[24] = {HM_64_LN2, -HM_LN2_64_HI, -HM_LN2_64_LO, HM_EXP_Q3, HM_EXP_Q2,
  HM_EXP_Q1, HM_EXP_Q0, 0.0,
  HM_LOG_P7, HM_LOG_P6, HM_LOG_P5, HM_LOG_P4, HM_LOG_P3, HM_LOG_P2, HM_LOG_P1, 0.0, 0.0, 0.0, 0.0,
  6.93147180369123816490e-01, 1.90821492927058770002e-10, 0.0, 0.0, 0.0};
#endif
#if defined(__CUDA_ARCH__) && defined(HM_CONST_BANK_COEFFS)
#define HM_KC(i, lit) hm_kc[i]
#else
#define HM_KC(i, lit) (lit)
#endif
static const hm_d2 hm_exp2_tab_host[64] = {HM_EXP2_TABLE};

// hm_exp_core: NO argument check -- finite garbage (or inf / NaN) outside [-708, 709]; for callers that discard the
// result there anyway (a proposal outside the model's support, alpha of a log ratio below -708).
HM_HD double hm_exp_core(double x) {
  const double SHIFT = 6755399441055744.0;                 // 1.5 * 2^52: adding it rounds to the nearest integer
  const double t = hm_fma(x, HM_KC(0, HM_64_LN2), SHIFT);
  const double nf = t - SHIFT;
  double r = hm_fma(nf, HM_KC(1, -HM_LN2_64_HI), x);       // HM_LN2_64_HI has 32 significant bits: exact product
  r = hm_fma(nf, HM_KC(2, -HM_LN2_64_LO), r);
  const int n = (int)(uint32_t)(hm_d2bits(t) & 0xffffffffull);   // the integer sits in the low word of t
  const int j = n & 63, k = n >> 6;
#ifdef __CUDA_ARCH__
  const double2 tj = __ldg(reinterpret_cast<const double2*>(hm_exp2_tab_dev) + j);
  const double thi = tj.x, tlo = tj.y;
#else
  const double thi = hm_exp2_tab_host[j].hi, tlo = hm_exp2_tab_host[j].lo;
#endif
  double p = HM_KC(3, HM_EXP_Q3);                          // 4 near-minimax coefficients (gen_exp_table.py; absolute error
  p = hm_fma(p, r, HM_KC(4, HM_EXP_Q2));                   // 4.4e-18 on e^r - 1: 0.04 ulp of the e^r it becomes; the Taylor
  p = hm_fma(p, r, HM_KC(5, HM_EXP_Q1));                   // polynomial took 5) -- NOT for hm_expm1_nonpos below, which needs
  p = hm_fma(p, r, HM_KC(6, HM_EXP_Q0));                   // relative accuracy at small |x| and keeps the Taylor form
  p = p * r;
  p = hm_fma(p, r, r);                                     // e^r - 1
  const double y = thi + hm_fma(thi, p, tlo);              // T[j] e^r
  return hm_bits2d(hm_d2bits(y) + ((uint64_t)(int64_t)k << 52));
}
// e^x - 1 for x in [-708, 0] with full RELATIVE accuracy also at small |x| (1 - e^(-L/l) of the BB1 density at L << l):
// the same reduction as hm_exp_core; e^x - 1 = (s - 1) + s (e^r - 1) + 2^k T_lo with s = 2^k T_hi[j] in (0, 1]:
// s - 1 is exact for s >= 1/2 (Sterbenz) and, for |x| <= ln2/128, s = 1 and the result is the polynomial itself.
HM_HD double hm_expm1_nonpos(double x) {
  x = x < -708.0 ? -708.0 : x;
  const double SHIFT = 6755399441055744.0;
  const double t = hm_fma(x, HM_64_LN2, SHIFT);
  const double nf = t - SHIFT;
  double r = hm_fma(nf, -HM_LN2_64_HI, x);
  r = hm_fma(nf, -HM_LN2_64_LO, r);
  const int n = (int)(uint32_t)(hm_d2bits(t) & 0xffffffffull);
  const int j = n & 63, k = n >> 6;
#ifdef __CUDA_ARCH__
  const double2 tj = __ldg(reinterpret_cast<const double2*>(hm_exp2_tab_dev) + j);
  const double thi = tj.x, tlo = tj.y;
#else
  const double thi = hm_exp2_tab_host[j].hi, tlo = hm_exp2_tab_host[j].lo;
#endif
  double p = 1.3888888888888889e-03;
  p = hm_fma(p, r, 8.3333333333333332e-03);
  p = hm_fma(p, r, 4.1666666666666664e-02);
  p = hm_fma(p, r, 1.6666666666666666e-01);
  p = hm_fma(p, r, 0.5);
  p = p * r;
  p = hm_fma(p, r, r);                                     // e^r - 1
  const double scale = hm_bits2d((uint64_t)(int64_t)(k + 1023) << 52);   // 2^k, k in [-1022, 0]
  const double sh = thi * scale;                           // exact (power of two)
  return (sh - 1.0) + hm_fma(sh, p, tlo * scale);
}

HM_HD double hm_exp_fast(double x) {
  x = x < -708.0 ? -708.0 : (x > 709.0 ? 709.0 : x);       // (fmin / fmax cost 7 instructions each: NaN handling)
  return hm_exp_core(x);
}

// ln u for positive normal u: u = 2^e m, m in [sqrt(1/2), sqrt 2); ln m = 2 atanh(s), s = (m-1)/(m+1), |s| <= 0.1716,
// atanh(s)/s - 1 by 7 near-minimax coefficients in s^2 (log_coeffs.inc; the Taylor series needed 11 for the same 5e-18:
// 4 fewer DFMA on the serial chain and 8 fewer immediate moves per call); the quotient by a Newton-refined reciprocal.
// NEWTON: Newton steps on the seed before the correcting step (1 is enough, see hm_rcp_seed; 2 is the former code, kept
// because the on-chip p = 1 kernel is FASTER with it: C2 +0.6 %, C1 / C0 +0.5 % with one step -- code generation, the
// kernel is not issue-bound -- while the p = 2 streaming kernel gains 3.2 %).  A translation unit chooses with
// HM_NEWTON_STEPS (default 1); both variants are pinned on the host and on the device.
#ifndef HM_NEWTON_STEPS
#define HM_NEWTON_STEPS 1
#endif
template <int NEWTON>
HM_HD double hm_log_pos_n(double u) {
  uint64_t b = hm_d2bits(u);
  int e = (int)(b >> 52) - 1023;
  b = (b & 0x000fffffffffffffull) | 0x3ff0000000000000ull;
  double m = hm_bits2d(b);                                  // [1, 2)
  if (m > 1.4142135623730951) { m *= 0.5; e += 1; }
  const double a = m + 1.0, f = m - 1.0;
  double rc = hm_rcp_seed(a);
#pragma unroll
  for (int it = 0; it < NEWTON; ++it) {                     // 1/a to 2^-40 (2^-80)
    const double err = hm_fma(-a, rc, 1.0);
    rc = hm_fma(rc, err, rc);
  }
  double s = f * rc;
  s = hm_fma(hm_fma(-s, a, f), rc, s);                      // the correction squares the residual: s = f/a to ~0.5 ulp
  const double s2 = s * s;
  double p = HM_KC(8, HM_LOG_P7);                           // 7 near-minimax coefficients (gen_log_coeffs.py): 4.7e-18
  p = hm_fma(p, s2, HM_KC(9, HM_LOG_P6));
  p = hm_fma(p, s2, HM_KC(10, HM_LOG_P5));
  p = hm_fma(p, s2, HM_KC(11, HM_LOG_P4));
  p = hm_fma(p, s2, HM_KC(12, HM_LOG_P3));
  p = hm_fma(p, s2, HM_KC(13, HM_LOG_P2));
  p = hm_fma(p, s2, HM_KC(14, HM_LOG_P1));
  p = p * s2;                                               // atanh(s)/s - 1
  const double two_s = s + s;
  const double lm = hm_fma(two_s, p, two_s);                // ln m
  const double ed = (double)e;
  return hm_fma(ed, HM_KC(19, 6.93147180369123816490e-01), hm_fma(ed, HM_KC(20, 1.90821492927058770002e-10), lm));
}

HM_HD double hm_log_pos(double u) { return hm_log_pos_n<HM_NEWTON_STEPS>(u); }
HM_HD double hm_log_unit(double u) { return hm_log_pos(u); }   // u in [2^-53, 1)

// sqrt(w), w > 0 normal: Newton on (g, h) = (sqrt w, 1/(2 sqrt w)) from a 2^-23 reciprocal-root seed.
template <int NEWTON>
HM_HD double hm_sqrt_fast_n(double w) {
  const double y = hm_rsqrt_seed(w);
  double g = w * y, h = 0.5 * y;
#pragma unroll
  for (int it = 0; it < NEWTON; ++it) {                     // (g, h) to 2^-40 (2^-80)
    const double r = hm_fma(-g, h, 0.5);
    g = hm_fma(g, r, g); h = hm_fma(h, r, h);
  }
  return hm_fma(hm_fma(-g, g, w), h, g);                    // final correction: g + (w - g^2) h, residual squared
}
HM_HD double hm_sqrt_fast(double w) { return hm_sqrt_fast_n<HM_NEWTON_STEPS>(w); }

// sqrt(w) and 1/sqrt(w) together (the same Newton pair; 1/sqrt = 2 h after one more correction step), w > 0 normal
template <int NEWTON>
HM_HD void hm_sqrt_rsqrt_n(double w, double* root, double* inv_root) {
  const double y = hm_rsqrt_seed(w);
  double g = w * y, h = 0.5 * y;
  double r;
#pragma unroll
  for (int it = 0; it < NEWTON; ++it) {                     // (g, h) to 2^-40 (2^-80)
    r = hm_fma(-g, h, 0.5);
    g = hm_fma(g, r, g); h = hm_fma(h, r, h);
  }
  r = hm_fma(-g, h, 0.5);
  *root = hm_fma(hm_fma(-g, g, w), h, g);
  *inv_root = 2.0 * hm_fma(h, r, h);
}
HM_HD void hm_sqrt_rsqrt(double w, double* root, double* inv_root) { hm_sqrt_rsqrt_n<HM_NEWTON_STEPS>(w, root, inv_root); }

// exp / log of the theta tail: the specialised versions on the device (the tail is a serial chain on the critical
// path of every iteration), libm on the host (THETA_HOST).
HM_HD double hm_exp_any(double x) {
#ifdef __CUDA_ARCH__
  const double r = hm_exp_fast(x);
  return x < -708.0 ? 0.0 : r;
#else
  return std::exp(x);
#endif
}
// sin(2 pi u), cos(2 pi u) for u in [0, 1]: the Box-Muller angle of the plate draws (u on the sampler's 2^-32 or 2^-53
// grids, but any double in range works).  64 u is exact; adding 1.5 * 2^52 rounds it to the nearest integer n (low word
// of the sum) and d = 64 u - n in [-1/2, 1/2] is exact, so the angle is 2 pi n / 64 + phi with phi = d pi / 32,
// |phi| <= pi / 64 = 0.0491.  T[n & 63] = (S, C) = (sin, cos)(2 pi n / 64) from a 64-entry table (1 KB, stays in L1), rounded
// to nearest and EXACTLY 0 / +-1 at the quarter turns, so that near the zeros of sin and cos the result is C sin(phi)
// (resp. -S sin(phi)) with full relative accuracy.  sin(phi) by its Taylor polynomial through phi^9 (truncation
// phi^10 / 11! < 3e-21 relative), cos(phi) - 1 through phi^8 (phi^10 / 10! < 3e-20), then
//   sin = S + (S (cos phi - 1) + C sin phi),  cos = C + (C (cos phi - 1) - S sin phi).
// Error: half an ulp of the table entry, half an ulp of the last sum, and the roundings of the small bracket: <= 2 ulp,
// pinned in tests/test_fastmath_host.py against mpmath.  Half the instructions of the library sincospi on this argument
// range (26 + 11 fp64 immediates against 38 + 15), and a dependent chain of 4 DFMA instead of 7.
#include "sincos_table.inc"
#ifdef __CUDACC__
__device__ const hm_d2 hm_sincos64_tab_dev[64] = {HM_SINCOS64_TABLE};
#endif
static const hm_d2 hm_sincos64_tab_host[64] = {HM_SINCOS64_TABLE};
HM_HD void hm_sincos2pi(double u, double* s, double* c) {
  const double SHIFT = 6755399441055744.0;                 // 1.5 * 2^52
  const double t = hm_fma(u, 64.0, SHIFT);                 // n = rint(64 u) in the low word
  const double d = hm_fma(u, 64.0, -(t - SHIFT));          // 64 u - n, exact
  const int j = (int)(uint32_t)(hm_d2bits(t) & 63ull);
#ifdef __CUDA_ARCH__
  const double2 tj = __ldg(reinterpret_cast<const double2*>(hm_sincos64_tab_dev) + j);
  const double S = tj.x, C = tj.y;
#else
  const double S = hm_sincos64_tab_host[j].hi, C = hm_sincos64_tab_host[j].lo;
#endif
  const double phi = d * HM_PI_32;
  const double p2 = phi * phi;
  double sp = 2.7557319223985893e-06;                      // 1/9!
  sp = hm_fma(sp, p2, -1.9841269841269841e-04);            // -1/7!
  sp = hm_fma(sp, p2, 8.3333333333333332e-03);             // 1/5!
  sp = hm_fma(sp, p2, -1.6666666666666666e-01);            // -1/3!
  const double sphi = hm_fma(sp * p2, phi, phi);           // sin(phi)
  double cp = 2.4801587301587302e-05;                      // 1/8!
  cp = hm_fma(cp, p2, -1.3888888888888889e-03);            // -1/6!
  cp = hm_fma(cp, p2, 4.1666666666666664e-02);             // 1/4!
  cp = hm_fma(cp, p2, -0.5);
  const double cm = cp * p2;                               // cos(phi) - 1
  *s = S + hm_fma(S, cm, C * sphi);
  *c = C + hm_fma(C, cm, -(S * sphi));
}

HM_HD double hm_log_any_pos(double x) {
#ifdef __CUDA_ARCH__
  return hm_log_pos(x);
#else
  return std::log(x);
#endif
}

}  // namespace hm
