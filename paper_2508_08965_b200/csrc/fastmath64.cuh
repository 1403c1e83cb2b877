// fastmath64.cuh -- branch-free fp64 reciprocal, reciprocal square root, exponential and half-space Maxwellian moments
// for the flux kernel.  CUDA's libm versions carry slow-path branches that split the kernel body into basic blocks and
// keep ptxas from overlapping their long dependent chains with the neighbouring moment arithmetic (with two warps per
// scheduler those chains idled the FP64 pipe; profiles/r01c).  These versions are straight-line code with ~1-2 ulp
// error (not correctly rounded), valid for the finite, normal arguments of the flux kernel.
#pragma once
#include "math_gen.cuh"

namespace cgks {

// 1/x: MUFU.RCP64H seed (about 20 bits) + two Newton steps (error 2^-20 -> 2^-40 -> 2^-80, i.e. rounding only)
__device__ __forceinline__ double drcp(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  double e = fma(-x, r, 1.0); r = fma(r, e, r);
  e = fma(-x, r, 1.0); r = fma(r, e, r);
  return r;
}

// a/b with one residual correction of the quotient
__device__ __forceinline__ double ddiv(double a, double b) {
  const double r = drcp(b);
  const double q = a * r;
  return fma(fma(-b, q, a), r, q);
}

// 1/sqrt(x): MUFU.RSQ64H seed + Newton steps; sqrt(x) = x * drsqrt(x) with a residual correction
__device__ __forceinline__ double drsqrt(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double hx = 0.5 * x;
  double e = fma(-hx * y, y, 0.5); y = fma(y, e, y);
  e = fma(-hx * y, y, 0.5); y = fma(y, e, y);
  return y;
}

// exp(x) for x <= ~700 (clamped below at -1000 -> 0): Cody-Waite reduction by ln 2, Taylor polynomial of degree 13 on
// |r| <= ln2/2 (remainder < 4e-18), scaling by 2^n in two halves so that the result may underflow gradually
__device__ __forceinline__ double dexp(double x) {
  x = fmax(x, -1000.0);
  const double t = fma(x, 1.4426950408889634, 6755399441055744.0);        // 1.5 * 2^52: integer part lands in the low word
  const int n = __double2loint(t);
  const double nf = t - 6755399441055744.0;
  double r = fma(nf, -6.93147180559945290e-01, x);
  r = fma(nf, -2.31904681384629956e-17, r);
  const double r2 = r * r;
  // even and odd parts of sum_{k<=13} r^k/k! evaluated separately (two independent Horner chains in r^2)
  double pe = 1.0 / 479001600.0;                  // 1/12!
  pe = fma(pe, r2, 1.0 / 3628800.0);              // 1/10!
  pe = fma(pe, r2, 1.0 / 40320.0);
  pe = fma(pe, r2, 1.0 / 720.0);
  pe = fma(pe, r2, 1.0 / 24.0);
  pe = fma(pe, r2, 0.5);
  pe = fma(pe, r2, 1.0);
  double po = 1.0 / 6227020800.0;                 // 1/13!
  po = fma(po, r2, 1.0 / 39916800.0);             // 1/11!
  po = fma(po, r2, 1.0 / 362880.0);
  po = fma(po, r2, 1.0 / 5040.0);
  po = fma(po, r2, 1.0 / 120.0);
  po = fma(po, r2, 1.0 / 6.0);
  po = fma(po, r2, 1.0);
  const double p = fma(po, r, pe);
  const int n1 = n >> 1, n2 = n - n1;
  const double s1 = __hiloint2double((1023 + n1) << 20, 0), s2 = __hiloint2double((1023 + n2) << 20, 0);
  return (p * s1) * s2;
}

// log(x) for positive, finite, normal x: x = m 2^e with m in [1/sqrt 2, sqrt 2), log m = 2 atanh(f), f = (m-1)/(m+1),
// |f| <= 0.1716, odd series up to f^23 (next term < 6e-19); e ln 2 with ln 2 split in two.  Used for the viscosity power
// law (T/T_ref)^omega = exp(omega log(T/T_ref)); CUDA's log carries slow-path branches (see the header of this file).
__device__ __forceinline__ double dlog(double x) {
  int hi = __double2hiint(x);
  const int lo = __double2loint(x);
  int e = (hi >> 20) - 1023;
  hi = (hi & 0x000fffff) | 0x3ff00000;
  double m = __hiloint2double(hi, lo);                     // [1, 2)
  const bool big = m > 1.4142135623730951;
  m = big ? 0.5 * m : m;
  e += big ? 1 : 0;
  const double f = (m - 1.0) * drcp(m + 1.0), f2 = f * f;
  // two interleaved Horner chains in f^4 for sum_{k>=1} f2^k/(2k+1), k = 1..11
  const double f4 = f2 * f2;
  double pa = 1.0 / 23.0;                                  // k = 11, 9, 7, 5, 3, 1
  pa = fma(pa, f4, 1.0 / 19.0);
  pa = fma(pa, f4, 1.0 / 15.0);
  pa = fma(pa, f4, 1.0 / 11.0);
  pa = fma(pa, f4, 1.0 / 7.0);
  pa = fma(pa, f4, 1.0 / 3.0);
  double pb = 1.0 / 21.0;                                  // k = 10, 8, 6, 4, 2
  pb = fma(pb, f4, 1.0 / 17.0);
  pb = fma(pb, f4, 1.0 / 13.0);
  pb = fma(pb, f4, 1.0 / 9.0);
  pb = fma(pb, f4, 1.0 / 5.0);
  const double p = f2 * fma(pb, f2, pa);                   // sum_{k>=1} f2^k/(2k+1)
  const double tf = 2.0 * f;
  const double lm = fma(tf, p, tf);
  const double de = (double)e;
  return fma(de, 6.93147180369123816490e-01, fma(de, 1.90821492927058770002e-10, lm));
}

// tanh(x) for x >= 0 (the path function of the GENO blend): (1 - e)/(1 + e), e = exp(-2x); absolute error ~1e-16
__device__ __forceinline__ double dtanh_pos(double x) {
  const double e = dexp(-2.0 * x);
  return (1.0 - e) * drcp(1.0 + e);
}

// erfc(|x|) * exp(x^2) * (1 + 2|x|) as a polynomial in t = (|x|-4)/(|x|+4): even/odd split, two Horner chains
__device__ __forceinline__ double erfcx_poly(double t) {
  const double CGKS_ERFCX_P[CGKS_ERFCX_NP] = { CGKS_ERFCX_P_LIST };
  const double t2 = t * t;
  double pe = CGKS_ERFCX_P[22], po = CGKS_ERFCX_P[21];
#pragma unroll
  for (int k = 20; k >= 0; k -= 2) pe = fma(pe, t2, CGKS_ERFCX_P[k]);
#pragma unroll
  for (int k = 19; k >= 1; k -= 2) po = fma(po, t2, CGKS_ERFCX_P[k]);
  return fma(po, t, pe);
}

// erfc(y) and exp(-y^2) together (they share the exponential); |y| up to ~26 before erfc underflows
__device__ __forceinline__ void derfc_exp(double y, double& erfc_y, double& exp_my2) {
  const double s = y * y, slo = fma(y, y, -s);           // y^2 = s + slo exactly
  double E = dexp(-s);
  E = fma(-E, slo, E);                                   // exp(-(s + slo))
  const double ay = fabs(y);
  const double t = (ay - 4.0) * drcp(ay + 4.0);
  const double c = erfcx_poly(t) * E * drcp(fma(2.0, ay, 1.0));      // erfc(|y|)
  erfc_y = (y >= 0.0) ? c : 2.0 - c;
  exp_my2 = E;
}

}  // namespace cgks
