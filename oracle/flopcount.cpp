/*
 * flopcount.cpp -- the CPU oracle compiled with a COUNTING double ("an instrumented count from
 * the oracle -- a counting double wrapper -- with FMA = 2 and div/sqrt/exp/erfc/tanh = 1 each").  TEST INFRASTRUCTURE ONLY.
 *
 * The whole of cgks_ref.c is included with the token `double` replaced by a class whose arithmetic operators count:
 * add, subtract, multiply = 1 flop each (the oracle is built without FMA contraction, so a multiply-add is 2), divide,
 * sqrt, exp, erfc, tanh, pow = 1 each; comparisons, negation and fabs = 0.  Two totals are kept: every operation, and
 * the operations whose operands are both non-zero (multiplications by a structural zero of the constant matrices M, E
 * and of the moment tables, and additions of such products, are not algorithmic work: SURVEY.md 8(d) counts "non-zeros
 * of M and E").  Built without OpenMP; oracle/flop_count.py drives it.
 */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

static long g_flops_all = 0, g_flops_nz = 0;

struct cdouble {
  double v;
  cdouble() = default;
  cdouble(double x) : v(x) {}
};
static inline void cnt(bool nz) { g_flops_all++; if (nz) g_flops_nz++; }
static inline cdouble operator+(const cdouble& a, const cdouble& b) { cnt(a.v != 0.0 && b.v != 0.0); return cdouble(a.v + b.v); }
static inline cdouble operator-(const cdouble& a, const cdouble& b) { cnt(a.v != 0.0 && b.v != 0.0); return cdouble(a.v - b.v); }
static inline cdouble operator*(const cdouble& a, const cdouble& b) { cnt(a.v != 0.0 && b.v != 0.0); return cdouble(a.v * b.v); }
static inline cdouble operator/(const cdouble& a, const cdouble& b) { cnt(a.v != 0.0); return cdouble(a.v / b.v); }
static inline cdouble operator-(const cdouble& a) { return cdouble(-a.v); }
static inline cdouble& operator+=(cdouble& a, const cdouble& b) { a = a + b; return a; }
static inline cdouble& operator-=(cdouble& a, const cdouble& b) { a = a - b; return a; }
static inline cdouble& operator*=(cdouble& a, const cdouble& b) { a = a * b; return a; }
static inline cdouble& operator/=(cdouble& a, const cdouble& b) { a = a / b; return a; }
static inline bool operator<(const cdouble& a, const cdouble& b) { return a.v < b.v; }
static inline bool operator>(const cdouble& a, const cdouble& b) { return a.v > b.v; }
static inline bool operator<=(const cdouble& a, const cdouble& b) { return a.v <= b.v; }
static inline bool operator>=(const cdouble& a, const cdouble& b) { return a.v >= b.v; }
static inline bool operator==(const cdouble& a, const cdouble& b) { return a.v == b.v; }
static inline bool operator!=(const cdouble& a, const cdouble& b) { return a.v != b.v; }
static inline cdouble sqrt(const cdouble& a) { cnt(true); return cdouble(sqrt(a.v)); }
static inline cdouble exp(const cdouble& a) { cnt(true); return cdouble(exp(a.v)); }
static inline cdouble erfc(const cdouble& a) { cnt(true); return cdouble(erfc(a.v)); }
static inline cdouble tanh(const cdouble& a) { cnt(true); return cdouble(tanh(a.v)); }
static inline cdouble pow(const cdouble& a, const cdouble& b) { cnt(true); return cdouble(pow(a.v, b.v)); }
static inline cdouble pow(const cdouble& a, int b) { cnt(true); return cdouble(pow(a.v, (double)b)); }
static inline cdouble fabs(const cdouble& a) { return cdouble(fabs(a.v)); }

extern "C" void cgks_ref_flops_reset(void) { g_flops_all = 0; g_flops_nz = 0; }
extern "C" void cgks_ref_flops_get(long* all, long* nonzero) { *all = g_flops_all; *nonzero = g_flops_nz; }

extern "C" {
#define double cdouble
#include "cgks_ref.c"
#undef double
}
