// gks_flux.cuh -- gas-kinetic interface solver at one face Gauss point, in the face frame (n, t1, t2).
//
// Computes, from the left/right reconstructed states and slopes, the second-order integral solution of the BGK
// equation (Eq. 5), its time integrals over [0,dt] and [0,dt/2] and the time linearisation
// (Eq. 6-7): F^n, F_t^n, and the one-sided interface values Q^{l,r}, Q_t^{l,r}.
// Collision time per PAPER.md:344-352.  Readings of the paper's gaps: DESIGN.md section 3 (F1-F3, T1-T2).
//
// Formulation (differs from the CPU oracle on purpose).  Every term of Eq. 5 is a moment
// <(a.psi) u^I v^J w^K psi_alpha> of a Maxwellian, psi = (1, u, v, w, (u^2+v^2+w^2+xi^2)/2).  For each Maxwellian the
// tangential velocities are measured from its own mean, c_v = v - V, c_w = w - W, T = c_v^2 + c_w^2 + xi^2, and slopes and
// moments are carried in the basis psi' = (1, u, c_v, c_w, (u^2 + T)/2) ("primed"):
//     psi = B psi',  B = [1; u; V + c_v; W + c_w; psi'_4 + V c_v + W c_w + (V^2+W^2)/2].
// In that basis the (c_v, c_w, xi) integrals are the central moments <c_v^2> = 1/(2 lam), <T> = (K+2)/(2 lam), ... so no
// moment tables are needed: a slope leaves ONE quadratic in u (weight 1) plus two constants (weights c_v, c_w), and the
// spatial-divergence combination a_x u + a_y v + a_z w of Eq. 5 leaves one cubic and two quadratics.  The micro-slope
// solve is done directly in the primed basis (its tangential part decouples: a'_2 = 2 lam h'_2), the compatibility
// condition hands its primed moments straight to the solve of the time slope, and only what is summed over BOTH sides
// (different V, W) is converted to the laboratory basis, 10 FMAs per moment vector.
#pragma once
#include <math.h>
#include "fastmath64.cuh"

namespace cgks {

struct GasConst {
  double K;            // internal degrees of freedom N = (5-3 gamma)/(gamma-1)
  double inv_K3;       // 1/(K+3)
  double Pr_fix;       // 1/Pr - 1, 0 when inviscid
  double mu_ref, omega, inv_T_ref;
  double c1, c2;       // tau = mu/p + c1 dt + c2 |pl-pr|/|pl+pr| dt
};

// Maxwellian (per unit density) and the constants of its primed basis
struct Maxw {
  double rho, irho, U, V, W, lam, hil;   // hil = 1/(2 lam) = p/rho
  double hsU;                            // (U^2 + (K+3)/(2 lam))/2
  double c4;                             // 4 lam^2/(K+3)
  double q2;                             // (V^2 + W^2)/2
  double t1;                             // <T> = (K+2)/(2 lam)
};

// scalars of the Maxwellian of the conservative state Wc.  ONE division: with re = rho E - |m|^2/2 = rho (rho e),
// r = 1/(rho re) gives 1/rho = re r and 1/re = rho r; lambda = (K+3) rho/(4 rho e) = (K+3) rho^2/(4 re).
__device__ __forceinline__ void maxw_scalars(Maxw& g, const double* Wc, const GasConst& gc) {
  g.rho = Wc[0];
  const double re = Wc[0] * Wc[4] - 0.5 * (Wc[1] * Wc[1] + Wc[2] * Wc[2] + Wc[3] * Wc[3]);     // rho * (rho e)
  const double r = drcp(Wc[0] * re);
  g.irho = re * r;
  const double ire = Wc[0] * r;
  g.U = Wc[1] * g.irho; g.V = Wc[2] * g.irho; g.W = Wc[3] * g.irho;
  g.hil = 2.0 * gc.inv_K3 * re * (g.irho * g.irho);          // 1/(2 lam) = 2 (rho e)/((K+3) rho) = p/rho
  g.lam = 0.25 * (gc.K + 3.0) * (Wc[0] * Wc[0]) * ire;
  g.hsU = 0.5 * fma(g.U, g.U, (gc.K + 3.0) * g.hil);
  g.c4 = 4.0 * g.lam * g.lam * gc.inv_K3;
  g.q2 = 0.5 * fma(g.V, g.V, g.W * g.W);
  g.t1 = (gc.K + 2.0) * g.hil;
}

// first two half-space moments (times rho) of a Maxwellian: SGN = +1 -> u > 0, -1 -> u < 0
__device__ __forceinline__ void half_moments(const Maxw& g, double SGN, double& mh0, double& mh1) {
  const double sl = drsqrt(2.0 * g.hil), isl = 2.0 * g.hil * sl;               // sqrt(lam), 1/sqrt(lam)
  double ec, E;
  derfc_exp(-SGN * (sl * g.U), ec, E);                                         // erfc(-+ sqrt(lam) U), exp(-lam U^2)
  const double ex = 0.28209479177387814347 * E * isl;                          // 1/2 e^{-lam U^2}/sqrt(pi lam)
  mh0 = g.rho * (0.5 * ec);
  mh1 = g.U * mh0 + SGN * (g.rho * ex);
}

// <u^0..u^(N-1)> from the first two
template <int N>
__device__ __forceinline__ void mom_recur(double* m, double U, double hil) {
#pragma unroll
  for (int n = 0; n + 2 < N; n++) m[n + 2] = U * m[n + 1] + (n + 1) * hil * m[n];
}

// Micro slope in the primed basis from the PRIMED moments hp[alpha] = <(a.psi) psi'_alpha> per unit density (
// the standard GKS relation with V = W = 0).  With a.psi = a'.psi', the slope is carried as
//     a = (a'_0, a_1, a'_2/(2 lam), a'_3/(2 lam), a_4/2):
// the tangential components only ever appear divided by 2 lam (and then a'_2/(2 lam) = h'_2: no arithmetic at all), and
// a_4 only halved or times 1/(2 lam).
__device__ __forceinline__ void micro_slope_primed(const Maxw& g, const double* hp, double* a) {
  const double R1 = fma(-g.U, hp[0], hp[1]);
  const double R4h = fma(-g.hsU, hp[0], hp[4]);                  // (2 h'_4 - (U^2 + (K+3)/(2 lam)) h'_0)/2
  a[4] = g.c4 * fma(-g.U, R1, R4h);                               // a_4/2 = (4 lam^2/(K+3)) (R_4 - 2 U R_1)/2
  a[1] = fma(-2.0 * g.U, a[4], (2.0 * g.lam) * R1);
  a[2] = hp[2];
  a[3] = hp[3];
  a[0] = fma(-2.0 * g.hsU, a[4], fma(-g.U, a[1], hp[0]));
}

// the same from LABORATORY moments rho h[alpha] = rho <(a.psi) psi_alpha> (the slope of the conservative variables):
// psi' = B^-1 psi first, the factor 1/rho applied to the five primed moments
__device__ __forceinline__ void micro_slope_lab(const Maxw& g, const double* S, double* a) {
  double hp[5];
  const double s2 = fma(-g.V, S[0], S[2]), s3 = fma(-g.W, S[0], S[3]);
  const double s4 = fma(-g.q2, S[0], fma(-g.W, s3, fma(-g.V, s2, S[4])));
  hp[0] = S[0] * g.irho; hp[1] = S[1] * g.irho; hp[2] = s2 * g.irho; hp[3] = s3 * g.irho; hp[4] = s4 * g.irho;
  micro_slope_primed(g, hp, a);
}

// out (laboratory basis) (+)= B M (primed moments M); ACC = false overwrites (the first contribution to a sum)
template <bool ACC = true>
__device__ __forceinline__ void lab_acc(const Maxw& g, const double* M, double* out) {
  if (ACC) {
    out[0] += M[0];
    out[1] += M[1];
    out[2] = fma(g.V, M[0], out[2] + M[2]);
    out[3] = fma(g.W, M[0], out[3] + M[3]);
    out[4] = fma(g.q2, M[0], fma(g.W, M[3], fma(g.V, M[2], out[4] + M[4])));
  } else {
    out[0] = M[0];
    out[1] = M[1];
    out[2] = fma(g.V, M[0], M[2]);
    out[3] = fma(g.W, M[0], M[3]);
    out[4] = fma(g.q2, M[0], fma(g.W, M[3], fma(g.V, M[2], M[4])));
  }
}

// polynomial in u left by a primed slope after the (c_v, c_w, xi) integrals
struct SlopePoly { double p[3]; double cv, cw, e4; };      // weight 1: p0 + p1 u + p2 u^2; weights c_v, c_w: constants; e4 = a_4/(2 lam)

__device__ __forceinline__ void make_slope_poly(SlopePoly& P, const Maxw& g, const double* a) {
  P.p[0] = fma(a[4], g.t1, a[0]); P.p[1] = a[1]; P.p[2] = a[4];
  P.cv = a[2]; P.cw = a[3]; P.e4 = (2.0 * g.hil) * a[4];
}

template <int N>
__device__ __forceinline__ double pdot(const double* c, const double* mu) {
  double s = c[0] * mu[0];
#pragma unroll
  for (int k = 1; k < N; k++) s = fma(c[k], mu[k], s);
  return s;
}

// primed moments M[alpha] = <(a.psi) u^I psi'_alpha> with the u-moments m (full or half, possibly pre-scaled by rho)
template <int I>
__device__ __forceinline__ void apply_slope(const Maxw& g, const SlopePoly& P, const double* m, double* M) {
  const double d0 = pdot<3>(P.p, m + I), d1 = pdot<3>(P.p, m + I + 1), d2 = pdot<3>(P.p, m + I + 2);
  M[0] = d0; M[1] = d1; M[2] = P.cv * m[I]; M[3] = P.cw * m[I];
  M[4] = 0.5 * fma(g.t1, fma(P.e4, m[I], d0), d2);
}

// shift 0 (conserved moments, MQ) and shift 1 (flux moments, MF) together: the dots d1, d2 are shared
__device__ __forceinline__ void apply_slope_QF(const Maxw& g, const SlopePoly& P, const double* m, double* MQ, double* MF) {
  const double d0 = pdot<3>(P.p, m), d1 = pdot<3>(P.p, m + 1), d2 = pdot<3>(P.p, m + 2), d3 = pdot<3>(P.p, m + 3);
  MQ[0] = d0; MQ[1] = d1; MQ[2] = P.cv * m[0]; MQ[3] = P.cw * m[0];
  MQ[4] = 0.5 * fma(g.t1, fma(P.e4, m[0], d0), d2);
  MF[0] = d1; MF[1] = d2; MF[2] = P.cv * m[1]; MF[3] = P.cw * m[1];
  MF[4] = 0.5 * fma(g.t1, fma(P.e4, m[1], d1), d3);
}

// The spatial-divergence combination (a_x.psi) u + (a_y.psi) v + (a_z.psi) w of Eq. 5 after the (c_v, c_w, xi) integrals:
// with v = V + c_v, w = W + c_w and b = V a_y + W a_z it is u (a_x.psi) + (b.psi) + c_v (a_y.psi) + c_w (a_z.psi), which
// leaves a cubic e(u) for weight 1, quadratics dv(u), dw(u) for weights c_v, c_w and, for weight T,
// t1 e(u) + (g1 u + g0)/(2 lam).
struct DivPoly { double e[4], dv[3], dw[3], g0, g1; };

__device__ __forceinline__ void make_div_poly(DivPoly& D, const Maxw& g, const double* ax, const double* ay, const double* az) {
  // slopes as carried by micro_slope_primed: (a'_0, a_1, a'_2 h, a'_3 h, a_4/2), h = 1/(2 lam); b = V a_y + W a_z in the same form
  const double h = g.hil;
  double b[5];
#pragma unroll
  for (int k = 0; k < 5; k++) b[k] = fma(g.V, ay[k], g.W * az[k]);
  const double htr = ay[2] + az[3];                         // h (a'_y2 + a'_z3)
  D.e[0] = fma(b[4], g.t1, b[0]) + htr;
  D.e[1] = fma(ax[4], g.t1, ax[0]) + b[1];
  D.e[2] = ax[1] + b[4];
  D.e[3] = ax[4];
  const double t1p = fma(2.0, h, g.t1);                     // <c_v^2 T>/<c_v^2> = (K+4)/(2 lam)
  D.dv[0] = fma(h, fma(ay[4], t1p, ay[0]), b[2]); D.dv[1] = fma(h, ay[1], ax[2]); D.dv[2] = h * ay[4];
  D.dw[0] = fma(h, fma(az[4], t1p, az[0]), b[3]); D.dw[1] = fma(h, az[1], ax[3]); D.dw[2] = h * az[4];
  const double ht1x2 = 2.0 * (h * g.t1);
  D.g1 = ht1x2 * ax[4];
  D.g0 = fma(ht1x2, b[4], 2.0 * (h * htr));
}

template <int I>
__device__ __forceinline__ void apply_div(const Maxw& g, const DivPoly& D, const double* m, double* M) {
  const double e0 = pdot<4>(D.e, m + I), e1 = pdot<4>(D.e, m + I + 1), e2 = pdot<4>(D.e, m + I + 2);
  M[0] = e0; M[1] = e1; M[2] = pdot<3>(D.dv, m + I); M[3] = pdot<3>(D.dw, m + I);
  M[4] = 0.5 * fma(g.t1, e0, fma(D.g1, m[I + 1], fma(D.g0, m[I], e2)));
}

__device__ __forceinline__ void apply_div_QF(const Maxw& g, const DivPoly& D, const double* m, double* MQ, double* MF) {
  const double e0 = pdot<4>(D.e, m), e1 = pdot<4>(D.e, m + 1), e2 = pdot<4>(D.e, m + 2), e3 = pdot<4>(D.e, m + 3);
  MQ[0] = e0; MQ[1] = e1; MQ[2] = pdot<3>(D.dv, m); MQ[3] = pdot<3>(D.dw, m);
  MQ[4] = 0.5 * fma(g.t1, e0, fma(D.g1, m[1], fma(D.g0, m[0], e2)));
  MF[0] = e1; MF[1] = e2; MF[2] = pdot<3>(D.dv, m + 1); MF[3] = pdot<3>(D.dw, m + 1);
  MF[4] = 0.5 * fma(g.t1, e1, fma(D.g1, m[2], fma(D.g0, m[1], e3)));
}

// out[alpha] (laboratory basis) += <u^I psi_alpha> of the plain Maxwellian with (scaled) u-moments mu
template <int I, bool ACC = true>
__device__ __forceinline__ void add_plain(const Maxw& g, const double* mu, double* out) {
  const double et = fma(0.5, g.t1, g.q2);
  if (ACC) {
    out[0] += mu[I];
    out[1] += mu[I + 1];
    out[2] = fma(g.V, mu[I], out[2]);
    out[3] = fma(g.W, mu[I], out[3]);
    out[4] = fma(et, mu[I], fma(0.5, mu[I + 2], out[4]));
  } else {
    out[0] = mu[I];
    out[1] = mu[I + 1];
    out[2] = g.V * mu[I];
    out[3] = g.W * mu[I];
    out[4] = fma(et, mu[I], 0.5 * mu[I + 2]);
  }
}

struct Groups {        // moments of the groups of Eq. 5 that are shared between both sides (all times rho, laboratory basis)
  double W0[5];        // int_{u>0} g_l psi + int_{u<0} g_r psi   (= conserved moments of group 4)
  double dW0[3][5];    // kinetic-weighted slopes of W0 (reading F1)
  double G4F[5];
  double G5Q[5], G5F[5];
  double G6Q[5], G6F[5];
};

// one side (left state with the u > 0 half moments, right state with the u < 0 ones); ACC = false: the first side, which
// initialises the sums over both sides
template <bool ACC>
__device__ __forceinline__ void gks_side(const Maxw& g, double mh0, double mh1, const double (*S)[5], Groups& G, double* dQs) {
  double mu[6], mh[7];
  mu[0] = 1.0; mu[1] = g.U; mom_recur<6>(mu, g.U, g.hil);
  mh[0] = mh0; mh[1] = mh1;                      // half-space moments, pre-scaled by rho
  mom_recur<7>(mh, g.U, g.hil);
  add_plain<0, ACC>(g, mh, G.W0);
  add_plain<1, ACC>(g, mh, G.G4F);
  // micro slopes of the one-sided Maxwellian (primed basis); their half-space moments feed the slopes of W0
  double a[3][5], M[5], MF[5];
#pragma unroll
  for (int d = 0; d < 3; d++) {
    micro_slope_lab(g, S[d], a[d]);
    SlopePoly P; make_slope_poly(P, g, a[d]);
    apply_slope<0>(g, P, mh, M);
    lab_acc<ACC>(g, M, G.dW0[d]);
  }
  DivPoly D; make_div_poly(D, g, a[0], a[1], a[2]);
  // time slope from the compatibility condition <a_x u + a_y v + a_z w + A> = 0 (full velocity space): the primed
  // moments go straight into the primed solve
  apply_div<0>(g, D, mu, M);
#pragma unroll
  for (int v = 0; v < 5; v++) M[v] = -M[v];
  lab_acc<false>(g, M, dQs);
#pragma unroll
  for (int v = 0; v < 5; v++) dQs[v] *= g.rho;                                // d/dt of the one-sided Maxwellian's moments
  double A[5]; micro_slope_primed(g, M, A);
  apply_div_QF(g, D, mh, M, MF);
  lab_acc<ACC>(g, M, G.G5Q); lab_acc<ACC>(g, MF, G.G5F);
  SlopePoly PA; make_slope_poly(PA, g, A);
  apply_slope_QF(g, PA, mh, M, MF);
  lab_acc<ACC>(g, M, G.G6Q); lab_acc<ACC>(g, MF, G.G6F);
}

// Full solver in the face frame.  WL/WR[5] and SL/SR[3][5] are the rotated states and (n, t1, t2) slopes.
// Outputs (face frame): Fn, Ft, VL, DL, VR, DR, each [5].  STAGE2: only the time derivatives Ft, DL, DR (reading T4).
template <bool STAGE2>
__device__ __forceinline__ void gks_flux_local(const GasConst& gc, double dt, double idt, const double* WL, const double (*SL)[5],
                                               const double* WR, const double (*SR)[5],
                                               double* Fn, double* Ft, double* VL, double* DL, double* VR, double* DR) {
  Groups G;
  // scalars and half-space moments of both sides first: the two erfc/exp/sqrt/reciprocal chains are independent and
  // overlap in the FP64 pipe; the slopes of each side follow
  double pl, pr;
  {
    Maxw gl, gr;
    double hl0, hl1, hr0, hr1;
    maxw_scalars(gl, WL, gc); maxw_scalars(gr, WR, gc);
    half_moments(gl, 1.0, hl0, hl1); half_moments(gr, -1.0, hr0, hr1);
    pl = gl.rho * gl.hil; pr = gr.rho * gr.hil;
    gks_side<false>(gl, hl0, hl1, SL, G, DL);     // DL, DR hold the one-sided time derivatives for now
    gks_side<true>(gr, hr0, hr1, SR, G, DR);
  }
  // equilibrium state g0 and its slopes
  Maxw g0; maxw_scalars(g0, G.W0, gc);
  double mu[7];
  mu[0] = g0.rho; mu[1] = g0.rho * g0.U; mom_recur<7>(mu, g0.U, g0.hil);     // full moments times rho0
  double G1F[5], G2Q[5], G2F[5], G3F[5];
  add_plain<1, false>(g0, mu, G1F);
  {
    double a[3][5], h[5], MQ[5], MF[5];
#pragma unroll
    for (int d = 0; d < 3; d++) {
      micro_slope_lab(g0, G.dW0[d], a[d]);
    }
    DivPoly D; make_div_poly(D, g0, a[0], a[1], a[2]);
    apply_div_QF(g0, D, mu, MQ, MF);
    lab_acc<false>(g0, MQ, G2Q); lab_acc<false>(g0, MF, G2F);
    // Abar from <abar.u + Abar> = 0: its primed conserved moments are -MQ
#pragma unroll
    for (int v = 0; v < 5; v++) h[v] = -MQ[v] * g0.irho;
    double A[5]; micro_slope_primed(g0, h, A);
    SlopePoly PA; make_slope_poly(PA, g0, A);
    apply_slope<1>(g0, PA, mu, MF);
    lab_acc<false>(g0, MF, G3F);
  }
  // collision time
  // branch-free: an inviscid run (mu_ref = 0, T_ref possibly unset) evaluates the power law at T/T_ref = 1
  const double Trel = (gc.mu_ref > 0.0) ? g0.hil * gc.inv_T_ref : 1.0;
  const double visc = gc.mu_ref * dexp(gc.omega * dlog(Trel));                    // mu_ref (T/T_ref)^omega, T = p/rho
  const double tau_phys = visc * (2.0 * g0.lam * g0.irho);                        // mu / p0
  const double dpr = ddiv(fabs(pl - pr), fabs(pl + pr));
  const double tau = tau_phys + gc.c1 * dt + gc.c2 * dpr * dt;
  // Time-integrated coefficients of the six groups of Eq. 5 over [0, dt] and [0, dt/2], combined as
  // f^n = (4 fbar(dt/2) - fbar(dt))/dt and f_t^n = 4 (fbar(dt) - 2 fbar(dt/2))/dt^2, in closed form: with
  // E = exp(-dt/(2 tau)), x = 1 - E, y = tau/dt, w = 4 y x^2/dt, u = 4 y E x, z = y x (3 - E), s = E (2 - E)
  //   c_t = [ w, u - 2 tau w, 1 - tau w, -w, 2 tau w - u, tau w ]           (so the W0 coefficient c_t0 + c_t3 vanishes)
  //   c_n = [ 1 - z, tau (2z - s - 1), -tau (1 - z), z, tau (s - 2z), -tau z ]   (and c_n0 + c_n3 = 1)
  // which avoids the cancellation between the two time integrals.  tau = 0 (reading T2): f = g0 (1 + Abar t).
  // evaluated without a branch: with tau = 0 the exponential is replaced by its limit E = 0 and y = 0, which gives exactly the
  // coefficients of the tau = 0 solution, c_n = [1, 0, 0, 0, 0, 0] and c_t = [0, 0, 1, 0, 0, 0]
  double cn[6], ct[6];
  {
    const bool tz = (tau == 0.0);
    double E = dexp(-0.5 * dt * drcp(tz ? 1.0 : tau));
    E = tz ? 0.0 : E;
    const double x = 1.0 - E, y = tau * idt;
    const double w = 4.0 * (y * idt) * (x * x), u = 4.0 * y * (E * x), tw = tau * w;
    ct[0] = w; ct[1] = u - 2.0 * tw; ct[2] = 1.0 - tw; ct[3] = -w; ct[4] = -ct[1]; ct[5] = tw;
    if (!STAGE2) {
      const double z = y * x * (3.0 - E), sE = E * (2.0 - E);
      cn[0] = 1.0 - z; cn[1] = tau * (2.0 * z - sE - 1.0); cn[2] = -tau * cn[0]; cn[3] = z; cn[4] = tau * (sE - 2.0 * z); cn[5] = -tau * z;
    }
  }
  double Qn[5], Qt[5];
  const double cnG = cn[1] - cn[2], ctG = ct[1] - ct[2];       // the conserved moments of group 3 are minus those of group 2
#pragma unroll
  for (int v = 0; v < 5; v++) {
    Qt[v] = ctG * G2Q[v] + ct[4] * G.G5Q[v] + ct[5] * G.G6Q[v];
    Ft[v] = ct[0] * G1F[v] + ct[1] * G2F[v] + ct[2] * G3F[v] + ct[3] * G.G4F[v] + ct[4] * G.G5F[v] + ct[5] * G.G6F[v];
    if (!STAGE2) {
      Qn[v] = G.W0[v] + cnG * G2Q[v] + cn[4] * G.G5Q[v] + cn[5] * G.G6Q[v];
      Fn[v] = cn[0] * G1F[v] + cn[1] * G2F[v] + cn[2] * G3F[v] + cn[3] * G.G4F[v] + cn[4] * G.G5F[v] + cn[5] * G.G6F[v];
    }
  }
  // Prandtl number fix (reading F2): energy flux += (1/Pr - 1) q, q the heat flux of the same distribution
  {
    const double U0 = g0.U, V0 = g0.V, W0 = g0.W, ke = 0.5 * (U0 * U0 + V0 * V0 + W0 * W0);
    const double qt = Ft[4] - U0 * Qt[4] - U0 * (Ft[1] - U0 * Qt[1]) - V0 * (Ft[2] - U0 * Qt[2]) - W0 * (Ft[3] - U0 * Qt[3]) + ke * (Ft[0] - U0 * Qt[0]);
    Ft[4] += gc.Pr_fix * qt;
    if (!STAGE2) {
      const double qn = Fn[4] - U0 * Qn[4] - U0 * (Fn[1] - U0 * Qn[1]) - V0 * (Fn[2] - U0 * Qn[2]) - W0 * (Fn[3] - U0 * Qn[3]) + ke * (Fn[0] - U0 * Qn[0]);
      Fn[4] += gc.Pr_fix * qn;
    }
  }
  // one-sided interface values (reading F3): weight exp(-dt/tau0), tau0 = c2 |dp|/|sum p| dt
  // (the weight is < 1e-300 when c2 dpr < 1/700: skipped there, which changes nothing above the 300th digit)
  double wgt = 0.0;
  if (gc.c2 * dpr > 1.0 / 700.0) wgt = dexp(-drcp(gc.c2 * dpr));
  const double om = 1.0 - wgt;
#pragma unroll
  for (int v = 0; v < 5; v++) {
    DL[v] = om * Qt[v] + wgt * DL[v];
    DR[v] = om * Qt[v] + wgt * DR[v];
    if (!STAGE2) { VL[v] = om * Qn[v] + wgt * WL[v]; VR[v] = om * Qn[v] + wgt * WR[v]; }
  }
}

}  // namespace cgks
