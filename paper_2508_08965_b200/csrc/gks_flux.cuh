// gks_flux.cuh -- gas-kinetic interface solver at one face Gauss point, in the face frame (n, t1, t2).
//
// Computes, from the left/right reconstructed states and slopes, the second-order integral solution of the BGK
// equation (Eq. 5), its time integrals over [0,dt] and [0,dt/2] and the time linearisation
// (Eq. 6-7): F^n, F_t^n, and the one-sided interface values Q^{l,r}, Q_t^{l,r}.
// Collision time per PAPER.md:344-352.  Readings of the paper's gaps: DESIGN.md section 3 (F1-F3, T1-T2).
//
// Formulation (differs from the CPU oracle on purpose).  With psi = (1, u, v, w, (u^2+T2)/2),
// T2 = v^2 + w^2 + xi^2, every term of Eq. 5 is a moment <(a.psi) u^I v^J w^K psi_alpha> of a Maxwellian.  The
// tangential velocities and xi are integrated out FIRST with three small tables per Maxwellian
//     P0[q][r] = <v^q w^r>,  P2[q][r] = <T2 v^q w^r>,  P4[q][r] = <T2^2 v^q w^r>,
// which leaves, per weight phi in {1, v, w, T2}, a polynomial in u ("UPoly"); the spatial-divergence combination
// a_x u + a_y v + a_z w of Eq. 5 is summed as ONE cubic per weight before any u-moment is applied, and the same cubic
// serves the compatibility condition (full u-moments), the conserved moments (shift 0) and the flux moments (shift 1).
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

// Maxwellian per unit density with the tangential tables
struct Maxw {
  double rho, irho, U, V, W, lam, hil;   // hil = 1/(2 lam) = p/rho
  double s;                              // U^2+V^2+W^2 + (K+3)/(2 lam)
  double c4;                             // 4 lam^2/(K+3)
  double P0[4][4];                       // q + r <= 3 used
  double P2[3][3];                       // q + r <= 2 used
  double P4[2][2];                       // q + r <= 1 used
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
  const double k3h = (gc.K + 3.0) * g.hil;
  g.s = g.U * g.U + g.V * g.V + g.W * g.W + k3h;
  g.c4 = 4.0 * g.lam * g.lam * gc.inv_K3;
}

__device__ __forceinline__ void maxw_tables(Maxw& g, const GasConst& gc) {
  double mv[6], mw[6];
  mv[0] = 1.0; mv[1] = g.V; mw[0] = 1.0; mw[1] = g.W;
#pragma unroll
  for (int n = 0; n < 4; n++) { mv[n + 2] = g.V * mv[n + 1] + (n + 1) * g.hil * mv[n]; mw[n + 2] = g.W * mw[n + 1] + (n + 1) * g.hil * mw[n]; }
  const double x2 = gc.K * g.hil, x4 = gc.K * (gc.K + 2.0) * g.hil * g.hil;
#pragma unroll
  for (int q = 0; q < 4; q++)
#pragma unroll
    for (int r = 0; r + q < 4; r++) g.P0[q][r] = mv[q] * mw[r];
#pragma unroll
  for (int q = 0; q < 3; q++)
#pragma unroll
    for (int r = 0; r + q < 3; r++) g.P2[q][r] = mv[q + 2] * mw[r] + mv[q] * mw[r + 2] + x2 * g.P0[q][r];
#pragma unroll
  for (int q = 0; q < 2; q++)
#pragma unroll
    for (int r = 0; r + q < 2; r++)
      g.P4[q][r] = mv[q + 4] * mw[r] + mv[q] * mw[r + 4] + x4 * g.P0[q][r]
                 + 2.0 * (mv[q + 2] * mw[r + 2] + x2 * (mv[q + 2] * mw[r] + mv[q] * mw[r + 2]));
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

// solves <(a.psi) psi> = h for the micro slope a (standard GKS relation)
__device__ __forceinline__ void micro_slope(const Maxw& g, const double* h, double* a) {
  const double R1 = h[1] - g.U * h[0], R2 = h[2] - g.V * h[0], R3 = h[3] - g.W * h[0];
  const double R4 = 2.0 * h[4] - g.s * h[0];
  const double tl = 2.0 * g.lam;
  a[4] = g.c4 * (R4 - 2.0 * (g.U * R1 + g.V * R2 + g.W * R3));
  a[1] = tl * R1 - g.U * a[4];
  a[2] = tl * R2 - g.V * a[4];
  a[3] = tl * R3 - g.W * a[4];
  a[0] = h[0] - g.U * a[1] - g.V * a[2] - g.W * a[3] - 0.5 * a[4] * g.s;
}

// polynomial in u per weight phi = 0:1, 1:v, 2:w, 3:T2 of  <(a.psi) phi v^J w^K>_{v,w,xi} = c[phi][0] + c[phi][1] u + c[phi][2] u^2
struct UPoly { double c[4][3]; };

template <int J, int Kw>
__device__ __forceinline__ void make_upoly(UPoly& p, const Maxw& g, const double* a) {
  const double h4 = 0.5 * a[4];
  // phi = 1
  p.c[0][0] = a[0] * g.P0[J][Kw] + a[2] * g.P0[J + 1][Kw] + a[3] * g.P0[J][Kw + 1] + h4 * g.P2[J][Kw];
  p.c[0][1] = a[1] * g.P0[J][Kw];               p.c[0][2] = h4 * g.P0[J][Kw];
  // phi = v
  p.c[1][0] = a[0] * g.P0[J + 1][Kw] + a[2] * g.P0[J + 2][Kw] + a[3] * g.P0[J + 1][Kw + 1] + h4 * g.P2[J + 1][Kw];
  p.c[1][1] = a[1] * g.P0[J + 1][Kw];           p.c[1][2] = h4 * g.P0[J + 1][Kw];
  // phi = w
  p.c[2][0] = a[0] * g.P0[J][Kw + 1] + a[2] * g.P0[J + 1][Kw + 1] + a[3] * g.P0[J][Kw + 2] + h4 * g.P2[J][Kw + 1];
  p.c[2][1] = a[1] * g.P0[J][Kw + 1];           p.c[2][2] = h4 * g.P0[J][Kw + 1];
  // phi = T2
  p.c[3][0] = a[0] * g.P2[J][Kw] + a[2] * g.P2[J + 1][Kw] + a[3] * g.P2[J][Kw + 1] + h4 * g.P4[J][Kw];
  p.c[3][1] = a[1] * g.P2[J][Kw];               p.c[3][2] = h4 * g.P2[J][Kw];
}

// cubic per weight: u * Px + Py + Pz  (the a_x u + a_y v + a_z w combination of Eq. 5)
struct UCubic { double d[4][4]; };

__device__ __forceinline__ void make_cubic(UCubic& D, const UPoly& px, const UPoly& py, const UPoly& pz) {
#pragma unroll
  for (int f = 0; f < 4; f++) {
    D.d[f][0] = py.c[f][0] + pz.c[f][0];
    D.d[f][1] = px.c[f][0] + (py.c[f][1] + pz.c[f][1]);
    D.d[f][2] = px.c[f][1] + (py.c[f][2] + pz.c[f][2]);
    D.d[f][3] = px.c[f][2];
  }
}

template <int N>
__device__ __forceinline__ double pdot(const double* c, const double* mu) {
  double s = c[0] * mu[0];
#pragma unroll
  for (int k = 1; k < N; k++) s = fma(c[k], mu[k], s);
  return s;
}

// init + sum_k c[k] mu[k] as one FMA chain
template <int N>
__device__ __forceinline__ double pdot_acc(const double* c, const double* mu, double init) {
#pragma unroll
  for (int k = 0; k < N; k++) init = fma(c[k], mu[k], init);
  return init;
}

// out[alpha] (+)= < poly u^I psi_alpha > with u-moments mu (full or half, possibly pre-scaled by rho); N = 3 or 4 coefficients.
// Accumulating variants continue the FMA chain from the accumulator (no separate add).
template <int N, int I, bool ACC>
__device__ __forceinline__ void apply_poly(const double (*c)[N], const double* mu, double* out) {
  const double r4 = pdot_acc<N>(c[3], mu + I, pdot<N>(c[0], mu + I + 2));      // <u^2 .> + <T2 .>
  if (ACC) {
    out[0] = pdot_acc<N>(c[0], mu + I, out[0]); out[1] = pdot_acc<N>(c[0], mu + I + 1, out[1]);
    out[2] = pdot_acc<N>(c[1], mu + I, out[2]); out[3] = pdot_acc<N>(c[2], mu + I, out[3]);
    out[4] = fma(0.5, r4, out[4]);
  } else {
    out[0] = pdot<N>(c[0], mu + I); out[1] = pdot<N>(c[0], mu + I + 1); out[2] = pdot<N>(c[1], mu + I); out[3] = pdot<N>(c[2], mu + I);
    out[4] = 0.5 * r4;
  }
}

// moments of shift 0 (conserved, outQ) and shift 1 (flux, outF) together: the phi = 1 moments are shared
template <int N, bool ACC>
__device__ __forceinline__ void apply_poly_QF(const double (*c)[N], const double* mu, double* outQ, double* outF) {
  const double e1 = pdot<N>(c[0], mu + 1), e2 = pdot<N>(c[0], mu + 2);
  const double q4 = pdot_acc<N>(c[3], mu, e2);                                   // <u^2 .> + <T2 .>, shift 0
  const double f4 = pdot_acc<N>(c[3], mu + 1, pdot<N>(c[0], mu + 3));            // shift 1
  if (ACC) {
    outQ[0] = pdot_acc<N>(c[0], mu, outQ[0]); outQ[1] += e1;
    outQ[2] = pdot_acc<N>(c[1], mu, outQ[2]); outQ[3] = pdot_acc<N>(c[2], mu, outQ[3]); outQ[4] = fma(0.5, q4, outQ[4]);
    outF[0] += e1; outF[1] += e2;
    outF[2] = pdot_acc<N>(c[1], mu + 1, outF[2]); outF[3] = pdot_acc<N>(c[2], mu + 1, outF[3]); outF[4] = fma(0.5, f4, outF[4]);
  } else {
    outQ[0] = pdot<N>(c[0], mu); outQ[1] = e1; outQ[2] = pdot<N>(c[1], mu); outQ[3] = pdot<N>(c[2], mu); outQ[4] = 0.5 * q4;
    outF[0] = e1; outF[1] = e2; outF[2] = pdot<N>(c[1], mu + 1); outF[3] = pdot<N>(c[2], mu + 1); outF[4] = 0.5 * f4;
  }
}

// out[alpha] += <u^I psi_alpha> of the plain Maxwellian with (scaled) u-moments mu
template <int I>
__device__ __forceinline__ void add_plain(const Maxw& g, const double* mu, double* out) {
  out[0] += mu[I];
  out[1] += mu[I + 1];
  out[2] += g.V * mu[I];
  out[3] += g.W * mu[I];
  out[4] += 0.5 * (mu[I + 2] + g.P2[0][0] * mu[I]);
}

struct Groups {        // moments of the groups of Eq. 5 that are shared between both sides (all times rho)
  double W0[5];        // int_{u>0} g_l psi + int_{u<0} g_r psi   (= conserved moments of group 4)
  double dW0[3][5];    // kinetic-weighted slopes of W0 (reading F1)
  double G4F[5];
  double G5Q[5], G5F[5];
  double G6Q[5], G6F[5];
};

// one side (SGN = +1: left state, u > 0; SGN = -1: right state, u < 0)
__device__ __forceinline__ void gks_side(Maxw& g, double mh0, double mh1, const GasConst& gc, const double (*S)[5], Groups& G,
                                         double* dQs) {
  maxw_tables(g, gc);
  double mu[6], mh[7];
  mu[0] = 1.0; mu[1] = g.U; mom_recur<6>(mu, g.U, g.hil);
  mh[0] = mh0; mh[1] = mh1;                      // half-space moments, pre-scaled by rho
  mom_recur<7>(mh, g.U, g.hil);
  add_plain<0>(g, mh, G.W0);
  add_plain<1>(g, mh, G.G4F);
  // micro slopes of the one-sided Maxwellian; divergence cubic
  double a[5], h[5];
  UCubic D;
  {
    UPoly px, py, pz;
#pragma unroll
    for (int v = 0; v < 5; v++) h[v] = S[0][v] * g.irho;
    micro_slope(g, h, a); make_upoly<0, 0>(px, g, a);
    apply_poly<3, 0, true>(px.c, mh, G.dW0[0]);
#pragma unroll
    for (int v = 0; v < 5; v++) h[v] = S[1][v] * g.irho;
    micro_slope(g, h, a); make_upoly<0, 0>(py, g, a);
    apply_poly<3, 0, true>(py.c, mh, G.dW0[1]);
    make_upoly<1, 0>(py, g, a);
#pragma unroll
    for (int v = 0; v < 5; v++) h[v] = S[2][v] * g.irho;
    micro_slope(g, h, a); make_upoly<0, 0>(pz, g, a);
    apply_poly<3, 0, true>(pz.c, mh, G.dW0[2]);
    make_upoly<0, 1>(pz, g, a);
    make_cubic(D, px, py, pz);
  }
  // time slope from the compatibility condition <a_x u + a_y v + a_z w + A> = 0 (full velocity space)
  apply_poly<4, 0, false>(D.d, mu, h);
#pragma unroll
  for (int v = 0; v < 5; v++) { h[v] = -h[v]; dQs[v] = g.rho * h[v]; }     // d/dt of the one-sided Maxwellian's moments
  apply_poly_QF<4, true>(D.d, mh, G.G5Q, G.G5F);
  micro_slope(g, h, a);
  UPoly pa; make_upoly<0, 0>(pa, g, a);
  apply_poly_QF<3, true>(pa.c, mh, G.G6Q, G.G6F);
}

// time-integrated coefficients of the six groups of Eq. 5 over [0,T]
__device__ __forceinline__ void time_coef(double T, double tau, double E, double* cf) {
  const double ome = 1.0 - E;
  cf[0] = T - tau * ome;
  cf[1] = 2.0 * tau * tau * ome - tau * T * (1.0 + E);
  cf[2] = 0.5 * T * T - tau * T + tau * tau * ome;
  cf[3] = tau * ome;
  cf[4] = tau * T * E - 2.0 * tau * tau * ome;
  cf[5] = -tau * tau * ome;
}

// Full solver in the face frame.  WL/WR[5] and SL/SR[3][5] are the rotated states and (n, t1, t2) slopes.
// Outputs (face frame): Fn, Ft, VL, DL, VR, DR, each [5].  STAGE2: only the time derivatives Ft, DL, DR (reading T4).
template <bool STAGE2>
__device__ __forceinline__ void gks_flux_local(const GasConst& gc, double dt, double idt, const double* WL, const double (*SL)[5],
                                               const double* WR, const double (*SR)[5],
                                               double* Fn, double* Ft, double* VL, double* DL, double* VR, double* DR) {
  Groups G;
#pragma unroll
  for (int v = 0; v < 5; v++) {
    G.W0[v] = 0; G.G4F[v] = 0; G.G5Q[v] = 0; G.G5F[v] = 0; G.G6Q[v] = 0; G.G6F[v] = 0;
    G.dW0[0][v] = 0; G.dW0[1][v] = 0; G.dW0[2][v] = 0;
  }
  // scalars and half-space moments of both sides first: the two erfc/exp/sqrt/reciprocal chains are independent and
  // overlap in the FP64 pipe; the tables and slopes of each side follow
  double pl, pr;
  {
    Maxw gl, gr;
    double hl0, hl1, hr0, hr1;
    maxw_scalars(gl, WL, gc); maxw_scalars(gr, WR, gc);
    half_moments(gl, 1.0, hl0, hl1); half_moments(gr, -1.0, hr0, hr1);
    pl = gl.rho * gl.hil; pr = gr.rho * gr.hil;
    gks_side(gl, hl0, hl1, gc, SL, G, DL);     // DL, DR hold the one-sided time derivatives for now
    gks_side(gr, hr0, hr1, gc, SR, G, DR);
  }
  // equilibrium state g0 and its slopes
  Maxw g0; maxw_scalars(g0, G.W0, gc); maxw_tables(g0, gc);
  double mu[7];
  mu[0] = g0.rho; mu[1] = g0.rho * g0.U; mom_recur<7>(mu, g0.U, g0.hil);     // full moments times rho0
  double G1F[5] = { 0, 0, 0, 0, 0 }, G2Q[5], G2F[5], G3F[5];
  add_plain<1>(g0, mu, G1F);
  double a[5], h[5];
  {
    UCubic D; UPoly px, py, pz;
#pragma unroll
    for (int v = 0; v < 5; v++) h[v] = G.dW0[0][v] * g0.irho;
    micro_slope(g0, h, a); make_upoly<0, 0>(px, g0, a);
#pragma unroll
    for (int v = 0; v < 5; v++) h[v] = G.dW0[1][v] * g0.irho;
    micro_slope(g0, h, a); make_upoly<1, 0>(py, g0, a);
#pragma unroll
    for (int v = 0; v < 5; v++) h[v] = G.dW0[2][v] * g0.irho;
    micro_slope(g0, h, a); make_upoly<0, 1>(pz, g0, a);
    make_cubic(D, px, py, pz);
    apply_poly_QF<4, false>(D.d, mu, G2Q, G2F);
  }
  // Abar from <abar.u + Abar> = 0; its conserved moments are -G2Q
#pragma unroll
  for (int v = 0; v < 5; v++) h[v] = -G2Q[v] * g0.irho;
  micro_slope(g0, h, a);
  { UPoly pa; make_upoly<0, 0>(pa, g0, a); apply_poly<3, 1, false>(pa.c, mu, G3F); }
  // collision time
  double tau_phys = 0.0;
  if (gc.mu_ref > 0.0) {
    double visc = gc.mu_ref;
    if (gc.omega != 0.0) visc *= dexp(gc.omega * log(g0.hil * gc.inv_T_ref));      // (T/T_ref)^omega, T = p/rho
    tau_phys = visc * (2.0 * g0.lam * g0.irho);                                    // mu / p0
  }
  const double dpr = ddiv(fabs(pl - pr), fabs(pl + pr));
  const double tau = tau_phys + gc.c1 * dt + gc.c2 * dpr * dt;
  double c1[6], c2[6];
  if (tau == 0.0) {     // reading T2: f = g0 (1 + Abar t)
    c1[0] = dt; c1[1] = 0; c1[2] = 0.5 * dt * dt; c1[3] = c1[4] = c1[5] = 0;
    c2[0] = 0.5 * dt; c2[1] = 0; c2[2] = 0.125 * dt * dt; c2[3] = c2[4] = c2[5] = 0;
  } else {
    const double E2 = dexp(-0.5 * dt * drcp(tau)), E1 = E2 * E2;
    time_coef(dt, tau, E1, c1); time_coef(0.5 * dt, tau, E2, c2);
  }
  // f^n = (4 fbar(dt/2) - fbar(dt))/dt,  f_t^n = 4 (fbar(dt) - 2 fbar(dt/2))/dt^2
  double cn[6], ct[6];
#pragma unroll
  for (int q = 0; q < 6; q++) { cn[q] = (4.0 * c2[q] - c1[q]) * idt; ct[q] = 4.0 * (c1[q] - 2.0 * c2[q]) * idt * idt; }
  double Qn[5], Qt[5];
  const double cnW = cn[0] + cn[3], cnG = cn[1] - cn[2], ctW = ct[0] + ct[3], ctG = ct[1] - ct[2];
#pragma unroll
  for (int v = 0; v < 5; v++) {
    Qt[v] = ctW * G.W0[v] + ctG * G2Q[v] + ct[4] * G.G5Q[v] + ct[5] * G.G6Q[v];
    Ft[v] = ct[0] * G1F[v] + ct[1] * G2F[v] + ct[2] * G3F[v] + ct[3] * G.G4F[v] + ct[4] * G.G5F[v] + ct[5] * G.G6F[v];
    if (!STAGE2) {
      Qn[v] = cnW * G.W0[v] + cnG * G2Q[v] + cn[4] * G.G5Q[v] + cn[5] * G.G6Q[v];
      Fn[v] = cn[0] * G1F[v] + cn[1] * G2F[v] + cn[2] * G3F[v] + cn[3] * G.G4F[v] + cn[4] * G.G5F[v] + cn[5] * G.G6F[v];
    }
  }
  // Prandtl number fix (reading F2): energy flux += (1/Pr - 1) q, q the heat flux of the same distribution
  if (gc.Pr_fix != 0.0) {
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
