// gks_flux.cuh -- gas-kinetic interface solver at one face Gauss point, in the face frame (n, t1, t2).
//
// Computes, from the left/right reconstructed states and slopes, the second-order integral solution of the BGK
// equation (Eq. 5), its time integrals over [0,dt] and [0,dt/2] and the time linearisation
// (Eq. 6-7): F^n, F_t^n, and the one-sided interface values Q^{l,r}, Q_t^{l,r}.
// Collision time per PAPER.md:344-352.  Readings of the paper's gaps: DESIGN.md section 3 (F1-F3, T1-T2).
//
// Formulation (differs from the CPU oracle on purpose): every moment <(a.psi) u^p v^q w^r psi_alpha> is evaluated
// by first integrating v, w and xi out, which leaves a quadratic c0 + c1 u + c2 u^2 per (q, r, xi-power); the
// u-moments (full or half space, any shift p) are applied last, so one set of "triples" per slope vector serves the
// compatibility condition (full space), the conserved moments (shift p) and the flux moments (shift p+1).
#pragma once
#include <math.h>

namespace cgks {

struct GasConst {
  double K;            // internal degrees of freedom N = (5-3 gamma)/(gamma-1)
  double Pr_fix;       // 1/Pr - 1, 0 when inviscid
  double mu_ref, omega, T_ref;
  double c1, c2;       // tau = mu/p + c1 dt + c2 |pl-pr|/|pl+pr| dt
};

// solves <(a.psi) psi> = h for the micro slope a, Maxwellian (U,V,W,lam) per unit density
__device__ __forceinline__ void micro_slope(const double* h, double U, double V, double W, double lam, double K, double* a) {
  const double s = U * U + V * V + W * W + (K + 3.0) / (2.0 * lam);
  const double R1 = h[1] - U * h[0], R2 = h[2] - V * h[0], R3 = h[3] - W * h[0];
  const double R4 = 2.0 * h[4] - s * h[0];
  a[4] = 4.0 * lam * lam / (K + 3.0) * (R4 - 2.0 * U * R1 - 2.0 * V * R2 - 2.0 * W * R3);
  a[1] = 2.0 * lam * R1 - U * a[4];
  a[2] = 2.0 * lam * R2 - V * a[4];
  a[3] = 2.0 * lam * R3 - W * a[4];
  a[0] = h[0] - U * a[1] - V * a[2] - W * a[3] - 0.5 * a[4] * s;
}

// <x^0..x^(N-1)> of a 1-D Maxwellian from the first two
template <int N>
__device__ __forceinline__ void mom_recur(double* m, double U, double half_inv_lam) {
#pragma unroll
  for (int n = 0; n + 2 < N; n++) m[n + 2] = U * m[n + 1] + (n + 1) * half_inv_lam * m[n];
}

struct Maxw {
  double rho, U, V, W, lam, p;
  double mv[6], mw[6];   // full moments of v and w
  double x2, x4;         // <xi^2>, <xi^4>
};

__device__ __forceinline__ void maxw_init(Maxw& g, const double* Wc, double K) {
  g.rho = Wc[0];
  const double inv = 1.0 / Wc[0];
  g.U = Wc[1] * inv; g.V = Wc[2] * inv; g.W = Wc[3] * inv;
  const double e = Wc[4] - 0.5 * (Wc[1] * Wc[1] + Wc[2] * Wc[2] + Wc[3] * Wc[3]) * inv;
  g.lam = (K + 3.0) * Wc[0] / (4.0 * e);
  g.p = g.rho / (2.0 * g.lam);
  const double hil = 0.5 / g.lam;
  g.mv[0] = 1.0; g.mv[1] = g.V; mom_recur<6>(g.mv, g.V, hil);
  g.mw[0] = 1.0; g.mw[1] = g.W; mom_recur<6>(g.mw, g.W, hil);
  g.x2 = K * hil; g.x4 = K * (K + 2.0) * hil * hil;
}

// six triples (c0,c1,c2) of the slope a for tangential powers (J,Kw):
//   0:(J,Kw,xi^0) 1:(J+1,Kw) 2:(J,Kw+1) 3:(J+2,Kw) 4:(J,Kw+2) 5:(J,Kw,xi^2)
struct Trip { double c0[6], c1[6], c2[6]; };

__device__ __forceinline__ double nprod(const Maxw& g, int q, int r, int s) {
  const double x = (s == 0) ? 1.0 : ((s == 1) ? g.x2 : g.x4);
  return g.mv[q] * g.mw[r] * x;
}

template <int J, int Kw>
__device__ __forceinline__ void make_trip(Trip& t, const Maxw& g, const double* a) {
  const int Q[6] = { J, J + 1, J, J + 2, J, J }, R[6] = { Kw, Kw, Kw + 1, Kw, Kw + 2, Kw }, S[6] = { 0, 0, 0, 0, 0, 1 };
  const double ha4 = 0.5 * a[4];
#pragma unroll
  for (int c = 0; c < 6; c++) {
    const int q = Q[c], r = R[c], s = S[c];
    const double n0 = nprod(g, q, r, s);
    t.c0[c] = a[0] * n0 + a[2] * nprod(g, q + 1, r, s) + a[3] * nprod(g, q, r + 1, s)
            + ha4 * (nprod(g, q + 2, r, s) + nprod(g, q, r + 2, s) + nprod(g, q, r, s + 1));
    t.c1[c] = a[1] * n0;
    t.c2[c] = ha4 * n0;
  }
}

__device__ __forceinline__ double tmom(const Trip& t, int c, const double* mu, int p) {
  return t.c0[c] * mu[p] + t.c1[c] * mu[p + 1] + t.c2[c] * mu[p + 2];
}

// out[alpha] (+)= scale * <(a.psi) u^I v^J w^Kw psi_alpha>, u-moments mu (full or half)
template <int I, bool ACC>
__device__ __forceinline__ void apply_trip(const Trip& t, const double* mu, double scale, double* out) {
  const double r0 = tmom(t, 0, mu, I), r1 = tmom(t, 0, mu, I + 1), r2 = tmom(t, 1, mu, I), r3 = tmom(t, 2, mu, I);
  const double r4 = 0.5 * (tmom(t, 0, mu, I + 2) + tmom(t, 3, mu, I) + tmom(t, 4, mu, I) + tmom(t, 5, mu, I));
  if (ACC) { out[0] += scale * r0; out[1] += scale * r1; out[2] += scale * r2; out[3] += scale * r3; out[4] += scale * r4; }
  else { out[0] = scale * r0; out[1] = scale * r1; out[2] = scale * r2; out[3] = scale * r3; out[4] = scale * r4; }
}

// out[alpha] += scale * <u^I psi_alpha> for the plain Maxwellian (a = (1,0,0,0,0))
template <int I>
__device__ __forceinline__ void add_plain(const Maxw& g, const double* mu, double scale, double* out) {
  const double tw = g.mv[2] + g.mw[2] + g.x2;
  out[0] += scale * mu[I];
  out[1] += scale * mu[I + 1];
  out[2] += scale * (g.V * mu[I]);
  out[3] += scale * (g.W * mu[I]);
  out[4] += scale * (0.5 * (mu[I + 2] + tw * mu[I]));
}

struct Groups {        // moments of the groups of Eq. 5 that are shared between both sides
  double W0[5];        // int_{u>0} g_l psi + int_{u<0} g_r psi   (= conserved moments of group 4)
  double dW0[3][5];    // kinetic-weighted slopes of W0 (reading F1)
  double G4F[5];
  double G5Q[5], G5F[5];
  double G6Q[5], G6F[5];
};

// one side (SGN = +1: left state, u > 0; SGN = -1: right state, u < 0)
template <int SGN>
__device__ __forceinline__ void gks_side(const GasConst& gc, const double* Wc, const double (*S)[5], Groups& G,
                                         double* dQs, double& p_side) {
  Maxw g; maxw_init(g, Wc, gc.K);
  p_side = g.p;
  const double hil = 0.5 / g.lam;
  double mu[7], mh[7];
  mu[0] = 1.0; mu[1] = g.U; mom_recur<7>(mu, g.U, hil);
  const double sl = sqrt(g.lam);
  const double ex = 0.5 * exp(-g.lam * g.U * g.U) / (sl * 1.7724538509055160273);   // 1/2 e^{-lam U^2}/sqrt(pi lam)
  mh[0] = 0.5 * erfc(-SGN * sl * g.U);
  mh[1] = g.U * mh[0] + SGN * ex;
  mom_recur<7>(mh, g.U, hil);
  // micro slopes of the one-sided Maxwellian
  double a[3][5], h[5];
  const double irho = 1.0 / g.rho;
#pragma unroll
  for (int d = 0; d < 3; d++) {
#pragma unroll
    for (int v = 0; v < 5; v++) h[v] = S[d][v] * irho;
    micro_slope(h, g.U, g.V, g.W, g.lam, gc.K, a[d]);
  }
  Trip t0, t1, t1v, t2, t2w;
  make_trip<0, 0>(t0, g, a[0]);
  make_trip<0, 0>(t1, g, a[1]); make_trip<1, 0>(t1v, g, a[1]);
  make_trip<0, 0>(t2, g, a[2]); make_trip<0, 1>(t2w, g, a[2]);
  // time slope from the compatibility condition <a1 u + a2 v + a3 w + A> = 0 (full velocity space)
  apply_trip<1, false>(t0, mu, -1.0, h); apply_trip<0, true>(t1v, mu, -1.0, h); apply_trip<0, true>(t2w, mu, -1.0, h);
#pragma unroll
  for (int v = 0; v < 5; v++) dQs[v] = g.rho * h[v];       // d/dt of the one-sided Maxwellian's moments
  double A[5]; micro_slope(h, g.U, g.V, g.W, g.lam, gc.K, A);
  Trip tA; make_trip<0, 0>(tA, g, A);
  // half-space contributions
  add_plain<0>(g, mh, g.rho, G.W0);
  add_plain<1>(g, mh, g.rho, G.G4F);
  apply_trip<0, true>(t0, mh, g.rho, G.dW0[0]); apply_trip<0, true>(t1, mh, g.rho, G.dW0[1]); apply_trip<0, true>(t2, mh, g.rho, G.dW0[2]);
  apply_trip<1, true>(t0, mh, g.rho, G.G5Q); apply_trip<0, true>(t1v, mh, g.rho, G.G5Q); apply_trip<0, true>(t2w, mh, g.rho, G.G5Q);
  apply_trip<2, true>(t0, mh, g.rho, G.G5F); apply_trip<1, true>(t1v, mh, g.rho, G.G5F); apply_trip<1, true>(t2w, mh, g.rho, G.G5F);
  apply_trip<0, true>(tA, mh, g.rho, G.G6Q); apply_trip<1, true>(tA, mh, g.rho, G.G6F);
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
// Outputs (face frame): Fn, Ft, VL, DL, VR, DR, each [5].
__device__ __forceinline__ void gks_flux_local(const GasConst& gc, double dt, const double* WL, const double (*SL)[5],
                                               const double* WR, const double (*SR)[5],
                                               double* Fn, double* Ft, double* VL, double* DL, double* VR, double* DR) {
  Groups G;
#pragma unroll
  for (int v = 0; v < 5; v++) {
    G.W0[v] = 0; G.G4F[v] = 0; G.G5Q[v] = 0; G.G5F[v] = 0; G.G6Q[v] = 0; G.G6F[v] = 0;
    G.dW0[0][v] = 0; G.dW0[1][v] = 0; G.dW0[2][v] = 0;
  }
  double pl, pr;
  gks_side<+1>(gc, WL, SL, G, DL, pl);     // DL, DR hold the one-sided time derivatives for now
  gks_side<-1>(gc, WR, SR, G, DR, pr);
  // equilibrium state g0 and its slopes
  Maxw g0; maxw_init(g0, G.W0, gc.K);
  double mu[7];
  mu[0] = 1.0; mu[1] = g0.U; mom_recur<7>(mu, g0.U, 0.5 / g0.lam);
  double ab[3][5], h[5];
  const double irho = 1.0 / g0.rho;
#pragma unroll
  for (int d = 0; d < 3; d++) {
#pragma unroll
    for (int v = 0; v < 5; v++) h[v] = G.dW0[d][v] * irho;
    micro_slope(h, g0.U, g0.V, g0.W, g0.lam, gc.K, ab[d]);
  }
  double G1F[5] = { 0, 0, 0, 0, 0 }, G2Q[5], G2F[5], G3F[5];
  add_plain<1>(g0, mu, g0.rho, G1F);
  {
    Trip t0, t1v, t2w;
    make_trip<0, 0>(t0, g0, ab[0]); make_trip<1, 0>(t1v, g0, ab[1]); make_trip<0, 1>(t2w, g0, ab[2]);
    apply_trip<1, false>(t0, mu, g0.rho, G2Q); apply_trip<0, true>(t1v, mu, g0.rho, G2Q); apply_trip<0, true>(t2w, mu, g0.rho, G2Q);
    apply_trip<2, false>(t0, mu, g0.rho, G2F); apply_trip<1, true>(t1v, mu, g0.rho, G2F); apply_trip<1, true>(t2w, mu, g0.rho, G2F);
  }
  // Abar from <abar.u + Abar> = 0; its conserved moments are -G2Q
#pragma unroll
  for (int v = 0; v < 5; v++) h[v] = -G2Q[v] * irho;
  double Ab[5]; micro_slope(h, g0.U, g0.V, g0.W, g0.lam, gc.K, Ab);
  { Trip tA; make_trip<0, 0>(tA, g0, Ab); apply_trip<1, false>(tA, mu, g0.rho, G3F); }
  // collision time
  double visc = 0.0;
  if (gc.mu_ref > 0.0) {
    visc = gc.mu_ref;
    if (gc.omega != 0.0) visc *= pow((g0.p / g0.rho) / gc.T_ref, gc.omega);
  }
  const double dpr = fabs(pl - pr) / fabs(pl + pr);
  const double tau = visc / g0.p + gc.c1 * dt + gc.c2 * dpr * dt;
  double c1[6], c2[6];
  if (tau == 0.0) {     // reading T2: f = g0 (1 + Abar t)
    c1[0] = dt; c1[1] = 0; c1[2] = 0.5 * dt * dt; c1[3] = c1[4] = c1[5] = 0;
    c2[0] = 0.5 * dt; c2[1] = 0; c2[2] = 0.125 * dt * dt; c2[3] = c2[4] = c2[5] = 0;
  } else {
    const double E2 = exp(-0.5 * dt / tau), E1 = exp(-dt / tau);
    time_coef(dt, tau, E1, c1); time_coef(0.5 * dt, tau, E2, c2);
  }
  // f^n = (4 fbar(dt/2) - fbar(dt))/dt,  f_t^n = 4 (fbar(dt) - 2 fbar(dt/2))/dt^2
  double cn[6], ct[6];
  const double idt = 1.0 / dt;
#pragma unroll
  for (int q = 0; q < 6; q++) { cn[q] = (4.0 * c2[q] - c1[q]) * idt; ct[q] = 4.0 * (c1[q] - 2.0 * c2[q]) * idt * idt; }
  double Qn[5], Qt[5];
#pragma unroll
  for (int v = 0; v < 5; v++) {
    Qn[v] = cn[0] * G.W0[v] + cn[1] * G2Q[v] - cn[2] * G2Q[v] + cn[3] * G.W0[v] + cn[4] * G.G5Q[v] + cn[5] * G.G6Q[v];
    Qt[v] = ct[0] * G.W0[v] + ct[1] * G2Q[v] - ct[2] * G2Q[v] + ct[3] * G.W0[v] + ct[4] * G.G5Q[v] + ct[5] * G.G6Q[v];
    Fn[v] = cn[0] * G1F[v] + cn[1] * G2F[v] + cn[2] * G3F[v] + cn[3] * G.G4F[v] + cn[4] * G.G5F[v] + cn[5] * G.G6F[v];
    Ft[v] = ct[0] * G1F[v] + ct[1] * G2F[v] + ct[2] * G3F[v] + ct[3] * G.G4F[v] + ct[4] * G.G5F[v] + ct[5] * G.G6F[v];
  }
  // Prandtl number fix (reading F2): energy flux += (1/Pr - 1) q, q the heat flux of the same distribution
  if (gc.Pr_fix != 0.0) {
    const double U0 = g0.U, V0 = g0.V, W0 = g0.W, ke = 0.5 * (U0 * U0 + V0 * V0 + W0 * W0);
    const double qn = Fn[4] - U0 * Qn[4] - U0 * (Fn[1] - U0 * Qn[1]) - V0 * (Fn[2] - U0 * Qn[2]) - W0 * (Fn[3] - U0 * Qn[3]) + ke * (Fn[0] - U0 * Qn[0]);
    const double qt = Ft[4] - U0 * Qt[4] - U0 * (Ft[1] - U0 * Qt[1]) - V0 * (Ft[2] - U0 * Qt[2]) - W0 * (Ft[3] - U0 * Qt[3]) + ke * (Ft[0] - U0 * Qt[0]);
    Fn[4] += gc.Pr_fix * qn; Ft[4] += gc.Pr_fix * qt;
  }
  // one-sided interface values (reading F3): weight exp(-dt/tau0), tau0 = c2 |dp|/|sum p| dt
  double wgt = 0.0;
  if (gc.c2 > 0.0 && dpr > 0.0) wgt = exp(-1.0 / (gc.c2 * dpr));
  const double om = 1.0 - wgt;
#pragma unroll
  for (int v = 0; v < 5; v++) {
    VL[v] = om * Qn[v] + wgt * WL[v]; DL[v] = om * Qt[v] + wgt * DL[v];
    VR[v] = om * Qn[v] + wgt * WR[v]; DR[v] = om * Qt[v] + wgt * DR[v];
  }
}

}  // namespace cgks
