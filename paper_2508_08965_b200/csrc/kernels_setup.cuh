// kernels_setup.cuh -- create-time and boundary kernels: mesh metrics, state copy / bootstrap, CFL reduction.
#pragma once
#include "cgks_common.cuh"

namespace cgks {

__device__ __forceinline__ void cross3(const double* a, const double* b, double* o) {
  o[0] = a[1] * b[2] - a[2] * b[1]; o[1] = a[2] * b[0] - a[0] * b[2]; o[2] = a[0] * b[1] - a[1] * b[0];
}
__device__ __forceinline__ double det3(const double* m) {
  return m[0] * (m[4] * m[8] - m[5] * m[7]) - m[1] * (m[3] * m[8] - m[5] * m[6]) + m[2] * (m[3] * m[7] - m[4] * m[6]);
}

struct NodeView {
  const double* p; int ni1, nj1, nk1;
  __device__ __forceinline__ void get(int i, int j, int k, double* x) const {
    const long s = (long)ni1 * nj1 * nk1; const long o = ((long)k * nj1 + j) * ni1 + i;
    x[0] = p[o]; x[1] = p[s + o]; x[2] = p[2 * s + o];
  }
};

// flags[0] |= 1 if any cell's J0 differs from diag(period/n)  (-> general metrics needed)
// flags[1] |= 1 if det J0 <= 0 or volume <= 0;  flags[2] |= 1 if the node array is not periodic
// The node array is that of the GLOBAL periodic mesh (nk planes of cells); the context holds nkl planes of it starting at
// global plane kofs (wrapped): nkl = nk, kofs = 0 for a whole-mesh context, a slab with its halo planes for a sub-domain.
// A cell's metrics are computed from the same eight node values whichever context holds it.
__global__ void geometry_kernel(int ni, int nj, int nk, int nkl, int kofs, const double* __restrict__ nodes, double* __restrict__ met,
                                int* __restrict__ flags) {
  const long n = (long)ni * nj * nkl;
  const long c = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= n) return;
  const int i = (int)(c % ni), j = (int)((c / ni) % nj);
  int k = (int)(c / ((long)ni * nj)) + kofs;
  k %= nk; if (k < 0) k += nk;
  NodeView nv{ nodes, ni + 1, nj + 1, nk + 1 };
  double X[8][3];     // index 4*di + 2*dj + dk
#pragma unroll
  for (int v = 0; v < 8; v++) nv.get(i + ((v >> 2) & 1), j + ((v >> 1) & 1), k + (v & 1), X[v]);
  // J0 = [N2-N1 | N3-N1 | N4-N1], N1 = node(i,j,k)  (Eq. 18, reading R1); row-major J[3r+a] = dx_r/dxi_a
  double J[9];
#pragma unroll
  for (int r = 0; r < 3; r++) { J[3 * r] = X[4][r] - X[0][r]; J[3 * r + 1] = X[2][r] - X[0][r]; J[3 * r + 2] = X[1][r] - X[0][r]; }
  const double dj = det3(J);
  // uniform-Cartesian test against period/n
  double O[3], Pi[3], Pj[3], Pk[3];
  nv.get(0, 0, 0, O); nv.get(ni, 0, 0, Pi); nv.get(0, nj, 0, Pj); nv.get(0, 0, nk, Pk);
  const double h[3] = { (Pi[0] - O[0]) / ni, (Pj[1] - O[1]) / nj, (Pk[2] - O[2]) / nk };
  const double hm = fmax(fabs(h[0]), fmax(fabs(h[1]), fabs(h[2])));
  bool uni = true;
#pragma unroll
  for (int r = 0; r < 3; r++)
#pragma unroll
    for (int a = 0; a < 3; a++) uni = uni && (fabs(J[3 * r + a] - (r == a ? h[r] : 0.0)) <= 1e-11 * hm);
  // the other five nodes must also sit on the lattice
#pragma unroll
  for (int v = 0; v < 8; v++)
#pragma unroll
    for (int r = 0; r < 3; r++) {
      const int off = (r == 0) ? ((v >> 2) & 1) : ((r == 1) ? ((v >> 1) & 1) : (v & 1));
      uni = uni && (fabs(X[v][r] - X[0][r] - off * h[r]) <= 1e-11 * hm);
    }
  if (!uni) atomicOr(&flags[0], 1);
  // periodicity of the node array: boundary cells compare their outer nodes with the period vectors
  if (i == ni - 1 || j == nj - 1 || k == nk - 1) {
    double a[3], b[3]; bool per = true;
    const double tol = 1e-11 * (fabs(Pi[0] - O[0]) + fabs(Pj[1] - O[1]) + fabs(Pk[2] - O[2]));
    if (i == ni - 1) { nv.get(ni, j, k, a); nv.get(0, j, k, b); for (int r = 0; r < 3; r++) per = per && fabs(a[r] - b[r] - (Pi[r] - O[r])) <= tol; }
    if (j == nj - 1) { nv.get(i, nj, k, a); nv.get(i, 0, k, b); for (int r = 0; r < 3; r++) per = per && fabs(a[r] - b[r] - (Pj[r] - O[r])) <= tol; }
    if (k == nk - 1) { nv.get(i, j, nk, a); nv.get(i, j, 0, b); for (int r = 0; r < 3; r++) per = per && fabs(a[r] - b[r] - (Pk[r] - O[r])) <= tol; }
    if (!per) atomicOr(&flags[2], 1);
  }
  // volume: trilinear map, 3x3x3 Gauss quadrature (Appendix)
  const double gq[3] = { -0.5 * sqrt(0.6), 0.0, 0.5 * sqrt(0.6) }, wq[3] = { 5.0 / 18.0, 8.0 / 18.0, 5.0 / 18.0 };
  double vol = 0.0;
  for (int l = 0; l < 3; l++) for (int mm = 0; mm < 3; mm++) for (int nn = 0; nn < 3; nn++) {
    const double xi[3] = { gq[l], gq[mm], gq[nn] };
    double Jm[9] = { 0, 0, 0, 0, 0, 0, 0, 0, 0 };
#pragma unroll
    for (int v = 0; v < 8; v++) {
      const double s0 = ((v >> 2) & 1) ? 1.0 : -1.0, s1 = ((v >> 1) & 1) ? 1.0 : -1.0, s2 = (v & 1) ? 1.0 : -1.0;
      const double f0 = 0.5 + s0 * xi[0], f1 = 0.5 + s1 * xi[1], f2 = 0.5 + s2 * xi[2];
      const double dp[3] = { s0 * f1 * f2, f0 * s1 * f2, f0 * f1 * s2 };
#pragma unroll
      for (int r = 0; r < 3; r++)
#pragma unroll
        for (int a = 0; a < 3; a++) Jm[3 * r + a] += X[v][r] * dp[a];
    }
    vol += wq[l] * wq[mm] * wq[nn] * fabs(det3(Jm));
  }
  if (!(dj > 0.0) || !(vol > 0.0)) atomicOr(&flags[1], 1);
  if (met == nullptr) return;
#pragma unroll
  for (int q = 0; q < 9; q++) met[(MET_J0 + q) * n + c] = J[q];
  const double id = 1.0 / dj;
  double Ji[9];
  Ji[0] = (J[4] * J[8] - J[5] * J[7]) * id; Ji[1] = (J[2] * J[7] - J[1] * J[8]) * id; Ji[2] = (J[1] * J[5] - J[2] * J[4]) * id;
  Ji[3] = (J[5] * J[6] - J[3] * J[8]) * id; Ji[4] = (J[0] * J[8] - J[2] * J[6]) * id; Ji[5] = (J[2] * J[3] - J[0] * J[5]) * id;
  Ji[6] = (J[3] * J[7] - J[4] * J[6]) * id; Ji[7] = (J[1] * J[6] - J[0] * J[7]) * id; Ji[8] = (J[0] * J[4] - J[1] * J[3]) * id;
#pragma unroll
  for (int q = 0; q < 9; q++) met[(MET_J0INV + q) * n + c] = Ji[q];
  met[MET_VOL * n + c] = vol;
  // + faces: vector area = half the cross product of the diagonals, first tangent along the first in-face edge
  // (reading R2).  Node index v = 4 di + 2 dj + dk.
  const int FA[3][4] = { { 4, 6, 7, 5 }, { 2, 3, 7, 6 }, { 1, 5, 7, 3 } };   // a, b(+e1), c(+e1+e2), d(+e2); (ax,e1,e2) cyclic
#pragma unroll
  for (int ax = 0; ax < 3; ax++) {
    const double* a = X[FA[ax][0]]; const double* b = X[FA[ax][1]]; const double* cc = X[FA[ax][2]]; const double* d = X[FA[ax][3]];
    double d1[3], d2[3], A[3];
#pragma unroll
    for (int r = 0; r < 3; r++) { d1[r] = cc[r] - a[r]; d2[r] = d[r] - b[r]; }
    cross3(d1, d2, A);
#pragma unroll
    for (int r = 0; r < 3; r++) A[r] *= 0.5;
    const double S = sqrt(A[0] * A[0] + A[1] * A[1] + A[2] * A[2]);
    const double nr[3] = { A[0] / S, A[1] / S, A[2] / S };
    double e[3] = { b[0] - a[0], b[1] - a[1], b[2] - a[2] };
    const double en = e[0] * nr[0] + e[1] * nr[1] + e[2] * nr[2];
#pragma unroll
    for (int r = 0; r < 3; r++) e[r] -= en * nr[r];
    const double el = sqrt(e[0] * e[0] + e[1] * e[1] + e[2] * e[2]);
#pragma unroll
    for (int r = 0; r < 3; r++) { met[(MET_AREA + 3 * ax + r) * n + c] = A[r]; met[(MET_TAN + 3 * ax + r) * n + c] = e[r] / el; }
  }
}

// state copy-in, with bootstrap of missing derivative dof (reading S2).  Thread per (cell, variable).
__global__ void set_state_kernel(Mesh m, const double* __restrict__ Qin, const double* __restrict__ Gin,
                                 const double* __restrict__ Din, double* __restrict__ W) {
  const long c = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= m.n) return;
  const int v = blockIdx.y;
  const int i = (int)(c % m.ni), j = (int)((c / m.ni) % m.nj), k = (int)(c / m.plane);
  const double* q = Qin + (long)v * m.n;
  double* qg = W + iQG(v, c, m.n);
  qg[0] = q[c];
  double dr[3] = { 0, 0, 0 };
  if (Gin == nullptr || Din == nullptr) {
    const int ii[5] = { wrap(i - 2, m.ni), wrap(i - 1, m.ni), i, wrap(i + 1, m.ni), wrap(i + 2, m.ni) };
    const int jj[5] = { wrap(j - 2, m.nj), wrap(j - 1, m.nj), j, wrap(j + 1, m.nj), wrap(j + 2, m.nj) };
    const int kk[5] = { wrap(k - 2, m.nk), wrap(k - 1, m.nk), k, wrap(k + 1, m.nk), wrap(k + 2, m.nk) };
    dr[0] = (8.0 * (q[cell_at(m, ii[3], j, k)] - q[cell_at(m, ii[1], j, k)]) - (q[cell_at(m, ii[4], j, k)] - q[cell_at(m, ii[0], j, k)])) / 12.0;
    dr[1] = (8.0 * (q[cell_at(m, i, jj[3], k)] - q[cell_at(m, i, jj[1], k)]) - (q[cell_at(m, i, jj[4], k)] - q[cell_at(m, i, jj[0], k)])) / 12.0;
    dr[2] = (8.0 * (q[cell_at(m, i, j, kk[3])] - q[cell_at(m, i, j, kk[1])]) - (q[cell_at(m, i, j, kk[4])] - q[cell_at(m, i, j, kk[0])])) / 12.0;
  }
  if (Gin != nullptr) {
#pragma unroll
    for (int r = 0; r < 3; r++) qg[1 + r] = Gin[(long)(3 * v + r) * m.n + c];
  } else {
#pragma unroll
    for (int r = 0; r < 3; r++) {       // grad = J0^-T grad'
      double g;
      if (m.cart) g = dr[r] / m.h[r];
      else g = m.met[(MET_J0INV + 0 + r) * m.n + c] * dr[0] + m.met[(MET_J0INV + 3 + r) * m.n + c] * dr[1] + m.met[(MET_J0INV + 6 + r) * m.n + c] * dr[2];
      qg[1 + r] = g;
    }
  }
  if (Din != nullptr) {
#pragma unroll
    for (int s = 0; s < 12; s++) W[iD(v, s / 4, c, m.n) + s % 4] = Din[(long)(12 * v + s) * m.n + c];
  } else {
#pragma unroll
    for (int s = 0; s < 12; s++) W[iD(v, s / 4, c, m.n) + s % 4] = dr[s / 4];
  }
}

__global__ void get_state_kernel(Mesh m, const double* __restrict__ W, double* __restrict__ Qo, double* __restrict__ Go,
                                 double* __restrict__ Do) {
  const long c = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= m.n) return;
  const int v = blockIdx.y;
  const double* qg = W + iQG(v, c, m.n);
  if (Qo) Qo[(long)v * m.n + c] = qg[0];
  if (Go) for (int r = 0; r < 3; r++) Go[(long)(3 * v + r) * m.n + c] = qg[1 + r];
  if (Do) for (int s = 0; s < 12; s++) Do[(long)(12 * v + s) * m.n + c] = W[iD(v, s / 4, c, m.n) + s % 4];
}

// time step (reading S3): dt = min over cells of cfl / sum_d (|U.n_d| + c)/h_d and of the viscous cap.
// Warp-shuffle min, one atomicMin per block on the bit pattern (positive doubles order like unsigned integers).
struct CflPrm { double gamma, mu_ref, omega, T_ref, cfl; };

// Cells of the planes [kA, kA + cnt) only (a sub-domain reduces over the planes it owns).
__global__ void cfl_kernel(Mesh m, const double* __restrict__ W, CflPrm p, unsigned long long* __restrict__ dt_bits,
                           int* __restrict__ flag, int kA, int cnt) {
  double dtmin = INFINITY;
  bool bad = false;
  const long c0 = (long)kA * m.plane, c1 = c0 + (long)cnt * m.plane;
  for (long c = c0 + (long)blockIdx.x * blockDim.x + threadIdx.x; c < c1; c += (long)gridDim.x * blockDim.x) {
    const double rho = W[iQG(0, c, m.n)], mx = W[iQG(1, c, m.n)], my = W[iQG(2, c, m.n)], mz = W[iQG(3, c, m.n)], E = W[iQG(4, c, m.n)];
    const double U[3] = { mx / rho, my / rho, mz / rho };
    const double pr = (p.gamma - 1.0) * (E - 0.5 * rho * (U[0] * U[0] + U[1] * U[1] + U[2] * U[2]));
    if (!(rho > 0.0) || !(pr > 0.0)) { bad = true; continue; }
    const double cs = sqrt(p.gamma * pr / rho);
    double rate = 0.0, hmin = INFINITY;
    if (m.cart) {
#pragma unroll
      for (int ax = 0; ax < 3; ax++) { rate += (fabs(U[ax]) + cs) / m.h[ax]; hmin = fmin(hmin, m.h[ax]); }
    } else {
      const int i = (int)(c % m.ni), j = (int)((c / m.ni) % m.nj), k = (int)(c / m.plane);
      const double vol = m.met[MET_VOL * m.n + c];
#pragma unroll
      for (int ax = 0; ax < 3; ax++) {
        const long cm = (ax == 0) ? cell_at(m, wrap(i - 1, m.ni), j, k) : ((ax == 1) ? cell_at(m, i, wrap(j - 1, m.nj), k) : cell_at(m, i, j, wrap(k - 1, m.nk)));
        double Ap[3], Am[3];
#pragma unroll
        for (int r = 0; r < 3; r++) { Ap[r] = m.met[(MET_AREA + 3 * ax + r) * m.n + c]; Am[r] = m.met[(MET_AREA + 3 * ax + r) * m.n + cm]; }
        const double Sp = sqrt(Ap[0] * Ap[0] + Ap[1] * Ap[1] + Ap[2] * Ap[2]), Sm = sqrt(Am[0] * Am[0] + Am[1] * Am[1] + Am[2] * Am[2]);
        const double nb[3] = { Ap[0] + Am[0], Ap[1] + Am[1], Ap[2] + Am[2] };
        const double nl = sqrt(nb[0] * nb[0] + nb[1] * nb[1] + nb[2] * nb[2]);
        const double h = vol / (0.5 * (Sp + Sm));
        const double un = fabs(U[0] * nb[0] + U[1] * nb[1] + U[2] * nb[2]) / nl;
        rate += (un + cs) / h; hmin = fmin(hmin, h);
      }
    }
    dtmin = fmin(dtmin, p.cfl / rate);
    if (p.mu_ref > 0.0) {
      double mu = p.mu_ref;
      if (p.omega != 0.0) mu *= pow((pr / rho) / p.T_ref, p.omega);
      dtmin = fmin(dtmin, p.cfl * hmin * hmin / (3.0 * mu / rho));
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) dtmin = fmin(dtmin, __shfl_xor_sync(0xffffffffu, dtmin, o));
  __shared__ double sm[32];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (lane == 0) sm[wid] = dtmin;
  __syncthreads();
  if (wid == 0) {
    dtmin = (lane < (int)(blockDim.x >> 5)) ? sm[lane] : INFINITY;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) dtmin = fmin(dtmin, __shfl_xor_sync(0xffffffffu, dtmin, o));
    if (lane == 0) atomicMin(dt_bits, (unsigned long long)__double_as_longlong(dtmin));
  }
  if (bad) atomicOr(flag, 1);
}

// Halo planes of a sub-domain: `np` k-planes of all 80 state fields between the state
// buffer W [80][n] and a contiguous buffer [80][np][plane].  PACK: W -> buf, else buf -> W.
template <bool PACK>
__global__ void halo_kernel(double* __restrict__ W, double* __restrict__ buf, long n, long plane, int kfirst, int np) {
  // the planes [kfirst, kfirst + np) of every record array (5 of { Q, G }, 15 of the line differences of one axis) are one
  // contiguous run of 4 np plane doubles; the buffer holds the 20 runs one after the other
  const long run = 4L * np * plane;
  const long tot = 20 * run;
  for (long t = (long)blockIdx.x * blockDim.x + threadIdx.x; t < tot; t += (long)gridDim.x * blockDim.x) {
    const int a = (int)(t / run); const long r = t - a * run;
    double* w = W + (a < 5 ? iQG(a, (long)kfirst * plane, n) : iD((a - 5) / 3, (a - 5) % 3, (long)kfirst * plane, n)) + r;
    if (PACK) buf[t] = *w; else *w = buf[t];
  }
}

// Boundary conditions in k for a sub-domain context (the paper names its boundary types, PAPER.md:494
// and 536, without formulas: DESIGN.md reading B1): the two halo planes of one side are filled from the owned planes.
//   kind 0 slip wall / symmetry plane: mirror image about the boundary face; the normal momentum is odd, everything else even
//   kind 1 no-slip adiabatic wall: mirror image with ALL momentum components odd (zero velocity, zero normal
//          temperature gradient at the face)
//   kind 2 outflow: the outermost owned plane copied into both halo planes with its k-derivative dof set to zero
//   kind 3 far field: a given uniform state, zero derivative dof
// Mirror rules for the derivative dof of a field of parity s: G_r -> s G_r (r = i, j), -s G_k; line differences along i or j
// swap the two lines that differ in their k position (index bit b) with sign s; line differences along k keep their
// index and get the sign -s.  Uniform Cartesian meshes only (the halo cells' metrics are those of the periodic image).
struct BcPrm { int side, kind; double far[5]; };

__global__ void bc_halo_kernel(double* __restrict__ W, long n, long plane, int nkl, BcPrm bc) {
  const long ij = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (ij >= plane) return;
  const int f = blockIdx.y, hp = blockIdx.z;             // field 0..79, halo plane 0 (next to the boundary) or 1
  const int kt = bc.side ? nkl - 2 + hp : 1 - hp;
  int ks = bc.side ? nkl - 3 - hp : 2 + hp;              // mirror image
  if (bc.kind == 2) ks = bc.side ? nkl - 3 : 2;
  int v, fs = f; double sgn = 1.0; bool kderiv = false;
  if (f < 5) v = f;
  else if (f < 20) { v = (f - 5) / 3; const int r = (f - 5) % 3; kderiv = (r == 2); if (r == 2) sgn = -1.0; }
  else {
    v = (f - 20) / 12; const int s_ = (f - 20) % 12, ax = s_ / 4;
    if (ax == 2) { sgn = -1.0; kderiv = true; }
    else fs = 20 + 12 * v + (s_ ^ 1);                    // bit b = position along the second other axis = k for lines along i or j
  }
  double out;
  if (bc.kind <= 1) {
    const bool odd = (v == 3) || (bc.kind == 1 && (v == 1 || v == 2));
    out = (odd ? -sgn : sgn) * W[iField(fs, (long)ks * plane + ij, n)];
  } else if (bc.kind == 2) {
    out = kderiv ? 0.0 : W[iField(f, (long)ks * plane + ij, n)];
  } else {
    out = (f < 5) ? bc.far[f] : 0.0;
  }
  W[iField(f, (long)kt * plane + ij, n)] = out;
}

}  // namespace cgks
