// kernels_stage.cuh -- the three per-stage kernels of the S2O4 step:
//   recon_kernel   compact reconstruction on the reference cell + GENO blend -> values/gradients at 24 face points
//   flux_kernel    gas-kinetic flux + interface values at the 12 owned face Gauss points of each cell
//   update_kernel  accumulate L, dL/dt, gradient and line sums; S2O4 stage combine
// All index the mesh periodically and work on a slab of k-planes (see Slab).
#pragma once
#include "cgks_common.cuh"
#include "gks_flux.cuh"
#include "recon_gen.cuh"

namespace cgks {

struct ReconPrm { int nonlinear; double C, eps, inv_tanhC, gamma; };
// pv and fx are written once and read once by the next kernel, far beyond the L2 capacity: streaming (evict-first) stores.
// (Streaming LOADS of fx in the update kernel were 24 % slower: the face values shared with the neighbours do hit in L2.)
#define ST_STREAM(p, v) __stcs((p), (v))
// pv record of one (Gauss point p, variable v, cell slot): { value, d/dx, d/dy, d/dz } = 32 contiguous bytes, written with ONE
// 256-bit streaming store and read by the flux kernel with two 16-byte cp.async (a quarter / half of the memory instructions of
// a plane-per-component layout, and 1 KB contiguous per warp).  Index of the record's first double:
__device__ __forceinline__ long pv_index(const Slab& sl, int p, int v, long off) { return ((long)(p * NVAR + v) * sl.stride_pv + off) * 4; }
__device__ __forceinline__ void st_stream4(double* dst, double a, double b, double c, double d) {
  asm volatile("st.global.cs.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(__cvta_generic_to_global(dst)), "d"(a), "d"(b), "d"(c), "d"(d) : "memory");
}
#ifndef FLUX_MINB
#define FLUX_MINB 2
#endif

// ------------------------------------------------------------------------------------------------ reconstruction
// Thread per (cell, variable).  PAPER.md:134-246 (Eq. 11-16), 250-300 (Eq. 17-19).
// The 72 data of Eq. 19 are consumed neighbour group by neighbour group (face pairs, edge quads, line quads): each
// group's raw data are turned into reflection-parity combinations and accumulated into the 34 coefficients with the
// block-diagonal form of M (recon_gen.cuh), so the data vector is never held as a whole.
template <int AX> __device__ __forceinline__ void acc_face(const double* x, double* a) {
  if (AX == 0) recon_acc_face0(x, a); else if (AX == 1) recon_acc_face1(x, a); else recon_acc_face2(x, a);
}
template <int AX> __device__ __forceinline__ void acc_edge(const double* x, double* a) {
  if (AX == 0) recon_acc_edge0(x, a); else if (AX == 1) recon_acc_edge1(x, a); else recon_acc_edge2(x, a);
}
template <int AX> __device__ __forceinline__ void acc_line(const double* x, double* a) {
  if (AX == 0) recon_acc_line0(x, a); else if (AX == 1) recon_acc_line1(x, a); else recon_acc_line2(x, a);
}
template <int AX> __device__ __forceinline__ void eval_axis(const double* a, double* o) {
  if (AX == 0) recon_eval_axis0(a, o); else if (AX == 1) recon_eval_axis1(a, o); else recon_eval_axis2(a, o);
}

template <bool CART>
struct ReconCell {
  const Mesh& m; const double* qg;      // records { Q, G (3) } of this variable, [n][4]
  unsigned long long pol;               // L2 policy of the gathers
  double J[9];
  // average difference and (grad Q)' = J0^T grad Q of neighbour cn with the TARGET cell's J0: one 256-bit load
  __device__ __forceinline__ void neighbour(long cn, double q0, double& dq, double* gr) const {
    double q, g0, g1, g2;
    ld4_ro_keep(qg + 4 * cn, pol, q, g0, g1, g2);
    dq = q - q0;
    if (CART) { gr[0] = m.h[0] * g0; gr[1] = m.h[1] * g1; gr[2] = m.h[2] * g2; }
    else {
#pragma unroll
      for (int a = 0; a < 3; a++) gr[a] = J[a] * g0 + J[3 + a] * g1 + J[6 + a] * g2;
    }
  }
};

template <bool CART, int AX>
__device__ __forceinline__ void recon_gather_axis(const ReconCell<CART>& rc, const int* ii, const int* jj, const int* kk,
                                                  double q0, double* a, double* dface) {
  const Mesh& m = rc.m;
  {   // face pair of axis AX: x = { dq+, dq-, gr'+ (3), gr'- (3) }
    int op[3] = { 1, 1, 1 }, om[3] = { 1, 1, 1 };
    op[AX] = 2; om[AX] = 0;
    const long cp = cell_at(m, ii[op[0]], jj[op[1]], kk[op[2]]), cm = cell_at(m, ii[om[0]], jj[om[1]], kk[om[2]]);
    double x[8];
    rc.neighbour(cp, q0, x[0], x + 2); rc.neighbour(cm, q0, x[1], x + 5);
    dface[2 * AX] = x[0]; dface[2 * AX + 1] = x[1];
    acc_face<AX>(x, a);
  }
  {   // the four edge neighbours around axis AX: x = { dq_t (4), (gr'[AX], o.gr')_t (4 x 2) }
    const int o1 = (AX == 0) ? 1 : 0, o2 = (AX == 2) ? 1 : 2;
    double x[12];
#pragma unroll
    for (int t = 0; t < 4; t++) {
      int o[3] = { 1, 1, 1 };
      const int s1 = ((t >> 1) & 1) ? 1 : -1, s2 = (t & 1) ? 1 : -1;
      o[o1] += s1; o[o2] += s2;
      const long cn = cell_at(m, ii[o[0]], jj[o[1]], kk[o[2]]);
      double gr[3]; rc.neighbour(cn, q0, x[t], gr);
      x[4 + 2 * t] = gr[AX];
      x[5 + 2 * t] = s1 * gr[o1] + s2 * gr[o2];
    }
    acc_edge<AX>(x, a);
  }
}

// VOLUME = true: the same polynomial evaluated at the 8 interior points (+-g, +-g, +-g) of the 2x2x2 Gauss rule instead
// (pv planes 0..7, used by the diagnostics of PAPER.md:428-454).
// NL: the GENO blend is compiled in (nonlinear = 1, the paper's default) or out (linear scheme), so that the thread is one block of
// straight-line code either way.
// launch grid of recon_kernel over nthreads cells with blocks of tpb threads (see the index computation in the kernel)
template <bool CART>
inline dim3 recon_grid(long nthreads, int tpb) {
  const unsigned tiles = (unsigned)((nthreads + tpb - 1) / tpb);
  return CART ? dim3(tiles, 5) : dim3(tiles * 5u, 1);
}

template <bool CART, bool VOLUME = false, bool NL = true>
__global__ void __launch_bounds__(128, 3) recon_kernel(Mesh m, Slab sl, const double* __restrict__ W, double* __restrict__ pv,
                                                    double* __restrict__ chi_out, ReconPrm rp, int kA, long nthreads,
                                                    int* __restrict__ flag) {
  // Cartesian: grid (tiles, 5), v = blockIdx.y.  General meshes: grid (5 tiles), the five variable-blocks of a tile ADJACENT in launch
  // order (v = blockIdx.x % 5), so that the 18 doubles of J0 / J0^-1 per cell, which all five read, come from DRAM once and from L2
  // four times (with v = blockIdx.y the five readers run a whole grid row apart and every read misses: profiles/r03a_curvilinear.md)
  const unsigned tile = CART ? blockIdx.x : blockIdx.x / 5u;
  const int v = CART ? (int)blockIdx.y : (int)(blockIdx.x - 5u * tile);
  const long t = (long)tile * blockDim.x + threadIdx.x;
  if (t >= nthreads) return;
  const CellIdx x = cell_of(m, t, kA);
  const long n = m.n;
  if (v == 0) {      // physical admissibility of the incoming cell average (reported by cgks_status / cgks_compute_dt)
    const double w5[5] = { W[iQG(0, x.c, n)], W[iQG(1, x.c, n)], W[iQG(2, x.c, n)], W[iQG(3, x.c, n)], W[iQG(4, x.c, n)] };
    if (!admissible(w5)) atomicOr(flag, 1);      // rho > 0 and rho E - |m|^2/2 > 0: no division
  }
  const int ii[3] = { wrap(x.i - 1, m.ni), x.i, wrap(x.i + 1, m.ni) };
  const int jj[3] = { wrap(x.j - 1, m.nj), x.j, wrap(x.j + 1, m.nj) };
  const int kk[3] = { wrap(x.k - 1, m.nk), x.k, wrap(x.k + 1, m.nk) };
  ReconCell<CART> rc{ m, W + iQG(v, 0, n), l2_policy_evict_last(), {} };
  if (!CART) {
#pragma unroll
    for (int q = 0; q < 9; q++) rc.J[q] = m.met[(MET_J0 + q) * n + x.c];
  }
  const double q0 = rc.qg[4 * x.c];
  double a[34], dface[6], la[3];
#pragma unroll
  for (int b = 0; b < 34; b++) a[b] = 0.0;
  recon_gather_axis<CART, 0>(rc, ii, jj, kk, q0, a, dface);
  recon_gather_axis<CART, 1>(rc, ii, jj, kk, q0, a, dface);
  recon_gather_axis<CART, 2>(rc, ii, jj, kk, q0, a, dface);
  {   // line differences (Eq. 10): raw D, the factor h3' is folded into the coefficients; three 256-bit loads
    double Dl[4];
    ld4_ro(W + iD(v, 0, x.c, n), Dl[0], Dl[1], Dl[2], Dl[3]);
    la[0] = 0.25 * (Dl[0] + Dl[1] + Dl[2] + Dl[3]); acc_line<0>(Dl, a);
    ld4_ro(W + iD(v, 1, x.c, n), Dl[0], Dl[1], Dl[2], Dl[3]);
    la[1] = 0.25 * (Dl[0] + Dl[1] + Dl[2] + Dl[3]); acc_line<1>(Dl, a);
    ld4_ro(W + iD(v, 2, x.c, n), Dl[0], Dl[1], Dl[2], Dl[3]);
    la[2] = 0.25 * (Dl[0] + Dl[1] + Dl[2] + Dl[3]); acc_line<2>(Dl, a);
  }
  double chi = 1.0;
  if (NL) {
    // six linear polynomials (Eq. 15): normal slope = average difference, tangential = mean line difference
    double wsum = 0.0, bw[3] = { 0, 0, 0 };
#pragma unroll
    for (int mm = 0; mm < 6; mm++) {
      double b[3] = { la[0], la[1], la[2] };
      b[mm / 2] = (mm % 2 == 0) ? dface[mm] : -dface[mm];
      const double IS = b[0] * b[0] + b[1] * b[1] + b[2] * b[2];
      const double tt = IS + rp.eps, t2 = tt * tt;
      const double wb = (1.0 / 6.0) * drcp(t2 * t2 * tt);           // d_m/(IS_m + eps)^5
      wsum += wb; bw[0] += wb * b[0]; bw[1] += wb * b[1]; bw[2] += wb * b[2];
    }
    // path function (readings G2, G3); divisions and tanh are the branch-free ones of fastmath64.cuh
    const double IS1 = recon_IS1(a), IS2 = recon_IS2(a), ISt = recon_IS34(a);
    const double ISH = IS1 + IS2 + ISt;
    const double rH = ddiv(ISt, ISH + rp.eps), rL = ddiv(ISt, IS1 + rp.eps);
    const double aH = 1.0 + rH * rH, aL = 1.0 + rL * rL;
    const double alpha = ddiv(2.0 * aH, aH + aL);
    chi = dtanh_pos(rp.C * alpha) * rp.inv_tanhC;
    // Eq. 16 as one polynomial: chi P4 + (1-chi) sum_m omega_m P1_m
    const double w1 = ddiv(1.0 - chi, wsum);
#pragma unroll
    for (int b = 0; b < 3; b++) a[b] = chi * a[b] + w1 * bw[b];
#pragma unroll
    for (int b = 3; b < 34; b++) a[b] *= chi;
  }
  if (chi_out) chi_out[(long)v * n + x.c] = chi;
  // values and gradients at the 24 face Gauss points, back-transformed
  const long off = (long)slot_of(m, sl, x.k) * m.plane + x.ij;
  double Ji[9];
  if (!CART) {
#pragma unroll
    for (int q = 0; q < 9; q++) Ji[q] = m.met[(MET_J0INV + q) * n + x.c];
  }
  const double ih[3] = { drcp(m.h[0]), drcp(m.h[1]), drcp(m.h[2]) };
  auto store_axis = [&](int ax, const double* o) {
#pragma unroll
    for (int l = 0; l < 8; l++) {
      const int p = 8 * ax + l;            // = 4 * (2 ax + sgn) + 2a + b
      double g[3];
      if (CART) { g[0] = o[4 * l + 1] * ih[0]; g[1] = o[4 * l + 2] * ih[1]; g[2] = o[4 * l + 3] * ih[2]; }
      else {
#pragma unroll
        for (int r = 0; r < 3; r++) g[r] = Ji[r] * o[4 * l + 1] + Ji[3 + r] * o[4 * l + 2] + Ji[6 + r] * o[4 * l + 3];
      }
      st_stream4(pv + pv_index(sl, p, v, off), q0 + o[4 * l], g[0], g[1], g[2]);
    }
  };
  if (VOLUME) { double o[32]; recon_eval_volume(a, o); store_axis(0, o); return; }
  { double o[32]; eval_axis<0>(a, o); store_axis(0, o); }
  { double o[32]; eval_axis<1>(a, o); store_axis(1, o); }
  { double o[32]; eval_axis<2>(a, o); store_axis(2, o); }
}

// test tap: pv records -> planes [480][n] in the documented order (plane (4m+q)*20 + c: c = v value, 5+3v+r gradient)
__global__ void pv_unpack_kernel(Slab sl, long n, const double* __restrict__ pv, double* __restrict__ out) {
  const long c = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= n) return;
  const int pvv = blockIdx.y, p = pvv / NVAR, v = pvv - p * NVAR;
  const double* src = pv + pv_index(sl, p, v, c);
  out[(long)(p * 20 + v) * n + c] = src[0];
#pragma unroll
  for (int r = 0; r < 3; r++) out[(long)(p * 20 + 5 + 3 * v + r) * n + c] = src[1 + r];
}

// ------------------------------------------------------------------------------------------------ diagnostics
// E_k = int rho |U|^2/2 dV / |Omega|, enstrophy = int mu |curl U|^2 dV / |Omega| by the 2x2x2 Gauss rule
// with the reconstructed polynomial (reading X1).  Thread per cell over the 8 points staged in pv by
// recon_kernel<CART, true>; deterministic block tree reduction, one partial triple (E_k, enstrophy, volume) per block.
struct DiagPrm { double gamma, mu_ref, omega, inv_T_ref; };

template <bool CART>
__global__ void __launch_bounds__(128) diag_kernel(Mesh m, Slab sl, const double* __restrict__ W, const double* __restrict__ pv,
                                                   DiagPrm dp, int kA, long nthreads, double* __restrict__ partial) {
  __shared__ double red[3][128];
  const long t = (long)blockIdx.x * blockDim.x + threadIdx.x;
  double ek = 0.0, en = 0.0, vol = 0.0;
  if (t < nthreads) {
    const CellIdx x = cell_of(m, t, kA);
    const long off = (long)slot_of(m, sl, x.k) * m.plane + x.ij;
    vol = CART ? m.h[0] * m.h[1] * m.h[2] : m.met[MET_VOL * m.n + x.c];
#pragma unroll 1
    for (int p = 0; p < 8; p++) {
      double w[5], g[4][3];
#pragma unroll
      for (int c = 0; c < 5; c++) {
        const double* src = pv + pv_index(sl, p, c, off);
        w[c] = src[0];
        if (c < 4) { g[c][0] = src[1]; g[c][1] = src[2]; g[c][2] = src[3]; }
      }
      double pe = w[4] - 0.5 * (w[1] * w[1] + w[2] * w[2] + w[3] * w[3]) / w[0];
      if (!admissible(w)) {                    // positivity fallback (reading R9): cell average, zero gradient
#pragma unroll
        for (int c = 0; c < 5; c++) w[c] = W[iQG(c, x.c, m.n)];
#pragma unroll
        for (int c = 0; c < 4; c++) { g[c][0] = 0.0; g[c][1] = 0.0; g[c][2] = 0.0; }
        pe = w[4] - 0.5 * (w[1] * w[1] + w[2] * w[2] + w[3] * w[3]) / w[0];
      }
      const double ir = 1.0 / w[0];
      const double U[3] = { w[1] * ir, w[2] * ir, w[3] * ir };
      double dU[3][3];      // dU[a][r] = d U_a / d x_r
#pragma unroll
      for (int a = 0; a < 3; a++)
#pragma unroll
        for (int r = 0; r < 3; r++) dU[a][r] = (g[1 + a][r] - U[a] * g[0][r]) * ir;
      const double c0 = dU[2][1] - dU[1][2], c1 = dU[0][2] - dU[2][0], c2 = dU[1][0] - dU[0][1];
      double mu = dp.mu_ref;
      if (dp.mu_ref > 0.0 && dp.omega != 0.0) mu *= pow(((dp.gamma - 1.0) * pe * ir) * dp.inv_T_ref, dp.omega);
      ek += 0.5 * w[0] * (U[0] * U[0] + U[1] * U[1] + U[2] * U[2]);
      en += mu * (c0 * c0 + c1 * c1 + c2 * c2);
    }
    ek *= 0.125 * vol; en *= 0.125 * vol;
  }
  red[0][threadIdx.x] = ek; red[1][threadIdx.x] = en; red[2][threadIdx.x] = vol;
  __syncthreads();
  for (int s2 = 64; s2 > 0; s2 >>= 1) {
    if (threadIdx.x < s2) {
#pragma unroll
      for (int c = 0; c < 3; c++) red[c][threadIdx.x] += red[c][threadIdx.x + s2];
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) { partial[3 * (long)blockIdx.x] = red[0][0]; partial[3 * (long)blockIdx.x + 1] = red[1][0]; partial[3 * (long)blockIdx.x + 2] = red[2][0]; }
}

// sums the per-block partial triples in a fixed order (one block) and ADDS them to acc[0..2]
__global__ void __launch_bounds__(256) diag_reduce_kernel(const double* __restrict__ partial, long nblocks, double* __restrict__ acc) {
  __shared__ double red[3][256];
  double s0 = 0.0, s1 = 0.0, s2 = 0.0;
  for (long b = threadIdx.x; b < nblocks; b += 256) { s0 += partial[3 * b]; s1 += partial[3 * b + 1]; s2 += partial[3 * b + 2]; }
  red[0][threadIdx.x] = s0; red[1][threadIdx.x] = s1; red[2][threadIdx.x] = s2;
  __syncthreads();
  for (int w = 128; w > 0; w >>= 1) {
    if (threadIdx.x < w) {
#pragma unroll
      for (int c = 0; c < 3; c++) red[c][threadIdx.x] += red[c][threadIdx.x + w];
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) { acc[0] += red[0][0]; acc[1] += red[1][0]; acc[2] += red[2][0]; }
}

// ------------------------------------------------------------------------------------------------ flux
// Thread per (cell, Gauss point q of the + face of AXIS); blockIdx.y = q.  PAPER.md:33-92, 330-352.
// stage 2 stores only the time derivatives (reading T4).
// Persistent blocks: each block walks over tiles of FLUX_TPB points (cells x Gauss point q of the + face of AXIS).
// The 2 x 20 inputs of a point are staged by the owning thread itself with cp.async into its own column of a
// shared-memory tile (refilled for the next tile as soon as it has been read into registers), one tile ahead, so the DRAM latency of the loads is hidden
// behind the ~2000 FP64 instructions of the previous point (no block-level synchronisation is needed: a thread only
// reads what it copied).
__device__ __forceinline__ void cp_async16(double* smem_dst, const double* gsrc) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
  const size_t ga = __cvta_generic_to_global(gsrc);          // the instruction takes a .global address, not a generic one
  asm volatile("cp.async.ca.shared.global [%0], [%1], 16;\n" ::"r"(sa), "l"(ga) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

constexpr int FLUX_TPB = 128;
constexpr int FLUX_SMEM_BYTES = 40 * FLUX_TPB * 8;      // one tile: a thread refills its column right after reading it

struct FluxPoint { int q; long t; CellIdx x; int ir, jr, kr; long offL, offR; };

template <int AXIS>
__device__ __forceinline__ bool flux_point(const Mesh& m, const Slab& sl, long tile, long tiles_per_q, long ncells, int kA, FluxPoint& f) {
  const unsigned tq = (unsigned)tile / (unsigned)tiles_per_q;
  f.q = (int)tq;
  f.t = (long)(((unsigned)tile - tq * (unsigned)tiles_per_q) * (unsigned)FLUX_TPB + threadIdx.x);
  if (f.t >= ncells) return false;
  f.x = cell_of(m, f.t, kA);
  f.ir = f.x.i; f.jr = f.x.j; f.kr = f.x.k;
  if (AXIS == 0) f.ir = wrap(f.x.i + 1, m.ni); else if (AXIS == 1) f.jr = wrap(f.x.j + 1, m.nj); else f.kr = wrap(f.x.k + 1, m.nk);
  f.offL = (long)slot_of(m, sl, f.x.k) * m.plane + f.x.ij;
  f.offR = (long)slot_of(m, sl, f.kr) * m.plane + (long)f.jr * m.ni + f.ir;
  return true;
}

template <bool CART, int AXIS, bool STAGE2>
__global__ void __launch_bounds__(FLUX_TPB, FLUX_MINB) flux_kernel(Mesh m, Slab sl, const double* __restrict__ W, const double* __restrict__ pv,
                                                   double* __restrict__ fx, GasConst gc, double dt, double idt, int kA, long ncells) {
  extern __shared__ __align__(16) double smf[];       // [20 chunks][FLUX_TPB][2]
  const long tiles_per_q = (ncells + FLUX_TPB - 1) / FLUX_TPB;
  const long ntiles = 4 * tiles_per_q;
  // returns whether this thread has a point in `tile`; its q and left offset are carried to the compute phase
  auto issue = [&](long tile, int& q_out, long& offL_out, long& c_out) -> bool {
    FluxPoint f;
    const bool act = tile < ntiles && flux_point<AXIS>(m, sl, tile, tiles_per_q, ncells, kA, f);
    if (act) {
      // chunk (side, variable, half) = 16 bytes: { value, d/dx } or { d/dy, d/dz }; tile layout [20 chunks][FLUX_TPB][2]
      const double* pL = pv + pv_index(sl, 4 * (2 * AXIS) + f.q, 0, f.offL);
      const double* pR = pv + pv_index(sl, 4 * (2 * AXIS + 1) + f.q, 0, f.offR);
      double* dst = smf + 2 * threadIdx.x;
#pragma unroll
      for (int c = 0; c < 10; c++) cp_async16(dst + c * (2 * FLUX_TPB), pL + (long)(c >> 1) * (4 * sl.stride_pv) + 2 * (c & 1));
#pragma unroll
      for (int c = 0; c < 10; c++) cp_async16(dst + (10 + c) * (2 * FLUX_TPB), pR + (long)(c >> 1) * (4 * sl.stride_pv) + 2 * (c & 1));
      q_out = f.q; offL_out = f.offL; c_out = f.x.c;
    }
    cp_async_commit();
    return act;
  };
  int q = 0, qn = 0;
  long offL = 0, offLn = 0, cL = 0, cLn = 0;
  bool active = issue(blockIdx.x, q, offL, cL), activen = false;
#pragma unroll 1
  for (long tile = blockIdx.x; tile < ntiles; tile += gridDim.x, q = qn, offL = offLn, cL = cLn, active = activen) {
  cp_async_wait<0>();
  const double2* sL = reinterpret_cast<const double2*>(smf) + threadIdx.x;
  double WLg[5], WRg[5], gL[15], gR[15];
#pragma unroll
  for (int v = 0; v < 5; v++) {
    const double2 l0 = sL[(2 * v) * FLUX_TPB], l1 = sL[(2 * v + 1) * FLUX_TPB];
    const double2 r0 = sL[(10 + 2 * v) * FLUX_TPB], r1 = sL[(11 + 2 * v) * FLUX_TPB];
    WLg[v] = l0.x; gL[3 * v] = l0.y; gL[3 * v + 1] = l1.x; gL[3 * v + 2] = l1.y;
    WRg[v] = r0.x; gR[3 * v] = r0.y; gR[3 * v + 1] = r1.x; gR[3 * v + 2] = r1.y;
  }
  activen = issue(tile + gridDim.x, qn, offLn, cLn);      // next tile's inputs stream in while this point is computed
  if (!active) continue;
  // positivity (reading R9, point-wise): a non-physical reconstructed state falls back to the cell average
  {
    if (!admissible(WLg)) {
#pragma unroll
      for (int c = 0; c < 5; c++) WLg[c] = W[iQG(c, cL, m.n)];
#pragma unroll
      for (int c = 0; c < 15; c++) gL[c] = 0.0;
    }
    if (!admissible(WRg)) {
      FluxPoint fp; flux_point<AXIS>(m, sl, tile, tiles_per_q, ncells, kA, fp);
      const long cr = cell_at(m, fp.ir, fp.jr, fp.kr);
#pragma unroll
      for (int c = 0; c < 5; c++) WRg[c] = W[iQG(c, cr, m.n)];
#pragma unroll
      for (int c = 0; c < 15; c++) gR[c] = 0.0;
    }
  }
  double WL[5], WR[5], SL[3][5], SR[3][5];
  double fr[3][3];       // rows: n, t1, t2 (general meshes)
  if (CART) {
    // face frame = cyclic permutation of the axes: n = e_AXIS, t1 = e_(AXIS+1), t2 = e_(AXIS+2)
    const int p0 = AXIS, p1 = (AXIS + 1) % 3, p2 = (AXIS + 2) % 3;
    const int pm[3] = { p0, p1, p2 };
    WL[0] = WLg[0]; WL[4] = WLg[4]; WR[0] = WRg[0]; WR[4] = WRg[4];
#pragma unroll
    for (int a = 0; a < 3; a++) { WL[1 + a] = WLg[1 + pm[a]]; WR[1 + a] = WRg[1 + pm[a]]; }
#pragma unroll
    for (int dd = 0; dd < 3; dd++) {
      SL[dd][0] = gL[pm[dd]]; SL[dd][4] = gL[12 + pm[dd]]; SR[dd][0] = gR[pm[dd]]; SR[dd][4] = gR[12 + pm[dd]];
#pragma unroll
      for (int a = 0; a < 3; a++) { SL[dd][1 + a] = gL[3 * (1 + pm[a]) + pm[dd]]; SR[dd][1 + a] = gR[3 * (1 + pm[a]) + pm[dd]]; }
    }
  } else {
    double A[3];
#pragma unroll
    for (int r = 0; r < 3; r++) { A[r] = m.met[(MET_AREA + 3 * AXIS + r) * m.n + cL]; fr[1][r] = m.met[(MET_TAN + 3 * AXIS + r) * m.n + cL]; }
    const double S = sqrt(A[0] * A[0] + A[1] * A[1] + A[2] * A[2]);
#pragma unroll
    for (int r = 0; r < 3; r++) fr[0][r] = A[r] / S;
    fr[2][0] = fr[0][1] * fr[1][2] - fr[0][2] * fr[1][1];
    fr[2][1] = fr[0][2] * fr[1][0] - fr[0][0] * fr[1][2];
    fr[2][2] = fr[0][0] * fr[1][1] - fr[0][1] * fr[1][0];
#pragma unroll
    for (int side = 0; side < 2; side++) {
      const double* Wg = side ? WRg : WLg; const double* gg = side ? gR : gL;
      double* Wl = side ? WR : WL; double (*Sx)[5] = side ? SR : SL;
      Wl[0] = Wg[0]; Wl[4] = Wg[4];
#pragma unroll
      for (int a = 0; a < 3; a++) Wl[1 + a] = Wg[1] * fr[a][0] + Wg[2] * fr[a][1] + Wg[3] * fr[a][2];
#pragma unroll
      for (int dd = 0; dd < 3; dd++) {
        double dg[5];
#pragma unroll
        for (int vv = 0; vv < 5; vv++) dg[vv] = gg[3 * vv] * fr[dd][0] + gg[3 * vv + 1] * fr[dd][1] + gg[3 * vv + 2] * fr[dd][2];
        Sx[dd][0] = dg[0]; Sx[dd][4] = dg[4];
#pragma unroll
        for (int a = 0; a < 3; a++) Sx[dd][1 + a] = dg[1] * fr[a][0] + dg[2] * fr[a][1] + dg[3] * fr[a][2];
      }
    }
  }
  double out[6][5];      // Fn, Ft, VL, DL, VR, DR in the face frame
  gks_flux_local<STAGE2>(gc, dt, idt, WL, SL, WR, SR, out[0], out[1], out[2], out[3], out[4], out[5]);
  double* dst = fx + (long)((4 * AXIS + q) * 30) * sl.stride_fx + offL;
#pragma unroll
  for (int g = 0; g < 6; g++) {
    if (STAGE2 && (g == 0 || g == 2 || g == 4)) continue;
    double o3[3];
    if (CART) {
      const int p0 = AXIS, p1 = (AXIS + 1) % 3, p2 = (AXIS + 2) % 3;
      o3[p0] = out[g][1]; o3[p1] = out[g][2]; o3[p2] = out[g][3];
    } else {
#pragma unroll
      for (int r = 0; r < 3; r++) o3[r] = out[g][1] * fr[0][r] + out[g][2] * fr[1][r] + out[g][3] * fr[2][r];
    }
    ST_STREAM(dst + (long)(5 * g) * sl.stride_fx, out[g][0]);
    ST_STREAM(dst + (long)(5 * g + 1) * sl.stride_fx, o3[0]);
    ST_STREAM(dst + (long)(5 * g + 2) * sl.stride_fx, o3[1]);
    ST_STREAM(dst + (long)(5 * g + 3) * sl.stride_fx, o3[2]);
    ST_STREAM(dst + (long)(5 * g + 4) * sl.stride_fx, out[g][4]);
  }
  }   // tile loop
}

// ------------------------------------------------------------------------------------------------ update
// Thread per (cell, variable).  Eq. 8-10 and the S2O4 combine.
//   stage 1: Wstar = stage value at t_n + dt/2;  Wsave = { Q^n + dt L^n + dt^2/6 L_t^n,  G,D sums of V^n }
//   stage 2: Wsave <- { Wsave.Q + dt^2/3 L_t^*,  Wsave.GD + dt * (G,D sums of Dt^*) }   (in place) = state at t_n+1
template <bool CART, int STAGE>
__global__ void __launch_bounds__(128) update_kernel(Mesh m, Slab sl, const double* __restrict__ fx, const double* __restrict__ Wcur,
                                                     double* __restrict__ Wstar, double* __restrict__ Wsave, double dt,
                                                     int kA, long nthreads) {
  constexpr int stage = STAGE;
  const long t = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nthreads) return;
  const int v = blockIdx.y;
  const CellIdx x = cell_of(m, t, kA);
  const long n = m.n;
  const long offP = (long)slot_of(m, sl, x.k) * m.plane + x.ij;
  double L = 0, Lt = 0, SG0[3] = { 0, 0, 0 }, SG1[3] = { 0, 0, 0 }, SD0[12], SD1[12];
  double vol;
  if (CART) vol = m.h[0] * m.h[1] * m.h[2]; else vol = m.met[MET_VOL * n + x.c];
#pragma unroll
  for (int ax = 0; ax < 3; ax++) {
    int im = x.i, jm = x.j, km = x.k;
    if (ax == 0) im = wrap(x.i - 1, m.ni); else if (ax == 1) jm = wrap(x.j - 1, m.nj); else km = wrap(x.k - 1, m.nk);
    const long offM = (long)slot_of(m, sl, km) * m.plane + (long)jm * m.ni + im;
    double Ap[3] = { 0, 0, 0 }, Am[3] = { 0, 0, 0 }, Sp, Sm;
    if (CART) { Sp = Sm = vol / m.h[ax]; Ap[ax] = Sp; Am[ax] = Sm; }
    else {
      const long cm = cell_at(m, im, jm, km);
#pragma unroll
      for (int r = 0; r < 3; r++) { Ap[r] = m.met[(MET_AREA + 3 * ax + r) * n + x.c]; Am[r] = m.met[(MET_AREA + 3 * ax + r) * n + cm]; }
      Sp = sqrt(Ap[0] * Ap[0] + Ap[1] * Ap[1] + Ap[2] * Ap[2]); Sm = sqrt(Am[0] * Am[0] + Am[1] * Am[1] + Am[2] * Am[2]);
    }
#pragma unroll
    for (int q = 0; q < 4; q++) {
      const double* fp = fx + (long)((4 * ax + q) * 30) * sl.stride_fx + offP;    // + face: this cell is the left side
      const double* fm = fx + (long)((4 * ax + q) * 30) * sl.stride_fx + offM;    // - face: this cell is the right side
      const double Ftp = fp[(long)(5 + v) * sl.stride_fx], Ftm = fm[(long)(5 + v) * sl.stride_fx];
      const double Dp = fp[(long)(15 + v) * sl.stride_fx], Dm = fm[(long)(25 + v) * sl.stride_fx];
      Lt -= 0.25 * (Ftp * Sp - Ftm * Sm);
      SD1[4 * ax + q] = Dp - Dm;
      if (CART) SG1[ax] += 0.25 * (Dp * Sp - Dm * Sm);
      else {
#pragma unroll
        for (int r = 0; r < 3; r++) SG1[r] += 0.25 * (Dp * Ap[r] - Dm * Am[r]);
      }
      if (stage == 1) {
        const double Fp = fp[(long)v * sl.stride_fx], Fm = fm[(long)v * sl.stride_fx];
        const double Vp = fp[(long)(10 + v) * sl.stride_fx], Vm = fm[(long)(20 + v) * sl.stride_fx];
        L -= 0.25 * (Fp * Sp - Fm * Sm);
        SD0[4 * ax + q] = Vp - Vm;
        if (CART) SG0[ax] += 0.25 * (Vp * Sp - Vm * Sm);
        else {
#pragma unroll
          for (int r = 0; r < 3; r++) SG0[r] += 0.25 * (Vp * Ap[r] - Vm * Am[r]);
        }
      }
    }
  }
  const double iv = 1.0 / vol;
  Lt *= iv;
#pragma unroll
  for (int r = 0; r < 3; r++) SG1[r] *= iv;
  if (stage == 1) {
    L *= iv;
#pragma unroll
    for (int r = 0; r < 3; r++) SG0[r] *= iv;
    const double qn = Wcur[iQG(v, x.c, n)];
    const double hdt = 0.5 * dt;
    st4(Wstar + iQG(v, x.c, n), qn + hdt * L + 0.125 * dt * dt * Lt, SG0[0] + hdt * SG1[0], SG0[1] + hdt * SG1[1], SG0[2] + hdt * SG1[2]);
    st4(Wsave + iQG(v, x.c, n), qn + dt * L + (1.0 / 6.0) * dt * dt * Lt, SG0[0], SG0[1], SG0[2]);
#pragma unroll
    for (int s = 0; s < 12; s += 4) {
      double* ds = Wstar + iD(v, s / 4, x.c, n) - s; double* dv = Wsave + iD(v, s / 4, x.c, n) - s;
      st4(ds + s, SD0[s] + hdt * SD1[s], SD0[s + 1] + hdt * SD1[s + 1], SD0[s + 2] + hdt * SD1[s + 2], SD0[s + 3] + hdt * SD1[s + 3]);
      st4(dv + s, SD0[s], SD0[s + 1], SD0[s + 2], SD0[s + 3]);
    }
  } else {
    double* qg = Wsave + iQG(v, x.c, n);
    double a0, a1, a2, a3;
    ld4(qg, a0, a1, a2, a3);
    st4(qg, a0 + (1.0 / 3.0) * dt * dt * Lt, a1 + dt * SG1[0], a2 + dt * SG1[1], a3 + dt * SG1[2]);
#pragma unroll
    for (int s = 0; s < 12; s += 4) {
      double* dv = Wsave + iD(v, s / 4, x.c, n) - s;
      ld4(dv + s, a0, a1, a2, a3);
      st4(dv + s, a0 + dt * SD1[s], a1 + dt * SD1[s + 1], a2 + dt * SD1[s + 2], a3 + dt * SD1[s + 3]);
    }
  }
}

}  // namespace cgks
