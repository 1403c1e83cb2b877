// kernels_fused.cuh -- the gas-kinetic flux (row a4) and the update / S2O4 combine (row a5) of a stage as ONE sweep kernel per
// face direction: the interface results never go to HBM (the fx buffer of the three-kernel split, 2880 / 1440 B per cell
// and stage written and read back, is gone, and with it the update kernel).
//
//   sweep_kernel<CART, AXIS, STAGE>   PAPER.md:33-92, 330-352 (Eq. 1-7) at the Gauss points of the + faces of direction AXIS,
//                                     then Eq. 8-10 restricted to the two faces of that direction and the
//                                     S2O4 combine, accumulated into the state buffers direction by direction.
//
// Mapping.  A WARP owns a tile of 8 cells along i x the 4 Gauss points of their + face of direction AXIS (lane = 4 cell + q)
// and marches along a line of such tiles in the direction AXIS, one tile per step.  The face computed in the previous step
// is the - face of the cells of this step: what it hands over (F^n, F_t^n and the right-hand interface values, 20 numbers
// per point) stays in shared memory -- for AXIS = 1, 2 in the thread's own slot; for AXIS = 0 a lane takes the slot of the lane
// four to its left, and the first cell of a tile takes a copy that the last cell of the step before left in front slots of the
// warp's row (by step parity), so the exchange has no lane-dependent branch.  Every line starts with one extra step (the face
// below its first cell: for AXIS = 0 the periodic image of the row's last face, computed by four lanes).
// The sums over the four Gauss points of a face (Eq. 8-9) are a reduce-scatter inside the quad (two shuffle rounds); lane q then owns
// component q of the cell's record { Q, G_x, G_y, G_z } and line difference 4 AXIS + q of the 12 (Eq. 10): a quad reads and
// writes whole 32-byte sectors.  Direction 0 of stage 1 writes the records, the later directions (and every direction of stage
// 2, which updates the saved buffer in place) read-modify-write them; these operands are prefetched with cp.async together
// with the 2 x 20 reconstructed inputs of the next step, one step ahead of the arithmetic.  No block-level synchronisation,
// no atomics: the order of every floating-point sum is fixed, results are deterministic and independent of the slab depth.
// General meshes: the face frame comes from metrics staged the same way, the - face's vector area travels with the hand-over.
#pragma once
#include "kernels_stage.cuh"

namespace cgks {

constexpr int SW_TPB = 128;                  // 4 warps; FLUX_MINB blocks per SM (254 registers per thread)
constexpr int SW_CELLS = 8;                  // cells per warp tile
constexpr int SW_SMEM_IN = 40 * SW_TPB;      // doubles: staged inputs [20 chunks][SW_TPB][2]
// Shared memory of a block, in doubles (the sizes depend on the kernel: the Cartesian kernels must stay at or below 81 KB per block,
// the configuration that leaves 92 KB of L1; profiles/r02e_experiments.md):
//   staged inputs      [20 chunks][SW_TPB][2]
//   hand-over values   [rows][row length]: rows = 20 (stage 1) or 10 (stage 2: time derivatives only), + 4 on general meshes (vector
//                      area and area of the face); a row holds one slot per thread, and for AXIS = 0 per warp 8 more in front of its
//                      32: the values of its last cell of the step before, by step parity (the first cell of a tile takes them)
//   read-modify-write operands [2 (step parity)][rows][SW_TPB]: rows = 5 for the first direction of stage 1 (Q^n only), else 10
//   face metrics       general meshes only: [2 (step parity)][7][SW_TPB] (+ face vector area, tangent, cell volume)
__host__ __device__ constexpr int sw_x_warp(int axis) { return axis == 0 ? 40 : 32; }                 // hand-over slots per warp in a row
__host__ __device__ constexpr int sw_x_row(int axis) { return sw_x_warp(axis) * (SW_TPB / 32); }
__host__ __device__ constexpr int sw_x_rows(bool cart, int stage) { return (stage == 2 ? 10 : 20) + (cart ? 0 : 4); }
__host__ __device__ constexpr int sw_smem_x(bool cart, int axis, int stage) { return sw_x_rows(cart, stage) * sw_x_row(axis); }
__host__ __device__ constexpr int sw_rmw_rows(int axis, int stage) { return (axis == 0 && stage == 1) ? 5 : 10; }
__host__ __device__ constexpr int sw_smem_rmw(int axis, int stage) { return 2 * sw_rmw_rows(axis, stage) * SW_TPB; }
__host__ __device__ constexpr int sw_smem_met(bool cart) { return cart ? 0 : 2 * 7 * SW_TPB; }
__host__ __device__ constexpr int sw_smem_bytes(bool cart, int axis, int stage) {
  return (SW_SMEM_IN + sw_smem_x(cart, axis, stage) + sw_smem_rmw(axis, stage) + sw_smem_met(cart)) * 8;
}

struct SweepPrm {
  int kA, cnt;       // planes kA .. kA+cnt-1 (wrapped) are updated
  int seg, nseg;     // lines along AXIS = 1 (j) or 2 (k) are cut into nseg segments of seg cells
  int ntx;           // tiles per row: ceil(ni / 8)
  int nlines;
};

__device__ __forceinline__ void cp_async8(double* smem_dst, const double* gsrc) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
  const size_t ga = __cvta_generic_to_global(gsrc);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(sa), "l"(ga) : "memory");
}

// a line and this lane's cell at its step 0
struct SweepLine { int len, i, j, k; };

template <int AXIS>
__device__ __forceinline__ SweepLine sweep_line(const Mesh& m, const SweepPrm& sp, int line, int cl) {
  SweepLine L;
  const unsigned u = (unsigned)line;
  if (AXIS == 0) {
    const unsigned kk = u / (unsigned)m.nj;
    L.j = (int)(u - kk * (unsigned)m.nj); L.k = sp.kA + (int)kk; L.i = cl; L.len = sp.ntx;
  } else if (AXIS == 1) {
    const unsigned a = u / (unsigned)sp.ntx, tx = u - a * (unsigned)sp.ntx;
    const unsigned kk = a / (unsigned)sp.nseg, sg = a - kk * (unsigned)sp.nseg;
    L.i = (int)tx * SW_CELLS + cl; L.j = (int)sg * sp.seg; L.k = sp.kA + (int)kk;
    L.len = m.nj - L.j < sp.seg ? m.nj - L.j : sp.seg;
  } else {
    const unsigned a = u / (unsigned)sp.ntx, tx = u - a * (unsigned)sp.ntx;
    const unsigned sg = a / (unsigned)m.nj, j = a - sg * (unsigned)m.nj;
    const int kk0 = (int)sg * sp.seg;
    L.i = (int)tx * SW_CELLS + cl; L.j = (int)j; L.k = sp.kA + kk0;
    L.len = sp.cnt - kk0 < sp.seg ? sp.cnt - kk0 : sp.seg;
  }
  if (L.k >= m.nk) L.k -= m.nk;
  return L;
}

// this lane's left cell (cL), the cell across the + face (cR) and their slab offsets at step s (-1: the line's extra first face)
struct SweepPos { bool act; int cL, cR; long offL, offR; };

template <int AXIS>
__device__ __forceinline__ SweepPos sweep_pos(const Mesh& m, const Slab& sl, const SweepLine& L, int s, int cl) {
  SweepPos p;
  int i = L.i, j = L.j, k = L.k;
  if (AXIS == 0) {
    if (s < 0) { i = m.ni - 1; p.act = (cl == SW_CELLS - 1); }
    else { i = L.i + SW_CELLS * s; p.act = i < m.ni; }
  } else {
    p.act = i < m.ni;
    if (AXIS == 1) j = wrap(j + s, m.nj); else k = wrap(k + s, m.nk);
  }
  int ir = i, jr = j, kr = k;
  if (AXIS == 0) ir = wrap(i + 1, m.ni); else if (AXIS == 1) jr = wrap(j + 1, m.nj); else kr = wrap(k + 1, m.nk);
  const int ijL = j * m.ni + i, ijR = jr * m.ni + ir;
  p.cL = k * (int)m.plane + ijL; p.cR = kr * (int)m.plane + ijR;
  p.offL = (long)slot_of(m, sl, k) * m.plane + ijL;
  p.offR = (long)slot_of(m, sl, kr) * m.plane + ijR;
  return p;
}

template <bool CART, int AXIS, int STAGE>
__global__ void __launch_bounds__(SW_TPB, FLUX_MINB) sweep_kernel(Mesh m, Slab sl, SweepPrm sp, const double* __restrict__ Win,
                                                                  const double* __restrict__ pv, const double* Wcur, double* Wstar,
                                                                  double* Wsave, GasConst gc, double dt, double idt) {
  constexpr bool STAGE2 = (STAGE == 2);
  constexpr bool FIRST = (STAGE == 1 && AXIS == 0);      // writes the records instead of accumulating into them
  extern __shared__ __align__(16) double sm[];
  double* smf = sm;                                      // staged inputs
  double* smx = sm + SW_SMEM_IN;                         // hand-over values
  double* smr = sm + SW_SMEM_IN + sw_smem_x(CART, AXIS, STAGE);       // read-modify-write operands
  double* smm = smr + sw_smem_rmw(AXIS, STAGE);                       // face metrics of the step (general meshes)
  constexpr int RR = sw_rmw_rows(AXIS, STAGE);                        // rows of one parity of the read-modify-write operands
  constexpr int XR = sw_x_row(AXIS);                                  // row length of the hand-over buffer
  const int tid = threadIdx.x, lane = tid & 31, q = lane & 3, cl = lane >> 2;
  const int gw = blockIdx.x * (SW_TPB / 32) + (tid >> 5), nw = gridDim.x * (SW_TPB / 32);
  const long n = m.n;

  // ---- staging of one step's inputs: 2 x 5 records of the reconstruction + the operands of the read-modify-write
  auto issue = [&](const SweepPos& p, int s, int par) {
    if (p.act) {
      const double* pL = pv + pv_index(sl, 4 * (2 * AXIS) + q, 0, p.offL);
      const double* pR = pv + pv_index(sl, 4 * (2 * AXIS + 1) + q, 0, p.offR);
      double* dst = smf + 2 * tid;
#pragma unroll
      for (int c = 0; c < 10; c++) cp_async16(dst + c * (2 * SW_TPB), pL + (long)(c >> 1) * (4 * sl.stride_pv) + 2 * (c & 1));
#pragma unroll
      for (int c = 0; c < 10; c++) cp_async16(dst + (10 + c) * (2 * SW_TPB), pR + (long)(c >> 1) * (4 * sl.stride_pv) + 2 * (c & 1));
      if (!CART) {
        double* mt = smm + par * (7 * SW_TPB) + tid;
#pragma unroll
        for (int r = 0; r < 3; r++) {
          cp_async8(mt + r * SW_TPB, m.met + (MET_AREA + 3 * AXIS + r) * n + p.cL);
          cp_async8(mt + (3 + r) * SW_TPB, m.met + (MET_TAN + 3 * AXIS + r) * n + p.cL);
        }
        cp_async8(mt + 6 * SW_TPB, m.met + MET_VOL * n + p.cL);
      }
      if (s >= 0) {
        double* r = smr + par * (RR * SW_TPB) + tid;
        const long oq = 4 * (long)p.cL + q, sq = 4 * n;
        if (FIRST) {
          if (q == 0) {
#pragma unroll
            for (int v = 0; v < 5; v++) cp_async8(r + v * SW_TPB, Wcur + oq + v * sq);
          }
        } else if (!STAGE2) {
#pragma unroll
          for (int v = 0; v < 5; v++) { cp_async8(r + v * SW_TPB, Wstar + oq + v * sq); cp_async8(r + (5 + v) * SW_TPB, Wsave + oq + v * sq); }
        } else {
          const long od = iD(0, AXIS, p.cL, n) + q, sd = 12 * n;
#pragma unroll
          for (int v = 0; v < 5; v++) { cp_async8(r + v * SW_TPB, Wsave + oq + v * sq); cp_async8(r + (5 + v) * SW_TPB, Wsave + od + v * sd); }
        }
      }
    }
    cp_async_commit();
  };

  int line = gw, s = -1, par = 0;
  if (line >= sp.nlines) return;
  SweepLine L = sweep_line<AXIS>(m, sp, line, cl);
  SweepPos cur = sweep_pos<AXIS>(m, sl, L, s, cl);
  issue(cur, s, par);
#pragma unroll 1
  while (line < sp.nlines) {
    cp_async_wait<0>();
    const double2* sL = reinterpret_cast<const double2*>(smf) + tid;
    double WLg[5], WRg[5], gL[15], gR[15];
#pragma unroll
    for (int v = 0; v < 5; v++) {
      const double2 l0 = sL[(2 * v) * SW_TPB], l1 = sL[(2 * v + 1) * SW_TPB];
      const double2 r0 = sL[(10 + 2 * v) * SW_TPB], r1 = sL[(11 + 2 * v) * SW_TPB];
      WLg[v] = l0.x; gL[3 * v] = l0.y; gL[3 * v + 1] = l1.x; gL[3 * v + 2] = l1.y;
      WRg[v] = r0.x; gR[3 * v] = r0.y; gR[3 * v + 1] = r1.x; gR[3 * v + 2] = r1.y;
    }
    // general meshes: this face's frame (n, t1, t2), vector area A and area S from the staged metrics; built twice per step (before
    // and after the solver) instead of being carried through it in 26 registers
    auto face_frame = [&](double (*f)[3], double* A, double& S) {
      const double* mt = smm + par * (7 * SW_TPB) + tid;
#pragma unroll
      for (int r = 0; r < 3; r++) { A[r] = mt[r * SW_TPB]; f[1][r] = mt[(3 + r) * SW_TPB]; }
      const double AA = A[0] * A[0] + A[1] * A[1] + A[2] * A[2], iS = drsqrt(AA);     // branch-free; stale but finite on lanes without a cell
      S = AA * iS;
#pragma unroll
      for (int r = 0; r < 3; r++) f[0][r] = A[r] * iS;
      f[2][0] = f[0][1] * f[1][2] - f[0][2] * f[1][1];
      f[2][1] = f[0][2] * f[1][0] - f[0][0] * f[1][2];
      f[2][2] = f[0][0] * f[1][1] - f[0][1] * f[1][0];
    };
    // the step after this one (warp-uniform): its inputs stream in during the arithmetic of this one
    int nline = line, ns = s + 1;
    if (ns >= L.len) { nline = line + nw; ns = -1; if (nline < sp.nlines) L = sweep_line<AXIS>(m, sp, nline, cl); }
    SweepPos nxt; nxt.act = false; nxt.cL = 0; nxt.cR = 0; nxt.offL = 0; nxt.offR = 0;
    if (nline < sp.nlines) nxt = sweep_pos<AXIS>(m, sl, L, ns, cl);
    issue(nxt, ns, par ^ 1);

    // Lanes without a cell (ragged last tile, the extra first face of an i-line) run the arithmetic on whatever their staging
    // column holds and are masked at every global load and store: the warp stays converged, the shuffles need no mask logic.
    const bool act = cur.act;
    double P[4][5];       // this face, global frame: F^n, F_t^n, own-side (left) value and time derivative
    double R[2][5];       // right-hand interface value and time derivative: they belong to the next cell
    double A[3] = { 0, 0, 0 }, Sface = 0.0;      // general meshes: vector area and area of this face
    {
      // positivity (reading R9, point-wise): a non-physical reconstructed state falls back to the cell average
      if (act && !admissible(WLg)) {
#pragma unroll
        for (int c = 0; c < 5; c++) WLg[c] = Win[iQG(c, cur.cL, n)];
#pragma unroll
        for (int c = 0; c < 15; c++) gL[c] = 0.0;
      }
      if (act && !admissible(WRg)) {
#pragma unroll
        for (int c = 0; c < 5; c++) WRg[c] = Win[iQG(c, cur.cR, n)];
#pragma unroll
        for (int c = 0; c < 15; c++) gR[c] = 0.0;
      }
      double WL[5], WR[5], SL[3][5], SR[3][5];
      if (CART) {
        // face frame = cyclic permutation of the axes: n = e_AXIS, t1 = e_(AXIS+1), t2 = e_(AXIS+2)
        const int pm[3] = { AXIS, (AXIS + 1) % 3, (AXIS + 2) % 3 };
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
        double fr[3][3], A0[3], S0;
        face_frame(fr, A0, S0);
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
      // back to the global frame
      double fr[3][3];
      if (!CART) face_frame(fr, A, Sface);
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
        double* d = (g < 4) ? P[g] : R[g - 4];
        d[0] = out[g][0]; d[1] = o3[0]; d[2] = o3[1]; d[3] = o3[2]; d[4] = out[g][4];
      }
    }
    // ---- hand-over: M = what the face below this cell left (F^n, F_t^n, right-hand value and time derivative)
    double M[4][5];
    double Am[3] = { 0, 0, 0 }, Sm = 0;      // general meshes: vector area and area of the - face (the + face of the cell below)
    {
      // Unconditional: a lane without a cell hands over (and takes) numbers nobody uses.  AXIS = 1, 2: the thread's own slot.
      // AXIS = 0: the slot of the lane four to the left; the first cell of the tile takes the copy that the last cell of the step
      // before left in the warp's 2 x 4 front slots (by step parity): no lane-dependent branch around the loads.
      const int wslot = (tid >> 5) * sw_x_warp(AXIS);
      double* xs = smx + wslot + (AXIS == 0 ? 8 + lane : lane);
      auto put = [&](double* dst) {
        if (!CART) {
#pragma unroll
          for (int r = 0; r < 3; r++) dst[(sw_x_rows(true, STAGE) + r) * XR] = A[r];
          dst[(sw_x_rows(true, STAGE) + 3) * XR] = Sface;
        }
        if (!STAGE2) {
#pragma unroll
          for (int v = 0; v < 5; v++) { dst[v * XR] = P[0][v]; dst[(5 + v) * XR] = P[1][v]; dst[(10 + v) * XR] = R[0][v]; dst[(15 + v) * XR] = R[1][v]; }
        } else {
#pragma unroll
          for (int v = 0; v < 5; v++) { dst[v * XR] = P[1][v]; dst[(5 + v) * XR] = R[1][v]; }
        }
      };
      auto get = [&](const double* src) {
        if (!CART) {
#pragma unroll
          for (int r = 0; r < 3; r++) Am[r] = src[(sw_x_rows(true, STAGE) + r) * XR];
          Sm = src[(sw_x_rows(true, STAGE) + 3) * XR];
        }
        if (!STAGE2) {
#pragma unroll
          for (int v = 0; v < 5; v++) { M[0][v] = src[v * XR]; M[1][v] = src[(5 + v) * XR]; M[2][v] = src[(10 + v) * XR]; M[3][v] = src[(15 + v) * XR]; }
        } else {
#pragma unroll
          for (int v = 0; v < 5; v++) { M[1][v] = src[v * XR]; M[3][v] = src[(5 + v) * XR]; }
        }
      };
      if (AXIS == 0) {
        __syncwarp();      // the neighbours have taken what this lane left in the step before
        put(xs);
        if (cl == SW_CELLS - 1) put(smx + wslot + 4 * par + q);
        __syncwarp();
        get(cl == 0 ? smx + wslot + 4 * (par ^ 1) + q : xs - 4);
      } else {
        get(xs);
        put(xs);
      }
    }
    if (s >= 0) {
      // ---- Eq. 8-10 restricted to the two faces of this direction, S2O4 combine
      double cf;
      const double* Ap = A; const double Sp = Sface;
      if (CART) cf = 0.25 / m.h[AXIS]; else cf = 0.25 * drcp(smm[par * (7 * SW_TPB) + 6 * SW_TPB + tid]);      // 1/(4 |Omega|)
      const double hdt = 0.5 * dt;
      const double* rb = smr + par * (RR * SW_TPB) + tid;
      const int comp = q - 1;      // gradient component owned by this lane (q = 0: the cell average)
      // this lane's component of the records of variable 0; the next variable is 4 n (records) / 12 n (line differences) further
      const long oq = 4 * (long)cur.cL + q, od = iD(0, AXIS, cur.cL, n) + q;
      double* pq_star = Wstar + oq; double* pq_save = Wsave + oq; double* pd_star = Wstar + od; double* pd_save = Wsave + od;
      const long sq = 4 * n, sd = 12 * n;
      double o_q0[5], o_q1[5], o_d0[5], o_d1[5];      // what this lane writes: record component and line difference, W* and saved buffer
#pragma unroll
      for (int v = 0; v < 5; v++) {
        // sums over the four Gauss points of the face pair
        double sF = 0, sFt, sV[3] = { 0, 0, 0 }, sD[3];
        const double d1 = P[3][v] - M[3][v];
        double d0 = 0;
        if (!STAGE2) d0 = P[2][v] - M[2][v];
        if (CART) {
          // Only lane 0 of the quad needs the flux sums (its component is Q) and only lane 1 + AXIS the sums of the interface
          // values (its component is G_AXIS): a reduce-scatter.  Each lane keeps one of the two kinds and hands the other to
          // its xor-1 partner, then the two lanes that keep the same kind add up: half the shuffles of four full butterflies,
          // and the same order of additions, (q0 + q1) + (q2 + q3), in the lane that uses the sum.
          const bool keepF = (AXIS == 1) ? (q == 0 || q == 3) : ((q & 1) == 0);
          constexpr int PAIR = (AXIS == 1) ? 3 : 2;
          const double fT = P[1][v] - M[1][v];
          double kT = keepF ? fT : d1;
          kT += __shfl_xor_sync(0xffffffffu, keepF ? d1 : fT, 1);
          kT += __shfl_xor_sync(0xffffffffu, kT, PAIR);
          sFt = kT; sD[0] = kT;
          if (!STAGE2) {
            const double fN = P[0][v] - M[0][v];
            double kN = keepF ? fN : d0;
            kN += __shfl_xor_sync(0xffffffffu, keepF ? d0 : fN, 1);
            kN += __shfl_xor_sync(0xffffffffu, kN, PAIR);
            sF = kN; sV[0] = kN;
          }
        } else {
          // General meshes: lane 0 needs the two flux sums, lane 1 + r the sums of (interface value) x (component r of the
          // vector areas): four kinds, one per lane.  Reduce-scatter in two rounds: the halves of the quad exchange the two
          // kinds that belong to the other half (xor 2), then the partners exchange the other's kind (xor 1).
          double kT[4], kN[4];
          kT[0] = P[1][v] * Sp - M[1][v] * Sm;
#pragma unroll
          for (int r = 0; r < 3; r++) kT[1 + r] = P[3][v] * Ap[r] - M[3][v] * Am[r];
          if (!STAGE2) {
            kN[0] = P[0][v] * Sp - M[0][v] * Sm;
#pragma unroll
            for (int r = 0; r < 3; r++) kN[1 + r] = P[2][v] * Ap[r] - M[2][v] * Am[r];
          }
          const bool hi = (q & 2) != 0, odd = (q & 1) != 0;
          auto rs = [&](const double* k) {
            double a = hi ? k[2] : k[0], b = hi ? k[3] : k[1];            // kinds of my half
            a += __shfl_xor_sync(0xffffffffu, hi ? k[0] : k[2], 2);
            b += __shfl_xor_sync(0xffffffffu, hi ? k[1] : k[3], 2);
            double mine = odd ? b : a;
            mine += __shfl_xor_sync(0xffffffffu, odd ? a : b, 1);
            return mine;                                                  // kind q, summed over the quad
          };
          const double tT = rs(kT);
          sFt = tT; sD[0] = tT; sD[1] = tT; sD[2] = tT;
          if (!STAGE2) { const double tN = rs(kN); sF = tN; sV[0] = tN; sV[1] = tN; sV[2] = tN; }
        }
        // this lane's component of the record { Q, G_x, G_y, G_z }: the increments of both kinds are formed and selected (no branch)
        double gV = 0.0, gD = 0.0;      // gradient sums of the values / of the time derivatives, this lane's component
        if (CART) { gV = (comp == AXIS) ? sV[0] : 0.0; gD = (comp == AXIS) ? sD[0] : 0.0; }
        else { gV = sV[0]; gD = sD[0]; }      // the reduce-scatter left this lane's kind in every entry
        if (!STAGE2) {
          const double iq_star = -cf * (hdt * sF + 0.125 * dt * dt * sFt), iq_save = -cf * (dt * sF + (1.0 / 6.0) * dt * dt * sFt);
          const double ig_star = cf * (gV + hdt * gD), ig_save = cf * gV;
          const double b0 = rb[v * SW_TPB];
          const double b_star = FIRST ? (q == 0 ? b0 : 0.0) : b0;
          const double b_save = FIRST ? b_star : rb[(RR - 5 + v) * SW_TPB];
          o_q0[v] = b_star + (q == 0 ? iq_star : ig_star);
          o_q1[v] = b_save + (q == 0 ? iq_save : ig_save);
          o_d0[v] = d0 + hdt * d1;
          o_d1[v] = d0;
        } else {
          const double inc = (q == 0) ? -cf * ((1.0 / 3.0) * dt * dt * sFt) : cf * (dt * gD);
          o_q1[v] = rb[v * SW_TPB] + inc;
          o_d1[v] = rb[(5 + v) * SW_TPB] + dt * d1;
        }
      }
      if (act) {
#pragma unroll
        for (int v = 0; v < 5; v++) {
          if (!STAGE2) { pq_star[v * sq] = o_q0[v]; pd_star[v * sd] = o_d0[v]; }
          pq_save[v * sq] = o_q1[v]; pd_save[v * sd] = o_d1[v];
        }
      }
    }
    line = nline; s = ns; cur = nxt; par ^= 1;
  }
}

}  // namespace cgks
