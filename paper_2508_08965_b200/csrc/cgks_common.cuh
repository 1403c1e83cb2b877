// cgks_common.cuh -- shared device-side definitions of the CGKS-5 hot path: mesh indexing, HBM layout, metrics.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace cgks {

// ---- HBM layout (all fp64, structure-of-arrays, i fastest) ---------------------------------------------------------
// state buffer        [80][N]      planes: Q v (0..4) | G 5+3v+r (5..19) | D 20+12v+s (20..79)
// metrics (general)   [37][N]      J0 3r+a (0..8) | J0^-1 9+3a+r... see MET_* | vol | +face vector areas | +face tangents
// pv (slab)           [24*5][slots*plane][4]   record (point p = 4m+q, variable v, cell slot) = { value, physical gradient (3) }
// fx (slab)           [360][slots*plane]   plane (4ax+q)*30 + c : Fn 0..4 | Ft 5..9 | VL 10..14 | DL 15..19 | VR 20..24 | DR 25..29
enum { NVAR = 5, NSTATE = 80, NPV = 480, NFX = 360, NMET = 37 };
enum { MET_J0 = 0, MET_J0INV = 9, MET_VOL = 18, MET_AREA = 19, MET_TAN = 28 };
__host__ __device__ inline int planeQ(int v) { return v; }
__host__ __device__ inline int planeG(int v, int r) { return 5 + 3 * v + r; }
__host__ __device__ inline int planeD(int v, int s) { return 20 + 12 * v + s; }

struct Mesh {
  int ni, nj, nk;
  long plane;        // ni*nj
  long n;            // ni*nj*nk
  int cart;          // 1: uniform Cartesian, metrics are the constants below
  double h[3];       // cell sizes (cart)
  const double* met; // [37][n] (general)
};

struct Slab {
  int kbase;         // plane held by slot 0
  int slots_pv, slots_fx;
  long stride_pv, stride_fx;   // slots*plane
};

__device__ __forceinline__ int wrap(int i, int n) { return i < 0 ? i + n : (i >= n ? i - n : i); }
__device__ __forceinline__ int slot_of(const Mesh& m, const Slab& s, int k) { int t = k - s.kbase; return t < 0 ? t + m.nk : t; }

// Positivity test of a reconstructed state (reading R9): admissible iff rho > 0 and rho (rho e) = rho E - |m|^2/2 > 0.
// The expression is evaluated with individually rounded operations in this fixed order (no FMA contraction), so that the
// decision is taken on bit-identical arithmetic wherever it is made.
__device__ __forceinline__ bool admissible(const double* w) {
  const double m2 = __dadd_rn(__dadd_rn(__dmul_rn(w[1], w[1]), __dmul_rn(w[2], w[2])), __dmul_rn(w[3], w[3]));
  const double re = __dsub_rn(__dmul_rn(w[0], w[4]), __dmul_rn(0.5, m2));
  return (w[0] > 0.0) && (re > 0.0);
}

struct CellIdx { int i, j, k; long ij; long c; };
// thread t over `cnt` planes starting at plane kA (wrapped).  32-bit index arithmetic: cgks_create rejects meshes with
// 2^31 cells or more (far beyond 180 GB of state), and 64-bit integer division costs ~100 instructions on the SM.
__device__ __forceinline__ CellIdx cell_of(const Mesh& m, long t, int kA) {
  CellIdx x;
  const unsigned tu = (unsigned)t, pl = (unsigned)m.plane, ni = (unsigned)m.ni;
  const unsigned kk = tu / pl, ij = tu - kk * pl, j = ij / ni;
  x.ij = ij; x.j = (int)j; x.i = (int)(ij - j * ni);
  x.k = kA + (int)kk; if (x.k >= m.nk) x.k -= m.nk;
  x.c = (long)x.k * m.plane + x.ij;
  return x;
}
__device__ __forceinline__ long cell_at(const Mesh& m, int i, int j, int k) { return ((long)k * m.nj + j) * m.ni + i; }

}  // namespace cgks
