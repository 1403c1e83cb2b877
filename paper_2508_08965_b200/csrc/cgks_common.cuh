// cgks_common.cuh -- shared device-side definitions of the CGKS-5 hot path: mesh indexing, HBM layout, metrics.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace cgks {

// ---- HBM layout (all fp64, structure-of-arrays, i fastest) ---------------------------------------------------------
// state buffer        80 N doubles: [5][N][4] records { Q_v, G_v (3) } (32 B), then [5][3][N][4] records of the four line
//                     differences D_v of one axis (32 B).  A neighbour's average and gradient arrive with ONE 256-bit load
//                     (one 32-byte sector), a cell's 12 line differences with three: 22 loads per (cell, variable) in the
//                     reconstruction instead of 85 with one plane per component; a sweep kernel (kernels_fused.cuh) touches
//                     exactly the record of its own axis, contiguous from cell to cell.
// metrics (general)   [37][N]      J0 3r+a (0..8) | J0^-1 9+3a+r... see MET_* | vol | +face vector areas | +face tangents
// pv (slab)           [24*5][slots*plane][4]   record (point p = 4m+q, variable v, cell slot) = { value, physical gradient (3) }
// fx (slab)           [360][slots*plane]   plane (4ax+q)*30 + c : Fn 0..4 | Ft 5..9 | VL 10..14 | DL 15..19 | VR 20..24 | DR 25..29
enum { NVAR = 5, NSTATE = 80, NPV = 480, NFX = 360, NMET = 37 };
enum { MET_J0 = 0, MET_J0INV = 9, MET_VOL = 18, MET_AREA = 19, MET_TAN = 28 };
// index of the first double of the records of (variable v, cell c) in a state buffer of n cells
__host__ __device__ inline long iQG(int v, long c, long n) { return ((long)v * n + c) * 4; }             // + 0: Q, + 1 + r: G_r
__host__ __device__ inline long iD(int v, int ax, long c, long n) { return 20 * n + ((long)(3 * v + ax) * n + c) * 4; }   // + q: D_(4 ax + q)
// field number f = 0..79 in the user order (Q v | G 5+3v+r | D 20+12v+s) -> index in the state buffer
__host__ __device__ inline long iField(int f, long c, long n) {
  if (f < 5) return iQG(f, c, n);
  if (f < 20) return iQG((f - 5) / 3, c, n) + 1 + (f - 5) % 3;
  const int s = (f - 20) % 12;
  return iD((f - 20) / 12, s / 4, c, n) + s % 4;
}

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

// 256-bit global loads / stores of four consecutive doubles (32-byte aligned)
__device__ __forceinline__ void ld4(const double* p, double& a, double& b, double& c, double& d) {
  asm volatile("ld.global.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(__cvta_generic_to_global(p)) : "memory");
}
__device__ __forceinline__ void st4(double* p, double a, double b, double c, double d) {
  asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(__cvta_generic_to_global(p)), "d"(a), "d"(b), "d"(c), "d"(d) : "memory");
}

// the same load from data the kernel never writes: non-coherent path, free for the compiler to schedule
__device__ __forceinline__ void ld4_ro(const double* p, double& a, double& b, double& c, double& d) {
  asm("ld.global.nc.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(__cvta_generic_to_global(p)));
}

// the same with an L2 evict-last policy: records that neighbouring cells will gather again (one plane of output later)
__device__ __forceinline__ unsigned long long l2_policy_evict_last() {
  unsigned long long p;
  asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ void ld4_ro_keep(const double* p, unsigned long long pol, double& a, double& b, double& c, double& d) {
  asm("ld.global.nc.L2::cache_hint.v4.f64 {%0, %1, %2, %3}, [%4], %5;" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(__cvta_generic_to_global(p)), "l"(pol));
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
