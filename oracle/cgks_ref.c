/*
 * cgks_ref.c -- CPU ORACLE for the CGKS-5 / S2O4 hot path.  TEST INFRASTRUCTURE ONLY.
 * See cgks_ref.h for scope and parity status.  Plain C, fp64, compiled with
 * -ffp-contract=off.  Loops over cells may be OpenMP-parallel; nothing else is
 * blocked, fused or reordered relative to the paper's statement of the algorithm.
 *
 * Citations are PAPER.md line numbers (+ equation).  "Reading Xn" refers to DESIGN.md section 3.
 */
#include "cgks_ref.h"
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#define NV 5
#define NB 34
#define ND 72
#define NGP 24
#define NROW_E 96

/* ------------------------------------------------------------------ */
/* Reference-cell constants                                            */
/* ------------------------------------------------------------------ */

/* ordering conventions (free: the LS solution does not depend on them)
   faces  m = 2*axis + (0:+, 1:-)
   edges  n = 4*z0 + 2*(s1>0) + (s2>0): parallel to axis z0, offsets s1,s2 along the two other axes (ascending)
   lines  s = 4*axis + 2*a + b: along axis, at (-g/+g, -g/+g) on the two other axes (ascending)
   points p = 4*m + 2*a + b on face m                                                             */
static int    g_didx[NB][3];
static double g_gp[NGP][3];
static double g_M[NB][ND];       /* a = M d                                  (Eq. 14 / 19)   */
static double g_E[NROW_E][NB];   /* value + 3 reference derivatives at the 24 Gauss points  */
static double g_Gram[4][NB][NB]; /* int over unit cube of sum_{|l|=o+1} D^l p_i D^l p_j     */
static int    g_face_off[6][3], g_edge_off[12][3], g_edge_axis[12];
static int    g_ready = 0;
/* Alternative readings of the paper's gaps, selectable so that oracle/readings_table.py can
   compare each of them with Tables 1-2.  The defaults are the readings taken (R5 normalised tau2, S3 sum over
   directions, G2 variant B); nothing but that script and its test changes them. */
static int    g_r5_normalised = 1;   /* R5: 1 tau2 = o/sqrt 2 (unit vector), 0 tau2 = o                               */
static int    g_s3_sum = 1;          /* S3: 1 rate = sum over directions, 0 rate = max over directions               */
static int    g_g2_variant = 1;      /* G2: 1 (B) IS^tau = third+fourth derivative part, 0 (A) IS^tau = |IS^H - IS^L|, 2 fourth part only */
void cgks_ref_set_readings(int r5_normalised, int s3_sum, int g2_variant) {
  if (r5_normalised != g_r5_normalised) g_ready = 0;      /* M is rebuilt at the next use */
  g_r5_normalised = r5_normalised; g_s3_sum = s3_sum; g_g2_variant = g2_variant;
}

static double factorial(int n) { double f = 1; for (int i = 2; i <= n; i++) f *= i; return f; }
/* int_a^b x^d/d! dx */
static double I1(int d, double a, double b) { return (pow(b, d + 1) - pow(a, d + 1)) / ((d + 1) * factorial(d)); }
static void other_axes(int ax, int* o1, int* o2) { *o1 = (ax == 0) ? 1 : 0; *o2 = (ax == 2) ? 1 : 2; }

/* average over the unit cube at integer offset o of the zero-mean basis function p_d (Eq. 13, reading R4) */
static double cellavg(const int d[3], const int o[3]) {
  double a = 1, m = 1;
  for (int i = 0; i < 3; i++) { a *= I1(d[i], o[i] - 0.5, o[i] + 0.5); m *= I1(d[i], -0.5, 0.5); }
  return a - m;
}
/* average over that cube of d p_d / d xi_ax */
static double cellavg_der(const int d[3], const int o[3], int ax) {
  if (d[ax] == 0) return 0.0;
  int dd[3] = { d[0], d[1], d[2] }; dd[ax]--;
  double a = 1;
  for (int i = 0; i < 3; i++) a *= I1(dd[i], o[i] - 0.5, o[i] + 0.5);
  return a;
}
static double mono(const int d[3], const double x[3]) {
  double a = 1;
  for (int i = 0; i < 3; i++) a *= pow(x[i], d[i]) / factorial(d[i]);
  return a;
}
static double basis_pt(const int d[3], const double x[3]) {
  double m = 1; for (int i = 0; i < 3; i++) m *= I1(d[i], -0.5, 0.5);
  return mono(d, x) - m;
}
static double basis_dpt(const int d[3], const double x[3], int ax) {
  if (d[ax] == 0) return 0.0;
  int dd[3] = { d[0], d[1], d[2] }; dd[ax]--;
  return mono(dd, x);
}

/* dense Gaussian elimination with partial pivoting: A (n x n) X = B (n x m), in place */
static int solve_dense(int n, int m, double* A, double* B) {
  for (int c = 0; c < n; c++) {
    int piv = c; double best = fabs(A[c * n + c]);
    for (int r = c + 1; r < n; r++) if (fabs(A[r * n + c]) > best) { best = fabs(A[r * n + c]); piv = r; }
    if (best == 0.0) return -1;
    if (piv != c) {
      for (int k = 0; k < n; k++) { double t = A[c * n + k]; A[c * n + k] = A[piv * n + k]; A[piv * n + k] = t; }
      for (int k = 0; k < m; k++) { double t = B[c * m + k]; B[c * m + k] = B[piv * m + k]; B[piv * m + k] = t; }
    }
    for (int r = c + 1; r < n; r++) {
      double f = A[r * n + c] / A[c * n + c];
      if (f == 0.0) continue;
      for (int k = c; k < n; k++) A[r * n + k] -= f * A[c * n + k];
      for (int k = 0; k < m; k++) B[r * m + k] -= f * B[c * m + k];
    }
  }
  for (int c = n - 1; c >= 0; c--) {
    for (int k = 0; k < m; k++) {
      double s = B[c * m + k];
      for (int r = c + 1; r < n; r++) s -= A[c * n + r] * B[r * m + k];
      B[c * m + k] = s / A[c * n + c];
    }
  }
  return 0;
}

static void init_constants(void) {
  if (g_ready) return;
  const double g = 0.5 / sqrt(3.0);
  /* basis multi-indices 1 <= |d| <= 4 : 34 of them */
  int nb = 0;
  for (int tot = 1; tot <= 4; tot++)
    for (int d1 = tot; d1 >= 0; d1--)
      for (int d2 = tot - d1; d2 >= 0; d2--) { g_didx[nb][0] = d1; g_didx[nb][1] = d2; g_didx[nb][2] = tot - d1 - d2; nb++; }
  /* stencil offsets */
  for (int m = 0; m < 6; m++) { for (int i = 0; i < 3; i++) g_face_off[m][i] = 0; g_face_off[m][m / 2] = (m % 2 == 0) ? 1 : -1; }
  for (int n = 0; n < 12; n++) {
    int z0 = n / 4, o1, o2; other_axes(z0, &o1, &o2);
    g_edge_axis[n] = z0; g_edge_off[n][z0] = 0;
    g_edge_off[n][o1] = ((n >> 1) & 1) ? 1 : -1; g_edge_off[n][o2] = (n & 1) ? 1 : -1;
  }
  /* face Gauss points (K = 4 per face) */
  for (int m = 0; m < 6; m++) {
    int ax = m / 2, o1, o2; other_axes(ax, &o1, &o2);
    for (int a = 0; a < 2; a++) for (int b = 0; b < 2; b++) {
      int p = 4 * m + 2 * a + b;
      g_gp[p][ax] = (m % 2 == 0) ? 0.5 : -0.5; g_gp[p][o1] = a ? g : -g; g_gp[p][o2] = b ? g : -g;
    }
  }
  /* rows of Eq. 14/19 on the ideal lattice (reading R4), scalings h1'=2, h2'=1, h3'=3 */
  const double h1 = 2.0, h2 = 1.0, h3 = 3.0;
  static double C[6][NB], L[ND - 6][NB];
  for (int b = 0; b < NB; b++) {
    int r = 0;
    for (int m = 0; m < 6; m++) C[m][b] = cellavg(g_didx[b], g_face_off[m]);               /* strict  */
    for (int n = 0; n < 12; n++) L[r++][b] = cellavg(g_didx[b], g_edge_off[n]);             /* LS      */
    for (int m = 0; m < 6; m++) for (int ax = 0; ax < 3; ax++) L[r++][b] = h1 * cellavg_der(g_didx[b], g_face_off[m], ax);
    for (int n = 0; n < 12; n++) {
      /* tau1 parallel to the shared edge; tau2 unit vector towards the neighbour's centroid (reading R5) */
      L[r++][b] = h2 * cellavg_der(g_didx[b], g_edge_off[n], g_edge_axis[n]);
      double s = 0;
      for (int ax = 0; ax < 3; ax++) s += g_edge_off[n][ax] * cellavg_der(g_didx[b], g_edge_off[n], ax);
      L[r++][b] = h2 * s / (g_r5_normalised ? sqrt(2.0) : 1.0);
    }
    for (int ax = 0; ax < 3; ax++) {
      int o1, o2; other_axes(ax, &o1, &o2);
      for (int a = 0; a < 2; a++) for (int bb = 0; bb < 2; bb++) {
        double x1[3], x2[3];
        x1[ax] = -0.5; x2[ax] = 0.5; x1[o1] = x2[o1] = a ? g : -g; x1[o2] = x2[o2] = bb ? g : -g;
        L[r++][b] = h3 * (basis_pt(g_didx[b], x2) - basis_pt(g_didx[b], x1));   /* 4th row of Eq. 19 */
      }
    }
  }
  /* constrained least squares: min |L a - l|^2 s.t. C a = c, via the KKT system
       [L^T L  C^T] [a  ]   [L^T l]
       [C      0  ] [lam] = [c    ]     solved once for the 72 unit right-hand sides -> M            */
  enum { NK = NB + 6, NL = ND - 6 };
  static double K[NK * NK], R[NK * ND];
  memset(K, 0, sizeof K); memset(R, 0, sizeof R);
  for (int i = 0; i < NB; i++) for (int j = 0; j < NB; j++) { double s = 0; for (int r = 0; r < NL; r++) s += L[r][i] * L[r][j]; K[i * NK + j] = s; }
  for (int m = 0; m < 6; m++) for (int i = 0; i < NB; i++) { K[i * NK + NB + m] = C[m][i]; K[(NB + m) * NK + i] = C[m][i]; }
  for (int i = 0; i < NB; i++) for (int r = 0; r < NL; r++) R[i * ND + 6 + r] = L[r][i];
  for (int m = 0; m < 6; m++) R[(NB + m) * ND + m] = 1.0;
  if (solve_dense(NK, ND, K, R) != 0) { fprintf(stderr, "cgks_ref: singular KKT system\n"); abort(); }
  for (int i = 0; i < NB; i++) for (int c = 0; c < ND; c++) g_M[i][c] = R[i * ND + c];
  /* evaluation matrix */
  for (int p = 0; p < NGP; p++) for (int b = 0; b < NB; b++) {
    g_E[4 * p][b] = basis_pt(g_didx[b], g_gp[p]);
    for (int ax = 0; ax < 3; ax++) g_E[4 * p + 1 + ax][b] = basis_dpt(g_didx[b], g_gp[p], ax);
  }
  /* Gram matrices of the smoothness indicators (h = |Omega| = 1 in reference space):
     D^l p_d = xi^(d-l)/(d-l)! when d >= l componentwise, else 0 */
  memset(g_Gram, 0, sizeof g_Gram);
  for (int l0 = 0; l0 <= 4; l0++) for (int l1 = 0; l0 + l1 <= 4; l1++) for (int l2 = 0; l0 + l1 + l2 <= 4; l2++) {
    int l[3] = { l0, l1, l2 }, ord = l0 + l1 + l2;
    if (ord < 1) continue;
    for (int i = 0; i < NB; i++) for (int j = 0; j < NB; j++) {
      double v = 1;
      for (int ax = 0; ax < 3 && v != 0.0; ax++) {
        int ei = g_didx[i][ax] - l[ax], ej = g_didx[j][ax] - l[ax];
        if (ei < 0 || ej < 0) { v = 0; break; }
        /* int_{-1/2}^{1/2} x^ei/ei! x^ej/ej! dx */
        int e = ei + ej;
        v *= (e % 2) ? 0.0 : 2.0 * pow(0.5, e + 1) / ((e + 1) * factorial(ei) * factorial(ej));
      }
      g_Gram[ord - 1][i][j] += v;
    }
  }
  g_ready = 1;
}

void cgks_ref_matrices(double* M, double* E) {
  init_constants();
  if (M) memcpy(M, g_M, sizeof g_M);
  if (E) memcpy(E, g_E, sizeof g_E);
}
void cgks_ref_basis(int* didx, double* gp) {
  init_constants();
  if (didx) memcpy(didx, g_didx, sizeof g_didx);
  if (gp) memcpy(gp, g_gp, sizeof g_gp);
}
void cgks_ref_smoothness(const double* a, double* IS4) {
  init_constants();
  for (int o = 0; o < 4; o++) {
    double s = 0;
    for (int i = 0; i < NB; i++) for (int j = 0; j < NB; j++) s += a[i] * g_Gram[o][i][j] * a[j];
    IS4[o] = s;
  }
}

/* ------------------------------------------------------------------ */
/* Reconstruction in reference space for one (cell, variable)          */
/* ------------------------------------------------------------------ */
void cgks_ref_recon_reference(const cgks_ref_params* p, const double* d, double* a, double* b,
                              double* chi_out, double* omega, double* val, double* gref) {
  init_constants();
  /* quartic polynomial: a = M d (Eq. 14 / 19); val/gref are relative to Q0 */
  for (int i = 0; i < NB; i++) { double s = 0; for (int c = 0; c < ND; c++) s += g_M[i][c] * d[c]; a[i] = s; }
  /* six linear polynomials (Eq. 15): strict on Q_{1,m}; LS on the 8 line derivatives perpendicular to
     the centroid line -> each tangential slope is the mean of the 4 (unscaled) line differences of that axis */
  double lineavg[3];
  for (int ax = 0; ax < 3; ax++) {
    double s = 0; for (int q = 0; q < 4; q++) s += d[60 + 4 * ax + q] / 3.0;   /* undo h3' */
    lineavg[ax] = s / 4.0;
  }
  for (int m = 0; m < 6; m++) {
    int ax = m / 2; double sgn = (m % 2 == 0) ? 1.0 : -1.0;
    for (int e = 0; e < 3; e++) b[3 * m + e] = lineavg[e];
    b[3 * m + ax] = sgn * d[m];
  }
  double chi = 1.0;
  for (int m = 0; m < 6; m++) omega[m] = 1.0 / 6.0;
  if (p->nonlinear) {
    const double eps = p->geno_eps;
    /* omega_m: IS_m = int |grad P_m|^2 = |b^m|^2 */
    double wsum = 0, wb[6];
    for (int m = 0; m < 6; m++) {
      double IS = b[3 * m] * b[3 * m] + b[3 * m + 1] * b[3 * m + 1] + b[3 * m + 2] * b[3 * m + 2];
      wb[m] = (1.0 / 6.0) / pow(IS + eps, 5);
      wsum += wb[m];
    }
    for (int m = 0; m < 6; m++) omega[m] = wb[m] / wsum;
    /* path function (readings G2: IS^tau = third+fourth derivative part, G3: C = geno_C) */
    double IS4[4]; cgks_ref_smoothness(a, IS4);
    double ISH = IS4[0] + IS4[1] + IS4[2] + IS4[3], ISL = IS4[0], ISt = IS4[2] + IS4[3];
    if (g_g2_variant == 0) ISt = fabs(ISH - ISL);   /* alternative reading G2 (A); never the default */
    if (g_g2_variant == 2) ISt = IS4[3];            /* negative control of oracle/readings_table.py: fourth-derivative part only */
    double aH = 1.0 + pow(ISt / (ISH + eps), p->geno_r), aL = 1.0 + pow(ISt / (ISL + eps), p->geno_r);
    double alpha = 2.0 * aH / (aH + aL);
    chi = tanh(p->geno_C * alpha) / tanh(p->geno_C);
  }
  *chi_out = chi;
  /* Eq. 16 at the 24 Gauss points */
  for (int pnt = 0; pnt < NGP; pnt++) {
    double v4 = 0, g4[3] = { 0, 0, 0 };
    for (int i = 0; i < NB; i++) {
      v4 += g_E[4 * pnt][i] * a[i];
      for (int ax = 0; ax < 3; ax++) g4[ax] += g_E[4 * pnt + 1 + ax][i] * a[i];
    }
    double v1 = 0, g1[3] = { 0, 0, 0 };
    for (int m = 0; m < 6; m++) {
      double pm = b[3 * m] * g_gp[pnt][0] + b[3 * m + 1] * g_gp[pnt][1] + b[3 * m + 2] * g_gp[pnt][2];
      v1 += omega[m] * pm;
      for (int ax = 0; ax < 3; ax++) g1[ax] += omega[m] * b[3 * m + ax];
    }
    val[pnt] = chi * v4 + (1.0 - chi) * v1;
    for (int ax = 0; ax < 3; ax++) gref[3 * pnt + ax] = chi * g4[ax] + (1.0 - chi) * g1[ax];
  }
}

/* ------------------------------------------------------------------ */
/* Context                                                             */
/* ------------------------------------------------------------------ */
struct cgks_ref_ctx {
  int ni, nj, nk; long n;
  cgks_ref_params prm;
  double *J0, *J0inv, *vol;     /* [n][9], [n][9], [n] */
  double *area, *tan1;          /* [3][n][3]: vector area and first tangent of the + face of each axis */
  double *Q, *G, *D;            /* current state */
  double *Qn, *Ln, *Ltn, *SG0, *SD0;   /* saved by stage 1 */
  double *Qs, *Gs, *Ds;         /* stage output */
  double *pv;                   /* [n][24][20] */
  double *fx;                   /* [3][n][4][30] */
  double *chi;                  /* [5][n] */
  long   nfall;                 /* Gauss-point states replaced by the positivity fallback (reading R9) in the last reconstruction */
  double fall_rho, fall_pe;     /* most negative rho / |rho_cell| and (rho E - |m|^2/2) / (rho E)_cell among them (0 if none)      */
  char err[256];
};

static inline long cidx(const cgks_ref_ctx* c, int i, int j, int k) {
  i = (i % c->ni + c->ni) % c->ni; j = (j % c->nj + c->nj) % c->nj; k = (k % c->nk + c->nk) % c->nk;   /* periodic */
  return ((long)k * c->nj + j) * c->ni + i;
}
static inline const double* node(const cgks_ref_ctx* c, const double* nodes, int comp, int i, int j, int k) {
  return nodes + (((long)comp * (c->nk + 1) + k) * (c->nj + 1) + j) * (c->ni + 1) + i;
}
static void getnode(const cgks_ref_ctx* c, const double* nodes, int i, int j, int k, double x[3]) {
  for (int r = 0; r < 3; r++) x[r] = *node(c, nodes, r, i, j, k);
}
static void cross(const double a[3], const double b[3], double o[3]) {
  o[0] = a[1] * b[2] - a[2] * b[1]; o[1] = a[2] * b[0] - a[0] * b[2]; o[2] = a[0] * b[1] - a[1] * b[0];
}
static double det3(const double m[9]) {
  return m[0] * (m[4] * m[8] - m[5] * m[7]) - m[1] * (m[3] * m[8] - m[5] * m[6]) + m[2] * (m[3] * m[7] - m[4] * m[6]);
}
static void inv3(const double m[9], double o[9]) {
  double d = det3(m);
  o[0] = (m[4] * m[8] - m[5] * m[7]) / d; o[1] = (m[2] * m[7] - m[1] * m[8]) / d; o[2] = (m[1] * m[5] - m[2] * m[4]) / d;
  o[3] = (m[5] * m[6] - m[3] * m[8]) / d; o[4] = (m[0] * m[8] - m[2] * m[6]) / d; o[5] = (m[2] * m[3] - m[0] * m[5]) / d;
  o[6] = (m[3] * m[7] - m[4] * m[6]) / d; o[7] = (m[1] * m[6] - m[0] * m[7]) / d; o[8] = (m[0] * m[4] - m[1] * m[3]) / d;
}

/* hexahedron volume: trilinear map + 3x3x3 Gauss quadrature (Appendix) */
static double hexa_volume(double X[8][3]) {
  /* X index = 4*(xi side) + 2*(eta side) + (zeta side), sides 0:-1/2, 1:+1/2, as psi_1..psi_8 in the Appendix */
  const double gq[3] = { -0.5 * sqrt(0.6), 0.0, 0.5 * sqrt(0.6) }, wq[3] = { 5.0 / 18.0, 8.0 / 18.0, 5.0 / 18.0 };
  double vol = 0;
  for (int l = 0; l < 3; l++) for (int m = 0; m < 3; m++) for (int n = 0; n < 3; n++) {
    double xi[3] = { gq[l], gq[m], gq[n] }, Jm[9];
    for (int r = 0; r < 3; r++) for (int a = 0; a < 3; a++) Jm[3 * r + a] = 0;
    for (int v = 0; v < 8; v++) {
      int s[3] = { (v >> 2) & 1, (v >> 1) & 1, v & 1 };
      double f[3], df[3];
      for (int a = 0; a < 3; a++) { double sg = s[a] ? 1.0 : -1.0; f[a] = 0.5 * (1 + 2 * sg * xi[a]); df[a] = sg; }
      double dpsi[3] = { df[0] * f[1] * f[2], f[0] * df[1] * f[2], f[0] * f[1] * df[2] };
      for (int r = 0; r < 3; r++) for (int a = 0; a < 3; a++) Jm[3 * r + a] += X[v][r] * dpsi[a];
    }
    vol += wq[l] * wq[m] * wq[n] * fabs(det3(Jm));
  }
  return vol;
}

cgks_ref_ctx* cgks_ref_create(int ni, int nj, int nk, const double* nodes, const cgks_ref_params* p) {
  init_constants();
  if (ni < 4 || nj < 4 || nk < 4 || !nodes || !p) return NULL;
  cgks_ref_ctx* c = (cgks_ref_ctx*)calloc(1, sizeof *c);
  c->ni = ni; c->nj = nj; c->nk = nk; c->n = (long)ni * nj * nk; c->prm = *p;
  long n = c->n;
  c->J0 = malloc(sizeof(double) * 9 * n); c->J0inv = malloc(sizeof(double) * 9 * n); c->vol = malloc(sizeof(double) * n);
  c->area = malloc(sizeof(double) * 9 * n); c->tan1 = malloc(sizeof(double) * 9 * n);
  c->Q = calloc(5 * n, sizeof(double)); c->G = calloc(15 * n, sizeof(double)); c->D = calloc(60 * n, sizeof(double));
  c->Qs = calloc(5 * n, sizeof(double)); c->Gs = calloc(15 * n, sizeof(double)); c->Ds = calloc(60 * n, sizeof(double));
  c->Qn = calloc(5 * n, sizeof(double)); c->Ln = calloc(5 * n, sizeof(double)); c->Ltn = calloc(5 * n, sizeof(double));
  c->SG0 = calloc(15 * n, sizeof(double)); c->SD0 = calloc(60 * n, sizeof(double));
  c->pv = malloc(sizeof(double) * n * NGP * 20); c->fx = malloc(sizeof(double) * 3 * n * 4 * 30); c->chi = calloc(5 * n, sizeof(double));
  for (int k = 0; k < nk; k++) for (int j = 0; j < nj; j++) for (int i = 0; i < ni; i++) {
    long ci = cidx(c, i, j, k);
    double N1[3], N2[3], N3[3], N4[3];
    /* Eq. 18 with reading R1: N1 = node(i,j,k), N2,N3,N4 its +i,+j,+k neighbours */
    getnode(c, nodes, i, j, k, N1); getnode(c, nodes, i + 1, j, k, N2); getnode(c, nodes, i, j + 1, k, N3); getnode(c, nodes, i, j, k + 1, N4);
    double* J = c->J0 + 9 * ci;
    for (int r = 0; r < 3; r++) { J[3 * r] = N2[r] - N1[r]; J[3 * r + 1] = N3[r] - N1[r]; J[3 * r + 2] = N4[r] - N1[r]; }
    if (!(det3(J) > 0)) { snprintf(c->err, sizeof c->err, "non-positive det J0 at cell %d %d %d", i, j, k); }
    inv3(J, c->J0inv + 9 * ci);
    double X[8][3];
    for (int v = 0; v < 8; v++) getnode(c, nodes, i + ((v >> 2) & 1), j + ((v >> 1) & 1), k + (v & 1), X[v]);
    c->vol[ci] = hexa_volume(X);
    /* + faces: vector area = half cross product of the diagonals (reading R2) */
    for (int ax = 0; ax < 3; ax++) {
      int e1 = (ax + 1) % 3, e2 = (ax + 2) % 3;       /* (ax,e1,e2) right-handed */
      int o[3] = { i, j, k }; o[ax] += 1;
      int ia[3] = { o[0], o[1], o[2] }, ib[3] = { o[0], o[1], o[2] }, ic[3] = { o[0], o[1], o[2] }, id[3] = { o[0], o[1], o[2] };
      ib[e1] += 1; ic[e1] += 1; ic[e2] += 1; id[e2] += 1;
      double a[3], b[3], cc[3], d[3], d1[3], d2[3], A[3];
      getnode(c, nodes, ia[0], ia[1], ia[2], a); getnode(c, nodes, ib[0], ib[1], ib[2], b);
      getnode(c, nodes, ic[0], ic[1], ic[2], cc); getnode(c, nodes, id[0], id[1], id[2], d);
      for (int r = 0; r < 3; r++) { d1[r] = cc[r] - a[r]; d2[r] = d[r] - b[r]; }
      cross(d1, d2, A);
      double* Af = c->area + ((long)ax * n + ci) * 3; double* t1 = c->tan1 + ((long)ax * n + ci) * 3;
      for (int r = 0; r < 3; r++) Af[r] = 0.5 * A[r];
      double S = sqrt(Af[0] * Af[0] + Af[1] * Af[1] + Af[2] * Af[2]), nrm[3] = { Af[0] / S, Af[1] / S, Af[2] / S };
      double e[3] = { b[0] - a[0], b[1] - a[1], b[2] - a[2] };
      double en = e[0] * nrm[0] + e[1] * nrm[1] + e[2] * nrm[2];
      for (int r = 0; r < 3; r++) e[r] -= en * nrm[r];
      double el = sqrt(e[0] * e[0] + e[1] * e[1] + e[2] * e[2]);
      for (int r = 0; r < 3; r++) t1[r] = e[r] / el;
    }
  }
  return c;
}

void cgks_ref_destroy(cgks_ref_ctx* c) {
  if (!c) return;
  free(c->J0); free(c->J0inv); free(c->vol); free(c->area); free(c->tan1);
  free(c->Q); free(c->G); free(c->D); free(c->Qs); free(c->Gs); free(c->Ds);
  free(c->Qn); free(c->Ln); free(c->Ltn); free(c->SG0); free(c->SD0);
  free(c->pv); free(c->fx); free(c->chi); free(c);
}
const char* cgks_ref_last_error(const cgks_ref_ctx* c) { return c ? c->err : "null context"; }

void cgks_ref_geometry(cgks_ref_ctx* c, double* vol, double* J0, double* area) {
  if (vol) memcpy(vol, c->vol, sizeof(double) * c->n);
  if (J0) memcpy(J0, c->J0, sizeof(double) * 9 * c->n);
  if (area) memcpy(area, c->area, sizeof(double) * 9 * c->n);
}

int cgks_ref_set_state(cgks_ref_ctx* c, const double* Q, const double* G, const double* D) {
  long n = c->n;
  memcpy(c->Q, Q, sizeof(double) * 5 * n);
  if (G && D) { memcpy(c->G, G, sizeof(double) * 15 * n); memcpy(c->D, D, sizeof(double) * 60 * n); return 0; }
  /* bootstrap of the derivative dof (reading S2; the paper is silent on initialisation) */
  for (int v = 0; v < NV; v++)
    for (int k = 0; k < c->nk; k++) for (int j = 0; j < c->nj; j++) for (int i = 0; i < c->ni; i++) {
      long ci = cidx(c, i, j, k);
      const double* q = c->Q + v * n;
      double dr[3];
      for (int ax = 0; ax < 3; ax++) {
        int o[3] = { 0, 0, 0 }; o[ax] = 1;
        double p1 = q[cidx(c, i + o[0], j + o[1], k + o[2])], m1 = q[cidx(c, i - o[0], j - o[1], k - o[2])];
        double p2 = q[cidx(c, i + 2 * o[0], j + 2 * o[1], k + 2 * o[2])], m2 = q[cidx(c, i - 2 * o[0], j - 2 * o[1], k - 2 * o[2])];
        dr[ax] = (8.0 * (p1 - m1) - (p2 - m2)) / 12.0;
      }
      const double* Ji = c->J0inv + 9 * ci;     /* grad = J0^-T grad' */
      if (!G) for (int r = 0; r < 3; r++) c->G[(v * 3 + r) * n + ci] = Ji[0 * 3 + r] * dr[0] + Ji[1 * 3 + r] * dr[1] + Ji[2 * 3 + r] * dr[2];
      if (!D) for (int s = 0; s < 12; s++) c->D[(v * 12 + s) * n + ci] = dr[s / 4];
    }
  if (G) memcpy(c->G, G, sizeof(double) * 15 * n);
  if (D) memcpy(c->D, D, sizeof(double) * 60 * n);
  return 0;
}
int cgks_ref_get_state(cgks_ref_ctx* c, double* Q, double* G, double* D) {
  long n = c->n;
  if (Q) memcpy(Q, c->Q, sizeof(double) * 5 * n);
  if (G) memcpy(G, c->G, sizeof(double) * 15 * n);
  if (D) memcpy(D, c->D, sizeof(double) * 60 * n);
  return 0;
}

/* ------------------------------------------------------------------ */
/* Step 1-4: reconstruct all cells                                      */
/* ------------------------------------------------------------------ */
static void reconstruct_all(cgks_ref_ctx* c) {
  const long n = c->n;
  c->nfall = 0; c->fall_rho = 0.0; c->fall_pe = 0.0;
#pragma omp parallel for collapse(2) schedule(static)
  for (int k = 0; k < c->nk; k++) for (int j = 0; j < c->nj; j++) for (int i = 0; i < c->ni; i++) {
    long ci = cidx(c, i, j, k);
    const double* J = c->J0 + 9 * ci; const double* Ji = c->J0inv + 9 * ci;
    double* pv = c->pv + ci * NGP * 20;
    for (int v = 0; v < NV; v++) {
      const double* q = c->Q + v * n;
      double q0 = q[ci], d[ND];
      /* data vector in reference space (Eq. 19, C_k = 1 by reading R3) */
      for (int m = 0; m < 6; m++) d[m] = q[cidx(c, i + g_face_off[m][0], j + g_face_off[m][1], k + g_face_off[m][2])] - q0;
      for (int e = 0; e < 12; e++) d[6 + e] = q[cidx(c, i + g_edge_off[e][0], j + g_edge_off[e][1], k + g_edge_off[e][2])] - q0;
      for (int m = 0; m < 6; m++) {
        long nb = cidx(c, i + g_face_off[m][0], j + g_face_off[m][1], k + g_face_off[m][2]);
        for (int a = 0; a < 3; a++) {
          double s = 0;   /* (grad Q)' = J0^T grad Q with the TARGET cell's J0 */
          for (int r = 0; r < 3; r++) s += J[3 * r + a] * c->G[(v * 3 + r) * n + nb];
          d[18 + 3 * m + a] = 2.0 * s;
        }
      }
      for (int e = 0; e < 12; e++) {
        long nb = cidx(c, i + g_edge_off[e][0], j + g_edge_off[e][1], k + g_edge_off[e][2]);
        double gr[3];
        for (int a = 0; a < 3; a++) { double s = 0; for (int r = 0; r < 3; r++) s += J[3 * r + a] * c->G[(v * 3 + r) * n + nb]; gr[a] = s; }
        d[36 + 2 * e] = 1.0 * gr[g_edge_axis[e]];
        d[36 + 2 * e + 1] = 1.0 * (g_edge_off[e][0] * gr[0] + g_edge_off[e][1] * gr[1] + g_edge_off[e][2] * gr[2]) / (g_r5_normalised ? sqrt(2.0) : 1.0);
      }
      for (int s = 0; s < 12; s++) d[60 + s] = 3.0 * c->D[(v * 12 + s) * n + ci];
      double a[NB], b[18], chi, om[6], val[NGP], gref[NGP * 3];
      cgks_ref_recon_reference(&c->prm, d, a, b, &chi, om, val, gref);
      c->chi[v * n + ci] = chi;
      for (int p = 0; p < NGP; p++) {
        pv[p * 20 + v] = q0 + val[p];
        for (int r = 0; r < 3; r++)   /* back-transform */
          pv[p * 20 + 5 + 3 * v + r] = Ji[0 * 3 + r] * gref[3 * p] + Ji[1 * 3 + r] * gref[3 * p + 1] + Ji[2 * 3 + r] * gref[3 * p + 2];
      }
    }
    /* positivity (reading R9, point-wise): a non-physical reconstructed state falls back to the cell average.
       Admissible means rho > 0 and rho * (rho e) = rho E - |m|^2/2 > 0, evaluated in exactly this order of
       operations (R9: the decision is taken on the same fp64 expression on both sides). */
    for (int p = 0; p < NGP; p++) {
      double* w = pv + p * 20;
      double rho = w[0], pe = w[0] * w[4] - 0.5 * ((w[1] * w[1] + w[2] * w[2]) + w[3] * w[3]);
      if (!(rho > 0.0) || !(pe > 0.0)) {
#pragma omp critical
        {   /* statistics only (cgks_ref_fallback_stats): how far outside the admissible set the replaced state was */
          double r0 = c->Q[ci], e0 = c->Q[ci] * c->Q[4 * n + ci];
          c->nfall++;
          if (rho / r0 < c->fall_rho) c->fall_rho = rho / r0;
          if (pe / e0 < c->fall_pe) c->fall_pe = pe / e0;
        }
        for (int v = 0; v < NV; v++) w[v] = c->Q[v * n + ci];
        for (int q = 5; q < 20; q++) w[q] = 0.0;
      }
    }
  }
}

void cgks_ref_fallback_stats(const cgks_ref_ctx* c, long* npoints, double* min_rho_rel, double* min_pe_rel) {
  *npoints = c->nfall; *min_rho_rel = c->fall_rho; *min_pe_rel = c->fall_pe;
}

int cgks_ref_reconstruct(cgks_ref_ctx* c, double* pv, double* chi) {
  reconstruct_all(c);
  if (pv) memcpy(pv, c->pv, sizeof(double) * c->n * NGP * 20);
  if (chi) memcpy(chi, c->chi, sizeof(double) * 5 * c->n);
  return 0;
}

/* ------------------------------------------------------------------ */
/* Step 5: gas-kinetic solver at one Gauss point                        */
/* ------------------------------------------------------------------ */
typedef struct { double u[7], v[7], w[7], xi[3]; } mom_t;

void cgks_ref_moments(double U, double lam, double* full, double* pos, double* neg) {
  /* <u^0>=1, <u^1>=U, <u^(n+2)> = U<u^(n+1)> + (n+1)/(2 lam) <u^n>; half-space start values from erfc / exp */
  const double PI = 3.14159265358979323846;
  double e = exp(-lam * U * U) / sqrt(PI * lam);
  if (full) { full[0] = 1.0; full[1] = U; }
  if (pos) { pos[0] = 0.5 * erfc(-sqrt(lam) * U); pos[1] = U * pos[0] + 0.5 * e; }
  if (neg) { neg[0] = 0.5 * erfc(sqrt(lam) * U); neg[1] = U * neg[0] - 0.5 * e; }
  for (int n = 0; n < 5; n++) {
    if (full) full[n + 2] = U * full[n + 1] + (n + 1) / (2.0 * lam) * full[n];
    if (pos) pos[n + 2] = U * pos[n + 1] + (n + 1) / (2.0 * lam) * pos[n];
    if (neg) neg[n + 2] = U * neg[n + 1] + (n + 1) / (2.0 * lam) * neg[n];
  }
}
static void mom_set(mom_t* m, double U, double V, double W, double lam, double K, int half) {
  if (half == 0) cgks_ref_moments(U, lam, m->u, NULL, NULL);
  else if (half > 0) cgks_ref_moments(U, lam, NULL, m->u, NULL);
  else cgks_ref_moments(U, lam, NULL, NULL, m->u);
  cgks_ref_moments(V, lam, m->v, NULL, NULL);
  cgks_ref_moments(W, lam, m->w, NULL, NULL);
  m->xi[0] = 1.0; m->xi[1] = K / (2.0 * lam); m->xi[2] = K * (K + 2.0) / (4.0 * lam * lam);
}
static double Mp(const mom_t* m, int i, int j, int k, int l) { return m->u[i] * m->v[j] * m->w[k] * m->xi[l]; }
/* < (a.psi) u^i v^j w^k xi^2l > */
static double Acal(const mom_t* m, const double a[5], int i, int j, int k, int l) {
  return a[0] * Mp(m, i, j, k, l) + a[1] * Mp(m, i + 1, j, k, l) + a[2] * Mp(m, i, j + 1, k, l) + a[3] * Mp(m, i, j, k + 1, l)
       + 0.5 * a[4] * (Mp(m, i + 2, j, k, l) + Mp(m, i, j + 2, k, l) + Mp(m, i, j, k + 2, l) + Mp(m, i, j, k, l + 1));
}
/* < (a.psi) u^i v^j w^k psi > */
static void mom_apsi(const mom_t* m, const double a[5], int i, int j, int k, double out[5]) {
  out[0] = Acal(m, a, i, j, k, 0);
  out[1] = Acal(m, a, i + 1, j, k, 0);
  out[2] = Acal(m, a, i, j + 1, k, 0);
  out[3] = Acal(m, a, i, j, k + 1, 0);
  out[4] = 0.5 * (Acal(m, a, i + 2, j, k, 0) + Acal(m, a, i, j + 2, k, 0) + Acal(m, a, i, j, k + 2, 0) + Acal(m, a, i, j, k, 1));
}
void cgks_ref_moment_apsi(const double* a, int i, int j, int k, double U, double V, double W, double lam,
                          double K, int half, double* out) {
  mom_t m; mom_set(&m, U, V, W, lam, K, half); mom_apsi(&m, a, i, j, k, out);
}
void cgks_ref_microslope(const double* h, double U, double V, double W, double lam, double K, double* a) {
  /* solves <(a.psi) psi> = h for a (standard GKS, refs [16,17] of the paper) */
  double s = U * U + V * V + W * W + (K + 3.0) / (2.0 * lam);
  double R4 = 2.0 * h[4] - s * h[0], R1 = h[1] - U * h[0], R2 = h[2] - V * h[0], R3 = h[3] - W * h[0];
  a[4] = 4.0 * lam * lam / (K + 3.0) * (R4 - 2.0 * U * R1 - 2.0 * V * R2 - 2.0 * W * R3);
  a[1] = 2.0 * lam * R1 - U * a[4];
  a[2] = 2.0 * lam * R2 - V * a[4];
  a[3] = 2.0 * lam * R3 - W * a[4];
  a[0] = h[0] - U * a[1] - V * a[2] - W * a[3] - 0.5 * a[4] * s;
}
typedef struct { double rho, U, V, W, lam, p; } prim_t;
static prim_t prim_of(const double w[5], double K) {
  prim_t q; q.rho = w[0]; q.U = w[1] / w[0]; q.V = w[2] / w[0]; q.W = w[3] / w[0];
  double e = w[4] - 0.5 * (w[1] * w[1] + w[2] * w[2] + w[3] * w[3]) / w[0];
  q.lam = (K + 3.0) * w[0] / (4.0 * e); q.p = q.rho / (2.0 * q.lam);    /* lambda = rho/(2p) */
  return q;
}
/* time-integrated coefficients of the six groups of Eq. 5 over [0,T] */
static void time_coef(double T, double tau, double cf[6]) {
  if (tau == 0.0) { cf[0] = T; cf[1] = 0; cf[2] = 0.5 * T * T; cf[3] = cf[4] = cf[5] = 0; return; }   /* reading T2 */
  double E = exp(-T / tau);
  cf[0] = T - tau * (1.0 - E);
  cf[1] = 2.0 * tau * tau * (1.0 - E) - tau * T * (1.0 + E);
  cf[2] = 0.5 * T * T - tau * T + tau * tau * (1.0 - E);
  cf[3] = tau * (1.0 - E);
  cf[4] = tau * T * E - 2.0 * tau * tau * (1.0 - E);
  cf[5] = -tau * tau * (1.0 - E);
}

void cgks_ref_flux_point(const cgks_ref_params* prm, double dt, const double* WLg, const double* gLg,
                         const double* WRg, const double* gRg, const double* nrm, const double* t1,
                         double* out) {
  const double K = (5.0 - 3.0 * prm->gamma) / (prm->gamma - 1.0);     /* N of PAPER.md:41 */
  double t2[3]; cross(nrm, t1, t2);
  const double* fr[3] = { nrm, t1, t2 };
  /* 1. rotate states and slopes into the face frame (n, t1, t2) */
  double WL[5], WR[5], sL[3][5], sR[3][5];
  for (int side = 0; side < 2; side++) {
    const double* Wg = side ? WRg : WLg; const double* gg = side ? gRg : gLg;
    double* Wl = side ? WR : WL; double (*sl)[5] = side ? sR : sL;
    Wl[0] = Wg[0]; Wl[4] = Wg[4];
    for (int a = 0; a < 3; a++) Wl[1 + a] = Wg[1] * fr[a][0] + Wg[2] * fr[a][1] + Wg[3] * fr[a][2];
    for (int dir = 0; dir < 3; dir++) {
      double dg[5];
      for (int v = 0; v < 5; v++) dg[v] = gg[3 * v] * fr[dir][0] + gg[3 * v + 1] * fr[dir][1] + gg[3 * v + 2] * fr[dir][2];
      sl[dir][0] = dg[0]; sl[dir][4] = dg[4];
      for (int a = 0; a < 3; a++) sl[dir][1 + a] = dg[1] * fr[a][0] + dg[2] * fr[a][1] + dg[3] * fr[a][2];
    }
  }
  /* 2-3. Maxwellians g_l, g_r and their moments */
  prim_t pl = prim_of(WL, K), pr = prim_of(WR, K);
  mom_t mlf, mlp, mrf, mrn;
  mom_set(&mlf, pl.U, pl.V, pl.W, pl.lam, K, 0); mom_set(&mlp, pl.U, pl.V, pl.W, pl.lam, K, +1);
  mom_set(&mrf, pr.U, pr.V, pr.W, pr.lam, K, 0); mom_set(&mrn, pr.U, pr.V, pr.W, pr.lam, K, -1);
  const double one[5] = { 1, 0, 0, 0, 0 };
  /* 4. equilibrium state W0 = int_{u>0} g_l psi + int_{u<0} g_r psi */
  double W0[5], tl[5], tr[5];
  mom_apsi(&mlp, one, 0, 0, 0, tl); mom_apsi(&mrn, one, 0, 0, 0, tr);
  for (int v = 0; v < 5; v++) W0[v] = pl.rho * tl[v] + pr.rho * tr[v];
  prim_t p0 = prim_of(W0, K);
  mom_t m0; mom_set(&m0, p0.U, p0.V, p0.W, p0.lam, K, 0);
  /* 5. micro slopes a^l_i, a^r_i from the one-sided slopes; abar_i from kinetic weighting (reading F1) */
  double aL[3][5], aR[3][5], a0[3][5], h[5];
  for (int d = 0; d < 3; d++) {
    for (int v = 0; v < 5; v++) h[v] = sL[d][v] / pl.rho;
    cgks_ref_microslope(h, pl.U, pl.V, pl.W, pl.lam, K, aL[d]);
    for (int v = 0; v < 5; v++) h[v] = sR[d][v] / pr.rho;
    cgks_ref_microslope(h, pr.U, pr.V, pr.W, pr.lam, K, aR[d]);
  }
  for (int d = 0; d < 3; d++) {
    mom_apsi(&mlp, aL[d], 0, 0, 0, tl); mom_apsi(&mrn, aR[d], 0, 0, 0, tr);
    for (int v = 0; v < 5; v++) h[v] = (pl.rho * tl[v] + pr.rho * tr[v]) / p0.rho;
    cgks_ref_microslope(h, p0.U, p0.V, p0.W, p0.lam, K, a0[d]);
  }
  /* time slopes from the compatibility condition <a1 u + a2 v + a3 w + A> = 0 */
  double AL[5], AR[5], A0[5], x1[5], x2[5], x3[5];
  double dQL[5], dQR[5];       /* rho * <A psi> = time derivative of the one-sided Maxwellian's moments */
  mom_apsi(&mlf, aL[0], 1, 0, 0, x1); mom_apsi(&mlf, aL[1], 0, 1, 0, x2); mom_apsi(&mlf, aL[2], 0, 0, 1, x3);
  for (int v = 0; v < 5; v++) { h[v] = -(x1[v] + x2[v] + x3[v]); dQL[v] = pl.rho * h[v]; }
  cgks_ref_microslope(h, pl.U, pl.V, pl.W, pl.lam, K, AL);
  mom_apsi(&mrf, aR[0], 1, 0, 0, x1); mom_apsi(&mrf, aR[1], 0, 1, 0, x2); mom_apsi(&mrf, aR[2], 0, 0, 1, x3);
  for (int v = 0; v < 5; v++) { h[v] = -(x1[v] + x2[v] + x3[v]); dQR[v] = pr.rho * h[v]; }
  cgks_ref_microslope(h, pr.U, pr.V, pr.W, pr.lam, K, AR);
  mom_apsi(&m0, a0[0], 1, 0, 0, x1); mom_apsi(&m0, a0[1], 0, 1, 0, x2); mom_apsi(&m0, a0[2], 0, 0, 1, x3);
  for (int v = 0; v < 5; v++) h[v] = -(x1[v] + x2[v] + x3[v]);
  cgks_ref_microslope(h, p0.U, p0.V, p0.W, p0.lam, K, A0);
  /* 6. collision time (readings T1, T2) */
  double mu = 0.0;
  if (prm->mu_ref > 0.0) {
    mu = prm->mu_ref;
    if (prm->visc_omega != 0.0) mu *= pow((p0.p / p0.rho) / prm->T_ref, prm->visc_omega);
  }
  double dpr = fabs(pl.p - pr.p) / fabs(pl.p + pr.p);
  double tau = mu / p0.p + prm->tau_c1 * dt + prm->tau_c2 * dpr * dt;
  /* 7. moments of every group of Eq. 5: index 0 -> conserved moments (psi), 1 -> flux moments (u psi) */
  double G1[2][5], G2[2][5], G3[2][5], G4[2][5], G5[2][5], G6[2][5];
  for (int f = 0; f < 2; f++) {
    mom_apsi(&m0, one, f, 0, 0, x1); for (int v = 0; v < 5; v++) G1[f][v] = p0.rho * x1[v];
    mom_apsi(&m0, a0[0], f + 1, 0, 0, x1); mom_apsi(&m0, a0[1], f, 1, 0, x2); mom_apsi(&m0, a0[2], f, 0, 1, x3);
    for (int v = 0; v < 5; v++) G2[f][v] = p0.rho * (x1[v] + x2[v] + x3[v]);
    mom_apsi(&m0, A0, f, 0, 0, x1); for (int v = 0; v < 5; v++) G3[f][v] = p0.rho * x1[v];
    mom_apsi(&mlp, one, f, 0, 0, tl); mom_apsi(&mrn, one, f, 0, 0, tr);
    for (int v = 0; v < 5; v++) G4[f][v] = pl.rho * tl[v] + pr.rho * tr[v];
    double yl[5], yr[5];
    mom_apsi(&mlp, aL[0], f + 1, 0, 0, x1); mom_apsi(&mlp, aL[1], f, 1, 0, x2); mom_apsi(&mlp, aL[2], f, 0, 1, x3);
    for (int v = 0; v < 5; v++) yl[v] = x1[v] + x2[v] + x3[v];
    mom_apsi(&mrn, aR[0], f + 1, 0, 0, x1); mom_apsi(&mrn, aR[1], f, 1, 0, x2); mom_apsi(&mrn, aR[2], f, 0, 1, x3);
    for (int v = 0; v < 5; v++) yr[v] = x1[v] + x2[v] + x3[v];
    for (int v = 0; v < 5; v++) G5[f][v] = pl.rho * yl[v] + pr.rho * yr[v];
    mom_apsi(&mlp, AL, f, 0, 0, tl); mom_apsi(&mrn, AR, f, 0, 0, tr);
    for (int v = 0; v < 5; v++) G6[f][v] = pl.rho * tl[v] + pr.rho * tr[v];
  }
  /* time integrals over [0,dt] and [0,dt/2] */
  double IF[2][5], IQ[2][5];
  for (int q = 0; q < 2; q++) {
    double T = q ? 0.5 * dt : dt, cf[6];
    time_coef(T, tau, cf);
    for (int v = 0; v < 5; v++) {
      IQ[q][v] = cf[0] * G1[0][v] + cf[1] * G2[0][v] + cf[2] * G3[0][v] + cf[3] * G4[0][v] + cf[4] * G5[0][v] + cf[5] * G6[0][v];
      IF[q][v] = cf[0] * G1[1][v] + cf[1] * G2[1][v] + cf[2] * G3[1][v] + cf[3] * G4[1][v] + cf[4] * G5[1][v] + cf[5] * G6[1][v];
    }
    /* 9. Prandtl number fix (reading F2): energy flux += (1/Pr - 1) q */
    if (prm->mu_ref > 0.0 && prm->Pr != 1.0) {
      double U0[3] = { p0.U, p0.V, p0.W };
      double qh = IF[q][4] - U0[0] * IQ[q][4];
      for (int a = 0; a < 3; a++) qh -= U0[a] * (IF[q][1 + a] - U0[0] * IQ[q][1 + a]);
      qh += 0.5 * (U0[0] * U0[0] + U0[1] * U0[1] + U0[2] * U0[2]) * (IF[q][0] - U0[0] * IQ[q][0]);
      IF[q][4] += (1.0 / prm->Pr - 1.0) * qh;
    }
  }
  /* 8. linearisation in time (Eq. 6-7) */
  double Fn[5], Ft[5], Qn[5], Qt[5];
  for (int v = 0; v < 5; v++) {
    Fn[v] = (4.0 * IF[1][v] - IF[0][v]) / dt;  Ft[v] = 4.0 * (IF[0][v] - 2.0 * IF[1][v]) / (dt * dt);
    Qn[v] = (4.0 * IQ[1][v] - IQ[0][v]) / dt;  Qt[v] = 4.0 * (IQ[0][v] - 2.0 * IQ[1][v]) / (dt * dt);
  }
  /* 10. one-sided interface values (reading F3) */
  double wgt = 0.0;
  if (prm->tau_c2 > 0.0 && dpr > 0.0) wgt = exp(-1.0 / (prm->tau_c2 * dpr));   /* exp(-dt/tau0), tau0 = c2 dpr dt */
  double VL[5], VR[5], DL[5], DR[5];
  for (int v = 0; v < 5; v++) {
    VL[v] = (1.0 - wgt) * Qn[v] + wgt * WL[v];  DL[v] = (1.0 - wgt) * Qt[v] + wgt * dQL[v];
    VR[v] = (1.0 - wgt) * Qn[v] + wgt * WR[v];  DR[v] = (1.0 - wgt) * Qt[v] + wgt * dQR[v];
  }
  /* 11. rotate back */
  double* vec[6] = { Fn, Ft, VL, DL, VR, DR };
  for (int q = 0; q < 6; q++) {
    double* o = out + 5 * q; const double* x = vec[q];
    o[0] = x[0]; o[4] = x[4];
    for (int r = 0; r < 3; r++) o[1 + r] = x[1] * nrm[r] + x[2] * t1[r] + x[3] * t2[r];
  }
}

/* ------------------------------------------------------------------ */
/* Steps 5-6 over the mesh                                              */
/* ------------------------------------------------------------------ */
static void flux_all(cgks_ref_ctx* c, double dt) {
  const long n = c->n;
#pragma omp parallel for collapse(2) schedule(static)
  for (int k = 0; k < c->nk; k++) for (int j = 0; j < c->nj; j++) for (int i = 0; i < c->ni; i++) {
    long ci = cidx(c, i, j, k);
    for (int ax = 0; ax < 3; ax++) {
      int o[3] = { 0, 0, 0 }; o[ax] = 1;
      long cr = cidx(c, i + o[0], j + o[1], k + o[2]);
      const double* Af = c->area + ((long)ax * n + ci) * 3; const double* t1 = c->tan1 + ((long)ax * n + ci) * 3;
      double S = sqrt(Af[0] * Af[0] + Af[1] * Af[1] + Af[2] * Af[2]), nrm[3] = { Af[0] / S, Af[1] / S, Af[2] / S };
      for (int q = 0; q < 4; q++) {
        /* the left cell's point on its + face and the right cell's point on its - face coincide */
        const double* L = c->pv + (ci * NGP + 4 * (2 * ax) + q) * 20;
        const double* R = c->pv + (cr * NGP + 4 * (2 * ax + 1) + q) * 20;
        cgks_ref_flux_point(&c->prm, dt, L, L + 5, R, R + 5, nrm, t1, c->fx + (((long)ax * n + ci) * 4 + q) * 30);
      }
    }
  }
}

/* test tap: reconstruct + flux of the current state; fx [3][ncell][4][30] */
int cgks_ref_debug_flux(cgks_ref_ctx* c, double dt, double* fx) {
  reconstruct_all(c); flux_all(c, dt);
  memcpy(fx, c->fx, sizeof(double) * 3 * c->n * 4 * 30);
  return 0;
}

void cgks_ref_s2o4_stage1(double qn, double L, double Lt, double dt, double* qstar) {
  *qstar = qn + 0.5 * dt * L + 0.125 * dt * dt * Lt;
}
void cgks_ref_s2o4_stage2(double qn, double L, double Lt, double Ltstar, double dt, double* qnew) {
  *qnew = qn + dt * L + (1.0 / 6.0) * dt * dt * (Lt + 2.0 * Ltstar);
}

/* accumulate the operators of one cell from its 24 face points:
   Lop[5], Ltop[5]; SG0/SG1 [5][3] (Eq. 9 applied to V and Dt); SD0/SD1 [5][12] (Eq. 10 differences) */
static void accumulate_cell(const cgks_ref_ctx* c, int i, int j, int k, double Lop[5], double Ltop[5],
                            double SG0[15], double SG1[15], double SD0[60], double SD1[60]) {
  const long n = c->n; long ci = cidx(c, i, j, k);
  for (int v = 0; v < 5; v++) Lop[v] = Ltop[v] = 0;
  for (int q = 0; q < 15; q++) SG0[q] = SG1[q] = 0;
  for (int ax = 0; ax < 3; ax++) {
    int o[3] = { 0, 0, 0 }; o[ax] = 1;
    long cm = cidx(c, i - o[0], j - o[1], k - o[2]);
    const double* Ap = c->area + ((long)ax * n + ci) * 3; const double* Am = c->area + ((long)ax * n + cm) * 3;
    double Sp = sqrt(Ap[0] * Ap[0] + Ap[1] * Ap[1] + Ap[2] * Ap[2]), Sm = sqrt(Am[0] * Am[0] + Am[1] * Am[1] + Am[2] * Am[2]);
    for (int q = 0; q < 4; q++) {
      const double* fp = c->fx + (((long)ax * n + ci) * 4 + q) * 30;   /* + face: this cell is the left side  */
      const double* fm = c->fx + (((long)ax * n + cm) * 4 + q) * 30;   /* - face: this cell is the right side */
      for (int v = 0; v < 5; v++) {
        Lop[v] -= 0.25 * (fp[v] * Sp - fm[v] * Sm);                     /* Eq. 8, omega_k = 1/4 */
        Ltop[v] -= 0.25 * (fp[5 + v] * Sp - fm[5 + v] * Sm);
        for (int r = 0; r < 3; r++) {                                   /* Eq. 9 with own-side values */
          SG0[3 * v + r] += 0.25 * (fp[10 + v] * Ap[r] - fm[20 + v] * Am[r]);
          SG1[3 * v + r] += 0.25 * (fp[15 + v] * Ap[r] - fm[25 + v] * Am[r]);
        }
        SD0[12 * v + 4 * ax + q] = fp[10 + v] - fm[20 + v];             /* Eq. 10 / Eq. 19 row 4 */
        SD1[12 * v + 4 * ax + q] = fp[15 + v] - fm[25 + v];
      }
    }
  }
  double vol = c->vol[ci];
  for (int v = 0; v < 5; v++) { Lop[v] /= vol; Ltop[v] /= vol; }
  for (int q = 0; q < 15; q++) { SG0[q] /= vol; SG1[q] /= vol; }
}

static int check_physical(cgks_ref_ctx* c, const double* Q, const char* what) {
  const long n = c->n; long bad = -1;
  for (long ci = 0; ci < n; ci++) {
    double rho = Q[ci], e = Q[4 * n + ci] - 0.5 * (Q[n + ci] * Q[n + ci] + Q[2 * n + ci] * Q[2 * n + ci] + Q[3 * n + ci] * Q[3 * n + ci]) / rho;
    if (!(rho > 0.0) || !(e > 0.0)) { bad = ci; break; }
  }
  if (bad >= 0) { snprintf(c->err, sizeof c->err, "non-physical cell average after %s at cell %ld", what, bad); return -4; }
  return 0;
}

int cgks_ref_step(cgks_ref_ctx* c, double dt) {
  const long n = c->n;
  /* ---- stage 1 (state n) ---- */
  reconstruct_all(c);
  flux_all(c, dt);
#pragma omp parallel for collapse(2) schedule(static)
  for (int k = 0; k < c->nk; k++) for (int j = 0; j < c->nj; j++) for (int i = 0; i < c->ni; i++) {
    long ci = cidx(c, i, j, k);
    double Lop[5], Ltop[5], SG0[15], SG1[15], SD0[60], SD1[60];
    accumulate_cell(c, i, j, k, Lop, Ltop, SG0, SG1, SD0, SD1);
    for (int v = 0; v < 5; v++) {
      c->Qn[v * n + ci] = c->Q[v * n + ci]; c->Ln[v * n + ci] = Lop[v]; c->Ltn[v * n + ci] = Ltop[v];
      cgks_ref_s2o4_stage1(c->Q[v * n + ci], Lop[v], Ltop[v], dt, &c->Qs[v * n + ci]);
    }
    /* interface values at t* = tn + dt/2: Q* = Q^n + dt/2 (dQ/dt)^n, then Eq. 9-10 */
    for (int q = 0; q < 15; q++) { c->SG0[q * n + ci] = SG0[q]; c->Gs[q * n + ci] = SG0[q] + 0.5 * dt * SG1[q]; }
    for (int q = 0; q < 60; q++) { c->SD0[q * n + ci] = SD0[q]; c->Ds[q * n + ci] = SD0[q] + 0.5 * dt * SD1[q]; }
  }
  memcpy(c->Q, c->Qs, sizeof(double) * 5 * n); memcpy(c->G, c->Gs, sizeof(double) * 15 * n); memcpy(c->D, c->Ds, sizeof(double) * 60 * n);
  int rc = check_physical(c, c->Q, "stage 1"); if (rc) return rc;
  /* ---- stage 2 (state *) ---- */
  reconstruct_all(c);
  flux_all(c, dt);
#pragma omp parallel for collapse(2) schedule(static)
  for (int k = 0; k < c->nk; k++) for (int j = 0; j < c->nj; j++) for (int i = 0; i < c->ni; i++) {
    long ci = cidx(c, i, j, k);
    double Lop[5], Ltop[5], SG0[15], SG1[15], SD0[60], SD1[60];
    accumulate_cell(c, i, j, k, Lop, Ltop, SG0, SG1, SD0, SD1);
    for (int v = 0; v < 5; v++)
      cgks_ref_s2o4_stage2(c->Qn[v * n + ci], c->Ln[v * n + ci], c->Ltn[v * n + ci], Ltop[v], dt, &c->Qs[v * n + ci]);
    /* Q^{n+1} = Q^n + dt (dQ/dt)^* at the interfaces (reading T4) */
    for (int q = 0; q < 15; q++) c->Gs[q * n + ci] = c->SG0[q * n + ci] + dt * SG1[q];
    for (int q = 0; q < 60; q++) c->Ds[q * n + ci] = c->SD0[q * n + ci] + dt * SD1[q];
  }
  memcpy(c->Q, c->Qs, sizeof(double) * 5 * n); memcpy(c->G, c->Gs, sizeof(double) * 15 * n); memcpy(c->D, c->Ds, sizeof(double) * 60 * n);
  return check_physical(c, c->Q, "stage 2");
}

/* ------------------------------------------------------------------ */
/* Diagnostics: volume-averaged kinetic energy and   */
/* enstrophy, "calculated by numerical quadrature, and the velocity     */
/* derivative values at quadrature points are obtained by the compact   */
/* reconstruction".  Reading X1: 2x2x2 Gauss      */
/* points (+-g,+-g,+-g) of the reference cell, weights |Omega|/8, the   */
/* scheme's own (blended, Eq. 16) polynomial of the conservative        */
/* variables, U = m/rho, the solver's viscosity law for mu, point-wise  */
/* positivity fallback R9.  Returns the integrals divided by |Omega|    */
/* (rho_0 = 1 is left to the caller).                                   */
/* ------------------------------------------------------------------ */
int cgks_ref_diagnostics(cgks_ref_ctx* c, double* Ek_out, double* ens_out) {
  const long n = c->n; const double g = 0.5 / sqrt(3.0);
  double Ek = 0, ens = 0, vtot = 0;
#pragma omp parallel for collapse(2) schedule(static) reduction(+ : Ek, ens, vtot)
  for (int k = 0; k < c->nk; k++) for (int j = 0; j < c->nj; j++) for (int i = 0; i < c->ni; i++) {
    long ci = cidx(c, i, j, k);
    const double* J = c->J0 + 9 * ci; const double* Ji = c->J0inv + 9 * ci;
    double val[8][5], grd[8][5][3];
    for (int v = 0; v < NV; v++) {
      const double* q = c->Q + v * n;
      double q0 = q[ci], d[ND];
      for (int m = 0; m < 6; m++) d[m] = q[cidx(c, i + g_face_off[m][0], j + g_face_off[m][1], k + g_face_off[m][2])] - q0;
      for (int e = 0; e < 12; e++) d[6 + e] = q[cidx(c, i + g_edge_off[e][0], j + g_edge_off[e][1], k + g_edge_off[e][2])] - q0;
      for (int m = 0; m < 6; m++) {
        long nb = cidx(c, i + g_face_off[m][0], j + g_face_off[m][1], k + g_face_off[m][2]);
        for (int a = 0; a < 3; a++) {
          double s = 0; for (int r = 0; r < 3; r++) s += J[3 * r + a] * c->G[(v * 3 + r) * n + nb];
          d[18 + 3 * m + a] = 2.0 * s;
        }
      }
      for (int e = 0; e < 12; e++) {
        long nb = cidx(c, i + g_edge_off[e][0], j + g_edge_off[e][1], k + g_edge_off[e][2]);
        double gr[3];
        for (int a = 0; a < 3; a++) { double s = 0; for (int r = 0; r < 3; r++) s += J[3 * r + a] * c->G[(v * 3 + r) * n + nb]; gr[a] = s; }
        d[36 + 2 * e] = gr[g_edge_axis[e]];
        d[36 + 2 * e + 1] = (g_edge_off[e][0] * gr[0] + g_edge_off[e][1] * gr[1] + g_edge_off[e][2] * gr[2]) / (g_r5_normalised ? sqrt(2.0) : 1.0);
      }
      for (int s = 0; s < 12; s++) d[60 + s] = 3.0 * c->D[(v * 12 + s) * n + ci];
      double a[NB], b[18], chi, om[6], fval[NGP], fgref[NGP * 3];
      cgks_ref_recon_reference(&c->prm, d, a, b, &chi, om, fval, fgref);
      for (int p = 0; p < 8; p++) {
        double x[3] = { (p & 4) ? g : -g, (p & 2) ? g : -g, (p & 1) ? g : -g };
        double v4 = 0, g4[3] = { 0, 0, 0 }, v1 = 0, g1[3] = { 0, 0, 0 };
        for (int bb = 0; bb < NB; bb++) {
          v4 += a[bb] * basis_pt(g_didx[bb], x);
          for (int ax = 0; ax < 3; ax++) g4[ax] += a[bb] * basis_dpt(g_didx[bb], x, ax);
        }
        for (int m = 0; m < 6; m++) {
          v1 += om[m] * (b[3 * m] * x[0] + b[3 * m + 1] * x[1] + b[3 * m + 2] * x[2]);
          for (int ax = 0; ax < 3; ax++) g1[ax] += om[m] * b[3 * m + ax];
        }
        val[p][v] = q0 + chi * v4 + (1.0 - chi) * v1;
        double gr[3];
        for (int ax = 0; ax < 3; ax++) gr[ax] = chi * g4[ax] + (1.0 - chi) * g1[ax];
        for (int r = 0; r < 3; r++) grd[p][v][r] = Ji[0 * 3 + r] * gr[0] + Ji[1 * 3 + r] * gr[1] + Ji[2 * 3 + r] * gr[2];
      }
    }
    for (int p = 0; p < 8; p++) {
      double rho = val[p][0], pe = val[p][4] - 0.5 * (val[p][1] * val[p][1] + val[p][2] * val[p][2] + val[p][3] * val[p][3]) / rho;
      double adm = val[p][0] * val[p][4] - 0.5 * ((val[p][1] * val[p][1] + val[p][2] * val[p][2]) + val[p][3] * val[p][3]);   /* reading R9 */
      if (!(rho > 0.0) || !(adm > 0.0)) {
        for (int v = 0; v < NV; v++) { val[p][v] = c->Q[v * n + ci]; for (int r = 0; r < 3; r++) grd[p][v][r] = 0.0; }
        rho = val[p][0];
        pe = val[p][4] - 0.5 * (val[p][1] * val[p][1] + val[p][2] * val[p][2] + val[p][3] * val[p][3]) / rho;
      }
      double U[3] = { val[p][1] / rho, val[p][2] / rho, val[p][3] / rho };
      double dU[3][3];   /* dU[a][r] = d U_a / d x_r = (d m_a - U_a d rho)/rho */
      for (int a = 0; a < 3; a++) for (int r = 0; r < 3; r++) dU[a][r] = (grd[p][1 + a][r] - U[a] * grd[p][0][r]) / rho;
      double w[3] = { dU[2][1] - dU[1][2], dU[0][2] - dU[2][0], dU[1][0] - dU[0][1] };
      double pres = (c->prm.gamma - 1.0) * pe;
      double mu = c->prm.mu_ref;
      if (c->prm.mu_ref > 0.0 && c->prm.visc_omega != 0.0) mu *= pow((pres / rho) / c->prm.T_ref, c->prm.visc_omega);
      double wq = c->vol[ci] / 8.0;
      Ek += wq * 0.5 * rho * (U[0] * U[0] + U[1] * U[1] + U[2] * U[2]);
      ens += wq * mu * (w[0] * w[0] + w[1] * w[1] + w[2] * w[2]);
    }
    vtot += c->vol[ci];
  }
  *Ek_out = Ek / vtot; *ens_out = ens / vtot;
  return 0;
}

/* time step (reading S3): dt = CFL / max_cells sum_d (|U.n_d| + c)/h_d, h_d = |Omega|/S_d;
   viscous cap dt <= CFL min_d h_d^2 / (3 nu).  The sum over the three index directions is the
   reading that reproduces Table 1 (S3). */
int cgks_ref_compute_dt(cgks_ref_ctx* c, double cfl, double* dt_out) {
  const long n = c->n; const double gam = c->prm.gamma;
  double dtmin = INFINITY;
#pragma omp parallel for collapse(2) schedule(static) reduction(min : dtmin)
  for (int k = 0; k < c->nk; k++) for (int j = 0; j < c->nj; j++) for (int i = 0; i < c->ni; i++) {
    long ci = cidx(c, i, j, k);
    double rho = c->Q[ci], U[3] = { c->Q[n + ci] / rho, c->Q[2 * n + ci] / rho, c->Q[3 * n + ci] / rho };
    double p = (gam - 1.0) * (c->Q[4 * n + ci] - 0.5 * rho * (U[0] * U[0] + U[1] * U[1] + U[2] * U[2]));
    double cs = sqrt(gam * p / rho);
    double rate = 0.0, hmin = INFINITY;
    for (int ax = 0; ax < 3; ax++) {
      int o[3] = { 0, 0, 0 }; o[ax] = 1;
      long cm = cidx(c, i - o[0], j - o[1], k - o[2]);
      const double* Ap = c->area + ((long)ax * n + ci) * 3; const double* Am = c->area + ((long)ax * n + cm) * 3;
      double Sp = sqrt(Ap[0] * Ap[0] + Ap[1] * Ap[1] + Ap[2] * Ap[2]), Sm = sqrt(Am[0] * Am[0] + Am[1] * Am[1] + Am[2] * Am[2]);
      double nb[3] = { Ap[0] + Am[0], Ap[1] + Am[1], Ap[2] + Am[2] }, nl = sqrt(nb[0] * nb[0] + nb[1] * nb[1] + nb[2] * nb[2]);
      double h = c->vol[ci] / (0.5 * (Sp + Sm));
      double un = fabs(U[0] * nb[0] + U[1] * nb[1] + U[2] * nb[2]) / nl;
      if (g_s3_sum) rate += (un + cs) / h;
      else if ((un + cs) / h > rate) rate = (un + cs) / h;      /* alternative reading S3 (max); never the default */
      if (h < hmin) hmin = h;
    }
    double d = cfl / rate;
    if (d < dtmin) dtmin = d;
    if (c->prm.mu_ref > 0.0) {
      double mu = c->prm.mu_ref;
      if (c->prm.visc_omega != 0.0) mu *= pow((p / rho) / c->prm.T_ref, c->prm.visc_omega);
      double dv = cfl * hmin * hmin / (3.0 * mu / rho);
      if (dv < dtmin) dtmin = dv;
    }
  }
  *dt_out = dtmin;
  return 0;
}
