/*
 * cgks_ref.h -- CPU ORACLE for the CGKS-5 / S2O4 hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, step-by-step fp64 C implementation of what arxiv/paper_2508_08965
 * ("An effective implementation of high-order compact gas-kinetic scheme on
 * structured meshes for compressible flows") computes per S2O4 step, written from
 * PAPER.md and the readings listed in DESIGN.md section 3 (R1..R9, G1..G3, F1..F3,
 * S1..S3, T1..T4).  It shares no code, header, table or constant generator with the
 * CUDA path under paper_2508_08965_b200/csrc.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.
 *
 * Parity status of the individual functions (see DESIGN.md section 4 for the pins):
 *   reconstruction matrix, evaluation, S2O4 combine, GKS moments/flux ... pinned
 *   GENO path function reading G2/G3 ................ pinned only via Tables 1-2 (pattern)
 *   Prandtl fix F2, dt formula S3, positivity R9, bootstrap S2, the one-sided parts
 *   and the weight of the interface blend F3 ......... arithmetic pinned (tests/test_oracle_pins2.py);
 *                                                      the CHOICE of these readings: parity unpinned (paper silent)
 *
 * All pointers are HOST pointers.  Arrays are structure-of-arrays, i fastest:
 *   nodes [3][nk+1][nj+1][ni+1], Q [5][nk][nj][ni], G [5][3][nk][nj][ni],
 *   D [5][12][nk][nj][ni].
 */
#ifndef CGKS_REF_H
#define CGKS_REF_H
#ifdef __cplusplus
extern "C" {
#endif

typedef struct cgks_ref_ctx cgks_ref_ctx;

typedef struct {
  double gamma, Pr, mu_ref;      /* mu_ref = 0 -> inviscid                                        */
  double visc_omega, T_ref;      /* mu = mu_ref (T/T_ref)^omega, T = p/rho                       */
  double tau_c1, tau_c2;         /* tau = mu/p + c1 dt + c2 |pl-pr|/|pl+pr| dt */
  int    nonlinear;              /* 1 = GENO blend (Eq. 16), 0 = linear (chi = 1)                 */
  double geno_C, geno_eps;       /* tanh constant (reading G3), epsilon           */
  int    geno_r;                 /* exponent r                                     */
} cgks_ref_params;

/* sizes */
enum { CGKS_REF_NB = 34, CGKS_REF_ND = 72, CGKS_REF_NGP = 24 };

cgks_ref_ctx* cgks_ref_create(int ni, int nj, int nk, const double* nodes, const cgks_ref_params* p);
void   cgks_ref_destroy(cgks_ref_ctx*);
int    cgks_ref_set_state(cgks_ref_ctx*, const double* Q, const double* G, const double* D);
int    cgks_ref_get_state(cgks_ref_ctx*, double* Q, double* G, double* D);
int    cgks_ref_compute_dt(cgks_ref_ctx*, double cfl, double* dt);
int    cgks_ref_diagnostics(cgks_ref_ctx*, double* Ek, double* enstrophy);   /* PAPER.md:428-454, reading X1 */
int    cgks_ref_step(cgks_ref_ctx*, double dt);      /* 0 ok, -4 non-physical cell average */
const char* cgks_ref_last_error(const cgks_ref_ctx*);

/* Selects alternative readings of gaps in the paper for oracle/readings_table.py, which compares
   them with Tables 1-2: R5 (1: tau2 = unit vector towards the neighbour's centroid, 0: unnormalised offset), S3 (1: sum
   of the directional rates, 0: their maximum), G2 (1: variant B, 0: variant A).  Defaults (1, 1, 1) = the readings taken. */
void   cgks_ref_set_readings(int r5_normalised, int s3_sum, int g2_variant);

/* ---- pieces exposed so that tests can pin them against the paper ---- */
/* constant matrices: M [34][72] (a = M d, Eq. 14/19), E [96][34] (value, d/dxi, d/deta, d/dzeta at 24 points) */
void   cgks_ref_matrices(double* M, double* E);
/* basis multi-indices [34][3], Gauss points [24][3] in the reference cell */
void   cgks_ref_basis(int* didx, double* gp);
/* reference-space pieces for one (cell,variable): data vector d[72] -> a[34]; b[6][3]; chi, omega[6];
   val[24], gref[24][3] (blended value and reference-space gradient, Eq. 16) */
void   cgks_ref_recon_reference(const cgks_ref_params* p, const double* d, double* a, double* b,
                                double* chi, double* omega, double* val, double* gref);
/* smoothness indicators of a quartic with coefficients a[34]: IS[0..3] = sum over |l|=1..4 */
void   cgks_ref_smoothness(const double* a, double* IS4);
/* reconstruct every cell of the current state: pv [ncell][24][20] = (5 values, 15 physical
   gradient comps [v][dir]); chi [5][ncell] */
int    cgks_ref_reconstruct(cgks_ref_ctx*, double* pv, double* chi);
/* positivity fallback (reading R9) of the LAST reconstruction (cgks_ref_reconstruct or the second stage of cgks_ref_step):
   number of Gauss-point states replaced, and how far outside the admissible set they were: the most negative
   rho / rho_cell and (rho E - |m|^2/2) / (rho * rho E)_cell among the replaced states (0 when none was negative) */
void   cgks_ref_fallback_stats(const cgks_ref_ctx*, long* npoints, double* min_rho_rel, double* min_pe_rel);
/* reconstruct + flux of the current state: fx [3][ncell][4][30] = Fn, Ft, VL, DtL, VR, DtR per owned face point */
int    cgks_ref_debug_flux(cgks_ref_ctx*, double dt, double* fx);
/* gas-kinetic solver at one face Gauss point, global frame in/out.
   WL/WR[5], gL/gR[5][3] physical gradients, n,t1 unit vectors (t2 = n x t1).
   out[30] = Fn[5], Ft[5] (normal flux and its time derivative), VL[5], DtL[5], VR[5], DtR[5] */
void   cgks_ref_flux_point(const cgks_ref_params* p, double dt, const double* WL, const double* gL,
                           const double* WR, const double* gR, const double* n, const double* t1,
                           double* out);
/* Maxwellian moments <u^n>, n=0..6: full, u>0, u<0 */
void   cgks_ref_moments(double U, double lam, double* full, double* pos, double* neg);
/* micro-slope solve a = M^-1(h) for prim (U,V,W,lam), internal dof K */
void   cgks_ref_microslope(const double* h, double U, double V, double W, double lam, double K, double* a);
/* <(a.psi) u^i v^j w^k psi> per unit density of the Maxwellian (U,V,W,lam,K); half: 0 full, +1 u>0, -1 u<0 */
void   cgks_ref_moment_apsi(const double* a, int i, int j, int k, double U, double V, double W,
                            double lam, double K, int half, double* out);
/* geometry of the current mesh: vol[ncell], J0[ncell][9] (row-major dx_r/dxi_a), area [3][ncell][3] */
void   cgks_ref_geometry(cgks_ref_ctx*, double* vol, double* J0, double* area);
/* the S2O4 combine alone, for a scalar ODE: given L^n, Lt^n (stage 1) then Lt^* (stage 2) */
void   cgks_ref_s2o4_stage1(double qn, double L, double Lt, double dt, double* qstar);
void   cgks_ref_s2o4_stage2(double qn, double L, double Lt, double Ltstar, double dt, double* qnew);

#ifdef __cplusplus
}
#endif
#endif
