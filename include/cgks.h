/*
 * cgks.h -- C ABI of the B200-native CGKS-5 / S2O4 hot path (arxiv/paper_2508_08965).
 *
 * One S2O4 step of the fifth-order compact gas-kinetic scheme on a 3-D structured, periodic,
 * possibly non-orthogonal mesh: compact reconstruction on the reference cell (Eq. 11-15,
 * 17-19), GENO blend (Eq. 16), gas-kinetic flux and interface values at the face Gauss points
 * (Eq. 1-7), update of cell averages, cell-averaged gradients and line-averaged derivatives
 * (Eq. 8-10) and the two-stage fourth-order combine.
 *
 * Every step runs in hand-written fp64 CUDA kernels for sm_100a (paper_2508_08965_b200/csrc).  There is no CPU
 * fallback: every call fails with CGKS_ECUDA when no CUDA device / kernel image is usable.
 *
 * Conventions
 *  - All array arguments named d_* are DEVICE pointers owned by the caller, fp64, structure-of-arrays, i fastest:
 *      nodes [3][nk+1][nj+1][ni+1]   node coordinates (x, y, z planes)
 *      Q     [5][nk][nj][ni]         cell averages of (rho, rho U, rho V, rho W, rho E)
 *      G     [5][3][nk][nj][ni]      cell-averaged PHYSICAL gradients, index 3*v + dir         (Eq. 9)
 *      D     [5][12][nk][nj][ni]     line DIFFERENCES Q(x_G2) - Q(x_G1) (Eq. 10 times |l_G|, Eq. 19 row 4),
 *                                    index 12*v + s, s = 4*axis + 2*a + b, (a,b) in {0,1}^2 selecting -g/+g
 *                                    (g = 1/(2 sqrt 3)) along the two other axes in ascending axis order
 *  - Other pointers (params, dt_host, bytes, out) are HOST pointers.
 *  - The mesh is periodic in all three index directions; node planes 0 and n of each direction
 *    must differ by a constant vector (checked by cgks_create).
 *  - The library never allocates device memory: the caller passes one workspace (cgks_workspace_bytes) and keeps
 *    it alive until cgks_destroy.  The context itself (host memory) is owned by the library.
 *  - Calls enqueue work on the stream given to cgks_create and return without waiting, except cgks_create
 *    (validates the mesh), cgks_compute_dt (returns a host double) and cgks_status, which synchronise the stream.
 *  - Return value: 0 on success, negative error code otherwise; cgks_last_error gives a message.
 */
#ifndef CGKS_H
#define CGKS_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct cgks_ctx cgks_ctx;

enum {
  CGKS_OK = 0,
  CGKS_EINVAL = -1,        /* bad argument, ni/nj/nk < 4, non-periodic node array, det J0 <= 0 or volume <= 0 */
  CGKS_ENOMEM = -2,        /* workspace too small                                                              */
  CGKS_ECUDA = -3,         /* CUDA runtime error (including "no device")                                       */
  CGKS_ENONPHYSICAL = -4   /* a cell average with rho <= 0 or p <= 0 appeared after a stage                    */
};

typedef struct {
  double gamma, Pr, mu_ref;   /* mu_ref = 0 -> inviscid                                                        */
  double visc_omega, T_ref;   /* mu = mu_ref (T/T_ref)^omega, T = p/rho; omega = 0 -> constant                */
  double tau_c1, tau_c2;      /* tau = mu/p + c1 dt + c2 |pl-pr|/|pl+pr| dt: inviscid 0.05, 5;
                                 viscous 0, 5; accuracy test 0, 0 (tau = 0)                      */
  int    nonlinear;           /* 1 = GENO blend, 0 = linear reconstruction (chi = 1)            */
  double geno_C, geno_eps;    /* tanh constant C = 5 (reading G3), epsilon = 1e-15    */
  int    geno_r;              /* r = 2; only r = 2 is implemented                               */
} cgks_params;

/* Bytes of device workspace for a mesh of ni x nj x nk cells (state, stage buffers, metrics, and the slab buffer of
   reconstructed face values; when the whole mesh fits, also the face-flux buffer the test tap cgks_debug_stage needs).  `budget_bytes` = 0 asks for the default (largest useful slab up
   to ~48 GB of slab buffers); otherwise the slab depth is reduced so that the total stays below the budget, and
   CGKS_ENOMEM is returned when not even a slab of two k-planes fits under it.  (`budget_bytes` is an addition to
   the call list of SURVEY.md 8(b): the 384^3 case needs the caller to say how much of the device it may take.) */
int cgks_workspace_bytes(int ni, int nj, int nk, size_t budget_bytes, size_t* bytes);

/* Builds the mesh metrics (J0 of Eq. 18, cell volumes by the Appendix quadrature, face vector areas, DESIGN.md
   readings R1-R2) and the context.  d_nodes is read during the call only. */
int cgks_create(cgks_ctx** out, int ni, int nj, int nk, const double* d_nodes, const cgks_params* params,
                void* d_workspace, size_t workspace_bytes, void* cuda_stream);

/* Copies the state in.  d_G and/or d_D may be NULL: the missing derivative dof are bootstrapped from Q by
   fourth-order central differences in index space (reading S2). */
int cgks_set_state(cgks_ctx*, const double* d_Q, const double* d_G, const double* d_D);

/* Copies the state out (any pointer may be NULL). */
int cgks_get_state(cgks_ctx*, double* d_Q, double* d_G, double* d_D);

/* dt = cfl / max_cells sum_d (|U.n_d| + c)/h_d, capped by cfl h^2/(3 nu) for viscous flow (PAPER.md:342,
   DESIGN.md reading S3).  Synchronises; returns CGKS_ENONPHYSICAL if an earlier stage flagged a bad cell. */
int cgks_compute_dt(cgks_ctx*, double cfl, double* dt_host);

/* The same time step (reading S3) WITHOUT a context, a workspace or any device allocation, for
   callers that cannot get device memory: code that is handed a Q array inside a process whose framework allocator already
   holds all of HBM (a raw cudaMalloc fails there, and so would the workspace cgks_create needs), and time loops that must
   never stall (cudaMalloc / cudaFree synchronise the device).  The reduction's scratch memory is an array built into the
   library image: 33 024 bytes on every GPU that loads libcgks.so, held until the process exits.
     d_Q      DEVICE [5][nk][nj][ni] cell averages (rho, rho U, rho V, rho W, rho E), read only
     h_host   HOST   [3] cell sizes of a UNIFORM CARTESIAN mesh (period / n per direction, as cgks_create derives them);
                     general meshes need the metrics of a context: use cgks_compute_dt
     params   HOST   gamma, mu_ref, visc_omega, T_ref are used
     d_dt     DEVICE [1] result; +inf when no cell is admissible
     d_bad    DEVICE [1] or NULL: 1 if a cell average with rho <= 0 or p <= 0 was met (such cells are skipped), else 0
   Limit: ni * nj * nk <= CGKS_STATIC_MAX_CELLS (256^3); more returns CGKS_EINVAL with a message that says so.  The call
   enqueues one memset and two kernels on `cuda_stream` and returns without waiting; it calls no cudaMalloc, cudaFree or
   other allocating routine.  The result does not depend on the device's SM count (one partial minimum per 4096 cells) and
   is bit-identical to cgks_compute_dt on the same mesh and state as long as both compile to the same per-cell arithmetic
   (tested to 1e-13).
   Set-up: the first call on each device (with that device current) looks up the array's device address with
   cudaGetSymbolAddress, which may load the CUDA module; make that first call before any stream capture begins.
   Sharing: all calls on one device use the same array.  A call clears the one word that must start at zero and overwrites
   every partial it reads, so calls that follow each other on one stream are independent; calls that may OVERLAP on the
   GPU (different streams, or several host threads) race on it and give undefined results -- serialise them.
   Errors: CGKS_EINVAL / CGKS_ECUDA, message from cgks_static_last_error() (per host thread). */
enum { CGKS_STATIC_MAX_CELLS = 1 << 24 };
int cgks_compute_dt_static(int ni, int nj, int nk, const double* d_Q, const double* h_host, const cgks_params* params,
                           double cfl, double* d_dt, int* d_bad, void* cuda_stream);
const char* cgks_static_last_error(void);

/* One two-stage fourth-order step of size dt.  Asynchronous.
   Per stage: one reconstruction kernel (Eq. 11-19), then one sweep kernel per face direction that computes the gas-kinetic
   flux at the face Gauss points (Eq. 1-7) and accumulates Eq. 8-10 and the S2O4 combine into the state buffers.  (The
   three-kernel pipeline of the first rounds, flux -> face-flux buffer -> update, exists only in the test-only A/B build
   libcgks_ab.so and as the flux tap of cgks_debug_stage; nothing selects it at run time.) */
int cgks_step(cgks_ctx*, double dt);

/* One stage of the step (1: state n -> stage state; 2: stage state -> state n+1); cgks_step(dt) is
   cgks_stage(1, dt) followed by cgks_stage(2, dt).  Stages must alternate 1, 2.  Asynchronous. */
int cgks_stage(cgks_ctx*, int stage, double dt);

/* ---- Sub-domains of a slab decomposition along k (the paper's own parallelisation: "domain decomposed
   into slabs along one dimension", one rank per GPU) -------------------------------------
   A sub-domain context holds nk_owned k-planes of the global periodic mesh starting at global plane k0, plus TWO halo
   planes on each side (a cell's update needs the state of cells within index distance 2 per stage): its arrays have
   nk_owned + 4 planes, local plane 2 being global plane k0.  d_nodes is the node array of the WHOLE mesh
   [3][nk_global+1][nj+1][ni+1] (read during the call only), so that every cell has bit-identical metrics whichever
   context holds it.  Before EACH stage the halo planes of the stage's input state must be current:
       cgks_pack_halo(side) on the neighbour  ->  transport (NCCL / peer copy; the caller's)  ->  cgks_unpack_halo(side),
   side 0 = low k, 1 = high k; pack copies the two outermost OWNED planes of that side, unpack fills the two HALO planes
   of that side, all 80 fields.  The buffer (cgks_halo_bytes = 80 * 2 * nj * ni doubles) is OPAQUE: it is meant to be moved, not
   read.  (Its actual order is the library's internal record layout, 20 runs of [2][nj][ni][4]: runs 0..4 hold { Q_v, G_v } of
   variable v, runs 5..19 the four line differences of (variable, axis) = ((a-5)/3, (a-5)%3); it is NOT [80][2][nj][ni] in the user
   field order and may change between versions -- fill it only with cgks_pack_halo.)  Between cgks_stage(1) and cgks_stage(2)
   the calls act on the stage state, otherwise on the current state.  cgks_set_state / cgks_get_state take arrays of
   nk_owned + 4 planes (halo planes of Q should hold the neighbours' values so that the bootstrap of reading S2 is right
   on the owned planes; halo planes returned by cgks_get_state are not current).  cgks_compute_dt reduces over the owned
   planes only: the caller takes the minimum over sub-domains (one scalar all-reduce per step).  cgks_step,
   cgks_run_host, cgks_diagnostics and the debug taps need a whole-mesh context. */
int cgks_create_slab(cgks_ctx** out, int ni, int nj, int nk_global, int k0, int nk_owned, const double* d_nodes,
                     const cgks_params* params, void* d_workspace, size_t workspace_bytes, void* cuda_stream);
int cgks_halo_bytes(const cgks_ctx*, size_t* bytes);
int cgks_pack_halo(cgks_ctx*, int side, double* d_buf);
int cgks_unpack_halo(cgks_ctx*, int side, const double* d_buf);

/* Non-periodic boundary in k: instead of a neighbour's planes, the two halo planes of `side` of a
   sub-domain context are filled by a boundary rule applied to the owned planes of the stage's input state (call it before
   each stage, like the halo exchange).  The paper names its boundary types (no-slip adiabatic wall and far field,
   PAPER.md:494; non-reflecting) without formulas; reading B1:
     CGKS_BC_SLIP_WALL   mirror image about the boundary face, normal momentum odd (slip wall = symmetry plane)
     CGKS_BC_NOSLIP_WALL mirror image, all momentum components odd: zero velocity and zero normal temperature gradient at
                         the face (no-slip adiabatic wall)
     CGKS_BC_OUTFLOW     zero-gradient extrapolation of the outermost owned plane
     CGKS_BC_FARFIELD    the uniform state far_state_host[5] (host pointer: rho, rho U, rho V, rho W, rho E)
   Uniform Cartesian meshes only (CGKS_EINVAL otherwise).  A domain bounded in k on both sides is the sub-domain
   cgks_create_slab(..., k0 = 0, nk_owned = nk_global, ...) with this call on both sides.
   Initial state of a bounded domain: the bootstrap of cgks_set_state (G = D = NULL, reading S2) runs BEFORE any boundary rule
   and differences the Q the caller put in the halo planes.  The caller must therefore fill the halo planes of Q consistently
   with the boundary (mirror image for walls, copies for outflow, the far state), not with the periodic wrap: with periodic
   images across a wall, the derivative dof of the two owned planes next to it start from the wrong neighbour values unless the
   data happen to be mirror-symmetric.  Passing G and D explicitly avoids the question. */
enum { CGKS_BC_SLIP_WALL = 0, CGKS_BC_NOSLIP_WALL = 1, CGKS_BC_OUTFLOW = 2, CGKS_BC_FARFIELD = 3 };
int cgks_fill_halo_bc(cgks_ctx*, int side, int kind, const double* far_state_host);

/* Diagnostics of the current state: volume-averaged kinetic energy E_k = int rho |U|^2/2 dV / |Omega| and
   enstrophy int mu |curl U|^2 dV / |Omega| (rho_0 = 1), by the 2x2x2 Gauss rule on every cell with values and velocity
   derivatives from the compact reconstruction (the scheme's own polynomial, Eq. 16; reading X1); mu is the
   solver's viscosity law.  Synchronises; overwrites the slab buffers (not the chi tap).  Host pointers. */
int cgks_diagnostics(cgks_ctx*, double* ek_host, double* enstrophy_host);

/* Synchronises and returns CGKS_OK, CGKS_ECUDA or CGKS_ENONPHYSICAL for the work enqueued so far. */
int cgks_status(cgks_ctx*);

/* Same as cgks_set_state / cgks_step / cgks_get_state but with HOST buffers: copies the state host->device, runs
   `nsteps` steps with dt from the CFL condition each step, copies the state back (used for end-to-end timing). */
int cgks_run_host(cgks_ctx*, const double* h_Q, const double* h_G, const double* h_D, double cfl, int nsteps,
                  double* h_Q_out, double* h_G_out, double* h_D_out);

/* Depth in k-planes of the slab pipeline chosen by cgks_create from the workspace size (nk: whole mesh resident). */
int cgks_slab_depth(const cgks_ctx*);

/* Number of kernels launched by the library on this context so far (for bench.py's gpu_launches). */
long cgks_launch_count(const cgks_ctx*);

/* Device-side duration in milliseconds of the kernels of one class accumulated by the last cgks_step when profiling
   is switched on with cgks_set_profiling(ctx, 1): 0 reconstruction, 1 flux (the sweep kernels: flux + update), 2 update (three-kernel
   pipeline only), 3 cfl.  Profiling inserts
   CUDA events on the stream and synchronises at the end of the step. */
int cgks_set_profiling(cgks_ctx*, int on);
int cgks_kernel_ms(const cgks_ctx*, int which, double* ms, long* launches);

/* Debug/testing taps (device pointers, valid until the next cgks_step): reconstructed face values of slab-resident
   cells are not exposed; instead this returns chi of the last reconstruction, [5][nk][nj][ni], copied to d_chi. */
int cgks_get_chi(cgks_ctx*, double* d_chi);

/* Test tap: runs the reconstruction (and, if d_fx != NULL, the flux kernels with step size dt, stage 1) on the
   CURRENT state and copies the slab buffers out: d_pv [480][N] (plane (4m+q)*20 + c: c = v value, 5+3v+r physical
   gradient; NO positivity fallback applied), d_fx [360][N] (plane (4ax+q)*30 + c: Fn, Ft, VL, DtL, VR, DtR).
   Needs the whole mesh resident and, for d_fx, room for the face-flux buffer in the workspace (CGKS_ENOMEM otherwise); the flux tap
   runs the gas-kinetic solver through the thread-per-point kernel of the three-kernel pipeline.  The state is not modified. */
int cgks_debug_stage(cgks_ctx*, double dt, double* d_pv, double* d_fx);

/* Measures the device's FP64 FMA throughput with a register-resident DFMA micro-benchmark (8 independent chains
   per thread, three distinct rotating register operands, 8 blocks of 256 threads per multiprocessor) on `cuda_stream`; TFLOP/s (FMA = 2 flops) to *tflops (host).
   The only call that allocates device memory itself (8 bytes, freed before returning). */
int cgks_fp64_peak(void* cuda_stream, double* tflops);

/* Test tap for the branch-free fp64 special functions of the flux kernel (csrc/fastmath64.cuh): evaluates function
   `which` (0: 1/x, 1: 1/sqrt(x), 2: exp(x), 3: erfc(x), 4: exp(-x^2) as returned together with erfc, 5: log(x), 6: tanh(x) for x >= 0, used by the GENO blend) on n device values. */
int cgks_debug_math(int which, long n, const double* d_in, double* d_out, void* cuda_stream);

int cgks_destroy(cgks_ctx*);
/* Message of the last error on this context; with a NULL context, the same as cgks_last_create_error. */
const char* cgks_last_error(const cgks_ctx*);
/* Message of the last failed cgks_create of the calling thread (empty after a successful one). */
const char* cgks_last_create_error(void);
const char* cgks_version(void);

#ifdef __cplusplus
}
#endif
#endif
