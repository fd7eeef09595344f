/* tdgl.h -- C ABI of libtdgl: the per-time-step hot path of the large-lambda TDGL solver of
 * Sadovskyy, Koshelev, Phillips, Karpeyev, Glatz, "Stable large-scale solver for Ginzburg-Landau
 * equations for superconductors" (arXiv:1409.8340), hand-written CUDA for sm_100a (B200).
 *
 * Citations: "P:NNN" = PAPER.md line NNN; "Sxx" = a reading listed in DESIGN.md ("Readings of the
 * paper").  Everything a step computes runs in the library's own kernels; there is no CPU path.
 *
 * Memory model.  The CALLER owns all device memory: one workspace block handed over at create time
 * (size from tdgl_workspace_bytes), the output buffers of tdgl_get_psi_mu and the CUDA stream.  The
 * library never allocates device memory.  `tdgl_t` is a small host object freed by tdgl_destroy.
 * Pointers named *_dev are DEVICE pointers, pointers named *_host are HOST pointers that are only
 * read / written during the call.
 *
 * Data layout.  Site (i, j, k) of an nx x ny x nz mesh has the multi-index m = i + nx*(j + ny*k)
 * (x fastest).  psi is an array of N = nx*ny*nz interleaved (re, im) fp32 pairs, mu and eps
 * are fp32 arrays of N values.  nx must be even (rows are moved as 16-byte vectors); for a 3D mesh ny, nz <= 65535.
 *
 * Errors.  Every call returns an int: 0 = TDGL_OK, negative = error (nothing was done), positive =
 * warning (the call completed).  No exceptions, no aborts, nothing is printed.
 */
#ifndef TDGL_H
#define TDGL_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TDGL_OK            0
#define TDGL_EINVAL      (-1)   /* bad size / mesh / bc / pointer / struct_size                         */
#define TDGL_ENOMEM      (-2)   /* workspace too small or not 256-byte aligned                          */
#define TDGL_EINCOMPAT   (-3)   /* open x with Jx != 0; a field component the Landau gauge chosen  */
                                /* at create cannot carry (By in the xz gauge, Bx in the yz gauge or film) */
#define TDGL_ECUDA       (-4)   /* a CUDA runtime call failed; tdgl_last_cuda_error() has the code      */
#define TDGL_ESCRATCH    (-5)   /* tdgl_mean_abs2_static only: more sites than its built-in scratch array covers */
#define TDGL_WMAXSWEEPS    1    /* some step hit max_sweeps before max|r|^2 < eps_tol (S10)             */
#define TDGL_WMUCAP        2    /* TDGL_FLAG_MU_ITERATIVE / FP64: some mu solve stopped at max_outer or max_inner
                                   (tdgl_set_mu_solver) before eps_mu / eps_in was met: mu is not converged          */

#define TDGL_BC_PERIODIC   0    /* (quasi-)periodic                                          */
#define TDGL_BC_OPEN       1    /* open: n.(grad - iA)psi = 0, n.grad(mu) = 0            */

#define TDGL_FLAG_SOLVE_MU 1u   /* mu and K are active (S15).  Off: mu == 0, K == 0             */
#define TDGL_FLAG_GAUGE_YZ 4u   /* field in the yz plane: Landau gauge A = xbar [0, Bz, -By] (Eq. 24b),
                                   quasi-periodic jump in x.  set_field_current then takes By (Bx
                                   must be 0) and tdgl_obs.Bx_eff reports the effective B_y.  Not for films. */
#define TDGL_FLAG_MU_REFINE   8u /* always run one step of iterative refinement after the mu solve (below)       */
#define TDGL_FLAG_MU_NOREFINE 16u /* never run it.  Neither flag: automatic, iff tdgl_mu_gain() > TDGL_MU_REFINE_GAIN */
#define TDGL_MU_REFINE_GAIN 200.0
#define TDGL_FLAG_MU_ITERATIVE 32u /* solve mu by the paper's own iteration (Eq. 40: pseudo-time relaxation,
                                   Crank-Nicolson, Jacobi; readings S5, S20) instead of the direct transform solver.
                                   Host-driven loop.  Controls: tdgl_set_mu_solver.  Not with TDGL_FLAG_MU_REFINE. */
#define TDGL_FLAG_FP64 64u      /* the DOUBLE-PRECISION build (the paper ships and times SP and DP):
                                   psi, b, d, mu in double (104 B/site of workspace), every kernel of the step in fp64;
                                   mu is solved by the pseudo-time iteration in double, or directly with TDGL_FLAG_MU_DIRECT (the
                                   transform solver itself is fp32 only).  psi / mu buffers of tdgl_get_psi_mu, tdgl_set_state,
                                   tdgl_debug_* are then double (pairs). */
#define TDGL_FLAG_INSULATORS 128u /* insulating inclusions (P:511 (ii), reading S25): tdgl_set_insulators removes the sites
                                   inside a list of spheres and CUTS every link between a superconducting and a removed
                                   site ("no-current boundary conditions across internal grid edges").  Needs
                                   TDGL_FLAG_FP64 (the cut links are implemented in the precision-generic kernels; mu is
                                   then solved by the pseudo-time iteration, the transform solver does not apply). */
#define TDGL_FLAG_MU_DIRECT 256u /* with TDGL_FLAG_FP64: solve Delta_h mu = rho DIRECTLY in double precision -- the fp32 transform
                                   solver as an approximate inverse inside fp64 iterative refinement (residual rho - Delta_h mu
                                   in fp64; 3-4 passes reach its rounding floor) -- instead of the paper's pseudo-time iteration.
                                   Not with TDGL_FLAG_MU_ITERATIVE, TDGL_FLAG_MU_REFINE or TDGL_FLAG_INSULATORS. */
#define TDGL_FLAG_HOST_LOOP 2u  /* test/diagnostic: host-driven sweep loop instead of the CUDA-graph
                                   WHILE node (identical arithmetic)                                     */

typedef struct tdgl tdgl_t;

/* Problem statement of the paper (Fig. 1): mesh, time step, boundary type per axis,
 * Jacobi tolerance (Eq. 34), noise temperature (Eq. 39).  Plain C POD. */
typedef struct {
  uint32_t struct_size;      /* = sizeof(tdgl_params)                                                  */
  int32_t  nx, ny, nz;       /* mesh points per axis; nx, ny >= 2, nx even; nz >= 2, or nz = 1 for a FILM  */
                             /* (the paper's 2D mode: no z links, bc[2] and hz ignored except  */
                             /* that Eq. (39) and the free energy use the cell h_x h_y; Bx must be 0)      */
  float    hx, hy, hz;       /* mesh size in xi_0                                                      */
  float    dt;               /* real time step; h_t = dt/u (P:257 fn. 3, S1)                           */
  float    u;                /* relaxation-time ratio, > 0 (S1: 1)                                     */
  float    g;                /* anisotropy, z terms / g^2                                      */
  int32_t  bc[3];            /* per axis x,y,z: TDGL_BC_PERIODIC / TDGL_BC_OPEN                        */
  float    eps_tol;          /* threshold on max_m |r_m|^2, Eq. (34)                                   */
  int32_t  max_sweeps;       /* cap on Jacobi sweeps per step (S10), >= 1                              */
  int32_t  fixed_sweeps;     /* > 0: exactly this many sweeps per step, no test (S9 replay)            */
  float    temperature;      /* reduced T-bar of Eq. (39) (S12); 0 = no Langevin term                  */
  uint64_t seed;             /* Philox4x32-10 key (S11)                                                */
  float    init_amp;         /* psi0 = 1 + init_amp (N(0,1) + i N(0,1)), Philox stream 1 (S13)         */
  uint32_t flags;            /* TDGL_FLAG_*                                                            */
  void    *workspace_dev;    /* DEVICE memory, 256-byte aligned, >= tdgl_workspace_bytes()             */
  uint64_t workspace_bytes;
  void    *stream;           /* cudaStream_t the work is enqueued on (NULL = legacy default stream)    */
} tdgl_params;

/* A spherical inclusion: centre and radius in xi_0, domain coordinates (site i sits at x = i*hx). */
typedef struct { float cx, cy, cz, r; } tdgl_sphere;

typedef struct {
  double  t;                  /* steps * dt                                                            */
  double  K;                  /* gauge variable of Eq. (13)-(15), rewound                      */
  double  Ex;                 /* E_x = d_t K of the last step (Eq. 15); V = Ex * Lx                    */
  double  Jav;                /* J_av of the last step, Eq. (35)                                       */
  double  Ex_mean;            /* mean of Ex over the steps since the last tdgl_set_field_current       */
  double  free_energy;        /* discrete GL functional                      */
  double  mean_abs2;          /* <|psi|^2>                                                             */
  double  vortices_per_slice; /* signed sum of z-plaquette windings / nz                               */
  double  max_resid2;         /* max_m |r_m|^2 at the deciding sweep of the last step                  */
  float   Bx_eff, Bz_eff;     /* field after flux-quantum snapping                        */
  int64_t steps;              /* steps taken since create                                              */
  int64_t sweeps_total;       /* Jacobi sweeps since create                                            */
  int32_t sweeps_last;        /* sweeps of the last step                                               */
  int32_t status;             /* latched warnings since create: TDGL_WMAXSWEEPS | TDGL_WMUCAP (bits), 0 = none */
} tdgl_obs;

/* Bytes of device workspace tdgl_create needs for these params (0 if the params are invalid).
 * About 44 bytes per site (two psi buffers, b, d: 8 B each; mu, eps, one scratch: 4 B each). */
uint64_t tdgl_workspace_bytes(const tdgl_params *p_host);

/* Validates the params, carves the workspace, builds the transform tables and sets the initial
 * state psi0 (S13), mu = 0, K = 0, eps = 1, B = 0, J = 0.  Asynchronous on `stream`.
 * Errors: TDGL_EINVAL, TDGL_ENOMEM, TDGL_ECUDA. */
int tdgl_create(const tdgl_params *p_host, tdgl_t **out);
int tdgl_destroy(tdgl_t *h);

/* eps_m = eps_in if site m lies within distance r of any sphere centre (minimum image on periodic
 * axes), else eps_out (P:245, P:511 (i), S19).  `spheres_host` is copied during the call; n may be 0.
 * The workspace scratch array holds the device copy, so n <= N/4. */
int tdgl_set_pinning(tdgl_t *h, const tdgl_sphere *spheres_host, int64_t n, float eps_in, float eps_out);

/* Insulating inclusions (TDGL_FLAG_INSULATORS only, else TDGL_EINCOMPAT): every site within distance r of a sphere centre
 * (the inside test of tdgl_set_pinning) is REMOVED -- psi = 0 and mu = 0 there for good -- and every link between a
 * remaining and a removed site is cut: it carries no supercurrent and no normal current, and drops out of the covariant
 * Laplacian (Eq. 29), of M (the diagonal sums c_alpha over the links that exist), of rho and of the
 * Laplacian of mu.  External open faces keep the paper's mirror rule.  Replaces any earlier list; n may be 0.
 * J_av keeps the plain 1/N mean of Eq. (35) over the links that exist. */
int tdgl_set_insulators(tdgl_t *h, const tdgl_sphere *spheres_host, int64_t n);

/* Further generator shapes ("ellipsoids ... cylinders", Fig. 2(d) elliptical inclusions, Fig. 2(e) +-45 degree
 * columnar defects; reading S26).  Lengths in xi_0, domain coordinates; d = site position - c, minimum image on
 * periodic axes.  Inside tests, every operation a separately rounded fp64 operation in the order written:
 *   kind 0 sphere    : (d_x^2 + d_y^2) + d_z^2 <= a[0]^2
 *   kind 1 ellipsoid : ((d_x/a[0])^2 + (d_y/a[1])^2) + (d_z/a[2])^2 <= 1     (semi-axes along x, y, z)
 *   kind 2 cylinder  : t = (d_x n_x + d_y n_y) + d_z n_z with n = the given axis / its fp64 norm;
 *                      |t| <= a[1] (half-length) and ((d_x^2 + d_y^2) + d_z^2) - t^2 <= a[0]^2 (radius)
 * `kind` is stored as a float (0, 1, 2) so that a list is a plain float32 array of 10 columns. */
typedef struct { float kind; float c[3]; float a[3]; float n[3]; } tdgl_shape;

/* tdgl_set_pinning / tdgl_set_insulators with a list of shapes.  Same ownership and error rules; n <= N/10;
 * TDGL_EINVAL for an unknown kind, a non-positive radius / semi-axis / half-length or a zero cylinder axis. */
int tdgl_set_pinning_shapes(tdgl_t *h, const tdgl_shape *shapes_host, int64_t n, float eps_in, float eps_out);
int tdgl_set_insulator_shapes(tdgl_t *h, const tdgl_shape *shapes_host, int64_t n);

/* Applied field and transport current J_ext along x (Eq. 21).  The Landau gauge is fixed at create (S23):
 * xz gauge (default; Eq. 24a): B = (Bx, 0, Bz); yz gauge (TDGL_FLAG_GAUGE_YZ; Eq. 24b): B = (0, By, Bz).
 * B_z is snapped to 2 pi n_z/(Lx Ly) iff x and y are periodic; B_x to 2 pi n_x/(Ly Lz) iff y and z are; B_y to
 * 2 pi n_y/(Lx Lz) iff x and z are; the effective values are reported by tdgl_observables.
 * Resets Ex_mean.
 * Errors: TDGL_EINCOMPAT if By != 0 in the xz gauge, Bx != 0 in the yz gauge or for a film, or Jx != 0 with
 * open x. */
int tdgl_set_field_current(tdgl_t *h, float Bx, float By, float Bz, float Jx);

/* nsteps time steps in the paper's order "psi, then E, then mu": the implicit
 * Crank-Nicolson step (26) solved by Jacobi sweeps (33) to criterion (34), J_av (35) and the K update
 * (21), then rho = div j_s and the Poisson solve for mu (18).  Asynchronous on `stream`. */
int tdgl_step(tdgl_t *h, int32_t nsteps);

/* Device-to-device copy of the current state into caller buffers (either may be NULL):
 * psi_dev: N (re, im) fp32 pairs, 16-byte aligned; mu_dev: N fp32.  Asynchronous on `stream` (which of the two psi buffers
 * is current is device state; a copy kernel reads it on the device, the host never waits). */
int tdgl_get_psi_mu(tdgl_t *h, void *psi_dev, void *mu_dev);

/* Runs the reductions (a8) and fills *out_host.  Synchronises the stream.  Returns the latched warning, if any
 * (TDGL_WMAXSWEEPS before TDGL_WMUCAP when both are set; out_host->status carries both bits). */
int tdgl_observables(tdgl_t *h, tdgl_obs *out_host);

const char *tdgl_strerror(int code);
int tdgl_last_cuda_error(const tdgl_t *h);

/* Accuracy of the fp32 mu solve (Eq. 18).  The solver's own roundings and those of rho = div j_s are
 * white, and Delta_h^{-1} amplifies white noise by G = ((1/N) sum_{q != 0} 1/lambda_q^2)^{1/2} (lambda_q: eigenvalues
 * of the 7-point operator for this mesh and boundary types): |delta mu| ~ 2e-7 G rms(rho), measured.  G < 2 on the
 * 3D BASELINE grids, but it grows like L^{3/2} on quasi-one-dimensional meshes (500 on a 1026 x 3 film with open x).
 * With refinement on, every mu solve is followed by mu += Delta_h^{-1}(rho_64 - Delta_h mu), the residual being
 * evaluated in fp64 from psi (fp64 link variables): one more stencil pass and one more solve per step, 4 more
 * bytes of workspace per site.  tdgl_mu_gain returns G for these params (host arithmetic only; -1 if invalid). */
double tdgl_mu_gain(const tdgl_params *p_host);

/* The pseudo-time mu iteration (TDGL_FLAG_MU_ITERATIVE / TDGL_FLAG_FP64 only; else TDGL_EINVAL).  Per time step, warm-started
 * from the previous step's mu: outer iterations mu^- -> mu of one Crank-Nicolson step of d_tau mu = Delta_h mu - rho with
 * virtual step h_tau, N mu = c (Eq. 40) by Jacobi sweeps until max|N_mm (x^{l+1} - x^l)|^2 < eps_in, until
 * max|(mu - mu^-)/h_tau|^2 < eps_mu.  Defaults (S20): h_tau = 0.1, eps_mu = eps_in = 1e-6, max_outer = 1000,
 * max_inner = 100. */
int tdgl_set_mu_solver(tdgl_t *h, float h_tau, float eps_mu, float eps_in, int32_t max_outer, int32_t max_inner);
/* Log of the last `nsolves` mu solves (one per time step, and one per tdgl_debug_poisson call in this mode): outer_host[s] = outer iterations of solve s (oldest first);
 * inner_host = the Jacobi sweep counts of all those outer iterations in order (sum(outer_host) entries, at most
 * inner_cap, else TDGL_ENOMEM); *n_inner_host = that number.  Host arrays, any may be NULL.  Synchronises the stream. */
int tdgl_get_mu_log(tdgl_t *h, int32_t nsolves, int32_t *outer_host, int32_t *inner_host, int32_t inner_cap, int32_t *n_inner_host);
int tdgl_mu_refine_enabled(const tdgl_t *h);      /* 1 / 0 */

/* ---- extensions used by the tests and the bench (not part of the paper's problem statement) ---- */

/* Replace the state: psi_dev (N float pairs), mu_dev (N floats, may be NULL = keep) and K. */
int tdgl_set_state(tdgl_t *h, const void *psi_dev, const void *mu_dev, double K);
/* Change the solver controls between steps (S9 replay: fixed_sweeps > 0 runs exactly that many). */
int tdgl_set_solver(tdgl_t *h, float eps_tol, int32_t max_sweeps, int32_t fixed_sweeps);
/* Per-step replay of prescribed sweep counts: counts_host[s] sweeps in the s-th step from now on, for
 * n steps; after that the solver goes back to its own test.  n = 0 clears. n <= 65536. */
int tdgl_set_sweep_schedule(tdgl_t *h, const int32_t *counts_host, int32_t n);
/* Sweep counts and deciding max|r|^2 of the last n steps (oldest first) into host arrays
 * (either may be NULL).  n <= min(steps, 65536).  Synchronises the stream. */
int tdgl_get_sweep_log(tdgl_t *h, int32_t *counts_host, float *resid2_host, int32_t n);
/* Copy eps (N fp32) / the per-site Langevin term zeta of step index `step` (N float pairs) to caller
 * device buffers: bit-exactness checks of the inclusion kernel (a0) and of the Philox stream (a2). */
int tdgl_get_eps(tdgl_t *h, void *eps_dev);
int tdgl_debug_noise(tdgl_t *h, int64_t step, void *zeta_dev);
/* Single operators for kernel-level parity: one Poisson solve mu = Delta_h^{-1} rho (rho_dev and
 * mu_dev: N fp32, may alias), and rho = div j_s of the current state with the current K. */
int tdgl_debug_poisson(tdgl_t *h, const void *rho_dev, void *mu_dev);
int tdgl_debug_rho(tdgl_t *h, void *rho_dev);
/* Number of kernels the library has launched on this handle since create (bench: gpu_launches). */
int64_t tdgl_launch_count(const tdgl_t *h);
/* CUDA-event timing of the sweep kernels in HOST_LOOP mode: enable = 1 brackets every launch of the plain sweep kernel
 * by events on the stream, enable = 2 every launch of the fused two-sweep kernel (see tdgl_set_pair_mode); one kernel
 * at a time while timing is on.  The call returns the milliseconds and launches accumulated so far and, with enable > 0,
 * clears them.  Used by bench.py for the roofline figures. */
int tdgl_sweep_timing(tdgl_t *h, int32_t enable, double *ms_total_host, int64_t *launches_host);

/* TDGL_FLAG_MU_DIRECT: solves since create, refinement passes since create (each pass = one fp32 transform solve + one
 * fp64 residual), max |rho - Delta_h mu| of the last solve. */
int tdgl_get_mu_direct_stats(tdgl_t *h, int64_t *solves_host, int64_t *passes_host, double *resid_last_host);

/* Fused sweep pairs (temporal blocking of Eq. 33; march_pair.cu).  On meshes that admit it (xz gauge, fp32, nx % 128 == 0,
 * ny % 16 == 0, ny >= 32, nz >= 4) two Jacobi sweeps run as ONE pass over HBM whenever two more sweeps are certain
 * (prescribed counts) or predicted from the residual history.  Criterion (34) stays exact: both residuals are reduced,
 * and a pair whose first sweep already met the criterion is discarded and redone as a plain sweep, so psi, the sweep
 * counts, the residual log and J_av are bit-identical to plain sweeps.  mode: 0 never, 1 automatic (default), 2 whenever
 * the cap max_sweeps allows (tests: forces the redo path), 3 as 2 and a pair never sums the J_av links of its output (tests:
 * forces the separate pass k_jav_tiles, which otherwise runs only when a pair predicted not to end the step did end it).  tdgl_get_pair_stats: whether the mesh is eligible, pairs
 * launched, pairs discarded since create. */
int tdgl_set_pair_mode(tdgl_t *h, int32_t mode);
int tdgl_get_pair_stats(tdgl_t *h, int32_t *eligible_host, int64_t *pairs_host, int64_t *redone_host);

/* ---- for callers that cannot allocate device memory ---------------------------------------------------------------
 * <|psi|^2> (observable a8; the same per-site fp32 |psi_m|^2 summed in fp64 as tdgl_observables.mean_abs2) WITHOUT a
 * handle and WITHOUT a workspace.  Every other call needs the 44 B/site workspace the owner of the simulation allocated.
 * Code that merely sits beside a running solver and was handed a pointer to psi has none, and often cannot get any: an
 * in-situ monitor whose cudaMalloc / cudaFree would synchronise the device and stall the time-stepping stream, a plug-in
 * in a host application whose own pool reserved all of HBM at start-up (a cudaMalloc then fails), a component that is
 * forbidden to allocate after initialisation.  For them the scratch of the reduction (per-CTA partial sums and the
 * counter that elects the finishing CTA) lives in a fixed array inside the library image, and the call allocates
 * nothing -- no cudaMalloc, no cudaFree, no allocating library routine.
 *
 *   psi_dev   DEVICE, n_sites (re, im) fp32 pairs, 8-byte aligned (16-byte alignment takes the faster two-site loads); read only
 *   n_sites   1 ... TDGL_STATIC_MAX_SITES (2^29 = 1024 x 1024 x 512).  More: TDGL_ESCRATCH, nothing is enqueued or written
 *   mean_dev  DEVICE, one double, 8-byte aligned; written by the kernel, valid once the work enqueued on `stream` is done
 *   stream    cudaStream_t (NULL = legacy default stream) of the CURRENT device, which must own psi_dev and mean_dev
 *
 * What the built-in array implies:
 *   - TDGL_STATIC_SCRATCH_BYTES of device memory are held on every GPU that loads the library, until the process exits;
 *   - one array per device, shared by ALL calls: calls that can overlap on the GPU (different streams without an event
 *     between them, several host threads) race and return garbage.  Serialise them.  Calls on one stream are safe;
 *   - the array keeps the previous call's contents; what has to start at zero (the counter) is cleared on `stream` in
 *     front of every launch, so no call depends on how the previous one ended;
 *   - the FIRST call on each device resolves the array's device address (cudaGetSymbolAddress; the runtime may load the
 *     module on that device at this point).  Make that first call during start-up, before any stream capture begins.
 * Asynchronous.  Errors: TDGL_EINVAL (NULL / misaligned pointer, n_sites < 1), TDGL_ESCRATCH, TDGL_ECUDA (the runtime's
 * error is left in place for cudaGetLastError()).  The result does not depend on the number of SMs (fixed 65 536-site
 * chunks, partial sums added in index order). */
#define TDGL_STATIC_MAX_SITES     536870912
#define TDGL_STATIC_SCRATCH_BYTES 65792       /* 8192 fp64 partial sums + one 256-byte line for the counter */
int tdgl_mean_abs2_static(const void *psi_dev, int64_t n_sites, double *mean_dev, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* TDGL_H */
