// Device-side view of one TDGL problem: grid constants, workspace pointers and the control block.
// Shared by every kernel of libtdgl.  Citations: P:NNN = PAPER.md line, Sxx = DESIGN.md reading.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define TDGL_LOGCAP 65536            // ring of per-step sweep counts / residuals
#define TDGL_MAX_RESID_SLOTS 1024    // >= max_sweeps
#define TDGL_NPART 2048              // partial sums of the two-stage fp64 reductions
#define TDGL_MULOGCAP (1 << 18)      // ring of inner sweep counts of the pseudo-time mu iteration (one entry per outer iteration)

// Control block, resident in the workspace; written by kernels only (the host reads it back).
struct Ctl {
  double K;                 // gauge variable, Eq. (13)-(15)
  double Ex, Jav;           // last step
  double Ex_sum;            // running sum since set_field_current
  long long Ex_cnt;
  long long n;              // step index = Philox counter word 2 (S11)
  long long sweeps_total;
  int sweeps;               // sweeps done in the current step
  int done;                 // psi solve of the current step finished
  int use_pair;             // the next loop-body kernel to act is the fused two-sweep kernel (march_pair.cu), else the plain sweep
  int xbuf;                 // which psi buffer holds the latest iterate
  int status;               // latched warnings: bit 0 TDGL_WMAXSWEEPS, bit 1 TDGL_WMUCAP
  int sweeps_last;
  float resid_last;
  unsigned int ticket;      // last-block election of the sweep kernel
  unsigned int ticket2;     // ... of the reduction kernels
  // fused sweep pairs (march_pair.cu): 0 never, 1 when the residual history predicts that both sweeps are needed,
  // 2 whenever the cap allows (tests: exercises the redo path), 3 as 2 and never summing J_av inside a pair (tests:
  // exercises k_jav_tiles); residual of the previous sweep; statistics
  int pair_mode;
  int pair_jav;             // the next pair sums the J_av links of its output (it may be the last sweep of the step)
  int need_jav;             // the last sweep was a pair that did not: k_jav_tiles sums them
  float r_hist;
  long long pair_launches, pair_redone, body_launches;
  // solver controls (changed by tdgl_set_solver / tdgl_set_sweep_schedule)
  float eps_tol;
  int max_sweeps;
  int fixed_sweeps;
  int sched_n, sched_pos;   // prescribed per-step counts in sched[]
  double Jext;
  double Bx, Bz;            // effective field
  unsigned int resid_bits[TDGL_MAX_RESID_SLOTS];   // max |r|^2 of sweep l as uint bits (>= 0 floats order like uints)
  double obs[8];            // observables scratch
  // the paper's pseudo-time mu iteration (plain.cu; Eq. 40): controls, loop state, statistics
  float h_tau, eps_mu, eps_mu_in;
  int mu_max_outer, mu_max_inner;
  int mu_inner, mu_inner_done, mu_outer, mu_done;
  int mu_sched_n, mu_sched_pos;
  unsigned int mu_ticket;
  unsigned long long mu_r2bits;
  long long mu_log_pos, mu_solves, mu_outer_total, mu_inner_total;
  double mu_dt2_last;
  // direct mu solver of the double-precision build (TDGL_FLAG_MU_DIRECT: fp32 transform solver + fp64 iterative refinement)
  unsigned long long dref_rho_bits, dref_r_bits;   // max |rho|, max |rho - Delta_h mu| as fp64 bit patterns
  long long dref_solves, dref_passes;
  double dref_resid_last;
};

struct Dev {
  int nx, ny, nz;
  int bcx, bcy, bcz;        // 0 periodic, 1 open
  long long N;
  float cx, cy, cz;         // 1/hx^2, 1/hy^2, 1/(g hz)^2
  float ht2;                // h_t / 2
  float u;
  float csum2;              // 2 (cx + cy + cz)
  float zeta_max;           // Eq. (39); 0 = no noise
  double hx, hy, hz, dt, Lx, Ly, Lz;
  unsigned int seed_lo, seed_hi;
  int solve_mu;
  int zc;                   // planes per z-chunk of the marching kernels
  // workspace
  Ctl *ctl;
  float2 *psi[2];
  float2 *b, *d;
  float *mu, *eps, *scratch;
  float2 *Ux, *Uz;          // per-row link variables U_x(j), U_z(j)  (Eq. 27)
  float2 *Pi, *Pk;          // quasi-periodic jump P_{i,k} = Pi[i] conj(Pk[k])
  // yz Landau gauge (Eq. 24b, 29b): U_x = exp(i h_x K) for every row (Ux[] holds it), per-column
  // link variables U_y(i), U_z(i), jump in x  P_{j,k} = Pj[j] Pk[k]
  int gauge_yz;
  float2 *Uy, *Uzx, *Pj;
  // fp64 copies of all link / jump tables and the residual array of the mu refinement step (refine.cu)
  double2 *Ux64, *Uz64, *Pi64, *Pk64, *Uy64, *Uzx64, *Pj64;
  float *resid;             // N floats, only when mu_refine
  int mu_refine;            // one step of iterative refinement after every mu solve
  float *lam[3];            // eigenvalues of the 1-D operators per axis
  float2 *tw[3];            // FFT twiddles exp(-2 pi i m/n) per axis (power-of-two periodic axes)
  double *tab[3];           // generic transform tables: cas(2 pi m/n) or cos(pi m/(n-1))
  float2 *bT[3], *bC[3], *bH[3];   // Bluestein tables of the fast DCT-I per open axis (dct.cu)
  int bLB[3];               // its FFT length, 0 = axis not open / not supported
  const unsigned short *pfaT[3];   // index tables of the prime-factor DCT-I per open axis (dct_pfa.cu)
  int pfaK[3];              // its plan, -1 = none (the axis is periodic or its length has no plan)
  double *part;             // TDGL_NPART*4 partial sums
  double *jpart;            // one J_av partial sum per CTA of the marching kernels (in-tile x links of the new iterate)
  int *sweep_log; float *resid_log; int *sched;
  // double-precision build (TDGL_FLAG_FP64, plain.cu): the state in double, constants in double
  int fp64;
  double2 *psi64[2], *b64, *d64;
  double *mu64;
  double cx64, cy64, cz64, csum2_64, ht2_64, u64, zeta_max64;
  // insulating inclusions (TDGL_FLAG_INSULATORS, reading S25): 1 = superconducting site, 0 = removed; nullptr = none
  unsigned char *sc;
  // pseudo-time mu iteration (TDGL_FLAG_MU_ITERATIVE): rho, c, two Jacobi iterates (float or double), logs
  int mu_iterative;
  void *mu_rho, *mu_c, *mu_xa, *mu_xb;
  int *mu_log, *mu_outer_log, *mu_sched;
  int mu_direct64;          // TDGL_FLAG_MU_DIRECT: rho in mu_rho (double), residual / correction in resid (float)
  int pair_ok;              // the mesh admits the fused two-sweep kernel (march_pair.cu)
  unsigned long long cond_handle;   // cudaGraphConditionalHandle of the WHILE node (graph mode)
  int use_cond;
};

// SMs of the current device, cached per device (tdgl_api.cu): grid caps are multiples of it
int tdgl_sm_count();

// complex products with the contraction spelled out (one product, one FMA per component): the plain sweep and the
// fused pair kernel must round identically, whatever the compiler would choose in either context
__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
  return make_float2(__fmaf_rn(a.x, b.x, -__fmul_rn(a.y, b.y)), __fmaf_rn(a.x, b.y, __fmul_rn(a.y, b.x)));
}
__device__ __forceinline__ float2 cmulc(float2 a, float2 b) {   // conj(a) * b
  return make_float2(__fmaf_rn(a.x, b.x, __fmul_rn(a.y, b.y)), __fmaf_rn(a.x, b.y, -__fmul_rn(a.y, b.x)));
}
