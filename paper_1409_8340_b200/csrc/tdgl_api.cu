// C ABI of libtdgl (include/tdgl.h): parameter validation, workspace carving, the per-step launch
// sequence (host loop or CUDA graph with a WHILE node around the Jacobi sweep), read-back.
#include <atomic>
#include "../../include/tdgl.h"
#include "tdgl_dev.cuh"
#include "march_tma.h"
#include "march_film.h"
#include "march_pair.h"
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

// launchers defined in the kernel files
int jav_edge_blocks(const Dev &dv, int tile_w);
void launch_jav_edges(const Dev &dv, int tile_w, int nblocks, cudaStream_t st);
void launch_step_begin(const Dev &dv, cudaStream_t st);
void launch_step_finish(const Dev &dv, int ncta, int nedge, cudaStream_t st);
cudaError_t poisson_configure(int nx, int ny, int nz);
void launch_build_tables(float *lam, float2 *tw, double *tab, int n, int open, double c, cudaStream_t st);
int poisson_solve(const Dev &dv, float *data, bool thomas_open_z, cudaStream_t st);
int dct_fast_lb(int n);
cudaError_t dct_fast_configure(int LB);
void launch_build_bluestein(float2 *T, float2 *C, float2 *H, int n, int LB, cudaStream_t st);
int dct_pfa_kind(int n);
size_t dct_pfa_table_entries(int kind);
void dct_pfa_build_table(int kind, bool xpass, unsigned short *host_out);
cudaError_t dct_pfa_configure(int kind);
void launch_init_state(const Dev &dv, float amp, cudaStream_t st);
void launch_ctl_reset(const Dev &dv, float tol, int maxs, int fixed, cudaStream_t st);
void launch_ctl_solver(const Dev &dv, float tol, int maxs, int fixed, cudaStream_t st);
void launch_ctl_sched(const Dev &dv, int n, cudaStream_t st);
void launch_ctl_pair_mode(const Dev &dv, int mode, cudaStream_t st);
void launch_ctl_state(const Dev &dv, double K, cudaStream_t st);
void launch_set_field(const Dev &dv, double Bx, double Bz, double J, cudaStream_t st);
void launch_fill(float *p, long long n, float v, cudaStream_t st);
void launch_spheres(const Dev &dv, const float4 *sph, long long n, float eps_in, cudaStream_t st);
void launch_noise(const Dev &dv, long long step, float2 *out, cudaStream_t st);
int launch_obs(const Dev &dv, cudaStream_t st);
void launch_copy_psi(const Dev &dv, float2 *out, cudaStream_t st);
void launch_mu_residual(const Dev &dv, const float *rho, const float *mu, float *out, cudaStream_t st);
void launch_obs_final(const Dev &dv, int npart, cudaStream_t st);
// plain.cu: double-precision build and the pseudo-time mu iteration
void launch_march64(int mode, const Dev &dv, cudaStream_t st);
int launch_jav64(const Dev &dv, cudaStream_t st);
void launch_init_state64(const Dev &dv, double amp, cudaStream_t st);
void launch_noise64(const Dev &dv, long long step, double2 *out, cudaStream_t st);
void launch_copy_psi64(const Dev &dv, double2 *out, cudaStream_t st);
int launch_obs64(const Dev &dv, cudaStream_t st);
void launch_fill64(double *p, long long n, double v, cudaStream_t st);
void launch_mu_begin(const Dev &dv, cudaStream_t st);
void launch_mu_end(const Dev &dv, cudaStream_t st);
void launch_mu_rhs(const Dev &dv, void *mu, cudaStream_t st);
void launch_mu_sweep(const Dev &dv, void *mu, cudaStream_t st);
void launch_mu_finish(const Dev &dv, void *mu, cudaStream_t st);
void launch_mu_controls(const Dev &dv, float h_tau, float eps_mu, float eps_in, int max_outer, int max_inner, cudaStream_t st);
void launch_mu_sched(const Dev &dv, int n, cudaStream_t st);
void launch_dref_ctl(const Dev &dv, int what, cudaStream_t st);
void launch_dref_begin(const Dev &dv, cudaStream_t st);
void launch_dref_add(const Dev &dv, cudaStream_t st);
void launch_dref_resid(const Dev &dv, cudaStream_t st);
void launch_dref_zero_mean(const Dev &dv, cudaStream_t st);
void launch_spheres_mask(const Dev &dv, const float4 *sph, long long n, unsigned char *mask, cudaStream_t st);
void launch_shapes(const Dev &dv, const float *shp, long long n, float eps_in, unsigned char *mask, cudaStream_t st);
void launch_apply_mask64(const Dev &dv, cudaStream_t st);
void launch_fill_u8(unsigned char *p, long long n, unsigned char v, cudaStream_t st);
void launch_mu_add(const Dev &dv, float *mu, const float *delta, cudaStream_t st);

#define MODE_SWEEP 0
#define MODE_INIT 1
#define MODE_RHO 2

struct tdgl {
  tdgl_params p;
  Dev dv;
  cudaStream_t stream;
  dim3 mgrid;                  // grid of the marching kernels: 128 x 8 tiles x z chunks
  MarchMaps maps;              // TMA tensor maps of psi[0], psi[1], b, d
  PairMaps pmaps;              // ... of the fused two-sweep kernel (march_pair.cu), when dv.pair_ok
  bool film;                   // nz = 1: the paper's 2D mode (S22), kernels of march_film.cu
  Dev dvp;                     // the Poisson solver's view of the grid (film: y takes the role of z)
  int jav_blocks;
  int last_cuda;
  int64_t launches;            // host-counted kernel launches (graph launches are counted from the log)
  int64_t graph_steps;
  int fixed_per_step;          // kernels per step apart from the plain sweeps
  double Bx_eff, Bz_eff;
  // graph mode
  bool use_graph;
  cudaGraph_t graph;
  cudaGraphExec_t exec;
  cudaStream_t cap_stream;
  // host loop
  int *h_flag;                 // pinned: [0] done, [1] sweeps
  int pred_units;              // predicted iterations of the sweep loop (host loop: enqueued before the first flag read)
  int pred_mu_inner;           // pseudo-time mu iteration: predicted Jacobi sweeps per outer iteration
  int64_t dref_passes;         // TDGL_FLAG_MU_DIRECT: refinement passes since create
  // sweep timing
  int timing;                  // 0 off, 1 plain sweeps, 2 fused pairs
  double t_ms;
  int64_t t_launches;
  cudaEvent_t ev0, ev1;
};

static size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// SMs of the CURRENT device (B200: 148), queried once per device; the launch geometry is sized in multiples of it
int tdgl_sm_count() {
  static std::atomic<int> cached[64];
  int dev = 0, v = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return 148; }
  if (dev >= 0 && dev < 64 && (v = cached[dev].load(std::memory_order_relaxed)) > 0) return v;
  if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || v <= 0) { cudaGetLastError(); return 148; }
  if (dev >= 0 && dev < 64) cached[dev].store(v, std::memory_order_relaxed);
  return v;
}
static int sm_count() { return tdgl_sm_count(); }

// launch geometry of the marching kernels (march_tma.cu): 128 x 8 tiles, one warp per row; z chunks chosen
// so that there are enough CTAs for ~4 waves of 2 CTAs/SM, chunks of at least 8 planes
static void march_geometry(const tdgl_params *p, unsigned *gx, unsigned *gy, unsigned *gz, int *zc_out) {
  const long long nsm = sm_count();
  const long long want = nsm * 2 * 4;
  if (p->nz == 1) {            // film (march_film.cu): strips of 1024 sites in x, chunks of rows in y
    const int a = march_film_strips(p->nx);
    int yc = p->ny;
    while (yc > 8 && (long long)a * ((p->ny + yc - 1) / yc) < want) yc = (yc + 1) / 2;
    *gx = (unsigned)a; *gy = (unsigned)((p->ny + yc - 1) / yc); *gz = 1; *zc_out = yc;
    return;
  }
  int a, b;
  march_tma_grid(p->nx, p->ny, &a, &b);
  int zc = p->nz;
  // chunks of >= 32 planes while that still gives ~4 waves (each chunk re-reads two planes and pays a prologue);
  // shorter chunks only to put at least one CTA on every SM (measured on C3: 32 planes 0.584 ms/step, 8 planes 0.616)
  auto ctas = [&](int z) { return (long long)a * b * ((p->nz + z - 1) / z); };
  while (zc > 32 && ctas(zc) < want) zc = (zc + 1) / 2;
  while (zc > 8 && ctas(zc) < nsm) zc = (zc + 1) / 2;
  *gx = (unsigned)a; *gy = (unsigned)b; *gz = (unsigned)((p->nz + zc - 1) / zc); *zc_out = zc;
}

static bool params_ok(const tdgl_params *p) {
  if (!p || p->struct_size != sizeof(tdgl_params)) return false;
  if (p->nx < 2 || p->ny < 2 || p->nz < 1 || (p->nx & 1)) return false;      // nz = 1: film (2D mode, S22)
  if ((long long)p->nx * p->ny * p->nz > (1ll << 40)) return false;
  // the strided transform passes put the "other" extent into grid.y (<= 65535): ny, nz for a 3D mesh, none for a film
  if (p->nz > 1 && (p->ny > 65535 || p->nz > 65535)) return false;
  if (!(p->hx > 0.f) || !(p->hy > 0.f) || !(p->hz > 0.f) || !(p->dt > 0.f) || !(p->u > 0.f) || !(p->g > 0.f)) return false;
  for (int a = 0; a < 3; ++a)
    if (p->bc[a] != TDGL_BC_PERIODIC && p->bc[a] != TDGL_BC_OPEN) return false;
  if (!(p->eps_tol >= 0.f) || p->max_sweeps < 1 || p->max_sweeps > TDGL_MAX_RESID_SLOTS || p->fixed_sweeps < 0 ||
      p->fixed_sweeps > TDGL_MAX_RESID_SLOTS) return false;
  if (!(p->temperature >= 0.f)) return false;
  if ((p->flags & TDGL_FLAG_GAUGE_YZ) && p->nz == 1) return false;          // films use the xz gauge
  if ((p->flags & TDGL_FLAG_MU_REFINE) && (p->flags & (TDGL_FLAG_MU_ITERATIVE | TDGL_FLAG_FP64))) return false;
  if ((p->flags & TDGL_FLAG_INSULATORS) && !(p->flags & TDGL_FLAG_FP64)) return false;   // cut links: plain kernels only
  if ((p->flags & TDGL_FLAG_MU_DIRECT) && (!(p->flags & TDGL_FLAG_FP64) || (p->flags & (TDGL_FLAG_MU_ITERATIVE | TDGL_FLAG_MU_REFINE |
                                                                                      TDGL_FLAG_INSULATORS)))) return false;
  return true;
}

// White-noise gain of the discrete inverse Laplacian, G = ((1/N) sum_{q != 0} 1/lambda_q^2)^{1/2} (refine.cu): the factor
// by which the solve amplifies the (white) fp32 roundings of rho and of the transform passes.  1/lambda^2 falls like
// |q|^-4, so the 48 smallest eigenvalues per axis carry the sum.  Host, fp64, from the params alone.
static double mu_gain(const tdgl_params *p) {
  const bool film = p->nz == 1;
  const int ns[3] = {p->nx, p->ny, p->nz};
  const int bcs[3] = {p->bc[0], p->bc[1], film ? TDGL_BC_PERIODIC : p->bc[2]};
  const double cs[3] = {1.0 / ((double)p->hx * p->hx), 1.0 / ((double)p->hy * p->hy),
                        film ? 0.0 : 1.0 / ((double)p->g * p->g * (double)p->hz * p->hz)};
  const double pi = 3.14159265358979323846;
  std::vector<double> lam[3];
  for (int a = 0; a < 3; ++a) {
    const int n = ns[a], keep = n < 48 ? n : 48;
    // eigenvalues in ascending |lambda|: open q = 0, 1, 2, ...; periodic 0, then the pairs (q, n - q)
    for (int t = 0; t < keep; ++t) {
      double ang;
      if (n == 1) ang = 0.0;
      else if (bcs[a] == TDGL_BC_OPEN) ang = pi * t / (n - 1);
      else ang = 2.0 * pi * ((t + 1) / 2) / n;
      lam[a].push_back(cs[a] * (2.0 - 2.0 * std::cos(ang)));
    }
  }
  double sum = 0.0;
  for (double lx : lam[0]) for (double ly : lam[1]) for (double lz : lam[2]) {
    const double l = lx + ly + lz;
    if (l > 1e-14) sum += 1.0 / (l * l);
  }
  return std::sqrt(sum / ((double)p->nx * p->ny * p->nz));
}
// Refinement of the mu solve: forced by TDGL_FLAG_MU_REFINE, suppressed by TDGL_FLAG_MU_NOREFINE, otherwise
// automatic for meshes whose gain exceeds TDGL_MU_REFINE_GAIN (quasi-1D / thin long films; never the 3D BASELINE grids)
static bool is_fp64(const tdgl_params *p) { return (p->flags & TDGL_FLAG_FP64) != 0; }
// the pseudo-time iteration is the mu solver of the double-precision build (the direct solver is fp32 only)
static bool is_mu_direct64(const tdgl_params *p) { return is_fp64(p) && (p->flags & TDGL_FLAG_SOLVE_MU) && (p->flags & TDGL_FLAG_MU_DIRECT); }
static bool is_mu_iterative(const tdgl_params *p) {
  return (p->flags & TDGL_FLAG_SOLVE_MU) && (p->flags & (TDGL_FLAG_MU_ITERATIVE | TDGL_FLAG_FP64)) && !is_mu_direct64(p);
}
static bool want_refine(const tdgl_params *p) {
  if (!(p->flags & TDGL_FLAG_SOLVE_MU) || (p->flags & TDGL_FLAG_MU_NOREFINE) || is_mu_iterative(p)) return false;
  if (p->flags & TDGL_FLAG_MU_REFINE) return true;
  return mu_gain(p) > TDGL_MU_REFINE_GAIN;
}

// workspace carving; with base == nullptr only the size is computed
static size_t carve(const tdgl_params *p, char *base, Dev *dv) {
  const size_t N = (size_t)p->nx * p->ny * p->nz;
  size_t off = 0;
  auto take = [&](size_t bytes) { char *q = base ? base + off : nullptr; off = align_up(off + bytes, 256); return q; };
  char *q;
  q = take(sizeof(Ctl)); if (dv) dv->ctl = (Ctl *)q;
  q = take(p->ny * sizeof(float2)); if (dv) dv->Ux = (float2 *)q;
  q = take(p->ny * sizeof(float2)); if (dv) dv->Uz = (float2 *)q;
  q = take(p->nx * sizeof(float2)); if (dv) dv->Pi = (float2 *)q;
  q = take(p->nz * sizeof(float2)); if (dv) dv->Pk = (float2 *)q;
  q = take(p->nx * sizeof(float2)); if (dv) dv->Uy = (float2 *)q;
  q = take(p->nx * sizeof(float2)); if (dv) dv->Uzx = (float2 *)q;
  q = take(p->ny * sizeof(float2)); if (dv) dv->Pj = (float2 *)q;
  q = take(p->ny * sizeof(double2)); if (dv) dv->Ux64 = (double2 *)q;
  q = take(p->ny * sizeof(double2)); if (dv) dv->Uz64 = (double2 *)q;
  q = take(p->nx * sizeof(double2)); if (dv) dv->Pi64 = (double2 *)q;
  q = take(p->nz * sizeof(double2)); if (dv) dv->Pk64 = (double2 *)q;
  q = take(p->nx * sizeof(double2)); if (dv) dv->Uy64 = (double2 *)q;
  q = take(p->nx * sizeof(double2)); if (dv) dv->Uzx64 = (double2 *)q;
  q = take(p->ny * sizeof(double2)); if (dv) dv->Pj64 = (double2 *)q;
  const int ns[3] = {p->nx, p->ny, p->nz};
  for (int a = 0; a < 3; ++a) {
    q = take(ns[a] * sizeof(float)); if (dv) dv->lam[a] = (float *)q;
    q = take(ns[a] * sizeof(float2)); if (dv) dv->tw[a] = (float2 *)q;
    q = take(2 * (size_t)ns[a] * sizeof(double)); if (dv) dv->tab[a] = (double *)q;
    q = take(4096 * sizeof(float2)); if (dv) dv->bT[a] = (float2 *)q;
    q = take(4096 * sizeof(float2)); if (dv) dv->bC[a] = (float2 *)q;
    q = take(4096 * sizeof(float2)); if (dv) dv->bH[a] = (float2 *)q;
    // open x / y axis whose length has a prime-factor DCT-I plan (open z is solved by the Thomas algorithm)
    const bool open_xy = a < 2 && p->bc[a] == TDGL_BC_OPEN;
    const int kind = open_xy ? dct_pfa_kind(ns[a]) : -1;
    q = take(dct_pfa_table_entries(kind) * sizeof(unsigned short));
    if (dv) { dv->pfaK[a] = kind; dv->pfaT[a] = kind >= 0 ? (const unsigned short *)q : nullptr; }
  }
  q = take((size_t)TDGL_NPART * 4 * sizeof(double)); if (dv) dv->part = (double *)q;
  {
    unsigned gx, gy, gz; int zc;
    march_geometry(p, &gx, &gy, &gz, &zc);
    q = take((size_t)gx * gy * gz * sizeof(double)); if (dv) dv->jpart = (double *)q;
  }
  q = take(TDGL_LOGCAP * sizeof(int)); if (dv) dv->sweep_log = (int *)q;
  q = take(TDGL_LOGCAP * sizeof(float)); if (dv) dv->resid_log = (float *)q;
  q = take(TDGL_LOGCAP * sizeof(int)); if (dv) dv->sched = (int *)q;
  q = take(TDGL_MULOGCAP * sizeof(int)); if (dv) dv->mu_log = (int *)q;
  q = take(TDGL_LOGCAP * sizeof(int)); if (dv) dv->mu_outer_log = (int *)q;
  q = take(TDGL_LOGCAP * sizeof(int)); if (dv) dv->mu_sched = (int *)q;
  const bool f64 = is_fp64(p), iter = is_mu_iterative(p);
  if (f64) {                                   // double-precision state: 72 B/site + the iteration's 32 B/site
    q = take(N * sizeof(double2)); if (dv) dv->psi64[0] = (double2 *)q;
    q = take(N * sizeof(double2)); if (dv) dv->psi64[1] = (double2 *)q;
    q = take(N * sizeof(double2)); if (dv) dv->b64 = (double2 *)q;
    q = take(N * sizeof(double2)); if (dv) dv->d64 = (double2 *)q;
    q = take(N * sizeof(double)); if (dv) dv->mu64 = (double *)q;
    q = take(N * sizeof(float)); if (dv) dv->eps = (float *)q;
    q = take(N * sizeof(float)); if (dv) dv->scratch = (float *)q;          // sphere list of tdgl_set_pinning
    if (p->flags & TDGL_FLAG_INSULATORS) { q = take(N); if (dv) dv->sc = (unsigned char *)q; }
  } else {
    q = take(N * sizeof(float2)); if (dv) dv->psi[0] = (float2 *)q;
    q = take(N * sizeof(float2)); if (dv) dv->psi[1] = (float2 *)q;
    q = take(N * sizeof(float2)); if (dv) dv->b = (float2 *)q;
    q = take(N * sizeof(float2)); if (dv) dv->d = (float2 *)q;
    q = take(N * sizeof(float)); if (dv) dv->mu = (float *)q;
    q = take(N * sizeof(float)); if (dv) dv->eps = (float *)q;
    q = take(N * sizeof(float)); if (dv) dv->scratch = (float *)q;
    if (want_refine(p)) { q = take(N * sizeof(float)); if (dv) { dv->resid = (float *)q; dv->mu_refine = 1; } }
  }
  if (iter) {                                  // rho, c and the two Jacobi iterates of Eq. (40)
    const size_t es = f64 ? sizeof(double) : sizeof(float);
    q = take(N * es); if (dv) dv->mu_rho = q;
    q = take(N * es); if (dv) dv->mu_c = q;
    q = take(N * es); if (dv) dv->mu_xa = q;
    q = take(N * es); if (dv) dv->mu_xb = q;
    if (dv) dv->mu_iterative = 1;
  }
  if (is_mu_direct64(p)) {                     // rho in double, the residual / correction the fp32 solver works on
    q = take(N * sizeof(double)); if (dv) dv->mu_rho = q;
    q = take(N * sizeof(float)); if (dv) { dv->resid = (float *)q; dv->mu_direct64 = 1; }
  }
  if (dv) dv->fp64 = f64 ? 1 : 0;
  return off;
}

static int cuda_fail(tdgl_t *h, cudaError_t e) {
  if (getenv("TDGL_DEBUG")) fprintf(stderr, "libtdgl: CUDA error %d: %s\n", (int)e, cudaGetErrorString(e));
  if (h) h->last_cuda = (int)e;
  return TDGL_ECUDA;
}
#define CK(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(h, e_); } while (0)
#define CKL() do { cudaError_t e_ = cudaGetLastError(); if (e_ != cudaSuccess) return cuda_fail(h, e_); } while (0)

extern "C" uint64_t tdgl_workspace_bytes(const tdgl_params *p) {
  if (!params_ok(p)) return 0;
  return (uint64_t)carve(p, nullptr, nullptr);
}

static void march(tdgl_t *h, int mode, const Dev &dv, cudaStream_t st) {
  if (dv.fp64) launch_march64(mode, dv, st);
  else if (h->film) launch_march_film(mode, dv, h->mgrid, st);
  else launch_march_tma(mode, dv, h->maps, h->mgrid, st);
}

// one iteration of the sweep loop: the fused pair kernel (acts only when the device-side choice says so) and the plain
// sweep (acts otherwise); a kernel whose turn it is not returns at once
static int sweep_unit(tdgl_t *h, const Dev &dv, cudaStream_t st) {
  int n = 0;
  if (dv.pair_ok) { launch_march_pair(dv, h->pmaps, st); ++n; }
  march(h, MODE_SWEEP, dv, st); ++n;
  return n;
}

// One solve of the paper's pseudo-time mu iteration (Eq. 40; plain.cu), host-driven: per outer iteration the right side c,
// Jacobi sweeps until the device-side inner test passes (speculative launches return at once when it has), the outer
// update and test.  `mu` holds mu^- (warm start) and receives mu; rho is in dv.mu_rho.  Two 8-byte flag reads per outer
// iteration.  Returns the launches made, or -1 on a CUDA error.
static int mu_iterative_solve(tdgl_t *h, void *mu) {
  cudaStream_t st = h->stream;
  const Dev &dv = h->dv;
  int n = 0;
  launch_mu_begin(dv, st); ++n;
  for (;;) {
    launch_mu_rhs(dv, mu, st); ++n;
    int launched = 0;
    for (;;) {
      int burst = h->pred_mu_inner - launched;
      if (burst < 1) burst = 1;
      for (int s = 0; s < burst; ++s) { launch_mu_sweep(dv, mu, st); ++launched; ++n; }
      if (cudaMemcpyAsync(h->h_flag + 8, &dv.ctl->mu_inner, 2 * sizeof(int), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
          cudaStreamSynchronize(st) != cudaSuccess) return -1;
      if (h->h_flag[9]) break;
    }
    h->pred_mu_inner = h->h_flag[8] < 1 ? 1 : h->h_flag[8];
    launch_mu_finish(dv, mu, st); ++n;
    if (cudaMemcpyAsync(h->h_flag + 10, &dv.ctl->mu_done, sizeof(int), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess) return -1;
    if (h->h_flag[10]) break;
  }
  launch_mu_end(dv, st); ++n;
  return n;
}

// Direct mu solve of the double-precision build (TDGL_FLAG_MU_DIRECT; plain.cu (1b)): fp32 transform solves inside fp64
// iterative refinement, host-driven: one 16-byte read per pass (max |rho|, max |r|).  Stops at max |r| <= 2e-15 max(1, max |rho|),
// when a pass no longer halves the residual (its fp64 rounding floor), or after 8 passes.  rho is in dv.mu_rho.
static int mu_direct64_solve(tdgl_t *h, const Dev &dv) {
  cudaStream_t st = h->stream;
  int n = 0;
  launch_dref_ctl(dv, 0, st); ++n;
  launch_dref_begin(dv, st); ++n;
  double prev = -1.0;
  for (int pass = 0; pass < 8; ++pass) {
    n += poisson_solve(h->dvp, dv.resid, true, st);
    launch_dref_add(dv, st); ++n;
    launch_dref_ctl(dv, 1, st); ++n;
    launch_dref_resid(dv, st); ++n;
    unsigned long long bits[2];
    if (cudaMemcpyAsync(bits, &dv.ctl->dref_rho_bits, sizeof(bits), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess) return -1;
    double rho_max, r_max;
    memcpy(&rho_max, &bits[0], 8); memcpy(&r_max, &bits[1], 8);
    h->dref_passes += 1;
    if (r_max <= 2e-15 * (rho_max > 1.0 ? rho_max : 1.0)) break;
    if (prev >= 0.0 && r_max > 0.5 * prev) break;
    prev = r_max;
  }
  launch_dref_zero_mean(dv, st); n += 2;            // S7 in fp64 (the fp32 solves leave an offset of ~1e-9)
  launch_dref_ctl(dv, 2, st); ++n;
  return n;
}

// the kernels of one step after the psi solve: J_av + K (a5), rho (a6), mu (a7)
static int enqueue_after_solve(tdgl_t *h, cudaStream_t st) {
  int n = 0;
  const bool kact = h->dv.solve_mu && h->dv.bcx == 0;
  if (h->dv.fp64) {
    // double-precision build: J_av by its own pass over all x links (fp64 partials in dv.part)
    int np = 0;
    if (kact) { np = launch_jav64(h->dv, st); ++n; }
    launch_step_finish(h->dv, 0, np, st); ++n;
  } else {
    // J_av: the in-tile x links were summed by the last sweep (one partial per CTA); the links that cross a
    // tile edge are summed here
    if (kact && h->dv.pair_ok) { launch_jav_tiles(h->dv, st); ++n; }   // (acts only after a pair that skipped its J_av sums)
    if (kact) { launch_jav_edges(h->dv, march_tma_tile_w(), h->jav_blocks, st); ++n; }
    launch_step_finish(h->dv, (int)(h->mgrid.x * h->mgrid.y * h->mgrid.z), h->jav_blocks, st); ++n;
  }
  if (h->dv.solve_mu && h->dv.mu_direct64) {
    Dev d2 = h->dv;                               // the rho kernel writes where "mu" points: into the rho array
    d2.mu64 = (double *)h->dv.mu_rho;
    march(h, MODE_RHO, d2, st); ++n;
    const int m = mu_direct64_solve(h, h->dv);
    if (m < 0) return -1;
    n += m;
  } else if (h->dv.solve_mu && h->dv.mu_iterative) {
    Dev d2 = h->dv;                               // the rho kernel writes where "mu" points: into the iteration's rho array
    d2.mu = (float *)h->dv.mu_rho; d2.mu64 = (double *)h->dv.mu_rho;
    march(h, MODE_RHO, d2, st); ++n;
    const int m = mu_iterative_solve(h, h->dv.fp64 ? (void *)h->dv.mu64 : (void *)h->dv.mu);
    if (m < 0) return -1;
    n += m;
  } else if (h->dv.solve_mu) {
    march(h, MODE_RHO, h->dv, st); ++n;
    n += poisson_solve(h->dvp, h->dv.mu, true, st);
    if (h->dv.mu_refine) {                       // mu += S(rho_64 - Delta_h mu)  (refine.cu)
      launch_mu_residual(h->dv, nullptr, h->dv.mu, h->dv.resid, st); ++n;
      n += poisson_solve(h->dvp, h->dv.resid, true, st);
      launch_mu_add(h->dv, h->dv.mu, h->dv.resid, st); ++n;
    }
  }
  return n;
}

// inside a capture segment: a failing call (or a failed captured launch) ends the capture and discards what it built,
// so that tdgl_destroy never sees a stream that is still capturing
#define CKCAP(call) do { cudaError_t e_ = (call); if (e_ == cudaSuccess) e_ = cudaGetLastError(); \
    if (e_ != cudaSuccess) { cudaGraph_t junk_ = nullptr; cudaStreamEndCapture(cs, &junk_); cudaGetLastError(); \
      return cuda_fail(h, e_); } } while (0)

static int build_graph(tdgl_t *h) {
  CK(cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking));
  CK(cudaGraphCreate(&h->graph, 0));
  cudaGraphConditionalHandle handle;
  CK(cudaGraphConditionalHandleCreate(&handle, h->graph, 0, 0));
  h->dv.cond_handle = (unsigned long long)handle;
  h->dv.use_cond = 1;
  cudaStream_t cs = h->cap_stream;
  // segment A: begin + fused init/first sweep
  CK(cudaStreamBeginCaptureToGraph(cs, h->graph, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal));
  launch_step_begin(h->dv, cs);
  march(h, MODE_INIT, h->dv, cs);
  CKCAP(cudaSuccess);
  cudaStreamCaptureStatus status;
  const cudaGraphNode_t *deps = nullptr;
  size_t ndeps = 0;
  CKCAP(cudaStreamGetCaptureInfo(cs, &status, nullptr, nullptr, &deps, &ndeps));
  std::vector<cudaGraphNode_t> tail(deps, deps + ndeps);
  cudaGraph_t g2;
  CK(cudaStreamEndCapture(cs, &g2));
  // WHILE node: one plain sweep per iteration; the sweep's last CTA sets the condition
  cudaGraphNodeParams np = {cudaGraphNodeTypeConditional};
  np.type = cudaGraphNodeTypeConditional;
  np.conditional.handle = handle;
  np.conditional.type = cudaGraphCondTypeWhile;
  np.conditional.size = 1;
  cudaGraphNode_t cond;
  CK(cudaGraphAddNode(&cond, h->graph, tail.data(), tail.size(), &np));
  cudaGraph_t body = np.conditional.phGraph_out[0];
  CK(cudaStreamBeginCaptureToGraph(cs, body, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal));
  sweep_unit(h, h->dv, cs);
  CKCAP(cudaSuccess);
  CK(cudaStreamEndCapture(cs, &g2));
  // segment B: everything after the psi solve
  CK(cudaStreamBeginCaptureToGraph(cs, h->graph, &cond, nullptr, 1, cudaStreamCaptureModeThreadLocal));
  h->fixed_per_step = 2 + enqueue_after_solve(h, cs);
  CKCAP(cudaSuccess);
  CK(cudaStreamEndCapture(cs, &g2));
  CK(cudaGraphInstantiate(&h->exec, h->graph, 0));
  return TDGL_OK;
}

// inside tdgl_create a failing CUDA call releases the half-built handle (pinned flag word, events, graph objects)
// (TDGL_DEBUG in the environment: say which call failed; tdgl_create has no handle to leave the code in)
static void create_fail(cudaError_t e, int line) {
  if (getenv("TDGL_DEBUG")) fprintf(stderr, "tdgl_create: %s (tdgl_api.cu:%d)\n", cudaGetErrorString(e), line);
}
#define CKC(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { create_fail(e_, __LINE__); tdgl_destroy(h); return TDGL_ECUDA; } } while (0)
#define CKCL() do { cudaError_t e_ = cudaGetLastError(); if (e_ != cudaSuccess) { create_fail(e_, __LINE__); tdgl_destroy(h); return TDGL_ECUDA; } } while (0)
extern "C" int tdgl_destroy(tdgl_t *h);

extern "C" int tdgl_create(const tdgl_params *p, tdgl_t **out) {
  if (!out) return TDGL_EINVAL;
  *out = nullptr;
  if (!params_ok(p)) return TDGL_EINVAL;
  const size_t need = carve(p, nullptr, nullptr);
  if (!p->workspace_dev || ((uintptr_t)p->workspace_dev & 255) || p->workspace_bytes < need) return TDGL_ENOMEM;
  tdgl_t *h = new (std::nothrow) tdgl();
  if (!h) return TDGL_ENOMEM;
  memset(h, 0, sizeof(*h));
  h->p = *p;
  h->stream = (cudaStream_t)p->stream;
  Dev &dv = h->dv;
  memset(&dv, 0, sizeof(dv));
  carve(p, (char *)p->workspace_dev, &dv);
  // film (nz = 1): the paper's 2D mode: no z links, no z faces, d = 2 in Eq. (39) (S22)
  const bool film = p->nz == 1;
  h->film = film;
  const int bcs[3] = {p->bc[0], p->bc[1], film ? TDGL_BC_PERIODIC : p->bc[2]};
  dv.nx = p->nx; dv.ny = p->ny; dv.nz = p->nz;
  dv.bcx = bcs[0]; dv.bcy = bcs[1]; dv.bcz = bcs[2];
  dv.N = (long long)p->nx * p->ny * p->nz;
  dv.hx = p->hx; dv.hy = p->hy; dv.hz = p->hz; dv.dt = p->dt;
  const double cx = 1.0 / (dv.hx * dv.hx), cy = 1.0 / (dv.hy * dv.hy),
               cz = film ? 0.0 : 1.0 / ((double)p->g * p->g * dv.hz * dv.hz);
  dv.cx = (float)cx; dv.cy = (float)cy; dv.cz = (float)cz;
  dv.csum2 = (float)(2.0 * (cx + cy + cz));
  dv.ht2 = (float)(0.5 * dv.dt / (double)p->u);
  dv.u = p->u;
  dv.Lx = (p->nx - (p->bc[0] ? 1 : 0)) * dv.hx;
  dv.Ly = (p->ny - (p->bc[1] ? 1 : 0)) * dv.hy;
  dv.Lz = (p->nz - (bcs[2] ? 1 : 0)) * dv.hz;
  // Eq. (39), S12: zeta_max = (3 T u / (2 dt hx hy hz))^{1/2}
  dv.zeta_max = p->temperature > 0.f
                    ? (float)std::sqrt(3.0 * (double)p->temperature * (double)p->u /
                                       (2.0 * dv.dt * dv.hx * dv.hy * (film ? 1.0 : dv.hz)))
                    : 0.f;
  dv.seed_lo = (unsigned)(p->seed & 0xffffffffull);
  dv.seed_hi = (unsigned)(p->seed >> 32);
  dv.solve_mu = (p->flags & TDGL_FLAG_SOLVE_MU) ? 1 : 0;
  dv.gauge_yz = (p->flags & TDGL_FLAG_GAUGE_YZ) ? 1 : 0;
  // the same constants in double, from the fp32 values that crossed the ABI widened (R2): what the fp64 oracle uses
  dv.cx64 = cx; dv.cy64 = cy; dv.cz64 = cz;
  dv.csum2_64 = 2.0 * (cx + cy + cz);
  dv.ht2_64 = 0.5 * ((double)p->dt / (double)p->u);
  dv.u64 = (double)p->u;
  dv.zeta_max64 = p->temperature > 0.f ? std::sqrt(3.0 * (double)p->temperature * (double)p->u /
                                                   (2.0 * dv.dt * dv.hx * dv.hy * (film ? 1.0 : dv.hz))) : 0.0;

  {
    unsigned gx, gy, gz; int zc;
    march_geometry(p, &gx, &gy, &gz, &zc);
    dv.zc = zc;
    h->mgrid = dim3(gx, gy, gz);
  }
  h->jav_blocks = jav_edge_blocks(dv, march_tma_tile_w());
  h->pred_units = 0;
  h->pred_mu_inner = 1;
  if (dv.fp64) {
    // plain kernels: nothing to configure
  } else if (film) {
    CKC(march_film_configure());
  } else {
    CKC(march_tma_configure());
    if (march_tma_build_maps(dv, &h->maps) != 0) { tdgl_destroy(h); return TDGL_ECUDA; }
    if (march_pair_ok(p->nx, p->ny, p->nz, dv.gauge_yz != 0)) {
      CKC(march_pair_configure());
      { const int rc_ = march_pair_build_maps(dv, &h->pmaps); if (rc_ != 0) { create_fail(cudaErrorUnknown, -rc_); tdgl_destroy(h); return TDGL_ECUDA; } }
      dv.pair_ok = 1;
    }
  }
  if (film) CKC(poisson_configure(p->nx, 1, p->ny));
  else CKC(poisson_configure(p->nx, p->ny, p->nz));
  CKC(cudaMallocHost((void **)&h->h_flag, 64));
  CKC(cudaEventCreate(&h->ev0));
  CKC(cudaEventCreate(&h->ev1));

  cudaStream_t st = h->stream;
  launch_ctl_reset(dv, p->eps_tol, p->max_sweeps, p->fixed_sweeps, st);
  const int ns[3] = {p->nx, p->ny, p->nz};
  const double cs[3] = {cx, cy, cz};
  for (int a = 0; a < 3; ++a) launch_build_tables(dv.lam[a], dv.tw[a], dv.tab[a], ns[a], bcs[a], cs[a], st);
  for (int a = 0; a < 3; ++a) {
    if (dv.pfaK[a] >= 0) {                          // prime-factor DCT-I: index tables built on the host
      CKC(dct_pfa_configure(dv.pfaK[a]));
      std::vector<unsigned short> tab(dct_pfa_table_entries(dv.pfaK[a]));
      dct_pfa_build_table(dv.pfaK[a], a == 0, tab.data());
      CKC(cudaMemcpyAsync((void *)dv.pfaT[a], tab.data(), tab.size() * sizeof(unsigned short), cudaMemcpyHostToDevice, st));
      CKC(cudaStreamSynchronize(st));               // the host table dies at the end of this block
      continue;
    }
    // Bluestein DCT-I tables only for the axes that are transformed: x, and y of a 3D mesh (open z, and the open y of a
    // film, which takes the z role, are solved by the Thomas algorithm)
    const bool dct_axis = a == 0 || (a == 1 && !film);
    dv.bLB[a] = (bcs[a] == TDGL_BC_OPEN && dct_axis) ? dct_fast_lb(ns[a]) : 0;
    if (dv.bLB[a]) {
      CKC(dct_fast_configure(dv.bLB[a]));
      launch_build_bluestein(dv.bT[a], dv.bC[a], dv.bH[a], ns[a], dv.bLB[a], st);
      h->launches += 1;
    }
  }
  // the Poisson solver's view: a film (nx, ny, 1) is solved as the grid (nx, 1, ny) -- x transform, then the y
  // direction takes the role of z (transform + divide + transform back, or Thomas when y is open)
  h->dvp = dv;
  if (film) {
    Dev &q = h->dvp;
    q.ny = 1; q.nz = p->ny; q.bcy = TDGL_BC_PERIODIC; q.bcz = bcs[1]; q.cz = (float)cy;
    q.lam[1] = dv.lam[2]; q.lam[2] = dv.lam[1];        // lam of the length-1 periodic axis is {0}
    q.tw[2] = dv.tw[1]; q.tab[2] = dv.tab[1];
    q.bT[2] = dv.bT[1]; q.bC[2] = dv.bC[1]; q.bH[2] = dv.bH[1]; q.bLB[2] = dv.bLB[1]; q.bLB[1] = 0;
    q.pfaK[2] = dv.pfaK[1]; q.pfaT[2] = dv.pfaT[1]; q.pfaK[1] = -1; q.pfaT[1] = nullptr;
  }
  if (dv.fp64) launch_init_state64(dv, (double)p->init_amp, st);
  else launch_init_state(dv, p->init_amp, st);
  if (dv.sc) { launch_fill_u8(dv.sc, dv.N, 1, st); h->launches += 1; }      // no site removed yet
  launch_set_field(dv, 0.0, 0.0, 0.0, st);
  launch_step_begin(dv, st);
  h->launches += 7;
  CKCL();
  // the pseudo-time mu iteration has two nested data-dependent loops: it is driven from the host
  h->use_graph = !(p->flags & TDGL_FLAG_HOST_LOOP) && !dv.mu_iterative && !dv.fp64;
  if (h->use_graph) {
    int rc = build_graph(h);
    if (rc != TDGL_OK) { tdgl_destroy(h); return rc; }
  }
  *out = h;
  return TDGL_OK;
}

extern "C" int tdgl_destroy(tdgl_t *h) {
  if (!h) return TDGL_EINVAL;
  cudaStreamSynchronize(h->stream);
  if (h->exec) cudaGraphExecDestroy(h->exec);
  if (h->graph) cudaGraphDestroy(h->graph);
  if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
  if (h->h_flag) cudaFreeHost(h->h_flag);
  if (h->ev0) cudaEventDestroy(h->ev0);
  if (h->ev1) cudaEventDestroy(h->ev1);
  delete h;
  return TDGL_OK;
}

extern "C" int tdgl_set_pinning(tdgl_t *h, const tdgl_sphere *sph, int64_t n, float eps_in, float eps_out) {
  if (!h || n < 0 || (n > 0 && !sph) || n > h->dv.N / 4) return TDGL_EINVAL;
  launch_fill(h->dv.eps, h->dv.N, eps_out, h->stream);
  h->launches += 1;
  if (n > 0) {
    CK(cudaMemcpyAsync(h->dv.scratch, sph, (size_t)n * sizeof(tdgl_sphere), cudaMemcpyHostToDevice, h->stream));
    CK(cudaStreamSynchronize(h->stream));       // the host list may be freed on return
    launch_spheres(h->dv, (const float4 *)h->dv.scratch, n, eps_in, h->stream);
    h->launches += (n + (1 << 20) - 1) >> 20;
  }
  CKL();
  return TDGL_OK;
}

extern "C" int tdgl_set_insulators(tdgl_t *h, const tdgl_sphere *sph, int64_t n) {
  if (!h || n < 0 || (n > 0 && !sph) || n > h->dv.N / 4) return TDGL_EINVAL;
  if (!h->dv.sc) return TDGL_EINCOMPAT;                       // created without TDGL_FLAG_INSULATORS
  launch_fill_u8(h->dv.sc, h->dv.N, 1, h->stream);
  h->launches += 1;
  if (n > 0) {
    CK(cudaMemcpyAsync(h->dv.scratch, sph, (size_t)n * sizeof(tdgl_sphere), cudaMemcpyHostToDevice, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    launch_spheres_mask(h->dv, (const float4 *)h->dv.scratch, n, h->dv.sc, h->stream);
    h->launches += (n + (1 << 20) - 1) >> 20;
  }
  launch_apply_mask64(h->dv, h->stream);                      // psi = 0, mu = 0 on the removed sites
  h->launches += 1;
  CKL();
  return TDGL_OK;
}

static bool shapes_ok(const tdgl_shape *shp, int64_t n) {
  for (int64_t q = 0; q < n; ++q) {
    const tdgl_shape &s = shp[q];
    if (s.kind < 0.f || s.kind > 2.f || s.kind != (float)(int)s.kind || !(s.a[0] > 0.f)) return false;
    if (s.kind == 1.f && (!(s.a[1] > 0.f) || !(s.a[2] > 0.f))) return false;
    if (s.kind == 2.f && (!(s.a[1] > 0.f) || !(s.n[0] * s.n[0] + s.n[1] * s.n[1] + s.n[2] * s.n[2] > 0.f))) return false;
  }
  return true;
}

extern "C" int tdgl_set_pinning_shapes(tdgl_t *h, const tdgl_shape *shp, int64_t n, float eps_in, float eps_out) {
  if (!h || n < 0 || (n > 0 && !shp) || n > h->dv.N / 10 || !shapes_ok(shp, n)) return TDGL_EINVAL;
  launch_fill(h->dv.eps, h->dv.N, eps_out, h->stream);
  h->launches += 1;
  if (n > 0) {
    CK(cudaMemcpyAsync(h->dv.scratch, shp, (size_t)n * sizeof(tdgl_shape), cudaMemcpyHostToDevice, h->stream));
    CK(cudaStreamSynchronize(h->stream));       // the host list may be freed on return
    launch_shapes(h->dv, (const float *)h->dv.scratch, n, eps_in, nullptr, h->stream);
    h->launches += (n + (1 << 20) - 1) >> 20;
  }
  CKL();
  return TDGL_OK;
}

extern "C" int tdgl_set_insulator_shapes(tdgl_t *h, const tdgl_shape *shp, int64_t n) {
  if (!h || n < 0 || (n > 0 && !shp) || n > h->dv.N / 10 || !shapes_ok(shp, n)) return TDGL_EINVAL;
  if (!h->dv.sc) return TDGL_EINCOMPAT;                       // created without TDGL_FLAG_INSULATORS
  launch_fill_u8(h->dv.sc, h->dv.N, 1, h->stream);
  h->launches += 1;
  if (n > 0) {
    CK(cudaMemcpyAsync(h->dv.scratch, shp, (size_t)n * sizeof(tdgl_shape), cudaMemcpyHostToDevice, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    launch_shapes(h->dv, (const float *)h->dv.scratch, n, 0.f, h->dv.sc, h->stream);
    h->launches += (n + (1 << 20) - 1) >> 20;
  }
  launch_apply_mask64(h->dv, h->stream);                      // psi = 0, mu = 0 on the removed sites
  h->launches += 1;
  CKL();
  return TDGL_OK;
}

extern "C" int tdgl_set_field_current(tdgl_t *h, float Bx, float By, float Bz, float Jx) {
  if (!h) return TDGL_EINVAL;
  const bool yz = h->dv.gauge_yz != 0;
  if ((!yz && By != 0.f) || (yz && Bx != 0.f)) return TDGL_EINCOMPAT;   // one Landau gauge per field plane
  if (h->film && Bx != 0.f) return TDGL_EINCOMPAT;           // a film has no z links for B_x to act on
  if (Jx != 0.f && h->dv.bcx == 1) return TDGL_EINCOMPAT;
  double bx = yz ? By : Bx, bz = Bz;                         // bx: the in-plane component (B_x or B_y)
  const double twopi = 2.0 * 3.14159265358979323846;
  if (h->dv.bcx == 0 && h->dv.bcy == 0) {
    const double a = h->dv.Lx * h->dv.Ly;
    const double q = std::nearbyint(bz * a / twopi);
    bz = twopi * q / a;
  }
  if (!yz && h->dv.bcy == 0 && h->dv.bcz == 0) {
    const double a = h->dv.Ly * h->dv.Lz;
    const double q = std::nearbyint(bx * a / twopi);
    bx = twopi * q / a;
  }
  if (yz && h->dv.bcx == 0 && h->dv.bcz == 0) {  // B_y = 2 pi n/(L_x L_z): continuity of P_{j,k} in z
    const double a = h->dv.Lx * h->dv.Lz;
    const double q = std::nearbyint(bx * a / twopi);
    bx = twopi * q / a;
  }
  h->Bx_eff = bx;
  h->Bz_eff = bz;
  launch_set_field(h->dv, bx, bz, (double)Jx, h->stream);
  launch_step_begin(h->dv, h->stream);           // refresh U_x(j) for the new field
  h->launches += 2;
  CKL();
  return TDGL_OK;
}

static int step_host_loop(tdgl_t *h) {
  cudaStream_t st = h->stream;
  const Dev &dv = h->dv;
  launch_step_begin(dv, st);
  march(h, MODE_INIT, dv, st);
  h->launches += 2;
  int launched = 0;                             // loop iterations (sweep units) enqueued
  const int cap = TDGL_MAX_RESID_SLOTS;
  for (;;) {
    // speculative iterations (their kernels return at once when the solve is already done), then one flag read
    int burst = h->timing ? 0 : h->pred_units - launched;
    for (int s = 0; s < burst && launched < cap; ++s) {
      h->launches += sweep_unit(h, dv, st);
      ++launched;
    }
    CK(cudaMemcpyAsync(h->h_flag, &dv.ctl->sweeps, 3 * sizeof(int), cudaMemcpyDeviceToHost, st));   // sweeps, done, use_pair
    CK(cudaStreamSynchronize(st));
    if (h->h_flag[1] || launched >= cap) break;
    if (!h->timing) {
      h->launches += sweep_unit(h, dv, st);
    } else {
      // timing mode: exactly the kernel whose turn it is, bracketed by events (kind 1: plain sweeps, kind 2: pairs)
      const bool pair = dv.pair_ok && h->h_flag[2];
      const bool timed = pair ? h->timing == 2 : h->timing == 1;
      if (timed) CK(cudaEventRecord(h->ev0, st));
      if (pair) launch_march_pair(dv, h->pmaps, st);
      else march(h, MODE_SWEEP, dv, st);
      ++h->launches;
      if (timed) {
        CK(cudaEventRecord(h->ev1, st));
        CK(cudaEventSynchronize(h->ev1));
        float ms = 0.f;
        CK(cudaEventElapsedTime(&ms, h->ev0, h->ev1));
        h->t_ms += ms;
        h->t_launches += 1;
      }
    }
    ++launched;
  }
  h->pred_units = launched < 1 ? 1 : launched;
  {
    const int m = enqueue_after_solve(h, st);
    if (m < 0) return cuda_fail(h, cudaGetLastError());
    h->launches += m;
  }
  CKL();
  return TDGL_OK;
}

extern "C" int tdgl_step(tdgl_t *h, int32_t nsteps) {
  if (!h || nsteps < 0) return TDGL_EINVAL;
  for (int s = 0; s < nsteps; ++s) {
    if (h->use_graph) {
      CK(cudaGraphLaunch(h->exec, h->stream));
      h->graph_steps += 1;
    } else {
      int rc = step_host_loop(h);
      if (rc != TDGL_OK) return rc;
    }
  }
  return TDGL_OK;
}

extern "C" int tdgl_get_psi_mu(tdgl_t *h, void *psi_dev, void *mu_dev) {
  if (!h || ((uintptr_t)psi_dev & 15)) return TDGL_EINVAL;
  if (h->dv.fp64) {                                 // double-precision build: N double pairs / N doubles
    if (psi_dev) { launch_copy_psi64(h->dv, (double2 *)psi_dev, h->stream); h->launches += 1; CKL(); }
    if (mu_dev) CK(cudaMemcpyAsync(mu_dev, h->dv.mu64, (size_t)h->dv.N * sizeof(double), cudaMemcpyDeviceToDevice, h->stream));
    return TDGL_OK;
  }
  if (psi_dev) {
    // which buffer holds psi is device state (ctl->xbuf): the copy kernel reads it on the device
    launch_copy_psi(h->dv, (float2 *)psi_dev, h->stream);
    h->launches += 1;
    CKL();
  }
  if (mu_dev) CK(cudaMemcpyAsync(mu_dev, h->dv.mu, (size_t)h->dv.N * sizeof(float), cudaMemcpyDeviceToDevice, h->stream));
  return TDGL_OK;
}

extern "C" int tdgl_observables(tdgl_t *h, tdgl_obs *out) {
  if (!h || !out) return TDGL_EINVAL;
  if (h->dv.fp64) { launch_obs_final(h->dv, launch_obs64(h->dv, h->stream), h->stream); h->launches += 2; }
  else h->launches += launch_obs(h->dv, h->stream);
  CKL();
  Ctl c;
  CK(cudaMemcpyAsync(&c, h->dv.ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  memset(out, 0, sizeof(*out));
  out->t = (double)c.n * h->dv.dt;
  out->K = c.K; out->Ex = c.Ex; out->Jav = c.Jav;
  out->Ex_mean = c.Ex_cnt > 0 ? c.Ex_sum / (double)c.Ex_cnt : 0.0;
  out->mean_abs2 = c.obs[0] / (double)h->dv.N;
  out->free_energy = (c.obs[1] + c.obs[2]) * h->dv.hx * h->dv.hy * (h->film ? 1.0 : h->dv.hz);
  out->vortices_per_slice = c.obs[3] / (double)h->dv.nz;
  out->max_resid2 = c.resid_last;
  out->Bx_eff = (float)h->Bx_eff; out->Bz_eff = (float)h->Bz_eff;
  out->steps = c.n; out->sweeps_total = c.sweeps_total; out->sweeps_last = c.sweeps_last;
  out->status = ((c.status & 1) ? TDGL_WMAXSWEEPS : 0) | ((c.status & 2) ? TDGL_WMUCAP : 0);
  return (c.status & 1) ? TDGL_WMAXSWEEPS : ((c.status & 2) ? TDGL_WMUCAP : TDGL_OK);
}

extern "C" const char *tdgl_strerror(int code) {
  switch (code) {
    case TDGL_OK: return "ok";
    case TDGL_EINVAL: return "invalid argument (size, mesh, boundary type, pointer or struct_size)";
    case TDGL_ENOMEM: return "workspace too small or misaligned";
    case TDGL_EINCOMPAT: return "incompatible request (open x with a current, a field component the chosen Landau gauge cannot carry, or a call the mode chosen at create does not support)";
    case TDGL_ECUDA: return "CUDA runtime error";
    case TDGL_ESCRATCH: return "more sites than the built-in scratch array of tdgl_mean_abs2_static covers (TDGL_STATIC_MAX_SITES)";
    case TDGL_WMAXSWEEPS: return "warning: Jacobi iteration hit max_sweeps";
    case TDGL_WMUCAP: return "warning: the pseudo-time mu iteration stopped at max_outer / max_inner before its tolerance was met";
    default: return "unknown code";
  }
}
extern "C" int tdgl_last_cuda_error(const tdgl_t *h) { return h ? h->last_cuda : 0; }
extern "C" int tdgl_set_mu_solver(tdgl_t *h, float h_tau, float eps_mu, float eps_in, int32_t max_outer, int32_t max_inner) {
  if (!h || !h->dv.mu_iterative || !(h_tau > 0.f) || !(eps_mu >= 0.f) || !(eps_in >= 0.f) || max_outer < 1 || max_inner < 1) return TDGL_EINVAL;
  launch_mu_controls(h->dv, h_tau, eps_mu, eps_in, max_outer, max_inner, h->stream);
  h->launches += 1;
  CKL();
  return TDGL_OK;
}

extern "C" int tdgl_get_mu_log(tdgl_t *h, int32_t nsolves, int32_t *outer_host, int32_t *inner_host, int32_t inner_cap,
                               int32_t *n_inner_host) {
  if (!h || !h->dv.mu_iterative || nsolves < 0 || nsolves > TDGL_LOGCAP || inner_cap < 0) return TDGL_EINVAL;
  Ctl c;
  CK(cudaMemcpyAsync(&c, h->dv.ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  if (nsolves > c.mu_solves) return TDGL_EINVAL;
  std::vector<int> lo(TDGL_LOGCAP);
  CK(cudaMemcpyAsync(lo.data(), h->dv.mu_outer_log, TDGL_LOGCAP * sizeof(int), cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  long long total = 0;
  for (int s = 0; s < nsolves; ++s) {
    const int o = lo[(c.mu_solves - nsolves + s) % TDGL_LOGCAP];
    if (outer_host) outer_host[s] = o;
    total += o;
  }
  if (n_inner_host) *n_inner_host = (int32_t)total;
  if (total > TDGL_MULOGCAP) return TDGL_EINVAL;
  if (inner_host) {
    if (total > inner_cap) return TDGL_ENOMEM;
    std::vector<int> li(TDGL_MULOGCAP);
    CK(cudaMemcpyAsync(li.data(), h->dv.mu_log, (size_t)TDGL_MULOGCAP * sizeof(int), cudaMemcpyDeviceToHost, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    for (long long q = 0; q < total; ++q) inner_host[q] = li[(c.mu_log_pos - total + q) % TDGL_MULOGCAP];
  }
  return TDGL_OK;
}

extern "C" double tdgl_mu_gain(const tdgl_params *p) { return params_ok(p) ? mu_gain(p) : -1.0; }
extern "C" int tdgl_mu_refine_enabled(const tdgl_t *h) { return h ? h->dv.mu_refine : TDGL_EINVAL; }

extern "C" int tdgl_set_state(tdgl_t *h, const void *psi_dev, const void *mu_dev, double K) {
  if (!h || !psi_dev) return TDGL_EINVAL;
  if (h->dv.fp64) {
    CK(cudaMemcpyAsync(h->dv.psi64[0], psi_dev, (size_t)h->dv.N * sizeof(double2), cudaMemcpyDeviceToDevice, h->stream));
    if (mu_dev) CK(cudaMemcpyAsync(h->dv.mu64, mu_dev, (size_t)h->dv.N * sizeof(double), cudaMemcpyDeviceToDevice, h->stream));
  } else {
    CK(cudaMemcpyAsync(h->dv.psi[0], psi_dev, (size_t)h->dv.N * sizeof(float2), cudaMemcpyDeviceToDevice, h->stream));
    if (mu_dev) CK(cudaMemcpyAsync(h->dv.mu, mu_dev, (size_t)h->dv.N * sizeof(float), cudaMemcpyDeviceToDevice, h->stream));
  }
  launch_ctl_state(h->dv, K, h->stream);
  launch_step_begin(h->dv, h->stream);
  h->launches += 2;
  if (h->dv.sc) { launch_apply_mask64(h->dv, h->stream); h->launches += 1; }
  CKL();
  return TDGL_OK;
}

extern "C" int tdgl_set_solver(tdgl_t *h, float eps_tol, int32_t max_sweeps, int32_t fixed_sweeps) {
  if (!h || !(eps_tol >= 0.f) || max_sweeps < 1 || max_sweeps > TDGL_MAX_RESID_SLOTS || fixed_sweeps < 0 ||
      fixed_sweeps > TDGL_MAX_RESID_SLOTS) return TDGL_EINVAL;
  launch_ctl_solver(h->dv, eps_tol, max_sweeps, fixed_sweeps, h->stream);
  h->launches += 1;
  h->p.max_sweeps = max_sweeps;
  CKL();
  return TDGL_OK;
}

extern "C" int tdgl_set_sweep_schedule(tdgl_t *h, const int32_t *counts, int32_t n) {
  if (!h || n < 0 || n > TDGL_LOGCAP || (n > 0 && !counts)) return TDGL_EINVAL;
  for (int s = 0; s < n; ++s)
    if (counts[s] < 1 || counts[s] > TDGL_MAX_RESID_SLOTS) return TDGL_EINVAL;
  if (n > 0) {
    CK(cudaMemcpyAsync(h->dv.sched, counts, (size_t)n * sizeof(int), cudaMemcpyHostToDevice, h->stream));
    CK(cudaStreamSynchronize(h->stream));
  }
  launch_ctl_sched(h->dv, n, h->stream);
  h->launches += 1;
  CKL();
  return TDGL_OK;
}

extern "C" int tdgl_get_sweep_log(tdgl_t *h, int32_t *counts, float *resid2, int32_t n) {
  if (!h || n < 0 || n > TDGL_LOGCAP) return TDGL_EINVAL;
  long long steps = 0;
  CK(cudaMemcpyAsync(&steps, &h->dv.ctl->n, sizeof(long long), cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  if (n > steps) return TDGL_EINVAL;
  std::vector<int> lc(TDGL_LOGCAP);
  std::vector<float> lr(TDGL_LOGCAP);
  CK(cudaMemcpyAsync(lc.data(), h->dv.sweep_log, TDGL_LOGCAP * sizeof(int), cudaMemcpyDeviceToHost, h->stream));
  CK(cudaMemcpyAsync(lr.data(), h->dv.resid_log, TDGL_LOGCAP * sizeof(float), cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  for (int s = 0; s < n; ++s) {
    const long long step = steps - n + s;
    if (counts) counts[s] = lc[step % TDGL_LOGCAP];
    if (resid2) resid2[s] = lr[step % TDGL_LOGCAP];
  }
  return TDGL_OK;
}

extern "C" int tdgl_get_eps(tdgl_t *h, void *eps_dev) {
  if (!h || !eps_dev) return TDGL_EINVAL;
  CK(cudaMemcpyAsync(eps_dev, h->dv.eps, (size_t)h->dv.N * sizeof(float), cudaMemcpyDeviceToDevice, h->stream));
  return TDGL_OK;
}

extern "C" int tdgl_debug_noise(tdgl_t *h, int64_t step, void *zeta_dev) {
  if (!h || !zeta_dev) return TDGL_EINVAL;
  if (h->dv.fp64) launch_noise64(h->dv, step, (double2 *)zeta_dev, h->stream);
  else launch_noise(h->dv, step, (float2 *)zeta_dev, h->stream);
  h->launches += 1;
  CKL();
  return TDGL_OK;
}

extern "C" int tdgl_debug_poisson(tdgl_t *h, const void *rho_dev, void *mu_dev) {
  if (!h || !rho_dev || !mu_dev) return TDGL_EINVAL;
  if (h->dv.mu_direct64) {                        // rho, mu: N doubles; the state's own mu is left alone
    CK(cudaMemcpyAsync(h->dv.mu_rho, rho_dev, (size_t)h->dv.N * sizeof(double), cudaMemcpyDeviceToDevice, h->stream));
    Dev d2 = h->dv;
    d2.mu64 = (double *)mu_dev;
    const int m = mu_direct64_solve(h, d2);
    if (m < 0) return cuda_fail(h, cudaGetLastError());
    h->launches += m;
    CKL();
    return TDGL_OK;
  }
  if (h->dv.mu_iterative) {                       // the pseudo-time iteration from mu = 0 on the given rho
    const size_t es = h->dv.fp64 ? sizeof(double) : sizeof(float);
    CK(cudaMemcpyAsync(h->dv.mu_rho, rho_dev, (size_t)h->dv.N * es, cudaMemcpyDeviceToDevice, h->stream));
    CK(cudaMemsetAsync(mu_dev, 0, (size_t)h->dv.N * es, h->stream));
    const int m = mu_iterative_solve(h, mu_dev);
    if (m < 0) return cuda_fail(h, cudaGetLastError());
    h->launches += m;
    CKL();
    return TDGL_OK;
  }
  if (h->dv.mu_refine)                            // keep rho: the residual needs it after the in-place solve
    CK(cudaMemcpyAsync(h->dv.resid, rho_dev, (size_t)h->dv.N * sizeof(float), cudaMemcpyDeviceToDevice, h->stream));
  if (rho_dev != mu_dev)
    CK(cudaMemcpyAsync(mu_dev, rho_dev, (size_t)h->dv.N * sizeof(float), cudaMemcpyDeviceToDevice, h->stream));
  h->launches += poisson_solve(h->dvp, (float *)mu_dev, true, h->stream);
  if (h->dv.mu_refine) {
    launch_mu_residual(h->dv, h->dv.resid, (const float *)mu_dev, h->dv.resid, h->stream);
    h->launches += 2 + poisson_solve(h->dvp, h->dv.resid, true, h->stream);
    launch_mu_add(h->dv, (float *)mu_dev, h->dv.resid, h->stream);
  }
  CKL();
  return TDGL_OK;
}

extern "C" int tdgl_debug_rho(tdgl_t *h, void *rho_dev) {
  if (!h || !rho_dev) return TDGL_EINVAL;
  Dev d2 = h->dv;
  d2.mu = (float *)rho_dev;                       // the rho kernel writes where mu lives
  d2.mu64 = (double *)rho_dev;
  march(h, MODE_RHO, d2, h->stream);
  h->launches += 1;
  CKL();
  return TDGL_OK;
}

extern "C" int64_t tdgl_launch_count(const tdgl_t *h) {
  if (!h) return 0;
  int64_t n = h->launches;
  if (h->use_graph && h->graph_steps > 0) {
    long long body = 0;
    if (cudaMemcpyAsync(&body, &h->dv.ctl->body_launches, sizeof(long long), cudaMemcpyDeviceToHost, h->stream) != cudaSuccess ||
        cudaStreamSynchronize(h->stream) != cudaSuccess)
      return -1;
    // per graph step: fixed_per_step kernels (begin, init+sweep 1, ...) + the kernels of the sweep loop (counted on the device)
    n += h->graph_steps * (int64_t)h->fixed_per_step + body;
  }
  return n;
}

extern "C" int tdgl_get_mu_direct_stats(tdgl_t *h, int64_t *solves, int64_t *passes, double *resid_last) {
  if (!h) return TDGL_EINVAL;
  if (!h->dv.mu_direct64) return TDGL_EINVAL;
  long long sv = 0; double rl = 0.0;
  CK(cudaMemcpyAsync(&sv, &h->dv.ctl->dref_solves, sizeof(sv), cudaMemcpyDeviceToHost, h->stream));
  CK(cudaMemcpyAsync(&rl, &h->dv.ctl->dref_resid_last, sizeof(rl), cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  if (solves) *solves = sv;
  if (passes) *passes = h->dref_passes;
  if (resid_last) *resid_last = rl;
  return TDGL_OK;
}

extern "C" int tdgl_set_pair_mode(tdgl_t *h, int32_t mode) {
  if (!h || mode < 0 || mode > 3) return TDGL_EINVAL;
  launch_ctl_pair_mode(h->dv, mode, h->stream);
  h->launches += 1;
  CKL();
  return TDGL_OK;
}

extern "C" int tdgl_get_pair_stats(tdgl_t *h, int32_t *eligible, int64_t *pairs, int64_t *redone) {
  if (!h) return TDGL_EINVAL;
  long long v[2] = {0, 0};
  CK(cudaMemcpyAsync(v, &h->dv.ctl->pair_launches, 2 * sizeof(long long), cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  if (eligible) *eligible = h->dv.pair_ok;
  if (pairs) *pairs = v[0];
  if (redone) *redone = v[1];
  return TDGL_OK;
}

extern "C" int tdgl_sweep_timing(tdgl_t *h, int32_t enable, double *ms_total, int64_t *launches) {
  if (!h) return TDGL_EINVAL;
  if (ms_total) *ms_total = h->t_ms;
  if (launches) *launches = h->t_launches;
  h->timing = enable < 0 ? 0 : (enable > 2 ? 1 : enable);
  if (enable) { h->t_ms = 0.0; h->t_launches = 0; }
  return TDGL_OK;
}
