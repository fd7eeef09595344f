// Set-up and on-request kernels: initial state (S13), inclusion pattern (a0), field tables (a1),
// observables (a8), control-block setters, Langevin-term dump for the Philox bit-exactness test.
#include "tdgl_dev.cuh"
#include "philox.cuh"

// psi0 = 1 + amp (N(0,1) + i N(0,1)): Box-Muller on Philox stream 1 words (S13); mu = 0; eps = 1.
__global__ void k_init_state(const __grid_constant__ Dev dv, float amp) {
  for (long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x; m < dv.N; m += (long long)gridDim.x * blockDim.x) {
    const PhiloxOut p = philox4x32_10((uint32_t)m, (uint32_t)((unsigned long long)m >> 32), 0u, 1u, dv.seed_lo, dv.seed_hi);
    const double u1 = u32_to_01(p.x0), u2 = u32_to_01(p.x1);
    const double rad = sqrt(-2.0 * log(u1));
    double s, c;
    sincospi(2.0 * u2, &s, &c);
    dv.psi[0][m] = make_float2((float)(1.0 + (double)amp * rad * c), (float)((double)amp * rad * s));
    dv.mu[m] = 0.f;
    dv.eps[m] = 1.f;
  }
}

__global__ void k_ctl_reset(const __grid_constant__ Dev dv, float eps_tol, int max_sweeps, int fixed_sweeps) {
  Ctl *c = dv.ctl;
  c->K = 0.0; c->Ex = 0.0; c->Jav = 0.0; c->Ex_sum = 0.0; c->Ex_cnt = 0; c->n = 0; c->sweeps_total = 0;
  c->sweeps = 0; c->done = 0; c->xbuf = 0; c->status = 0; c->sweeps_last = 0; c->resid_last = 0.f;
  c->ticket = 0u; c->ticket2 = 0u; c->use_pair = 0; c->pair_mode = 1; c->pair_jav = 1; c->need_jav = 0; c->r_hist = 0.f;
  c->pair_launches = 0; c->pair_redone = 0; c->body_launches = 0;
  c->eps_tol = eps_tol; c->max_sweeps = max_sweeps; c->fixed_sweeps = fixed_sweeps;
  c->sched_n = 0; c->sched_pos = 0; c->Jext = 0.0; c->Bx = 0.0; c->Bz = 0.0;
  c->h_tau = 0.1f; c->eps_mu = 1e-6f; c->eps_mu_in = 1e-6f; c->mu_max_outer = 1000; c->mu_max_inner = 100;   // S20
  c->mu_inner = 0; c->mu_inner_done = 0; c->mu_outer = 0; c->mu_done = 0; c->mu_sched_n = 0; c->mu_sched_pos = 0;
  c->mu_ticket = 0u; c->mu_r2bits = 0ull; c->mu_log_pos = 0; c->mu_solves = 0; c->mu_outer_total = 0; c->mu_inner_total = 0;
  c->mu_dt2_last = 0.0;
  c->dref_rho_bits = 0ull; c->dref_r_bits = 0ull; c->dref_solves = 0; c->dref_passes = 0; c->dref_resid_last = 0.0;
}
__global__ void k_ctl_solver(const __grid_constant__ Dev dv, float eps_tol, int max_sweeps, int fixed_sweeps) {
  dv.ctl->eps_tol = eps_tol; dv.ctl->max_sweeps = max_sweeps; dv.ctl->fixed_sweeps = fixed_sweeps;
}
__global__ void k_ctl_sched(const __grid_constant__ Dev dv, int n) { dv.ctl->sched_n = n; dv.ctl->sched_pos = 0; }
__global__ void k_ctl_pair_mode(const __grid_constant__ Dev dv, int mode) { dv.ctl->pair_mode = mode; }
__global__ void k_ctl_state(const __grid_constant__ Dev dv, double K) { dv.ctl->K = K; dv.ctl->xbuf = 0; }

// a1: the K-independent phase tables of the xz Landau gauge (Eq. 24a, 27):
//   U_z(j) = exp(-i h_z B_x ybar_j),  Pi[i] = exp(i i h_x L_y B_z),  Pk[k] = exp(i k h_z L_y B_x),
//   P_{i,k} = Pi[i] conj(Pk[k]).  fp64 trigonometry, fp32 tables.
__global__ void k_set_field(const __grid_constant__ Dev dv, double Bx, double Bz, double Jext) {
  const int tid = threadIdx.x, nth = blockDim.x;
  if (tid == 0) {
    dv.ctl->Bx = Bx; dv.ctl->Bz = Bz; dv.ctl->Jext = Jext; dv.ctl->Ex_sum = 0.0; dv.ctl->Ex_cnt = 0;
  }
  double s, c;
  if (dv.gauge_yz) {
    // yz gauge (Eq. 24b; "Bx" carries B_y): U_y(i) = exp(-i h_y B_z xbar_i), U_z(i) = exp(+i h_z B_y xbar_i),
    // Pj[j] = exp(-i j h_y L_x B_z), Pk[k] = exp(+i k h_z L_x B_y), P_{j,k} = Pj[j] Pk[k]
    const double By = Bx;
    for (int i = tid; i < dv.nx; i += nth) {
      const double xbar = i * dv.hx - 0.5 * dv.Lx;
      sincos(-dv.hy * Bz * xbar, &s, &c);
      dv.Uy[i] = make_float2((float)c, (float)s);
      dv.Uy64[i] = make_double2(c, s);
      sincos(dv.hz * By * xbar, &s, &c);
      dv.Uzx[i] = make_float2((float)c, (float)s);
      dv.Uzx64[i] = make_double2(c, s);
    }
    for (int j = tid; j < dv.ny; j += nth) {
      sincos(-(double)j * dv.hy * dv.Lx * Bz, &s, &c);
      dv.Pj[j] = make_float2((float)c, (float)s);
      dv.Pj64[j] = make_double2(c, s);
    }
    for (int k = tid; k < dv.nz; k += nth) {
      sincos((double)k * dv.hz * dv.Lx * By, &s, &c);
      dv.Pk[k] = make_float2((float)c, (float)s);
      dv.Pk64[k] = make_double2(c, s);
    }
    return;
  }
  for (int j = tid; j < dv.ny; j += nth) {
    const double ybar = j * dv.hy - 0.5 * dv.Ly;
    sincos(-dv.hz * Bx * ybar, &s, &c);
    dv.Uz[j] = make_float2((float)c, (float)s);
    dv.Uz64[j] = make_double2(c, s);
  }
  for (int i = tid; i < dv.nx; i += nth) {
    sincos((double)i * dv.hx * dv.Ly * Bz, &s, &c);
    dv.Pi[i] = make_float2((float)c, (float)s);
    dv.Pi64[i] = make_double2(c, s);
  }
  for (int k = tid; k < dv.nz; k += nth) {
    sincos((double)k * dv.hz * dv.Ly * Bx, &s, &c);
    dv.Pk[k] = make_float2((float)c, (float)s);
    dv.Pk64[k] = make_double2(c, s);
  }
}

// tdgl_get_psi_mu: copy the CURRENT psi buffer (ctl->xbuf, device state) to the caller's array, 16 bytes per access
__global__ void __launch_bounds__(256) k_copy_psi(const __grid_constant__ Dev dv, float2 *__restrict__ out) {
  const float4 *__restrict__ src = reinterpret_cast<const float4 *>(dv.psi[dv.ctl->xbuf & 1]);
  float4 *dst = reinterpret_cast<float4 *>(out);
  const long long n2 = dv.N / 2;                      // nx is even
  for (long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x; m < n2; m += (long long)gridDim.x * blockDim.x)
    dst[m] = __ldcs(src + m);
}

__global__ void k_fill_f32(float *p, long long n, float v) {
  for (long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x; m < n; m += (long long)gridDim.x * blockDim.x) p[m] = v;
}

// a0: one CTA per sphere writes eps_in inside its bounding box (idempotent scatter; never N x n_s).
// Inside test (P:245, 511 (i), S19): d_x^2 + d_y^2 + d_z^2 <= r^2 with d the minimum-image distance on
// periodic axes, evaluated in fp64 with every product and sum rounded separately (no contraction), so
// the mask does not depend on how the compiler fuses operations.
// mask != nullptr: the sphere REMOVES its sites instead (insulating inclusion, S25): mask[m] = 0.
__global__ void __launch_bounds__(128) k_spheres(const __grid_constant__ Dev dv, const float4 *__restrict__ sph, float eps_in,
                                                 unsigned char *mask) {
  const float4 s = sph[blockIdx.x];
  const int n[3] = {dv.nx, dv.ny, dv.nz};
  const int bc[3] = {dv.bcx, dv.bcy, dv.bcz};
  const double h[3] = {dv.hx, dv.hy, dv.hz};
  const double cc[3] = {(double)s.x, (double)s.y, (double)s.z};
  const double r = (double)s.w;
  const double r2 = __dmul_rn(r, r);
  int lo[3], ext[3];
  for (int a = 0; a < 3; ++a) {
    int l = (int)floor((cc[a] - r) / h[a]) - 1, u = (int)ceil((cc[a] + r) / h[a]) + 1;
    if (bc[a] == 1) { l = max(l, 0); u = min(u, n[a] - 1); }
    else if (u - l + 1 >= n[a]) { l = 0; u = n[a] - 1; }
    lo[a] = l;
    ext[a] = max(0, u - l + 1);
  }
  const long long cnt = (long long)ext[0] * ext[1] * ext[2];
  for (long long t = threadIdx.x; t < cnt; t += blockDim.x) {
    const int qx = (int)(t % ext[0]);
    const long long rest = t / ext[0];
    const int qy = (int)(rest % ext[1]), qz = (int)(rest / ext[1]);
    const int q[3] = {lo[0] + qx, lo[1] + qy, lo[2] + qz};
    int idx[3];
    double d2[3];
    for (int a = 0; a < 3; ++a) {
      int ii = q[a] % n[a];
      if (ii < 0) ii += n[a];
      idx[a] = ii;
      double d = __dsub_rn(__dmul_rn((double)ii, h[a]), cc[a]);
      if (bc[a] == 0) {
        const double L = __dmul_rn((double)n[a], h[a]);
        d = __dsub_rn(d, __dmul_rn(L, rint(__ddiv_rn(d, L))));
      }
      d2[a] = __dmul_rn(d, d);
    }
    if (__dadd_rn(__dadd_rn(d2[0], d2[1]), d2[2]) <= r2) {
      const long long m = idx[0] + (long long)dv.nx * (idx[1] + (long long)dv.ny * idx[2]);
      if (mask) mask[m] = 0;
      else dv.eps[m] = eps_in;
    }
  }
}

// Further generator shapes (Fig. 2d/e; reading S26): one CTA per shape walks the shape's bounding box.
// A shape is 10 floats (kind, c[3], a[3], n[3]): 0 sphere (radius a0), 1 axis-aligned ellipsoid (semi-axes a),
// 2 capped cylinder (radius a0, half-length a1, axis n normalised here in fp64).  As in k_spheres every fp64
// operation of the inside test is rounded separately, in the order of include/tdgl.h.
__global__ void __launch_bounds__(128) k_shapes(const __grid_constant__ Dev dv, const float *__restrict__ shp, float eps_in,
                                                unsigned char *mask) {
  const float *s = shp + 10ll * blockIdx.x;
  const int kind = (int)s[0];
  const int n[3] = {dv.nx, dv.ny, dv.nz};
  const int bc[3] = {dv.bcx, dv.bcy, dv.bcz};
  const double h[3] = {dv.hx, dv.hy, dv.hz};
  const double cc[3] = {(double)s[1], (double)s[2], (double)s[3]};
  const double a[3] = {(double)s[4], (double)s[5], (double)s[6]};
  double nh[3] = {0.0, 0.0, 0.0};
  double ext[3] = {a[0], a[0], a[0]};
  if (kind == 1) { ext[1] = a[1]; ext[2] = a[2]; }
  if (kind == 2) {
    const double v[3] = {(double)s[7], (double)s[8], (double)s[9]};
    const double nn = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(v[0], v[0]), __dmul_rn(v[1], v[1])), __dmul_rn(v[2], v[2])));
    for (int q = 0; q < 3; ++q) {
      nh[q] = __ddiv_rn(v[q], nn);
      ext[q] = fabs(nh[q]) * a[1] + a[0] * sqrt(fmax(0.0, 1.0 - nh[q] * nh[q])) + 1e-9;   // box only: any cover will do
    }
  }
  if (kind < 0 || kind > 2) return;
  int lo[3], cnt3[3];
  for (int q = 0; q < 3; ++q) {
    int l = (int)floor((cc[q] - ext[q]) / h[q]) - 1, u = (int)ceil((cc[q] + ext[q]) / h[q]) + 1;
    if (bc[q] == 1) { l = max(l, 0); u = min(u, n[q] - 1); }
    else if (u - l + 1 >= n[q]) { l = 0; u = n[q] - 1; }
    lo[q] = l;
    cnt3[q] = max(0, u - l + 1);
  }
  const double r2 = __dmul_rn(a[0], a[0]);
  const long long cnt = (long long)cnt3[0] * cnt3[1] * cnt3[2];
  for (long long t = threadIdx.x; t < cnt; t += blockDim.x) {
    const int qx = (int)(t % cnt3[0]);
    const long long rest = t / cnt3[0];
    const int qq[3] = {lo[0] + qx, lo[1] + (int)(rest % cnt3[1]), lo[2] + (int)(rest / cnt3[1])};
    int idx[3];
    double d[3];
    for (int q = 0; q < 3; ++q) {
      int ii = qq[q] % n[q];
      if (ii < 0) ii += n[q];
      idx[q] = ii;
      double dd = __dsub_rn(__dmul_rn((double)ii, h[q]), cc[q]);
      if (bc[q] == 0) {
        const double L = __dmul_rn((double)n[q], h[q]);
        dd = __dsub_rn(dd, __dmul_rn(L, rint(__ddiv_rn(dd, L))));
      }
      d[q] = dd;
    }
    bool in;
    if (kind == 1) {
      const double ex = __ddiv_rn(d[0], a[0]), ey = __ddiv_rn(d[1], a[1]), ez = __ddiv_rn(d[2], a[2]);
      in = __dadd_rn(__dadd_rn(__dmul_rn(ex, ex), __dmul_rn(ey, ey)), __dmul_rn(ez, ez)) <= 1.0;
    } else {
      const double dsq = __dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2]));
      if (kind == 0) in = dsq <= r2;
      else {
        const double tt = __dadd_rn(__dadd_rn(__dmul_rn(d[0], nh[0]), __dmul_rn(d[1], nh[1])), __dmul_rn(d[2], nh[2]));
        in = fabs(tt) <= a[1] && __dsub_rn(dsq, __dmul_rn(tt, tt)) <= r2;
      }
    }
    if (in) {
      const long long m = idx[0] + (long long)dv.nx * (idx[1] + (long long)dv.ny * idx[2]);
      if (mask) mask[m] = 0;
      else dv.eps[m] = eps_in;
    }
  }
}

// zeta_m of step `step` (Eq. 39; S11') exactly as the init kernel draws it.
__global__ void k_noise(const __grid_constant__ Dev dv, long long step, float2 *out) {
  for (long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x; m < dv.N; m += (long long)gridDim.x * blockDim.x) {
    uint32_t wr, wi;
    langevin_words((unsigned long long)m, (uint32_t)step, dv.seed_lo, dv.seed_hi, wr, wi);
    out[m] = make_float2(dv.zeta_max * u32_to_pm1(wr), dv.zeta_max * u32_to_pm1(wi));
  }
}

// a8: observables.  Per-CTA fp64 partial sums of
//   [0] sum |psi|^2   [1] sum w (-eps |psi|^2 + |psi|^4/2)   [2] sum_alpha c_alpha sum_links w_link |S+ psi - psi|^2
//   [3] sum of rounded plaquette windings
// Free energy and winding definitions: DESIGN.md "Observables" (the paper only names F_GL).
__device__ __forceinline__ float face_w(int idx, int n, int open) { return (open && (idx == 0 || idx == n - 1)) ? 0.5f : 1.f; }

// Work item = 31 consecutive columns x OBS_RB consecutive rows of one plane, one WARP per item: lane q < 31 owns column
// 31 wc + q and walks down the rows, so that psi(i, j+1) and the x-link phase of row j + 1 are carried into the next row;
// lane q + 1 owns the EAST neighbour column, so psi(i+1, .) and the y-link phase of column i + 1 arrive by shuffle instead of
// by loads and a second arctangent.  The last lane of the warp (and the lane just past the last column: column 0 again when x
// is periodic) only supplies its column to its western neighbour and accumulates nothing.  Per site that leaves three 8-byte
// loads (psi of the next row, psi of the plane above, eps) and two arctangents.  Sums of a work item are formed in fp32
// (at most OBS_RB terms; the windings are small integers) and promoted to fp64 once per item.
#define OBS_RB 16
#define OBS_WC 31

// arg(x + i y) in (-pi, pi], absolute error 1.1e-7 rad (fp32 rounding level; the windings below are rint() of sums that are
// integers up to ~1e-6): octant reduction, one approximate division, atan(a)/a on [0, 1] as a degree-8 polynomial in a^2
// (Chebyshev fit, coefficients from a least-squares fit on 4000 Chebyshev nodes; max error checked in fp32 on 200 001 points).
__device__ __forceinline__ float obs_arg(float y, float x) {
  const float ax = fabsf(x), ay = fabsf(y);
  const float mx = fmaxf(fmaxf(ax, ay), 1.17549435e-38f), mn = fminf(ax, ay);      // arg(0) = 0, never NaN
  const float a = __fdividef(mn, mx), s = a * a;
  float r = 0.0028340641874819994f;
  r = fmaf(r, s, -0.016005029901862144f);
  r = fmaf(r, s, 0.042587608098983765f);
  r = fmaf(r, s, -0.07495445758104324f);
  r = fmaf(r, s, 0.10636754333972931f);
  r = fmaf(r, s, -0.14202570915222168f);
  r = fmaf(r, s, 0.19992484152317047f);
  r = fmaf(r, s, -0.3333306610584259f);
  r = fmaf(r, s, 1.0f);
  r *= a;
  if (ay > ax) r = 1.57079637f - r;
  if (x < 0.f) r = 3.14159274f - r;
  return copysignf(r, y);
}

template <bool YZ>
__global__ void __launch_bounds__(256, 4) k_obs_partial(const __grid_constant__ Dev dv) {
  const float2 *__restrict__ x = dv.psi[dv.ctl->xbuf];
  const int nx = dv.nx, ny = dv.ny, nz = dv.nz;
  const float inv2pi = 0.15915494309189535f;
  const float flux = (float)(dv.ctl->Bz * dv.hx * dv.hy);
  const bool px = dv.bcx == 0, py = dv.bcy == 0;
  const bool xjump = YZ && px, yjump = !YZ && py;
  const int lane = threadIdx.x & 31;
  const int nrb = (ny + OBS_RB - 1) / OBS_RB;
  const int ncw = (nx + OBS_WC - 1) / OBS_WC;
  const long long nitems = (long long)nrb * nz * ncw;
  const long long plane = (long long)nx * ny;
  double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
  for (long long item = (long long)blockIdx.x * 8 + (threadIdx.x >> 5); item < nitems; item += (long long)gridDim.x * 8) {
    const int wc = (int)(item % ncw);
    const long long blk = item / ncw;
    const int k = (int)(blk / nrb), jb = (int)(blk - (long long)k * nrb) * OBS_RB, je = min(ny, jb + OBS_RB);
    const int kp = (k + 1 == nz) ? 0 : k + 1;
    const bool hasz = dv.bcz == 0 || k + 1 < nz;
    const float wz = face_w(k, nz, dv.bcz);
    const float2 Pk = dv.Pk[k];
    const int ic = wc * OBS_WC + lane;
    const bool act = lane < OBS_WC && ic < nx;                       // this lane accumulates the sites of column ic
    const int col = ic < nx ? ic : ((px && ic == nx) ? 0 : nx - 1);  // the column it reads (helper lanes: the east neighbour's)
    const bool hasx = px || ic + 1 < nx, wrapx = ic + 1 == nx;
    const float wx = face_w(col, nx, dv.bcx);
    // row pointers advance by nx per row (no 64-bit index arithmetic in the loop); weights that do not change along the
    // walk are folded once per item: x links carry w_y w_z, y links w_x w_z, z links w_x w_y (O: DESIGN.md "Observables")
    const float2 *prow = x + plane * k + (long long)nx * jb + col;              // psi(col, j, k)
    const float2 *ptop = x + plane * kp + (long long)nx * jb + col;             // psi(col, j, k + 1)
    const float *erow = dv.eps + plane * k + (long long)nx * jb + col;
    const float2 *prow0 = x + plane * k + col;                                  // row 0 of the plane (wrap of j + 1)
    const float fx = hasx ? dv.cx * wz : 0.f, fy = dv.cy * wx * wz, fz = hasz ? dv.cz * wx : 0.f, fs = wx * wz;
    const float2 one = make_float2(1.f, 0.f);
    const float2 Uyc = YZ ? dv.Uy[col] : one, Uzc = YZ ? dv.Uzx[col] : one;
    const float2 Pic = yjump ? dv.Pi[col] : one;
    // x link of row j: psi*(i,j) U_x(j) psi(i+1,j) (times conj P_{j,k} on the yz-gauge seam); ee = psi(i+1, j)
    auto xlink = [&](int j, float2 ee) -> float2 {
      float2 e = cmul(dv.Ux[j], ee);
      if (xjump && wrapx) e = cmulc(cmul(dv.Pj[j], Pk), e);
      return e;
    };
    auto ylink = [&](int j, float2 v) -> float2 {                     // S+_y psi of the own column at row j
      if (YZ) return cmul(Uyc, v);
      if (yjump && j + 1 == ny) return cmulc(cmulc(Pk, Pic), v);
      return v;
    };
    float2 c = *prow;
    float2 er = make_float2(__shfl_down_sync(0xffffffffu, c.x, 1), __shfl_down_sync(0xffffffffu, c.y, 1));
    float2 e = xlink(jb, er);
    float gx0;
    { const float2 g = cmulc(c, e); gx0 = obs_arg(g.y, g.x); }
    float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
    // the three loads of a row are issued one row ahead (the walk is otherwise a chain of load -> use: 69 % of the stall
    // samples were long_scoreboard)
    int jn = (jb + 1 == ny) ? 0 : jb + 1;
    const float2 *pn = prow0 + (long long)nx * jn;                              // psi(col, j + 1, k)
    float2 nr = *pn, tz = *ptop;
    float ep = *erow;
    for (int j = jb; j < je; ++j) {
      const int jp = jn;
      float2 nr2 = nr, tz2 = tz;
      float ep2 = ep;
      if (j + 1 < je) {                                                         // (warp-uniform)
        jn = (jp + 1 == ny) ? 0 : jp + 1;
        pn = (jn == 0) ? prow0 : pn + nx;
        ptop += nx; erow += nx;
        nr2 = *pn; tz2 = *ptop; ep2 = *erow;
      }
      const bool hasy = py || j + 1 < ny;
      const float wy = face_w(j, ny, dv.bcy);
      const float2 ner = make_float2(__shfl_down_sync(0xffffffffu, nr.x, 1), __shfl_down_sync(0xffffffffu, nr.y, 1));
      const float2 t = cmul(YZ ? Uzc : dv.Uz[j], tz);
      const float2 nn = ylink(j, nr);
      const float ab = c.x * c.x + c.y * c.y;
      const float dxx = e.x - c.x, dxy = e.y - c.y, dyx = nn.x - c.x, dyy = nn.y - c.y, dzx = t.x - c.x, dzy = t.y - c.y;
      float g = fx * wy * (dxx * dxx + dxy * dxy);
      g += (hasy ? fy : 0.f) * (dyx * dyx + dyy * dyy);
      g += fz * wy * (dzx * dzx + dzy * dzy);
      // winding of the z-plaquette with corner (i, j):  g_x(i,j) + g_y(i+1,j) - g_x(i,j+1) - g_y(i,j) + B_z h_x h_y
      const float2 en = xlink(jp, ner);                               // row j+1
      float gx1, gy0;
      { const float2 q = cmulc(nr, en); gx1 = obs_arg(q.y, q.x); }
      { const float2 q = cmulc(c, nn); gy0 = obs_arg(q.y, q.x); }
      const float gy1 = __shfl_down_sync(0xffffffffu, gy0, 1);        // y-link phase of column i + 1, from its owner
      if (act) {
        s0 += ab;
        s1 += fs * wy * (ab * (0.5f * ab - ep));
        s2 += g;
        if (hasx && hasy) s3 += rintf((gx0 + gy1 - gx1 - gy0 + flux) * inv2pi);
      }
      c = nr; er = ner; e = en; gx0 = gx1;
      nr = nr2; tz = tz2; ep = ep2;
    }
    a0 += (double)s0; a1 += (double)s1; a2 += (double)s2; a3 += (double)s3;
  }
  __shared__ double sh[4][8];
  for (int o = 16; o > 0; o >>= 1) {
    a0 += __shfl_down_sync(0xffffffffu, a0, o);
    a1 += __shfl_down_sync(0xffffffffu, a1, o);
    a2 += __shfl_down_sync(0xffffffffu, a2, o);
    a3 += __shfl_down_sync(0xffffffffu, a3, o);
  }
  if ((threadIdx.x & 31) == 0) {
    sh[0][threadIdx.x >> 5] = a0; sh[1][threadIdx.x >> 5] = a1; sh[2][threadIdx.x >> 5] = a2; sh[3][threadIdx.x >> 5] = a3;
  }
  __syncthreads();
  if (threadIdx.x < 4) {
    double s = 0.0;
    for (int w = 0; w < 8; ++w) s += sh[threadIdx.x][w];
    dv.part[(size_t)threadIdx.x * TDGL_NPART + blockIdx.x] = s;
  }
}

__global__ void k_obs_final(const __grid_constant__ Dev dv, int npart) {
  __shared__ double sh[256];
  for (int q = 0; q < 4; ++q) {
    double s = 0.0;
    for (int p = threadIdx.x; p < npart; p += 256) s += dv.part[(size_t)q * TDGL_NPART + p];
    sh[threadIdx.x] = s;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
      if (threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
      __syncthreads();
    }
    if (threadIdx.x == 0) dv.ctl->obs[q] = sh[0];
    __syncthreads();
  }
}

// host-side launchers
static unsigned grid_for(long long n, int block, int cap) {
  long long g = (n + block - 1) / block;
  return (unsigned)(g < 1 ? 1 : (g > cap ? cap : g));
}
void launch_init_state(const Dev &dv, float amp, cudaStream_t st) { k_init_state<<<grid_for(dv.N, 256, tdgl_sm_count() * 16), 256, 0, st>>>(dv, amp); }
void launch_ctl_reset(const Dev &dv, float tol, int maxs, int fixed, cudaStream_t st) { k_ctl_reset<<<1, 1, 0, st>>>(dv, tol, maxs, fixed); }
void launch_ctl_solver(const Dev &dv, float tol, int maxs, int fixed, cudaStream_t st) { k_ctl_solver<<<1, 1, 0, st>>>(dv, tol, maxs, fixed); }
void launch_ctl_sched(const Dev &dv, int n, cudaStream_t st) { k_ctl_sched<<<1, 1, 0, st>>>(dv, n); }
void launch_ctl_pair_mode(const Dev &dv, int mode, cudaStream_t st) { k_ctl_pair_mode<<<1, 1, 0, st>>>(dv, mode); }
void launch_ctl_state(const Dev &dv, double K, cudaStream_t st) { k_ctl_state<<<1, 1, 0, st>>>(dv, K); }
void launch_set_field(const Dev &dv, double Bx, double Bz, double J, cudaStream_t st) { k_set_field<<<1, 256, 0, st>>>(dv, Bx, Bz, J); }
void launch_fill(float *p, long long n, float v, cudaStream_t st) { k_fill_f32<<<grid_for(n, 256, tdgl_sm_count() * 16), 256, 0, st>>>(p, n, v); }
static void spheres_impl(const Dev &dv, const float4 *sph, long long n, float eps_in, cudaStream_t st, unsigned char *mask) {
  for (long long off = 0; off < n; off += 1 << 20) {
    const unsigned g = (unsigned)((n - off) < (1 << 20) ? (n - off) : (1 << 20));
    k_spheres<<<g, 128, 0, st>>>(dv, sph + off, eps_in, mask);
  }
}
void launch_spheres(const Dev &dv, const float4 *sph, long long n, float eps_in, cudaStream_t st) { spheres_impl(dv, sph, n, eps_in, st, nullptr); }
void launch_spheres_mask(const Dev &dv, const float4 *sph, long long n, unsigned char *mask, cudaStream_t st) {
  spheres_impl(dv, sph, n, 0.f, st, mask);
}
void launch_shapes(const Dev &dv, const float *shp, long long n, float eps_in, unsigned char *mask, cudaStream_t st) {
  for (long long off = 0; off < n; off += 1 << 20) {
    const unsigned g = (unsigned)((n - off) < (1 << 20) ? (n - off) : (1 << 20));
    k_shapes<<<g, 128, 0, st>>>(dv, shp + 10 * off, eps_in, mask);
  }
}
void launch_copy_psi(const Dev &dv, float2 *out, cudaStream_t st) { k_copy_psi<<<grid_for(dv.N / 2, 256, tdgl_sm_count() * 16), 256, 0, st>>>(dv, out); }
void launch_noise(const Dev &dv, long long step, float2 *out, cudaStream_t st) { k_noise<<<grid_for(dv.N, 256, tdgl_sm_count() * 16), 256, 0, st>>>(dv, step, out); }
void launch_obs_final(const Dev &dv, int npart, cudaStream_t st) { k_obs_final<<<1, 256, 0, st>>>(dv, npart); }
int launch_obs(const Dev &dv, cudaStream_t st) {
  const long long nitems = (long long)((dv.ny + OBS_RB - 1) / OBS_RB) * dv.nz * ((dv.nx + OBS_WC - 1) / OBS_WC);   // one warp each
  const long long nblk = (nitems + 7) / 8;
  const int nb = (int)(nblk < TDGL_NPART ? nblk : TDGL_NPART);
  if (dv.gauge_yz) k_obs_partial<true><<<nb, 256, 0, st>>>(dv);
  else k_obs_partial<false><<<nb, 256, 0, st>>>(dv);
  k_obs_final<<<1, 256, 0, st>>>(dv, nb);
  return 2;
}
