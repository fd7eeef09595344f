// Precision-generic kernels of the hot path, templated on the real type T (float / double):
//
//  (1) the paper's OWN scalar-potential solver, TDGL_FLAG_MU_ITERATIVE (Eq. 40; readings S5, S20): pseudo-time
//      relaxation d_tau mu = Delta_h mu - rho, one Crank-Nicolson step of size h_tau per outer iteration, N mu = c solved
//      by Jacobi sweeps "like Eq. (33)", outer iterations until max|d_tau mu|^2 < eps_mu:
//         k_mu_rhs    c = mu^- + h_tau [ (Delta_h mu^-)/2 - rho ]                               12 B/site (T = float)
//         k_mu_sweep  x^{l+1} = (c + (h_tau/2) sum_alpha c_alpha (x^l_{+alpha} + x^l_{-alpha})) / N_mm, max residual, decision   12 B/site
//         k_mu_finish mu <- x, max |(x - mu^-)/h_tau|^2, outer decision, log                     12 B/site
//  (2) the DOUBLE-PRECISION build, TDGL_FLAG_FP64 (the paper ships SP and DP builds and times both: P:527, 579-581):
//      the marching stencil (fused init + first sweep, Jacobi sweep + max residual + decision, rho = div j_s; Eq. 26-35,
//      P:291-320, 383) on double2 fields with fp64 link variables, J_av, observables.  One thread per site, neighbours
//      through L1/L2 (three xy planes of the largest grids fit the 126 MB L2 many times): 64 B/site/sweep of HBM traffic.
//      Its mu solver is (1) in double.
// The neighbour operators are those of SURVEY 8(c): wrap, quasi-periodic jump, open faces with
// S- := S+ at the first site and S+ := S- at the last, both Landau gauges, films (no z links, S22).
#include "march_common.cuh"
#include "philox.cuh"

namespace {

template <class T> struct Vec2;
template <> struct Vec2<float> { typedef float2 type; };
template <> struct Vec2<double> { typedef double2 type; };

struct cd { double x, y; };
__device__ __forceinline__ cd mk(double x, double y) { cd r; r.x = x; r.y = y; return r; }
__device__ __forceinline__ cd cm(cd a, cd b) { return mk(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ cd cmc(cd a, cd b) { return mk(a.x * b.x + a.y * b.y, a.x * b.y - a.y * b.x); }   // conj(a) b
__device__ __forceinline__ cd ldc(const double2 *p) { const double2 v = *p; return mk(v.x, v.y); }
__device__ __forceinline__ cd ldt(const double2 *p) { const double2 v = __ldg(p); return mk(v.x, v.y); }

struct Site { int i, j, k, ie, iw, jn, js, kt, kb; bool xlo, xhi, ylo, yhi, zlo, zhi; };
__device__ __forceinline__ Site site_of(const Dev &dv, int i, int j, int k) {
  const int nx = dv.nx, ny = dv.ny, nz = dv.nz;
  const bool px = dv.bcx == 0, py = dv.bcy == 0, pz = dv.bcz == 0, film = nz == 1;
  Site s;
  s.i = i; s.j = j; s.k = k;
  s.xlo = !px && i == 0; s.xhi = !px && i == nx - 1;
  s.ylo = !py && j == 0; s.yhi = !py && j == ny - 1;
  s.zlo = !pz && k == 0; s.zhi = !pz && k == nz - 1;
  s.ie = (i + 1 < nx) ? i + 1 : (px ? 0 : nx - 2); s.iw = (i > 0) ? i - 1 : (px ? nx - 1 : 1);
  s.jn = (j + 1 < ny) ? j + 1 : (py ? 0 : ny - 2); s.js = (j > 0) ? j - 1 : (py ? ny - 1 : 1);
  s.kt = film ? 0 : ((k + 1 < nz) ? k + 1 : (pz ? 0 : nz - 2));
  s.kb = film ? 0 : ((k > 0) ? k - 1 : (pz ? nz - 1 : 1));
  return s;
}

// Insulating inclusions (S25): which of the six neighbour terms of a superconducting site exist.  A link to a removed
// site is cut; on an external open face the mirrored term exists iff the link it mirrors does.  bit 0/1: x +/-, 2/3: y, 4/5: z.
__device__ __forceinline__ unsigned link_bits(const Dev &dv, const Site &s) {
  if (!dv.sc) return 63u;
  const int nx = dv.nx, ny = dv.ny;
  const long long plane = (long long)nx * ny;
  const long long rowb = (long long)s.k * plane + (long long)s.j * nx;
  unsigned b = 0u;
  bool fw = dv.sc[rowb + s.ie] != 0, bw = dv.sc[rowb + s.iw] != 0;
  if (s.xlo) bw = fw;
  if (s.xhi) fw = bw;
  b |= (fw ? 1u : 0u) | (bw ? 2u : 0u);
  fw = dv.sc[(long long)s.k * plane + (long long)s.jn * nx + s.i] != 0; bw = dv.sc[(long long)s.k * plane + (long long)s.js * nx + s.i] != 0;
  if (s.ylo) bw = fw;
  if (s.yhi) fw = bw;
  b |= (fw ? 4u : 0u) | (bw ? 8u : 0u);
  if (dv.nz > 1) {
    fw = dv.sc[(long long)s.kt * plane + (long long)s.j * nx + s.i] != 0; bw = dv.sc[(long long)s.kb * plane + (long long)s.j * nx + s.i] != 0;
    if (s.zlo) bw = fw;
    if (s.zhi) fw = bw;
    b |= (fw ? 16u : 0u) | (bw ? 32u : 0u);
  }
  return b;
}
// sum over the existing links of site m of c_alpha: 2 (c_x + c_y + c_z) without inclusions (the "2 sum c" of M_mm)
__device__ __forceinline__ double link_diag(const Dev &dv, unsigned lb) {
  if (lb == 63u) return dv.csum2_64;
  return dv.cx64 * (double)__popc(lb & 3u) + dv.cy64 * (double)__popc(lb & 12u) + (dv.nz > 1 ? dv.cz64 * (double)__popc(lb & 48u) : 0.0);
}

// sum_alpha c_alpha (S+_alpha x + S-_alpha x)_m in fp64 (Eq. 29a / 29b without the -2 x term), fp64 link variables;
// `lb`: the terms that exist (link_bits)
__device__ __forceinline__ cd neighbour_sum(const Dev &dv, const double2 *__restrict__ x, const Site &s, unsigned lb = 63u) {
  const int nx = dv.nx, ny = dv.ny;
  const long long plane = (long long)nx * ny;
  const bool film = dv.nz == 1, yz = dv.gauge_yz != 0;
  const long long rowb = (long long)s.k * plane + (long long)s.j * nx;
  const cd Ux = ldt(dv.Ux64 + s.j);
  cd e = ldc(x + rowb + s.ie), w = ldc(x + rowb + s.iw);
  if (yz && dv.bcx == 0 && (s.i == nx - 1 || s.i == 0)) {          // jump in x: psi_{-1} = P_{j,k} psi_{nx-1}
    const cd P = cm(ldt(dv.Pj64 + s.j), ldt(dv.Pk64 + s.k));
    if (s.i == nx - 1) e = cmc(P, e);
    if (s.i == 0) w = cm(P, w);
  }
  cd sp = cm(Ux, e), sm = cmc(Ux, w);
  if (s.xlo) sm = sp;
  if (s.xhi) sp = sm;
  if (!(lb & 1u)) sp = mk(0.0, 0.0);
  if (!(lb & 2u)) sm = mk(0.0, 0.0);
  cd acc = mk(dv.cx64 * (sp.x + sm.x), dv.cx64 * (sp.y + sm.y));
  cd n = ldc(x + (long long)s.k * plane + (long long)s.jn * nx + s.i), so = ldc(x + (long long)s.k * plane + (long long)s.js * nx + s.i);
  if (!yz && dv.bcy == 0 && (s.j == ny - 1 || s.j == 0)) {         // jump in y: psi_{i,-1,k} = P_{i,k} psi_{i,ny-1,k}
    const cd P = cmc(ldt(dv.Pk64 + s.k), ldt(dv.Pi64 + s.i));
    if (s.j == ny - 1) n = cmc(P, n);
    if (s.j == 0) so = cm(P, so);
  }
  if (yz) { const cd Uy = ldt(dv.Uy64 + s.i); sp = cm(Uy, n); sm = cmc(Uy, so); }
  else { sp = n; sm = so; }
  if (s.ylo) sm = sp;
  if (s.yhi) sp = sm;
  if (!(lb & 4u)) sp = mk(0.0, 0.0);
  if (!(lb & 8u)) sm = mk(0.0, 0.0);
  acc.x += dv.cy64 * (sp.x + sm.x); acc.y += dv.cy64 * (sp.y + sm.y);
  if (!film) {
    const cd Uz = yz ? ldt(dv.Uzx64 + s.i) : ldt(dv.Uz64 + s.j);
    const cd t = ldc(x + (long long)s.kt * plane + (long long)s.j * nx + s.i), b = ldc(x + (long long)s.kb * plane + (long long)s.j * nx + s.i);
    sp = cm(Uz, t); sm = cmc(Uz, b);
    if (s.zlo) sm = sp;
    if (s.zhi) sp = sm;
    if (!(lb & 16u)) sp = mk(0.0, 0.0);
    if (!(lb & 32u)) sm = mk(0.0, 0.0);
    acc.x += dv.cz64 * (sp.x + sm.x); acc.y += dv.cz64 * (sp.y + sm.y);
  }
  return acc;
}

// Launch geometry of the one-thread-per-site kernels: 128 threads along x; a CTA walks a chunk of PLAIN_CH sites along
// the slowest axis that has an extent (z; y for a film), so that a 67 M-site grid launches 32 k CTAs, not 524 k: every
// CTA ends with two atomics on the same two words (max residual, ticket), which serialise in L2.
#define PLAIN_CH 16
struct Chunk { int i, j0, j1, k0, k1; };
__device__ __forceinline__ Chunk chunk_of(const Dev &dv) {
  Chunk c;
  c.i = blockIdx.x * 128 + threadIdx.x;
  if (dv.nz > 1) { c.j0 = blockIdx.y; c.j1 = c.j0 + 1; c.k0 = blockIdx.z * PLAIN_CH; c.k1 = min(dv.nz, c.k0 + PLAIN_CH); }
  else { c.j0 = blockIdx.y * PLAIN_CH; c.j1 = min(dv.ny, c.j0 + PLAIN_CH); c.k0 = 0; c.k1 = 1; }
  return c;
}

// CTA-wide max of a non-negative double -> thread 0 (blockDim.x <= 1024)
__device__ __forceinline__ double block_max(double v, double *sh) {
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_down_sync(0xffffffffu, v, o));
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
  __syncthreads();
  if (threadIdx.x == 0) {
    const int nw = (blockDim.x + 31) >> 5;
    for (int q = 1; q < nw; ++q) v = fmax(v, sh[q]);
  }
  return v;
}

// ------------------------------------------------------------------------------------------------------------------
// (2) double-precision marching stencil.  grid = (ceil(nx/128), ny, nz), 128 threads along x.
// ------------------------------------------------------------------------------------------------------------------
template <int MODE>
__global__ void __launch_bounds__(128) k_march64(const __grid_constant__ Dev dv) {
  Ctl *ctl = dv.ctl;
  int l = 0;
  if (MODE != MODE_RHO) {
    if (ctl->done) return;
    l = ctl->sweeps;
  }
  const int xb = ctl->xbuf;
  const double2 *__restrict__ xin = dv.psi64[xb];
  double2 *__restrict__ xout = dv.psi64[xb ^ 1];
  const Chunk ch = chunk_of(dv);
  const int i = ch.i;
  const bool act = i < dv.nx;
  double r2 = 0.0;
  if (act)
  for (int k = ch.k0; k < ch.k1; ++k)
  for (int j = ch.j0; j < ch.j1; ++j) {
    const Site s = site_of(dv, i, j, k);
    const long long m = (long long)i + (long long)dv.nx * (j + (long long)dv.ny * k);
    if (dv.sc && !dv.sc[m]) {                                             // a removed site (S25): psi = 0, rho = 0
      if (MODE == MODE_RHO) dv.mu64[m] = 0.0;
      else xout[m] = make_double2(0.0, 0.0);
      continue;
    }
    const unsigned lb = link_bits(dv, s);
    const cd c = ldc(xin + m);
    const cd ns = neighbour_sum(dv, xin, s, lb);
    if (MODE == MODE_RHO) {
      dv.mu64[m] = c.x * ns.y - c.y * ns.x;                                 // rho_m = Im[psi*_m sum (S+ + S-) psi]
    } else {
      const double ht2 = dv.ht2_64;
      cd b, d;
      if (MODE == MODE_INIT) {
        // d_m = 1 + (h_t/2)[|psi|^2 + 2 sum c - eps + i u mu];  b_m = psi (2 - d) + (h_t/2)(nsum + 2 zeta)  (Eq. 31)
        const double a = c.x * c.x + c.y * c.y;
        const double mu = dv.solve_mu ? dv.mu64[m] : 0.0;
        d = mk(1.0 + ht2 * (a + link_diag(dv, lb) - (double)dv.eps[m]), ht2 * dv.u64 * mu);
        cd z = mk(0.0, 0.0);
        if (dv.zeta_max64 > 0.0) {                                          // Langevin term, Eq. (39), S11
          const unsigned long long mm = (unsigned long long)m;
          uint32_t wr, wi;
          langevin_words(mm, (unsigned)ctl->n, dv.seed_lo, dv.seed_hi, wr, wi);
          z = mk(dv.zeta_max64 * (double)u32_to_pm1(wr), dv.zeta_max64 * (double)u32_to_pm1(wi));
        }
        const cd q = cm(c, mk(2.0 - d.x, -d.y));
        b = mk(q.x + ht2 * (ns.x + 2.0 * z.x), q.y + ht2 * (ns.y + 2.0 * z.y));
        dv.b64[m] = make_double2(b.x, b.y);
        dv.d64[m] = make_double2(d.x, d.y);
      } else {
        b = ldc(dv.b64 + m);
        d = ldc(dv.d64 + m);
      }
      // x^{l+1} = (b + (h_t/2) nsum) / d  (Eq. 33);  |r^l|^2 = |d|^2 |x^{l+1} - x^l|^2  (S8)
      const cd num = mk(b.x + ht2 * ns.x, b.y + ht2 * ns.y);
      const double m2 = d.x * d.x + d.y * d.y;
      const cd y = cmc(d, num);
      const cd out = mk(y.x / m2, y.y / m2);
      xout[m] = make_double2(out.x, out.y);
      const double ex = out.x - c.x, ey = out.y - c.y;
      r2 = fmax(r2, (ex * ex + ey * ey) * m2);
    }
  }
  if (MODE != MODE_RHO) {
    __shared__ double sh[4];
    const double bm = block_max(r2, sh);
    if (threadIdx.x == 0) {
      // the decision logic (Eq. 34, S8-S10) is the fp32 path's: the reduced residual is rounded to fp32 once
      atomicMax(&ctl->resid_bits[l], __float_as_uint((float)bm));
      __threadfence();
      const unsigned nb = gridDim.x * gridDim.y * gridDim.z;
      if (atomicAdd(&ctl->ticket, 1u) == nb - 1) {
        ctl->ticket = 0u;
        sweep_decide(dv, l);
      }
    }
  }
}

// J_av (Eq. 35): sum over ALL x links of Im[psi*_m U_x(j) psi_{m+x}] (x periodic), fp64, one partial per CTA -> dv.part
__global__ void __launch_bounds__(256) k_jav64(const __grid_constant__ Dev dv) {
  const double2 *__restrict__ x = dv.psi64[dv.ctl->xbuf];
  const int nx = dv.nx, ny = dv.ny;
  double acc = 0.0;
  for (long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x; m < dv.N; m += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(m % nx);
    const long long row = m / nx;
    const int j = (int)(row % ny), k = (int)(row / ny);
    const long long me = row * nx + (i + 1 == nx ? 0 : i + 1);
    if (dv.sc && !(dv.sc[m] && dv.sc[me])) continue;            // a cut link carries no current (S25)
    const cd a = ldc(x + m);
    cd b = ldc(x + me);
    if (dv.gauge_yz && i + 1 == nx) b = cmc(cm(ldt(dv.Pj64 + j), ldt(dv.Pk64 + k)), b);
    const cd ub = cm(ldt(dv.Ux64 + j), b);
    acc += a.x * ub.y - a.y * ub.x;
  }
  __shared__ double sh[8];
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x == 0) {
    double s = 0.0;
    for (int w = 0; w < 8; ++w) s += sh[w];
    dv.part[blockIdx.x] = s;
  }
}

// psi0 = 1 + amp (N(0,1) + i N(0,1)) (S13), mu = 0, eps = 1 -- the fp64 state
__global__ void k_init_state64(const __grid_constant__ Dev dv, double amp) {
  for (long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x; m < dv.N; m += (long long)gridDim.x * blockDim.x) {
    const PhiloxOut p = philox4x32_10((uint32_t)m, (uint32_t)((unsigned long long)m >> 32), 0u, 1u, dv.seed_lo, dv.seed_hi);
    const double u1 = u32_to_01(p.x0), u2 = u32_to_01(p.x1);
    const double rad = sqrt(-2.0 * log(u1));
    double s, c;
    sincospi(2.0 * u2, &s, &c);
    dv.psi64[0][m] = make_double2(1.0 + amp * rad * c, amp * rad * s);
    dv.mu64[m] = 0.0;
    dv.eps[m] = 1.f;
  }
}
__global__ void k_noise64(const __grid_constant__ Dev dv, long long step, double2 *out) {
  for (long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x; m < dv.N; m += (long long)gridDim.x * blockDim.x) {
    uint32_t wr, wi;
    langevin_words((unsigned long long)m, (uint32_t)step, dv.seed_lo, dv.seed_hi, wr, wi);
    out[m] = make_double2(dv.zeta_max64 * (double)u32_to_pm1(wr), dv.zeta_max64 * (double)u32_to_pm1(wi));
  }
}
__global__ void k_copy_psi64(const __grid_constant__ Dev dv, double2 *__restrict__ out) {
  const double2 *__restrict__ src = dv.psi64[dv.ctl->xbuf & 1];
  for (long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x; m < dv.N; m += (long long)gridDim.x * blockDim.x) out[m] = src[m];
}

// a8 in fp64: the sums of aux.cu (k_obs_partial) written site by site
//   [0] sum |psi|^2  [1] sum w (-eps |psi|^2 + |psi|^4/2)  [2] sum_alpha c_alpha sum_links w_link |S+ psi - psi|^2  [3] windings
__device__ __forceinline__ double face_w64(int idx, int n, int open) { return (open && (idx == 0 || idx == n - 1)) ? 0.5 : 1.0; }
__global__ void __launch_bounds__(256) k_obs64(const __grid_constant__ Dev dv) {
  const double2 *__restrict__ x = dv.psi64[dv.ctl->xbuf];
  const int nx = dv.nx, ny = dv.ny, nz = dv.nz;
  const bool yz = dv.gauge_yz != 0, film = nz == 1;
  const long long plane = (long long)nx * ny;
  const double flux = dv.ctl->Bz * dv.hx * dv.hy, twopi = 6.283185307179586476925286766559;
  double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
  for (long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x; m < dv.N; m += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(m % nx);
    const long long rest = m / nx;
    const int j = (int)(rest % ny), k = (int)(rest / ny);
    const int ip = (i + 1 == nx) ? 0 : i + 1, jp = (j + 1 == ny) ? 0 : j + 1, kp = (k + 1 == nz) ? 0 : k + 1;
    const bool hasx0 = dv.bcx == 0 || i + 1 < nx, hasy0 = dv.bcy == 0 || j + 1 < ny, hasz0 = !film && (dv.bcz == 0 || k + 1 < nz);
    const double wx = face_w64(i, nx, dv.bcx), wy = face_w64(j, ny, dv.bcy), wz = film ? 1.0 : face_w64(k, nz, dv.bcz);
    const cd Pk = ldt(dv.Pk64 + k);
    auto at = [&](int ii, int jj, int kk) { return ldc(x + (long long)kk * plane + (long long)jj * nx + ii); };
    auto xlink = [&](int ii, int jj) -> cd {                   // S+_x psi at (ii, jj, k)
      const int ie = (ii + 1 == nx) ? 0 : ii + 1;
      cd e = cm(ldt(dv.Ux64 + jj), at(ie, jj, k));
      if (yz && dv.bcx == 0 && ii + 1 == nx) e = cmc(cm(ldt(dv.Pj64 + jj), Pk), e);
      return e;
    };
    auto ylink = [&](int ii, int jj) -> cd {                   // S+_y psi at (ii, jj, k)
      const int jn = (jj + 1 == ny) ? 0 : jj + 1;
      const cd v = at(ii, jn, k);
      if (yz) return cm(ldt(dv.Uy64 + ii), v);
      if (dv.bcy == 0 && jj + 1 == ny) return cmc(cmc(Pk, ldt(dv.Pi64 + ii)), v);
      return v;
    };
    auto sc = [&](int ii, int jj, int kk) { return !dv.sc || dv.sc[(long long)kk * plane + (long long)jj * nx + ii] != 0; };
    if (!sc(i, j, k)) continue;                                  // removed sites and cut links carry nothing (S25)
    const bool hasx = hasx0 && sc(ip, j, k), hasy = hasy0 && sc(i, jp, k), hasz = hasz0 && sc(i, j, kp);
    const cd c = at(i, j, k);
    const double ab = c.x * c.x + c.y * c.y;
    const cd e = xlink(i, j), n = ylink(i, j);
    double g = 0.0;
    if (hasx) g += dv.cx64 * wy * wz * ((e.x - c.x) * (e.x - c.x) + (e.y - c.y) * (e.y - c.y));
    if (hasy) g += dv.cy64 * wx * wz * ((n.x - c.x) * (n.x - c.x) + (n.y - c.y) * (n.y - c.y));
    if (hasz) {
      const cd t = cm(yz ? ldt(dv.Uzx64 + i) : ldt(dv.Uz64 + j), at(i, j, kp));
      g += dv.cz64 * wx * wy * ((t.x - c.x) * (t.x - c.x) + (t.y - c.y) * (t.y - c.y));
    }
    a0 += ab;
    a1 += wx * wy * wz * (-(double)dv.eps[m] * ab + 0.5 * ab * ab);
    a2 += g;
    if (hasx && hasy && sc(ip, jp, k)) {                         // winding of the z-plaquette with corner (i, j)
      const cd cn = at(i, jp, k), ce = at(ip, j, k);
      const cd q0 = cmc(c, e), q1 = cmc(ce, ylink(ip, j)), q2 = cmc(cn, xlink(i, jp)), q3 = cmc(c, n);
      a3 += rint((atan2(q0.y, q0.x) + atan2(q1.y, q1.x) - atan2(q2.y, q2.x) - atan2(q3.y, q3.x) + flux) / twopi);
    }
  }
  __shared__ double sh[4][8];
  for (int o = 16; o > 0; o >>= 1) {
    a0 += __shfl_down_sync(0xffffffffu, a0, o); a1 += __shfl_down_sync(0xffffffffu, a1, o);
    a2 += __shfl_down_sync(0xffffffffu, a2, o); a3 += __shfl_down_sync(0xffffffffu, a3, o);
  }
  if ((threadIdx.x & 31) == 0) { sh[0][threadIdx.x >> 5] = a0; sh[1][threadIdx.x >> 5] = a1; sh[2][threadIdx.x >> 5] = a2; sh[3][threadIdx.x >> 5] = a3; }
  __syncthreads();
  if (threadIdx.x < 4) {
    double s = 0.0;
    for (int w = 0; w < 8; ++w) s += sh[threadIdx.x][w];
    dv.part[(size_t)threadIdx.x * TDGL_NPART + blockIdx.x] = s;
  }
}

// ------------------------------------------------------------------------------------------------------------------
// (1) the pseudo-time mu iteration.  Real 7-point operator, wrap or mirror ghost.  One thread per site.
// ------------------------------------------------------------------------------------------------------------------
template <class T> struct MuArrays { T *mu, *rho, *c, *xa, *xb; };

template <class T>
__device__ __forceinline__ double real_nsum(const Dev &dv, const T *__restrict__ x, const Site &s, double &centre, unsigned lb = 63u) {
  const int nx = dv.nx, ny = dv.ny;
  const long long plane = (long long)nx * ny;
  const long long rowb = (long long)s.k * plane + (long long)s.j * nx;
  centre = (double)x[rowb + s.i];
  // mirror ghost on external open faces (the clamped neighbour index IS the mirrored site); cut links contribute nothing
  double acc = dv.cx64 * (((lb & 1u) ? (double)x[rowb + s.ie] : 0.0) + ((lb & 2u) ? (double)x[rowb + s.iw] : 0.0)) +
               dv.cy64 * (((lb & 4u) ? (double)x[(long long)s.k * plane + (long long)s.jn * nx + s.i] : 0.0) +
                          ((lb & 8u) ? (double)x[(long long)s.k * plane + (long long)s.js * nx + s.i] : 0.0));
  if (dv.nz > 1)
    acc += dv.cz64 * (((lb & 16u) ? (double)x[(long long)s.kt * plane + (long long)s.j * nx + s.i] : 0.0) +
                      ((lb & 32u) ? (double)x[(long long)s.kb * plane + (long long)s.j * nx + s.i] : 0.0));
  return acc;
}

// c = mu^- + h_tau [ (Delta_h mu^-)/2 - rho ]   (P:409-419 with the stable sign, S5); resets the inner-loop state
template <class T>
__global__ void __launch_bounds__(128) k_mu_rhs(const __grid_constant__ Dev dv, MuArrays<T> A) {
  Ctl *ctl = dv.ctl;
  if (ctl->mu_done) return;
  const Chunk ch = chunk_of(dv);
  const int i = ch.i;
  if (i < dv.nx)
  for (int k = ch.k0; k < ch.k1; ++k)
  for (int j = ch.j0; j < ch.j1; ++j) {
    const Site s = site_of(dv, i, j, k);
    const long long m = (long long)i + (long long)dv.nx * (j + (long long)dv.ny * k);
    if (dv.sc && !dv.sc[m]) { A.c[m] = (T)0; continue; }
    const unsigned lb = link_bits(dv, s);
    double ctr;
    const double ns = real_nsum(dv, A.mu, s, ctr, lb);
    const double lap = ns - link_diag(dv, lb) * ctr;
    A.c[m] = (T)(ctr + (double)ctl->h_tau * (0.5 * lap - (double)A.rho[m]));
  }
  if (blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0 && threadIdx.x == 0) {
    ctl->mu_inner = 0; ctl->mu_inner_done = 0; ctl->mu_ticket = 0u; ctl->mu_r2bits = 0ull;
  }
}

// one Jacobi sweep of N mu = c ("a formulation like that in Eq. (33)"); x^0 = mu^-
template <class T>
__global__ void __launch_bounds__(128) k_mu_sweep(const __grid_constant__ Dev dv, MuArrays<T> A) {
  Ctl *ctl = dv.ctl;
  if (ctl->mu_done || ctl->mu_inner_done) return;
  const int l = ctl->mu_inner;
  const T *__restrict__ xin = (l == 0) ? A.mu : ((l & 1) ? A.xa : A.xb);
  T *__restrict__ xout = (l & 1) ? A.xb : A.xa;
  const Chunk ch = chunk_of(dv);
  const int i = ch.i;
  double r2 = 0.0;
  if (i < dv.nx)
  for (int k = ch.k0; k < ch.k1; ++k)
  for (int j = ch.j0; j < ch.j1; ++j) {
    const Site s = site_of(dv, i, j, k);
    const long long m = (long long)i + (long long)dv.nx * (j + (long long)dv.ny * k);
    if (dv.sc && !dv.sc[m]) { xout[m] = (T)0; continue; }
    const unsigned lb = link_bits(dv, s);
    double ctr;
    const double ns = real_nsum(dv, xin, s, ctr, lb);
    const double ht = (double)ctl->h_tau, d = 1.0 + 0.5 * ht * link_diag(dv, lb);
    const T xn = (T)(((double)A.c[m] + 0.5 * ht * ns) / d);
    xout[m] = xn;
    const double r = d * ((double)xn - ctr);
    r2 = fmax(r2, r * r);
  }
  __shared__ double sh[4];
  const double bm = block_max(r2, sh);
  if (threadIdx.x == 0) {
    atomicMax(&ctl->mu_r2bits, (unsigned long long)__double_as_longlong(bm));
    __threadfence();
    const unsigned nb = gridDim.x * gridDim.y * gridDim.z;
    if (atomicAdd(&ctl->mu_ticket, 1u) == nb - 1) {               // last CTA: the inner decision (rule S8 applied to Eq. 40)
      ctl->mu_ticket = 0u;
      const double r2max = __longlong_as_double((long long)atomicExch(&ctl->mu_r2bits, 0ull));
      const int sweeps = l + 1;
      ctl->mu_inner = sweeps;
      bool done;
      if (ctl->mu_sched_pos < ctl->mu_sched_n) done = sweeps >= dv.mu_sched[ctl->mu_sched_pos];
      else {
        done = r2max < (double)ctl->eps_mu_in || sweeps >= ctl->mu_max_inner;
        if (!(r2max < (double)ctl->eps_mu_in) && sweeps >= ctl->mu_max_inner) ctl->status |= 2;   // TDGL_WMUCAP: the cap, not the test, ended it
      }
      if (done) ctl->mu_inner_done = 1;
      __threadfence();
    }
  }
}

// end of an outer iteration: mu <- x, max |(x - mu^-)/h_tau|^2, outer decision, log
template <class T>
__global__ void __launch_bounds__(128) k_mu_finish(const __grid_constant__ Dev dv, MuArrays<T> A) {
  Ctl *ctl = dv.ctl;
  if (ctl->mu_done) return;
  const int l = ctl->mu_inner;                                    // >= 1 sweeps were done: the last wrote xa (l odd) / xb (l even)
  const T *__restrict__ x = (l & 1) ? A.xa : A.xb;
  const Chunk ch = chunk_of(dv);
  const int i = ch.i;
  double d2 = 0.0;
  if (i < dv.nx)
  for (int k = ch.k0; k < ch.k1; ++k)
  for (int j = ch.j0; j < ch.j1; ++j) {
    const long long m = (long long)i + (long long)dv.nx * (j + (long long)dv.ny * k);
    const T xn = x[m];
    const double dt = ((double)xn - (double)A.mu[m]) / (double)ctl->h_tau;
    A.mu[m] = xn;
    d2 = fmax(d2, dt * dt);
  }
  __shared__ double sh[4];
  const double bm = block_max(d2, sh);
  if (threadIdx.x == 0) {
    atomicMax(&ctl->mu_r2bits, (unsigned long long)__double_as_longlong(bm));
    __threadfence();
    const unsigned nb = gridDim.x * gridDim.y * gridDim.z;
    if (atomicAdd(&ctl->mu_ticket, 1u) == nb - 1) {
      ctl->mu_ticket = 0u;
      const double dt2 = __longlong_as_double((long long)atomicExch(&ctl->mu_r2bits, 0ull));
      dv.mu_log[ctl->mu_log_pos % TDGL_MULOGCAP] = l;             // inner sweeps of this outer iteration
      ctl->mu_log_pos += 1;
      ctl->mu_outer += 1;
      ctl->mu_inner_total += l;
      ctl->mu_dt2_last = dt2;
      bool done;
      if (ctl->mu_sched_pos < ctl->mu_sched_n) { ctl->mu_sched_pos += 1; done = ctl->mu_sched_pos >= ctl->mu_sched_n; }
      else {
        done = dt2 < (double)ctl->eps_mu || ctl->mu_outer >= ctl->mu_max_outer;
        if (!(dt2 < (double)ctl->eps_mu) && ctl->mu_outer >= ctl->mu_max_outer) ctl->status |= 2;   // TDGL_WMUCAP
      }
      if (done) ctl->mu_done = 1;
      __threadfence();
    }
  }
}

// start of a solve: clear the outer-loop state (one thread)
__global__ void k_mu_begin(const __grid_constant__ Dev dv) {
  Ctl *c = dv.ctl;
  c->mu_done = 0; c->mu_outer = 0; c->mu_inner = 0; c->mu_inner_done = 0; c->mu_ticket = 0u; c->mu_r2bits = 0ull;
}
// end of a solve: per-step log (outer iterations of this solve)
__global__ void k_mu_end(const __grid_constant__ Dev dv) {
  Ctl *c = dv.ctl;
  dv.mu_outer_log[c->mu_solves % TDGL_LOGCAP] = c->mu_outer;
  c->mu_solves += 1;
  c->mu_outer_total += c->mu_outer;
}
__global__ void k_mu_controls(const __grid_constant__ Dev dv, float h_tau, float eps_mu, float eps_in, int max_outer, int max_inner) {
  Ctl *c = dv.ctl;
  c->h_tau = h_tau; c->eps_mu = eps_mu; c->eps_mu_in = eps_in; c->mu_max_outer = max_outer; c->mu_max_inner = max_inner;
}
__global__ void k_mu_sched(const __grid_constant__ Dev dv, int n) { dv.ctl->mu_sched_n = n; dv.ctl->mu_sched_pos = 0; }

// ------------------------------------------------------------------------------------------------------------------
// (1b) direct mu solver of the double-precision build (TDGL_FLAG_MU_DIRECT).  Delta_h mu = rho (the
// fixed point of the paper's iteration) by mixed-precision iterative refinement: the fp32 transform solver S (poisson.cu)
// is an approximate inverse with relative error ~1e-6 G (G = white-noise gain, refine.cu), so
//     mu_0 = 0, r_0 = rho;   mu_{n+1} = mu_n + S(float(r_n)),   r_{n+1} = rho - Delta_h mu_{n+1}  (fp64)
// gains six to seven digits per pass and reaches the fp64 rounding floor of the residual in 3-4 passes.
// ------------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_dref_begin(const __grid_constant__ Dev dv) {
  const double *__restrict__ rho = (const double *)dv.mu_rho;
  double mx = 0.0;
  for (long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x; m < dv.N; m += (long long)gridDim.x * blockDim.x) {
    const double r = rho[m];
    dv.resid[m] = (float)r;
    dv.mu64[m] = 0.0;
    mx = fmax(mx, fabs(r));
  }
  __shared__ double sh[8];
  const double bm = block_max(mx, sh);
  if (threadIdx.x == 0) atomicMax(&dv.ctl->dref_rho_bits, (unsigned long long)__double_as_longlong(bm));
}
// mu += S(r) (the solver worked in place on resid), then nothing else: the residual needs the updated neighbours
__global__ void __launch_bounds__(256) k_dref_add(const __grid_constant__ Dev dv) {
  for (long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x; m < dv.N; m += (long long)gridDim.x * blockDim.x)
    dv.mu64[m] += (double)dv.resid[m];
}
// r = rho - Delta_h mu in fp64 (wrap / mirror ghost, S6), stored in fp32 for the next pass; max |r|
__global__ void __launch_bounds__(128) k_dref_resid(const __grid_constant__ Dev dv) {
  const double *__restrict__ rho = (const double *)dv.mu_rho;
  const Chunk ch = chunk_of(dv);
  const int i = ch.i;
  double mx = 0.0;
  if (i < dv.nx)
  for (int k = ch.k0; k < ch.k1; ++k)
  for (int j = ch.j0; j < ch.j1; ++j) {
    const Site s = site_of(dv, i, j, k);
    const long long m = (long long)i + (long long)dv.nx * (j + (long long)dv.ny * k);
    double ctr;
    const double ns = real_nsum(dv, dv.mu64, s, ctr, 63u);
    const double r = rho[m] - (ns - link_diag(dv, 63u) * ctr);
    dv.resid[m] = (float)r;
    mx = fmax(mx, fabs(r));
  }
  __shared__ double sh[4];
  const double bm = block_max(mx, sh);
  if (threadIdx.x == 0) atomicMax(&dv.ctl->dref_r_bits, (unsigned long long)__double_as_longlong(bm));
}
// S7: the solution is fixed by sum_m w_m mu_m = 0 (w = 1/2 per open face).  Every fp32 solve removes its own weighted mean
// only to fp32 accuracy and Delta_h cannot see a constant, so the accumulated mu carries an offset of ~1e-9: removed
// here in fp64.  Partial sums per CTA in a fixed grid, summed in a fixed order by every CTA of the second kernel.
#define DREF_NB 1024
__global__ void __launch_bounds__(256) k_dref_wsum(const __grid_constant__ Dev dv) {
  const int nx = dv.nx, ny = dv.ny, nz = dv.nz;
  double acc = 0.0;
  for (long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x; m < dv.N; m += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(m % nx);
    const long long rest = m / nx;
    const int j = (int)(rest % ny), k = (int)(rest / ny);
    double w = 1.0;
    if (dv.bcx && (i == 0 || i == nx - 1)) w *= 0.5;
    if (dv.bcy && (j == 0 || j == ny - 1)) w *= 0.5;
    if (nz > 1 && dv.bcz && (k == 0 || k == nz - 1)) w *= 0.5;
    acc += w * dv.mu64[m];
  }
  __shared__ double sh[8];
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int q = 0; q < 8; ++q) t += sh[q];
    dv.part[blockIdx.x] = t;
  }
}
__global__ void __launch_bounds__(256) k_dref_shift(const __grid_constant__ Dev dv) {
  __shared__ double mean;
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int q = 0; q < DREF_NB; ++q) t += dv.part[q];
    const double wsum = (double)(dv.nx - (dv.bcx ? 1 : 0)) * (double)(dv.ny - (dv.bcy ? 1 : 0)) *
                        (double)(dv.nz > 1 ? dv.nz - (dv.bcz ? 1 : 0) : 1);
    mean = t / wsum;
  }
  __syncthreads();
  const double mu0 = mean;
  for (long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x; m < dv.N; m += (long long)gridDim.x * blockDim.x)
    dv.mu64[m] -= mu0;
}
__global__ void k_dref_ctl(const __grid_constant__ Dev dv, int what) {
  Ctl *c = dv.ctl;
  if (what == 0) { c->dref_rho_bits = 0ull; c->dref_r_bits = 0ull; }           // start of a solve
  else if (what == 1) c->dref_r_bits = 0ull;                                    // before a residual pass
  else { c->dref_solves += 1; c->dref_resid_last = __longlong_as_double((long long)c->dref_r_bits); }   // end of a solve
}

// zero psi and mu on the removed sites (after tdgl_set_insulators / tdgl_set_state)
__global__ void k_apply_mask64(const __grid_constant__ Dev dv) {
  double2 *x = dv.psi64[dv.ctl->xbuf & 1];
  for (long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x; m < dv.N; m += (long long)gridDim.x * blockDim.x)
    if (!dv.sc[m]) { x[m] = make_double2(0.0, 0.0); dv.mu64[m] = 0.0; }
}
__global__ void k_fill_u8(unsigned char *p, long long n, unsigned char v) {
  for (long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x; m < n; m += (long long)gridDim.x * blockDim.x) p[m] = v;
}

template <class T> __global__ void k_fill_t(T *p, long long n, T v) {
  for (long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x; m < n; m += (long long)gridDim.x * blockDim.x) p[m] = v;
}

unsigned grid1(long long n, int block, int cap) {
  long long g = (n + block - 1) / block;
  return (unsigned)(g < 1 ? 1 : (g > cap ? cap : g));
}
dim3 grid3(const Dev &dv) {
  if (dv.nz > 1) return dim3((dv.nx + 127) / 128, dv.ny, (dv.nz + PLAIN_CH - 1) / PLAIN_CH);
  return dim3((dv.nx + 127) / 128, (dv.ny + PLAIN_CH - 1) / PLAIN_CH, 1);
}

template <class T> MuArrays<T> mu_arrays(const Dev &dv, void *mu) {
  MuArrays<T> A;
  A.mu = (T *)mu; A.rho = (T *)dv.mu_rho; A.c = (T *)dv.mu_c; A.xa = (T *)dv.mu_xa; A.xb = (T *)dv.mu_xb;
  return A;
}

}  // namespace

// ---- host-side launchers --------------------------------------------------------------------------------------------
void launch_march64(int mode, const Dev &dv, cudaStream_t st) {
  if (mode == MODE_SWEEP) k_march64<MODE_SWEEP><<<grid3(dv), 128, 0, st>>>(dv);
  else if (mode == MODE_INIT) k_march64<MODE_INIT><<<grid3(dv), 128, 0, st>>>(dv);
  else k_march64<MODE_RHO><<<grid3(dv), 128, 0, st>>>(dv);
}
int launch_jav64(const Dev &dv, cudaStream_t st) {                 // returns the number of partial sums written to dv.part
  const unsigned g = grid1(dv.N, 256, TDGL_NPART);
  k_jav64<<<g, 256, 0, st>>>(dv);
  return (int)g;
}
void launch_init_state64(const Dev &dv, double amp, cudaStream_t st) { k_init_state64<<<grid1(dv.N, 256, tdgl_sm_count() * 16), 256, 0, st>>>(dv, amp); }
void launch_noise64(const Dev &dv, long long step, double2 *out, cudaStream_t st) { k_noise64<<<grid1(dv.N, 256, tdgl_sm_count() * 16), 256, 0, st>>>(dv, step, out); }
void launch_copy_psi64(const Dev &dv, double2 *out, cudaStream_t st) { k_copy_psi64<<<grid1(dv.N, 256, tdgl_sm_count() * 16), 256, 0, st>>>(dv, out); }
int launch_obs64(const Dev &dv, cudaStream_t st) {                 // followed by k_obs_final (aux.cu): returns the partial count
  const unsigned g = grid1(dv.N, 256, TDGL_NPART);
  k_obs64<<<g, 256, 0, st>>>(dv);
  return (int)g;
}
void launch_apply_mask64(const Dev &dv, cudaStream_t st) { k_apply_mask64<<<grid1(dv.N, 256, tdgl_sm_count() * 16), 256, 0, st>>>(dv); }
void launch_fill_u8(unsigned char *p, long long n, unsigned char v, cudaStream_t st) { k_fill_u8<<<grid1(n, 256, tdgl_sm_count() * 16), 256, 0, st>>>(p, n, v); }
void launch_fill64(double *p, long long n, double v, cudaStream_t st) { k_fill_t<double><<<grid1(n, 256, tdgl_sm_count() * 16), 256, 0, st>>>(p, n, v); }

// the pieces of one pseudo-time solve; `mu` = the array that holds mu^- and receives mu (T = double iff dv.fp64)
void launch_mu_begin(const Dev &dv, cudaStream_t st) { k_mu_begin<<<1, 1, 0, st>>>(dv); }
void launch_mu_end(const Dev &dv, cudaStream_t st) { k_mu_end<<<1, 1, 0, st>>>(dv); }
void launch_mu_rhs(const Dev &dv, void *mu, cudaStream_t st) {
  if (dv.fp64) k_mu_rhs<double><<<grid3(dv), 128, 0, st>>>(dv, mu_arrays<double>(dv, mu));
  else k_mu_rhs<float><<<grid3(dv), 128, 0, st>>>(dv, mu_arrays<float>(dv, mu));
}
void launch_mu_sweep(const Dev &dv, void *mu, cudaStream_t st) {
  if (dv.fp64) k_mu_sweep<double><<<grid3(dv), 128, 0, st>>>(dv, mu_arrays<double>(dv, mu));
  else k_mu_sweep<float><<<grid3(dv), 128, 0, st>>>(dv, mu_arrays<float>(dv, mu));
}
void launch_mu_finish(const Dev &dv, void *mu, cudaStream_t st) {
  if (dv.fp64) k_mu_finish<double><<<grid3(dv), 128, 0, st>>>(dv, mu_arrays<double>(dv, mu));
  else k_mu_finish<float><<<grid3(dv), 128, 0, st>>>(dv, mu_arrays<float>(dv, mu));
}
void launch_mu_controls(const Dev &dv, float h_tau, float eps_mu, float eps_in, int max_outer, int max_inner, cudaStream_t st) {
  k_mu_controls<<<1, 1, 0, st>>>(dv, h_tau, eps_mu, eps_in, max_outer, max_inner);
}
void launch_mu_sched(const Dev &dv, int n, cudaStream_t st) { k_mu_sched<<<1, 1, 0, st>>>(dv, n); }

void launch_dref_ctl(const Dev &dv, int what, cudaStream_t st) { k_dref_ctl<<<1, 1, 0, st>>>(dv, what); }
void launch_dref_begin(const Dev &dv, cudaStream_t st) { k_dref_begin<<<tdgl_sm_count() * 8, 256, 0, st>>>(dv); }
void launch_dref_add(const Dev &dv, cudaStream_t st) { k_dref_add<<<tdgl_sm_count() * 8, 256, 0, st>>>(dv); }
void launch_dref_resid(const Dev &dv, cudaStream_t st) { k_dref_resid<<<grid3(dv), 128, 0, st>>>(dv); }
void launch_dref_zero_mean(const Dev &dv, cudaStream_t st) {
  k_dref_wsum<<<DREF_NB, 256, 0, st>>>(dv);
  k_dref_shift<<<tdgl_sm_count() * 8, 256, 0, st>>>(dv);
}
