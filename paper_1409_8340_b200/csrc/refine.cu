// a7, accuracy: one step of iterative refinement of the scalar-potential solve (Eq. 18 as discretised at P:379-383).
//
// The direct solver (poisson.cu) works in fp32: every transform pass rounds its coefficients to 6e-8 relative, and
// rho = div j_s itself is a sum of 24 fp32 products.  These roundings are white (they have no reason to be a
// discrete divergence), so the solve amplifies them by the white-noise gain of Delta_h^{-1},
//     G = ( (1/N) sum_{q != 0} 1/lambda_q^2 )^{1/2}:
// measured on B200, |delta mu| ~ 2e-7 G rms(rho).  G is below 2 for the 3D BASELINE grids (C4: 0.7, C5a: 2.0) but
// grows like L^{3/2} on quasi-one-dimensional meshes and like L on films (1026 x 3 film with open x: 499), where the
// error then exceeds the 2e-5 kernel gate for rough states.  The cure is textbook iterative
// refinement with the residual evaluated in HIGHER precision:
//     mu_1 = S(rho)                                  (fp32 solver)
//     r    = rho_64 - Delta_h mu_1                   (this file: fp64 arithmetic on the fp32 psi, mu_1; fp64 link
//                                                     variables; rho_64 = div j_s re-evaluated from psi)
//     mu   = mu_1 + S(r)                             (r is O(1e-6 |rho|): its own rounding no longer matters)
// after which the error is second order in the solver's error plus the fp32 rounding of mu itself.
#include "tdgl_dev.cuh"

namespace {

struct c64 { double x, y; };
__device__ __forceinline__ c64 mk(double x, double y) { c64 r; r.x = x; r.y = y; return r; }
__device__ __forceinline__ c64 cm(c64 a, c64 b) { return mk(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ c64 cmc(c64 a, c64 b) { return mk(a.x * b.x + a.y * b.y, a.x * b.y - a.y * b.x); }   // conj(a) b
__device__ __forceinline__ c64 ld(const float2 *p) { const float2 v = __ldg(p); return mk((double)v.x, (double)v.y); }
__device__ __forceinline__ c64 ldd(const double2 *p) { const double2 v = __ldg(p); return mk(v.x, v.y); }

// r_m = rho_m - (Delta_h mu)_m in fp64.  FROM_PSI: rho_m = sum_alpha c_alpha Im[psi*_m (S+ psi + S- psi)_m] with
// the neighbour operators of SURVEY 8(c) (wrap / quasi-periodic jump / open-face rule S- := S+), link variables
// from the fp64 tables; otherwise rho is read from `rho` (kernel-level test entry tdgl_debug_poisson).
template <bool FROM_PSI>
// `rho` and `out` MAY be the same array (tdgl_debug_poisson keeps rho in the residual buffer and overwrites it in place:
// each thread reads rho[m] before it writes out[m], and no other thread touches element m), so neither is __restrict__
// and rho is read with a plain load, not through the read-only path.
__global__ void __launch_bounds__(256) k_mu_residual(const __grid_constant__ Dev dv, const float *rho,
                                                     const float *__restrict__ mu, float *out) {
  const int nx = dv.nx, ny = dv.ny, nz = dv.nz;
  const bool px = dv.bcx == 0, py = dv.bcy == 0, pz = dv.bcz == 0, film = nz == 1, yz = dv.gauge_yz != 0;
  const long long plane = (long long)nx * ny;
  const double cx = (double)dv.cx, cy = (double)dv.cy, cz = (double)dv.cz;
  const float2 *__restrict__ x = FROM_PSI ? dv.psi[dv.ctl->xbuf & 1] : nullptr;
  for (long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x; m < dv.N; m += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(m % nx);
    const long long rest = m / nx;
    const int j = (int)(rest % ny), k = (int)(rest / ny);
    // neighbour indices: wrap or mirror; lo/hi = the site sits on the first/last layer of an open axis
    const bool xlo = !px && i == 0, xhi = !px && i == nx - 1;
    const bool ylo = !py && j == 0, yhi = !py && j == ny - 1;
    const bool zlo = !pz && k == 0, zhi = !pz && k == nz - 1;
    const int ie = (i + 1 < nx) ? i + 1 : (px ? 0 : nx - 2), iw = (i > 0) ? i - 1 : (px ? nx - 1 : 1);
    const int jn = (j + 1 < ny) ? j + 1 : (py ? 0 : ny - 2), js = (j > 0) ? j - 1 : (py ? ny - 1 : 1);
    const int kt = film ? 0 : ((k + 1 < nz) ? k + 1 : (pz ? 0 : nz - 2)), kb = film ? 0 : ((k > 0) ? k - 1 : (pz ? nz - 1 : 1));
    const long long rowb = (long long)k * plane + (long long)j * nx;
    double r;
    if (FROM_PSI) {
      const c64 c = ld(x + m);
      // link variables of the three forward links of this site (Eq. 27; gauge 24a or 24b)
      const c64 Ux = ldd(dv.Ux64 + j);
      const c64 Uy = yz ? ldd(dv.Uy64 + i) : mk(1.0, 0.0);
      const c64 Uz = film ? mk(1.0, 0.0) : (yz ? ldd(dv.Uzx64 + i) : ldd(dv.Uz64 + j));
      // x
      c64 e = ld(x + rowb + ie), w = ld(x + rowb + iw);
      if (yz && px && (i == nx - 1 || i == 0)) {           // quasi-periodic jump in x: psi_{-1} = P_{j,k} psi_{nx-1}
        const c64 P = cm(ldd(dv.Pj64 + j), ldd(dv.Pk64 + k));
        if (i == nx - 1) e = cmc(P, e);
        if (i == 0) w = cm(P, w);
      }
      c64 sp = cm(Ux, e), sm = cmc(Ux, w);
      if (xlo) sm = sp;                                     // open faces: S- := S+ at the first site, S+ := S- at the last
      if (xhi) sp = sm;
      c64 s = mk(cx * (sp.x + sm.x), cx * (sp.y + sm.y));
      // y
      c64 n = ld(x + (long long)k * plane + (long long)jn * nx + i), so = ld(x + (long long)k * plane + (long long)js * nx + i);
      if (!yz && py && (j == ny - 1 || j == 0)) {           // quasi-periodic jump in y: psi_{i,-1,k} = P_{i,k} psi_{i,ny-1,k}
        const c64 P = cmc(ldd(dv.Pk64 + k), ldd(dv.Pi64 + i));
        if (j == ny - 1) n = cmc(P, n);
        if (j == 0) so = cm(P, so);
      }
      sp = cm(Uy, n); sm = cmc(Uy, so);
      if (ylo) sm = sp;
      if (yhi) sp = sm;
      s.x += cy * (sp.x + sm.x); s.y += cy * (sp.y + sm.y);
      // z
      if (!film) {
        const c64 t = ld(x + (long long)kt * plane + (long long)j * nx + i), b = ld(x + (long long)kb * plane + (long long)j * nx + i);
        sp = cm(Uz, t); sm = cmc(Uz, b);
        if (zlo) sm = sp;
        if (zhi) sp = sm;
        s.x += cz * (sp.x + sm.x); s.y += cz * (sp.y + sm.y);
      }
      r = c.x * s.y - c.y * s.x;                            // Im[psi* s]
    } else {
      r = (double)rho[m];
    }
    // (Delta_h mu)_m with wrap / mirror ghost
    const double m0 = (double)__ldg(mu + m);
    double lap = cx * ((double)__ldg(mu + rowb + ie) + (double)__ldg(mu + rowb + iw) - 2.0 * m0) +
                 cy * ((double)__ldg(mu + (long long)k * plane + (long long)jn * nx + i) +
                       (double)__ldg(mu + (long long)k * plane + (long long)js * nx + i) - 2.0 * m0);
    if (!film)
      lap += cz * ((double)__ldg(mu + (long long)kt * plane + (long long)j * nx + i) +
                   (double)__ldg(mu + (long long)kb * plane + (long long)j * nx + i) - 2.0 * m0);
    out[m] = (float)(r - lap);
  }
}

// mu += delta, 16 bytes per access (N is even)
__global__ void __launch_bounds__(256) k_mu_add(float *__restrict__ mu, const float *__restrict__ delta, long long n4, long long n) {
  for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < n4; q += (long long)gridDim.x * blockDim.x) {
    float4 a = reinterpret_cast<float4 *>(mu)[q];
    const float4 b = __ldcs(reinterpret_cast<const float4 *>(delta) + q);
    a.x += b.x; a.y += b.y; a.z += b.z; a.w += b.w;
    reinterpret_cast<float4 *>(mu)[q] = a;
  }
  if (blockIdx.x == 0 && threadIdx.x == 0)
    for (long long m = 4 * n4; m < n; ++m) mu[m] += delta[m];
}

unsigned grid_for(long long n, int block, int cap) {
  long long g = (n + block - 1) / block;
  return (unsigned)(g < 1 ? 1 : (g > cap ? cap : g));
}

}  // namespace

// r = rho_64(psi, K) - Delta_h mu  ->  out      (rho == nullptr: rho from psi)
void launch_mu_residual(const Dev &dv, const float *rho, const float *mu, float *out, cudaStream_t st) {
  const unsigned g = grid_for(dv.N, 256, tdgl_sm_count() * 32);
  if (rho) k_mu_residual<false><<<g, 256, 0, st>>>(dv, rho, mu, out);
  else k_mu_residual<true><<<g, 256, 0, st>>>(dv, nullptr, mu, out);
}
void launch_mu_add(const Dev &dv, float *mu, const float *delta, cudaStream_t st) {
  k_mu_add<<<grid_for(dv.N / 4, 256, tdgl_sm_count() * 16), 256, 0, st>>>(mu, delta, dv.N / 4, dv.N);
}
