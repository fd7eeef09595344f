// The z-marching 7-point link-variable stencil: Jacobi sweep (a4), fused init + first sweep (a3),
// rho = div j_s (a6); plus the J_av reduction (a5) and the small per-step control kernels.
//
// One CTA owns an (2*bx) x by tile of the xy plane and marches through a chunk of z planes.  The psi
// planes k-1, k, k+1 live in a shared-memory ring filled by cp.async (16-byte vectors, ghost rows and
// columns included, wrapped or mirrored at the faces), two planes ahead of the arithmetic; every psi
// value is therefore read from HBM once per sweep (plus the tile halo), b and d once, and the new
// iterate is written once: 32 B/site/sweep.  x neighbours come from warp shuffles, y neighbours and
// z neighbours from shared memory.  Link variables U_x(j), U_z(j) are per-row constants read from a
// small table that a one-block kernel rewrites each step from K (fp64 sincos); the quasi-periodic jump
// P_{i,k} is applied only on rows j = 0 and j = ny-1.
#include "tdgl_dev.cuh"
#include "philox.cuh"
#include <cuda_device_runtime_api.h>

#define MODE_SWEEP 0
#define MODE_INIT  1
#define MODE_RHO   2

#define NBUF 5              // ring slots: planes k-1 .. k+2 resident, plane k+3 in flight

__device__ __forceinline__ void cp_async16(unsigned saddr, const void *g) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(saddr), "l"(g) : "memory");
}
__device__ __forceinline__ void cp_async8(unsigned saddr, const void *g) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(saddr), "l"(g) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory");
}

// The decision taken by the last CTA of a sweep (Eq. 34; S8: residual of the input iterate,
// keep the new one; S9/S10: prescribed counts, cap).
__device__ __noinline__ void sweep_decide(const Dev &dv, int l) {
  Ctl *c = dv.ctl;
  const float r2 = __uint_as_float(atomicMax(&c->resid_bits[l], 0u));
  const int sweeps = l + 1;
  c->sweeps = sweeps;
  c->xbuf ^= 1;
  int target = c->fixed_sweeps;
  if (c->sched_pos < c->sched_n) target = dv.sched[c->sched_pos];
  bool done;
  if (target > 0) {
    done = sweeps >= target;
  } else {
    done = (r2 < c->eps_tol) || sweeps >= c->max_sweeps;
    if (!(r2 < c->eps_tol) && sweeps >= c->max_sweeps) c->status = 1;
  }
  if (done) {
    c->done = 1;
    c->sweeps_last = sweeps;
    c->resid_last = r2;
  }
  if (dv.use_cond) cudaGraphSetConditional((cudaGraphConditionalHandle)dv.cond_handle, done ? 0u : 1u);
  __threadfence();
}

// BX thread columns (two sites each) x BY rows per CTA; tile = 2*BX x BY sites.
//
// Arithmetic per site (all modes): with W' = W, E' = E the x neighbours, S, N the y neighbours (jump
// phase applied on the wrap rows), B, T the z neighbours,
//   f . nsum = f cx [U_x E + U_x* W] + f cy [N + S] + f cz [U_z T + U_z* B]
//            = (f cx U_x).re (E + W) + i (f cx U_x).im (E - W) + f cy (N + S) + (f cz U_z).re (T + B) + i (...).im (T - B)
// with f = h_t/2 (sweep, init) or 1 (rho): 10 adds and 10 FMAs instead of four complex products.
// Open faces (S- := S+ at the first site, S+ := S- at the last) are folded into the
// neighbour itself: U* W' = U E  <=>  W' = U^2 E  (|U| = 1), likewise E' = U*^2 W, B' = U_z^2 T, T' = U_z*^2 B.
template <int MODE, int BX, int BY>
__global__ void __launch_bounds__(BX *BY, 1024 / (BX * BY)) k_march(const __grid_constant__ Dev dv) {
  constexpr int RP = 2 * BX + 4;            // row pitch in float2: [pad, W, 2*BX centre, E, pad]
  constexpr int SP = (BY + 2) * RP;         // slot pitch in float2
  constexpr unsigned SPB = SP * 8u;         // slot pitch in bytes
  extern __shared__ float4 smem4[];
  float2 *sm = reinterpret_cast<float2 *>(smem4);
  Ctl *ctl = dv.ctl;
  int l = 0;
  if (MODE != MODE_RHO) {
    if (ctl->done) return;
    l = ctl->sweeps;
  }
  const int xb = ctl->xbuf;
  const float2 *__restrict__ xin = dv.psi[xb];

  const int nx = dv.nx, ny = dv.ny, nz = dv.nz;
  const int tx = threadIdx.x, ty = threadIdx.y;
  const int lane = (ty * BX + tx) & 31;
  const int i0 = blockIdx.x * 2 * BX, j0 = blockIdx.y * BY;
  const int i = i0 + 2 * tx, j = j0 + ty;
  const int nvx = min(BX, (nx - i0) >> 1), nvy = min(BY, ny - j0);
  const bool actx = tx < nvx, acty = ty < nvy, act = actx && acty;
  const int k0 = blockIdx.z * dv.zc, k1 = min(nz, k0 + dv.zc);     // planes [k0, k1)
  const bool px = dv.bcx == 0, py = dv.bcy == 0, pz = dv.bcz == 0;
  const long long plane = (long long)nx * ny;
  const int r = ty + 1, c = 2 + 2 * tx;
  const unsigned sbase = (unsigned)__cvta_generic_to_shared(sm);

  // Copy roles, fixed for the whole march.  Every active thread copies its own 16-byte centre vector.
  // Ghost row j0-1 is copied by thread row 0, ghost row j0+nvy by thread row BY-1 (wrapped, or
  // mirrored); ghost column i0-1 by thread column 0, ghost column i0+2 nvx by thread column BX-1.
  const float2 *gC = xin + ((long long)min(j, ny - 1) * nx + min(i, nx - 2));
  const unsigned dC = sbase + (unsigned)(r * RP + c) * 8u;
  const float2 *gR = gC;
  unsigned dR = 0;
  bool hasR = false;
  if (actx && (ty == 0 || ty == BY - 1)) {
    int js, row;
    if (ty == 0) { js = j0 - 1; if (js < 0) js = py ? ny - 1 : 1; row = 0; }
    else { js = j0 + nvy; if (js >= ny) js = py ? 0 : ny - 2; row = nvy + 1; }
    gR = xin + ((long long)js * nx + i);
    dR = sbase + (unsigned)(row * RP + c) * 8u;
    hasR = true;
  }
  const float2 *gG = gC;
  unsigned dG = 0;
  bool hasG = false;
  if (acty && (tx == 0 || tx == BX - 1)) {
    int is, col;
    if (tx == 0) { is = i0 - 1; if (is < 0) is = px ? nx - 1 : 1; col = 1; }
    else { is = i0 + 2 * nvx; if (is >= nx) is = px ? 0 : nx - 2; col = 2 + 2 * nvx; }
    gG = xin + ((long long)j * nx + is);
    dG = sbase + (unsigned)(r * RP + col) * 8u;
    hasG = true;
  }

  // plane offset (elements) with the z wrap / mirror
  auto zoff = [&](int kp) -> long long {
    int kw = kp;
    if (kw < 0) kw = pz ? nz - 1 : 1;
    if (kw >= nz) kw = pz ? 0 : nz - 2;
    return (long long)kw * plane;
  };
  auto load_plane = [&](long long poff, unsigned slotb, bool ghosts) {
    if (act) cp_async16(dC + slotb, gC + poff);
    if (ghosts) {
      if (hasR) cp_async16(dR + slotb, gR + poff);
      if (hasG) cp_async8(dG + slotb, gG + poff);
    }
  };

  // prologue: planes k0-1, k0, k0+1 (slots 0, 1, 2) in one group, plane k0+2 (slot 3) in the next
  load_plane(zoff(k0 - 1), 0u, false);
  load_plane(zoff(k0), SPB, true);
  load_plane(zoff(k0 + 1), 2u * SPB, k0 + 1 < k1);
  cp_async_commit();
  if (k0 + 2 <= k1) load_plane(zoff(k0 + 2), 3u * SPB, k0 + 2 < k1);
  cp_async_commit();

  const int jc = min(j, ny - 1);
  const float f = (MODE == MODE_RHO) ? 1.f : dv.ht2;
  float2 hUx, hUz;
  {
    const float2 Ux = dv.Ux[jc], Uz = dv.Uz[jc];
    hUx = make_float2(f * dv.cx * Ux.x, f * dv.cx * Ux.y);
    hUz = make_float2(f * dv.cz * Uz.x, f * dv.cz * Uz.y);
  }
  const float hcy = f * dv.cy;
  const bool xlo0 = !px && i == 0, xhi1 = !px && (i + 1 == nx - 1);
  const bool ylo = py && j == 0, yhi = py && j == ny - 1;
  const bool wsm = (tx == 0 || lane == 0), esm = (tx >= nvx - 1 || lane == 31);
  float rmax = 0.f;
  unsigned nstep = 0;
  if (MODE == MODE_INIT) nstep = (unsigned)ctl->n;

  // running element index of this thread's pair of sites (float2 units)
  long long idx = (long long)k0 * plane + (long long)min(j, ny - 1) * nx + min(i, nx - 2);
  float2 *__restrict__ xout = dv.psi[xb ^ 1];
  // ring of 5 slots (element offsets): planes k-1, k, k+1, k+2 and the free slot that receives plane k+3
  unsigned oB = 0u, oC = SP, oT = 2u * SP, oU = 3u * SP, oF = 4u * SP;
  const float2 *sthr = sm + r * RP + c;       // this thread's centre position inside a slot

  for (int k = k0; k < k1; ++k) {
    cp_async_wait<1>();                     // planes <= k+1 have landed; plane k+2 may still be in flight
    __syncthreads();
    if (k + 3 <= k1) load_plane(zoff(k + 3), oF * 8u, k + 3 < k1);
    cp_async_commit();

    float4 bv = make_float4(0, 0, 0, 0), dvv = make_float4(1, 0, 1, 0);
    if (MODE == MODE_SWEEP && act) {                          // issued early, consumed after the stencil
      bv = __ldcs(reinterpret_cast<const float4 *>(dv.b + idx));
      dvv = __ldcs(reinterpret_cast<const float4 *>(dv.d + idx));
    }
    float2 muv = make_float2(0.f, 0.f), ev = make_float2(1.f, 1.f);
    if (MODE == MODE_INIT && act) {
      if (dv.solve_mu) muv = __ldcs(reinterpret_cast<const float2 *>(dv.mu + idx));
      ev = __ldg(reinterpret_cast<const float2 *>(dv.eps + idx));
    }

    const float2 *sC = sthr + oC;
    const float4 C = *reinterpret_cast<const float4 *>(sC);
    float4 Nn = *reinterpret_cast<const float4 *>(sC + RP);
    float4 Ss = *reinterpret_cast<const float4 *>(sC - RP);
    float4 T = *reinterpret_cast<const float4 *>(sthr + oT);
    float4 B = *reinterpret_cast<const float4 *>(sthr + oB);
    float2 W, E;
    W.x = __shfl_up_sync(0xffffffffu, C.z, 1);
    W.y = __shfl_up_sync(0xffffffffu, C.w, 1);
    E.x = __shfl_down_sync(0xffffffffu, C.x, 1);
    E.y = __shfl_down_sync(0xffffffffu, C.y, 1);
    if (wsm) W = sC[-1];
    if (esm) E = sC[2];
    const float2 c0 = make_float2(C.x, C.y), c1 = make_float2(C.z, C.w);

    if (ylo || yhi) {                          // quasi-periodic jump in y
      const float2 Pk = dv.Pk[k];
      const float4 Pij = *reinterpret_cast<const float4 *>(dv.Pi + min(i, nx - 2));
      const float2 P0 = cmulc(Pk, make_float2(Pij.x, Pij.y));   // P_{i,k} = Pi[i] conj(Pk[k])
      const float2 P1 = cmulc(Pk, make_float2(Pij.z, Pij.w));
      if (ylo) {                               // psi_{i,-1,k} = P psi_{i,ny-1,k}
        const float2 a = cmul(P0, make_float2(Ss.x, Ss.y)), bq = cmul(P1, make_float2(Ss.z, Ss.w));
        Ss = make_float4(a.x, a.y, bq.x, bq.y);
      }
      if (yhi) {                               // psi_{i,ny,k} = P* psi_{i,0,k}
        const float2 a = cmulc(P0, make_float2(Nn.x, Nn.y)), bq = cmulc(P1, make_float2(Nn.z, Nn.w));
        Nn = make_float4(a.x, a.y, bq.x, bq.y);
      }
    }
    if (xlo0 || xhi1) {
      const float2 Ux = dv.Ux[jc];
      if (xlo0) W = cmul(cmul(Ux, Ux), c1);                     // open x, first site: W' = U^2 E
      if (xhi1) E = cmulc(cmul(Ux, Ux), c0);                    // open x, last site:  E' = U*^2 W
    }
    if (!pz && (k == 0 || k == nz - 1)) {                       // open z faces (uniform over the CTA)
      const float2 Uz = dv.Uz[jc];
      const float2 U2 = cmul(Uz, Uz);
      if (k == 0) {
        const float2 a = cmul(U2, make_float2(T.x, T.y)), bq = cmul(U2, make_float2(T.z, T.w));
        B = make_float4(a.x, a.y, bq.x, bq.y);
      } else {
        const float2 a = cmulc(U2, make_float2(B.x, B.y)), bq = cmulc(U2, make_float2(B.z, B.w));
        T = make_float4(a.x, a.y, bq.x, bq.y);
      }
    }

    float2 b0 = make_float2(bv.x, bv.y), b1 = make_float2(bv.z, bv.w);
    // acc = start + f nsum;  start = b (sweep) or 0 (init, rho)
    float2 s0 = (MODE == MODE_SWEEP) ? b0 : make_float2(0.f, 0.f);
    float2 s1 = (MODE == MODE_SWEEP) ? b1 : make_float2(0.f, 0.f);
    // site 0: west W, east c1;  site 1: west c0, east E
    s0.x = fmaf(hUx.x, c1.x + W.x, s0.x);  s0.x = fmaf(-hUx.y, c1.y - W.y, s0.x);
    s0.y = fmaf(hUx.x, c1.y + W.y, s0.y);  s0.y = fmaf(hUx.y, c1.x - W.x, s0.y);
    s1.x = fmaf(hUx.x, E.x + c0.x, s1.x);  s1.x = fmaf(-hUx.y, E.y - c0.y, s1.x);
    s1.y = fmaf(hUx.x, E.y + c0.y, s1.y);  s1.y = fmaf(hUx.y, E.x - c0.x, s1.y);
    s0.x = fmaf(hcy, Nn.x + Ss.x, s0.x);   s0.y = fmaf(hcy, Nn.y + Ss.y, s0.y);
    s1.x = fmaf(hcy, Nn.z + Ss.z, s1.x);   s1.y = fmaf(hcy, Nn.w + Ss.w, s1.y);
    s0.x = fmaf(hUz.x, T.x + B.x, s0.x);   s0.x = fmaf(-hUz.y, T.y - B.y, s0.x);
    s0.y = fmaf(hUz.x, T.y + B.y, s0.y);   s0.y = fmaf(hUz.y, T.x - B.x, s0.y);
    s1.x = fmaf(hUz.x, T.z + B.z, s1.x);   s1.x = fmaf(-hUz.y, T.w - B.w, s1.x);
    s1.y = fmaf(hUz.x, T.w + B.w, s1.y);   s1.y = fmaf(hUz.y, T.z - B.z, s1.y);

    if (MODE == MODE_RHO) {
      // rho_m = sum_alpha c_alpha Im[psi*_m (S+ psi + S- psi)_m]
      if (act)
        *reinterpret_cast<float2 *>(dv.mu + idx) =
            make_float2(c0.x * s0.y - c0.y * s0.x, c1.x * s1.y - c1.y * s1.x);
    } else {
      float2 d0 = make_float2(dvv.x, dvv.y), d1 = make_float2(dvv.z, dvv.w);
      float2 n0 = s0, n1 = s1;                 // numerators b + (h_t/2) nsum
      if (MODE == MODE_INIT) {
        // d_m = 1 + (h_t/2)[|psi|^2 + 2 sum c - eps + i u mu]
        // b_m = psi (2 - d) + (h_t/2)(nsum + 2 zeta)            (Eq. 31, rearranged)
        const float ht2 = dv.ht2;
        const float a0 = c0.x * c0.x + c0.y * c0.y, a1 = c1.x * c1.x + c1.y * c1.y;
        d0 = make_float2(1.f + ht2 * (a0 + dv.csum2 - ev.x), ht2 * dv.u * muv.x);
        d1 = make_float2(1.f + ht2 * (a1 + dv.csum2 - ev.y), ht2 * dv.u * muv.y);
        float2 z0 = make_float2(0.f, 0.f), z1 = z0;
        if (dv.zeta_max > 0.f) {               // Langevin term, Eq. (39), S11
          const unsigned long long m = (unsigned long long)idx;
          const PhiloxOut p0 = philox4x32_10((uint32_t)m, (uint32_t)(m >> 32), nstep, 0u, dv.seed_lo, dv.seed_hi);
          const PhiloxOut p1 = philox4x32_10((uint32_t)(m + 1), (uint32_t)((m + 1) >> 32), nstep, 0u, dv.seed_lo, dv.seed_hi);
          const float zs = 2.f * ht2 * dv.zeta_max;
          z0 = make_float2(zs * u32_to_pm1(p0.x0), zs * u32_to_pm1(p0.x1));
          z1 = make_float2(zs * u32_to_pm1(p1.x0), zs * u32_to_pm1(p1.x1));
        }
        const float2 q0 = cmul(c0, make_float2(2.f - d0.x, -d0.y)), q1 = cmul(c1, make_float2(2.f - d1.x, -d1.y));
        b0 = make_float2(q0.x + s0.x + z0.x, q0.y + s0.y + z0.y);
        b1 = make_float2(q1.x + s1.x + z1.x, q1.y + s1.y + z1.y);
        n0 = make_float2(b0.x + s0.x, b0.y + s0.y);
        n1 = make_float2(b1.x + s1.x, b1.y + s1.y);
        if (act) {
          *reinterpret_cast<float4 *>(dv.b + idx) = make_float4(b0.x, b0.y, b1.x, b1.y);
          *reinterpret_cast<float4 *>(dv.d + idx) = make_float4(d0.x, d0.y, d1.x, d1.y);
        }
      }
      // x^{l+1}_m = (b_m + (h_t/2) nsum) / d_m   (Eq. 33);  |r^l_m|^2 = |d_m|^2 |x^{l+1}_m - x^l_m|^2  (S8)
      const float m0 = d0.x * d0.x + d0.y * d0.y, m1 = d1.x * d1.x + d1.y * d1.y;
      const float i0v = __fdividef(1.f, m0), i1v = __fdividef(1.f, m1);
      const float2 y0 = cmulc(d0, n0), y1 = cmulc(d1, n1);
      const float4 out = make_float4(y0.x * i0v, y0.y * i0v, y1.x * i1v, y1.y * i1v);
      if (act) {
        *reinterpret_cast<float4 *>(xout + idx) = out;
        const float e0x = out.x - c0.x, e0y = out.y - c0.y, e1x = out.z - c1.x, e1y = out.w - c1.y;
        rmax = fmaxf(rmax, fmaxf((e0x * e0x + e0y * e0y) * m0, (e1x * e1x + e1y * e1y) * m1));
      }
    }
    idx += plane;
    const unsigned t = oB; oB = oC; oC = oT; oT = oU; oU = oF; oF = t;     // rotate the ring
  }

  if (MODE != MODE_RHO) {
    // max-residual reduction: redux over the warp on the uint pattern (non-negative floats order like
    // uints), one shared atomic per warp, one global atomic per CTA; the last CTA decides (Eq. 34).
    __shared__ unsigned int s_max;
    const int tid = ty * BX + tx;
    if (tid == 0) s_max = 0u;
    __syncthreads();
    const unsigned int w = __reduce_max_sync(0xffffffffu, __float_as_uint(rmax));
    if (lane == 0) atomicMax(&s_max, w);
    __syncthreads();
    if (tid == 0) {
      atomicMax(&ctl->resid_bits[l], s_max);
      __threadfence();
      const unsigned int nb = gridDim.x * gridDim.y * gridDim.z;
      const unsigned int t = atomicAdd(&ctl->ticket, 1u);
      if (t == nb - 1) {
        ctl->ticket = 0u;
        sweep_decide(dv, l);
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------
// a5: J_av = 1/(2 N h_x) sum_m Im[psi*_m (U_x psi_{i+1} - U_x* psi_{i-1})]   (Eq. 35)
// Stage 1: fp64 partial sum per CTA (fixed grid => fixed summation order).
__global__ void __launch_bounds__(256) k_jav_partial(const __grid_constant__ Dev dv) {
  const float2 *__restrict__ x = dv.psi[dv.ctl->xbuf];
  const int hx2 = dv.nx >> 1;
  const long long npair = dv.N >> 1;
  double acc = 0.0;
  for (long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x; p < npair;
       p += (long long)gridDim.x * blockDim.x) {
    const long long row = p / hx2;
    const int i = 2 * (int)(p - row * hx2);
    const int j = (int)(row % dv.ny);
    const float2 *xr = x + row * dv.nx;
    const float4 C = *reinterpret_cast<const float4 *>(xr + i);
    const float2 W = xr[i == 0 ? dv.nx - 1 : i - 1];
    const float2 E = xr[i + 2 >= dv.nx ? 0 : i + 2];
    const float2 U = dv.Ux[j];
    const float2 c0 = make_float2(C.x, C.y), c1 = make_float2(C.z, C.w);
    // site i: E = c1, W = W; site i+1: E = E, W = c0
    const float2 up0 = cmul(U, c1), um0 = cmulc(U, W), up1 = cmul(U, E), um1 = cmulc(U, c0);
    const float t0 = c0.x * (up0.y - um0.y) - c0.y * (up0.x - um0.x);
    const float t1 = c1.x * (up1.y - um1.y) - c1.y * (up1.x - um1.x);
    acc += (double)t0 + (double)t1;
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

// Per-row link variables from K (Eq. 27; gauge 24a):  U_x(j) = exp(i h_x (K + B_z ybar_j)).
__device__ void write_Ux(const Dev &dv, double K, int tid, int nthreads) {
  const double Bz = dv.ctl->Bz;
  for (int j = tid; j < dv.ny; j += nthreads) {
    const double ybar = j * dv.hy - 0.5 * dv.Ly;
    double s, c;
    sincos(dv.hx * (K + Bz * ybar), &s, &c);
    dv.Ux[j] = make_float2((float)c, (float)s);
  }
}

// Start of a step: reset the sweep state, clear the residual slots, refresh U_x(j) with the lagged K (S2).
__global__ void k_step_begin(const __grid_constant__ Dev dv) {
  Ctl *c = dv.ctl;
  const int tid = threadIdx.x;
  for (int s = tid; s < TDGL_MAX_RESID_SLOTS; s += blockDim.x) c->resid_bits[s] = 0u;
  if (tid == 0) {
    c->sweeps = 0;
    c->done = 0;
    c->ticket = 0u;
  }
  write_Ux(dv, c->K, tid, blockDim.x);
}

// After the psi solve: finish the J_av sum, E_x = J_ext - J_av (Eq. 21 with d_t A = 0, Eq. 15), forward
// Euler for K (S3) and rewinding; refresh U_x(j) with the new K for rho (S4); log the step.
__global__ void k_step_finish(const __grid_constant__ Dev dv, int npart) {
  Ctl *c = dv.ctl;
  __shared__ double sh[256];
  __shared__ double Knew;
  const int tid = threadIdx.x;
  const bool kact = dv.solve_mu && dv.bcx == 0;
  if (kact) {
    double s = 0.0;
    for (int p = tid; p < npart; p += 256) s += dv.part[p];
    sh[tid] = s;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
      if (tid < o) sh[tid] += sh[tid + o];
      __syncthreads();
    }
  }
  if (tid == 0) {
    double K = c->K, Ex = 0.0, Jav = 0.0;
    if (kact) {
      Jav = sh[0] / (2.0 * (double)dv.N * dv.hx);
      Ex = c->Jext - Jav;
      K = K + dv.dt * Ex;
      const double q = 6.283185307179586476925286766559 / dv.hx;
      K = K - q * floor(K / q);
    }
    c->K = K; c->Ex = Ex; c->Jav = Jav;
    c->Ex_sum += Ex; c->Ex_cnt += 1;
    const long long n = c->n;
    dv.sweep_log[n % TDGL_LOGCAP] = c->sweeps_last;
    dv.resid_log[n % TDGL_LOGCAP] = c->resid_last;
    c->sweeps_total += c->sweeps_last;
    if (c->sched_pos < c->sched_n) c->sched_pos += 1;
    c->n = n + 1;
    Knew = K;
  }
  __syncthreads();
  if (kact) write_Ux(dv, Knew, tid, blockDim.x);
}

// ------------------------------------------------------------------------------------------------
// host-side launchers (called from tdgl_api.cu)
template <int BX, int BY>
static void launch_march_t(int mode, const Dev &dv, dim3 grid, size_t smem, cudaStream_t st) {
  const dim3 block(BX, BY, 1);
  if (mode == MODE_SWEEP) k_march<MODE_SWEEP, BX, BY><<<grid, block, smem, st>>>(dv);
  else if (mode == MODE_INIT) k_march<MODE_INIT, BX, BY><<<grid, block, smem, st>>>(dv);
  else k_march<MODE_RHO, BX, BY><<<grid, block, smem, st>>>(dv);
}
template <int BX, int BY>
static cudaError_t march_configure_t(size_t smem) {
  cudaError_t e = cudaFuncSetAttribute(k_march<MODE_SWEEP, BX, BY>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(k_march<MODE_INIT, BX, BY>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(k_march<MODE_RHO, BX, BY>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
}
// supported CTA shapes (thread columns x rows): 64x8, 32x16, 16x32
void launch_march(int mode, const Dev &dv, dim3 grid, dim3 block, size_t smem, cudaStream_t st) {
  if (block.x == 64) launch_march_t<64, 8>(mode, dv, grid, smem, st);
  else if (block.x == 32) launch_march_t<32, 16>(mode, dv, grid, smem, st);
  else launch_march_t<16, 32>(mode, dv, grid, smem, st);
}
size_t march_smem_bytes(dim3 block) { return (size_t)NBUF * (block.y + 2) * (2 * block.x + 4) * sizeof(float2); }
cudaError_t march_configure(dim3 block, size_t smem) {
  if (block.x == 64) return march_configure_t<64, 8>(smem);
  if (block.x == 32) return march_configure_t<32, 16>(smem);
  return march_configure_t<16, 32>(smem);
}
void launch_jav(const Dev &dv, int nblocks, cudaStream_t st) { k_jav_partial<<<nblocks, 256, 0, st>>>(dv); }
void launch_step_begin(const Dev &dv, cudaStream_t st) { k_step_begin<<<1, 256, 0, st>>>(dv); }
void launch_step_finish(const Dev &dv, int npart, cudaStream_t st) { k_step_finish<<<1, 256, 0, st>>>(dv, npart); }
