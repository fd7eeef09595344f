// The small per-step kernels around the marching stencil (march_tma.cu): the J_av reduction (a5), the
// per-row link variables U_x(j) from K (a1), the start-of-step and end-of-psi-solve control kernels.
#include "tdgl_dev.cuh"

// ------------------------------------------------------------------------------------------------
// a5: J_av = 1/(2 N h_x) sum_m Im[psi*_m (U_x psi_{i+1} - U_x* psi_{i-1})]   (Eq. 35)
// With x periodic the backward term of site m equals the forward term of site m-1, so
//   J_av = 1/(N h_x) sum over x links of Im[psi*_m U_x(j) psi_{m+x}].
// The links inside a 128-site tile row are summed by the marching kernel itself on the iterate it has
// just computed (one fp64 partial per CTA, dv.jpart).  This kernel adds the links that leave the last
// site of every tile row (wrapping to i = 0): one thread per (row, tile), fp64 partial per CTA, fixed
// grid => fixed summation order.
__global__ void __launch_bounds__(256) k_jav_edges(const __grid_constant__ Dev dv, int tile_w) {
  const float2 *__restrict__ x = dv.psi[dv.ctl->xbuf];
  const int ntx = (dv.nx + tile_w - 1) / tile_w;
  const long long nrows = (long long)dv.ny * dv.nz, total = nrows * ntx;
  double acc = 0.0;
  for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (long long)gridDim.x * blockDim.x) {
    const long long row = q / ntx;
    const int t = (int)(q - row * ntx);
    const int e = min(dv.nx, (t + 1) * tile_w) - 1;
    const int j = (int)(row % dv.ny);
    const float2 *xr = x + row * dv.nx;
    const float2 a = xr[e];
    float2 b = xr[e + 1 == dv.nx ? 0 : e + 1];
    if (dv.gauge_yz && e + 1 == dv.nx) b = cmulc(cmul(dv.Pj[j], dv.Pk[row / dv.ny]), b);   // psi_{nx} = P*_{j,k} psi_0
    const float2 ub = cmul(dv.Ux[j], b);
    acc += (double)(a.x * ub.y - a.y * ub.x);
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
  const double Bz = dv.gauge_yz ? 0.0 : dv.ctl->Bz;        // yz gauge: U_x = exp(i h_x K) on every row (Eq. 24b)
  for (int j = tid; j < dv.ny; j += nthreads) {
    const double ybar = j * dv.hy - 0.5 * dv.Ly;
    double s, c;
    sincos(dv.hx * (K + Bz * ybar), &s, &c);
    dv.Ux[j] = make_float2((float)c, (float)s);
    dv.Ux64[j] = make_double2(c, s);
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
    c->use_pair = 0;
    c->pair_jav = 1;
    c->need_jav = 0;
    c->ticket = 0u;
  }
  write_Ux(dv, c->K, tid, blockDim.x);
}

// After the psi solve: finish the J_av sum, E_x = J_ext - J_av (Eq. 21 with d_t A = 0, Eq. 15), forward
// Euler for K (S3) and rewinding; refresh U_x(j) with the new K for rho (S4); log the step.
__global__ void k_step_finish(const __grid_constant__ Dev dv, int ncta, int nedge) {
  Ctl *c = dv.ctl;
  __shared__ double sh[256];
  __shared__ double Knew;
  const int tid = threadIdx.x;
  const bool kact = dv.solve_mu && dv.bcx == 0;
  if (kact) {
    double s = 0.0;
    for (int p = tid; p < ncta; p += 256) s += dv.jpart[p];       // in-tile links (marching kernel)
    for (int p = tid; p < nedge; p += 256) s += dv.part[p];      // tile-crossing links (k_jav_edges)
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
      Jav = sh[0] / ((double)dv.N * dv.hx);
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
int jav_edge_blocks(const Dev &dv, int tile_w) {
  const long long total = (long long)dv.ny * dv.nz * ((dv.nx + tile_w - 1) / tile_w);
  const long long nb = (total + 255) / 256;
  return (int)(nb < 1 ? 1 : (nb > TDGL_NPART ? TDGL_NPART : nb));
}
void launch_jav_edges(const Dev &dv, int tile_w, int nblocks, cudaStream_t st) { k_jav_edges<<<nblocks, 256, 0, st>>>(dv, tile_w); }
void launch_step_begin(const Dev &dv, cudaStream_t st) { k_step_begin<<<1, 256, 0, st>>>(dv); }
void launch_step_finish(const Dev &dv, int ncta, int nedge, cudaStream_t st) { k_step_finish<<<1, 256, 0, st>>>(dv, ncta, nedge); }
