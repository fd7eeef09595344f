// a7: the scalar-potential solve  Delta_h mu = rho,  sum_m w_m mu_m = 0  (Eq. 18 as discretised at
// P:379-383; readings S5-S7), hand-written, no library.
//
// Delta_h is the 7-point operator with periodic wrap or mirror ghost per axis.  Its 1-D factors are
// diagonalised by REAL transforms, so the whole solve stays real and in place on the mu array:
//   periodic axis : discrete Hartley transform  H_q = sum_p x_p cas(2 pi q p/n)   (self-inverse up to 1/n;
//                   a symmetric circulant matrix is diagonal in the Hartley basis with the Fourier eigenvalues)
//   open axis     : DCT-I  X_q = x_0 + (-1)^q x_{n-1} + 2 sum x_p cos(pi q p/(n-1))   (self-inverse up to 1/(2(n-1)))
// x and y are transformed, z is either transformed + divided + transformed back inside one kernel
// (periodic z), or solved by the Thomas algorithm with the mirror rows (open z).
// Power-of-two Hartley transforms use a Stockham radix-4 FFT in shared memory on two real lines packed
// as one complex line; every other length takes the O(n^2) table path with fp64 accumulation.
#include "tdgl_dev.cuh"

// ---------------------------------------------------------------------------------------------
// batched Stockham FFT in shared memory; element (p, f) of FFT f lives at p*PS + f*FS
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void fft_stage(const float2 *__restrict__ in, float2 *__restrict__ out, int n, int Ns,
                                          int R, int nfft, int PS, int FS, const float2 *__restrict__ tw, int tid,
                                          int nth) {
  const int nb = n / R;
  const int tstep = n / (Ns * R);
  for (int w = tid; w < nfft * nb; w += nth) {
    int f, jj;
    if (FS == 1) { f = w % nfft; jj = w / nfft; } else { jj = w % nb; f = w / nb; }
    const int k = jj & (Ns - 1);
    const float2 *src = in + f * FS;
    float2 *dst = out + f * FS + (size_t)(((jj - k) * R) + k) * PS;
    if (R == 4) {
      float2 v0 = src[(jj)*PS], v1 = src[(jj + nb) * PS], v2 = src[(jj + 2 * nb) * PS], v3 = src[(jj + 3 * nb) * PS];
      if (k) {
        v1 = cmul(v1, tw[k * tstep]);
        v2 = cmul(v2, tw[2 * k * tstep]);
        v3 = cmul(v3, tw[3 * k * tstep]);
      }
      const float2 a0 = make_float2(v0.x + v2.x, v0.y + v2.y), a1 = make_float2(v0.x - v2.x, v0.y - v2.y);
      const float2 a2 = make_float2(v1.x + v3.x, v1.y + v3.y);
      const float2 a3 = make_float2(v1.y - v3.y, -(v1.x - v3.x));          // -i (v1 - v3)
      dst[0] = make_float2(a0.x + a2.x, a0.y + a2.y);
      dst[Ns * PS] = make_float2(a1.x + a3.x, a1.y + a3.y);
      dst[2 * Ns * PS] = make_float2(a0.x - a2.x, a0.y - a2.y);
      dst[3 * Ns * PS] = make_float2(a1.x - a3.x, a1.y - a3.y);
    } else {
      float2 v0 = src[jj * PS], v1 = src[(jj + nb) * PS];
      if (k) v1 = cmul(v1, tw[k * tstep]);
      dst[0] = make_float2(v0.x + v1.x, v0.y + v1.y);
      dst[Ns * PS] = make_float2(v0.x - v1.x, v0.y - v1.y);
    }
  }
}

// Hartley transforms of the two real lines packed as (re, im):  FFT, then
//   H^a_q = (Re Z_q + Re Z_{n-q} - Im Z_q + Im Z_{n-q})/2,  H^b_q = (Im Z_q + Im Z_{n-q} + Re Z_q - Re Z_{n-q})/2.
// Returns the buffer that holds the result.
__device__ float2 *dht_pairs(float2 *bufA, float2 *bufB, int n, int nfft, int PS, int FS, const float2 *tw, int tid,
                             int nth) {
  float2 *in = bufA, *out = bufB;
  for (int Ns = 1; Ns < n;) {
    const int R = (n / Ns >= 4) ? 4 : 2;
    fft_stage(in, out, n, Ns, R, nfft, PS, FS, tw, tid, nth);
    __syncthreads();
    float2 *t = in; in = out; out = t;
    Ns *= R;
  }
  const int half = n / 2 - 1;                 // pairs q = 1 .. n/2-1; q = 0 and n/2 are already H
  for (int w = tid; w < nfft * half; w += nth) {
    int f, q;
    if (FS == 1) { f = w % nfft; q = 1 + w / nfft; } else { q = 1 + w % half; f = w / half; }
    float2 *z = in + f * FS;
    const float2 u = z[q * PS], v = z[(n - q) * PS];
    z[q * PS] = make_float2(0.5f * (u.x + v.x - u.y + v.y), 0.5f * (u.y + v.y + u.x - v.x));
    z[(n - q) * PS] = make_float2(0.5f * (v.x + u.x - v.y + u.y), 0.5f * (v.y + u.y + v.x - u.x));
  }
  __syncthreads();
  return in;
}

// Hartley transform along x (contiguous rows), two rows per complex FFT.  grid.x = row-pair groups.
__global__ void __launch_bounds__(256) k_dht_x(float *__restrict__ data, int n, long long nrows, int nfft,
                                               const float2 *__restrict__ twg) {
  extern __shared__ float4 smem4[];
  float2 *tw = reinterpret_cast<float2 *>(smem4);
  float2 *A = tw + n, *Bf = A + (size_t)nfft * n;
  const int tid = threadIdx.x, nth = blockDim.x;
  for (int m = tid; m < n; m += nth) tw[m] = twg[m];
  const long long pair0 = (long long)blockIdx.x * nfft;
  for (int w = tid; w < nfft * n; w += nth) {
    const int f = w / n, p = w - f * n;
    const long long ra = 2 * (pair0 + f), rb = ra + 1;
    float2 v = make_float2(0.f, 0.f);
    if (ra < nrows) v.x = data[ra * n + p];
    if (rb < nrows) v.y = data[rb * n + p];
    A[f * n + p] = v;
  }
  __syncthreads();
  const float2 *res = dht_pairs(A, Bf, n, nfft, 1, n, tw, tid, nth);
  for (int w = tid; w < nfft * n; w += nth) {
    const int f = w / n, p = w - f * n;
    const long long ra = 2 * (pair0 + f), rb = ra + 1;
    const float2 v = res[f * n + p];
    if (ra < nrows) data[ra * n + p] = v.x;
    if (rb < nrows) data[rb * n + p] = v.y;
  }
}

// Hartley transform along a strided axis (y or z).  The real array is read as float2 columns (columns
// 2c, 2c+1 = re, im).  A CTA owns CC complex columns at a fixed "other" index o:
//   base = o*ostride + 2*(c0 + f),  element p at base + p*stride   (all in floats).
// divide != 0 (z axis, periodic): after the transform every coefficient is multiplied by
// scale / (lam_x[i] + lam_y[j] + lam_z[q]) (zero mode -> 0, S7) and transformed back.
__global__ void __launch_bounds__(256) k_dht_strided(float *__restrict__ data, int n, long long stride,
                                                     long long ostride, int ncolc, int CC,
                                                     const float2 *__restrict__ twg, int divide, float scale,
                                                     const float *__restrict__ lamx, const float *__restrict__ lamy,
                                                     const float *__restrict__ lamz) {
  extern __shared__ float4 smem4[];
  float2 *tw = reinterpret_cast<float2 *>(smem4);
  float2 *A = tw + n, *Bf = A + (size_t)CC * n;
  const int tid = threadIdx.x, nth = blockDim.x;
  for (int m = tid; m < n; m += nth) tw[m] = twg[m];
  const int c0 = blockIdx.x * CC;
  const long long o = blockIdx.y;
  float *base = data + o * ostride + 2 * (long long)c0;
  const int nv = min(CC, ncolc - c0);
  for (int w = tid; w < CC * n; w += nth) {
    const int p = w / CC, f = w - p * CC;
    float2 v = make_float2(0.f, 0.f);
    if (f < nv) v = *reinterpret_cast<const float2 *>(base + p * stride + 2 * f);
    A[p * CC + f] = v;
  }
  __syncthreads();
  float2 *res = dht_pairs(A, Bf, n, CC, CC, 1, tw, tid, nth);
  if (divide) {
    for (int w = tid; w < CC * n; w += nth) {
      const int q = w / CC, f = w - q * CC;
      const int i = 2 * (c0 + f);
      float2 v = res[q * CC + f];
      if (f < nv) {
        const float lyz = lamy[o] + lamz[q];
        const float la = lamx[i] + lyz, lb = lamx[i + 1] + lyz;
        v.x = (la != 0.f) ? v.x * (scale / la) : 0.f;
        v.y = (lb != 0.f) ? v.y * (scale / lb) : 0.f;
      }
      res[q * CC + f] = v;
    }
    __syncthreads();
    float2 *other = (res == A) ? Bf : A;
    res = dht_pairs(res, other, n, CC, CC, 1, tw, tid, nth);
  }
  for (int w = tid; w < CC * n; w += nth) {
    const int p = w / CC, f = w - p * CC;
    if (f < nv) *reinterpret_cast<float2 *>(base + p * stride + 2 * f) = res[p * CC + f];
  }
}

// Any length, any of the two transforms: out_q = sum_p w_p x_p tab[(q p) mod M], fp64 accumulation.
//   kind 0: Hartley, tab[m] = cas(2 pi m/n), M = n, w = 1
//   kind 1: DCT-I,   tab[m] = cos(pi m/(n-1)), M = 2(n-1), w = 1 at the ends, 2 inside
// A CTA owns TL lines.  contiguous != 0: line l = row (blockIdx.x*TL + l), elements adjacent.
// contiguous == 0: lines are adjacent columns i = blockIdx.x*TL + l at other index o = blockIdx.y.
__global__ void __launch_bounds__(256) k_transform_generic(float *__restrict__ data, int n, int kind, int contiguous,
                                                           long long nlines, long long stride, long long ostride,
                                                           int TL, const double *__restrict__ tabg, int divide,
                                                           float scale, const float *__restrict__ lamx,
                                                           const float *__restrict__ lamy,
                                                           const float *__restrict__ lamz) {
  extern __shared__ double smemd[];
  const int M = kind ? 2 * (n - 1) : n;
  double *tab = smemd;
  float *in = reinterpret_cast<float *>(tab + M);
  float *out = in + (size_t)TL * n;
  const int tid = threadIdx.x, nth = blockDim.x;
  for (int m = tid; m < M; m += nth) tab[m] = tabg[m];
  const long long l0 = (long long)blockIdx.x * TL;
  const long long o = blockIdx.y;
  const int nv = (int)min((long long)TL, nlines - l0);
  // smem layout: contiguous: [l][p]; strided: [p][l]
  for (int w = tid; w < TL * n; w += nth) {
    int l, p;
    if (contiguous) { l = w / n; p = w - l * n; } else { p = w / TL; l = w - p * TL; }
    float v = 0.f;
    if (l < nv) v = contiguous ? data[(l0 + l) * n + p] : data[o * ostride + p * stride + l0 + l];
    if (kind && p != 0 && p != n - 1) v *= 2.f;
    in[w] = v;
  }
  __syncthreads();
  for (int pass = 0; pass < (divide ? 2 : 1); ++pass) {
    for (int w = tid; w < TL * n; w += nth) {
      int l, q;
      if (contiguous) { l = w / n; q = w - l * n; } else { q = w / TL; l = w - q * TL; }
      double acc = 0.0;
      int idx = 0;
      const float *src = contiguous ? in + (size_t)l * n : in + l;
      const int ps = contiguous ? 1 : TL;
      for (int p = 0; p < n; ++p) {
        acc += (double)src[p * ps] * tab[idx];
        idx += q;
        if (idx >= M) idx -= M;
      }
      out[w] = (float)acc;
    }
    __syncthreads();
    if (divide && pass == 0) {        // strided z axis only: column i = l0 + l, row j = o
      for (int w = tid; w < TL * n; w += nth) {
        const int q = w / TL, l = w - q * TL;
        float v = out[w];
        if (l < nv) {
          const float la = lamx[l0 + l] + lamy[o] + lamz[q];
          v = (la != 0.f) ? v * (scale / la) : 0.f;
        }
        if (kind && q != 0 && q != n - 1) v *= 2.f;
        in[w] = v;
      }
      __syncthreads();
    }
  }
  for (int w = tid; w < TL * n; w += nth) {
    int l, p;
    if (contiguous) { l = w / n; p = w - l * n; } else { p = w / TL; l = w - p * TL; }
    if (l < nv) {
      if (contiguous) data[(l0 + l) * n + p] = out[w];
      else data[o * ostride + p * stride + l0 + l] = out[w];
    }
  }
}

// Open z: for every transformed (qx, qy) the mirror-row tridiagonal system
//   c_z (mu_{k+1} + mu_{k-1} - 2 mu_k) + (lam_x + lam_y) mu_k = rho_k,   mu_{-1} = mu_1, mu_{nz} = mu_{nz-2}  (S6)
// by the Thomas algorithm, one thread per line (adjacent threads = adjacent x: coalesced planes).
// Forward: pivots and modified right side (fp64 arithmetic, fp32 storage: c' -> scratch, d' in place).
// The (0,0) line is singular (Neumann): its last unknown is pinned to 0 and the z-weighted mean is
// removed afterwards (S7).
// Two adjacent lines (columns i, i+1: one 8-byte access) per thread: twice the loads in flight per thread and half
// the threads, so that the whole plane is resident in one wave (ncu: the one-line version ran 1.54 waves and was
// latency bound, 46 % of DRAM peak).
__global__ void __launch_bounds__(64) k_thomas_z(float *__restrict__ data, float *__restrict__ cp, int nx, int ny,
                                                 int nz, float cz, float scale, const float *__restrict__ lamx,
                                                 const float *__restrict__ lamy) {
  const long long pr = (long long)blockIdx.x * blockDim.x + threadIdx.x;     // pair index
  const long long plane = (long long)nx * ny;
  const long long col = 2 * pr;
  if (col >= plane) return;
  const int j = (int)(col / nx), i = (int)(col - (long long)j * nx);
  const double ly = (double)lamy[j];
  const double lam[2] = {(double)lamx[i] + ly, (double)lamx[i + 1] + ly};
  const bool zero[2] = {lam[0] == 0.0, lam[1] == 0.0};
  const double bq[2] = {-2.0 + lam[0] / (double)cz, -2.0 + lam[1] / (double)cz};   // diagonal / c_z
  const double rs = (double)scale / (double)cz;
  float2 *x = reinterpret_cast<float2 *>(data + col);
  float2 *c = reinterpret_cast<float2 *>(cp + col);
  const long long ps = plane / 2;                                            // plane stride in float2 units
  // forward elimination, 8 planes per batch so that 8 independent 8-byte loads are in flight per thread
  double cprev[2] = {0.0, 0.0}, dprev[2] = {0.0, 0.0};
  float2 xnext[8];                                       // the next batch is in flight while this one is eliminated
#pragma unroll
  for (int u = 0; u < 8; ++u) xnext[u] = (u < nz) ? __ldcs(x + (long long)u * ps) : make_float2(0.f, 0.f);
  for (int kb = 0; kb < nz; kb += 8) {
    float2 xin[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) xin[u] = xnext[u];
#pragma unroll
    for (int u = 0; u < 8; ++u) xnext[u] = (kb + 8 + u < nz) ? __ldcs(x + (long long)(kb + 8 + u) * ps) : make_float2(0.f, 0.f);
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int k = kb + u;
      if (k < nz) {
        const double rhs[2] = {(double)xin[u].x * rs, (double)xin[u].y * rs};
        float co[2], xo[2];
#pragma unroll
        for (int q = 0; q < 2; ++q) {
          double inv, dk;
          if (k == 0) {                                 // row 0: off-diagonal 2
            inv = 2.0 / bq[q];
            dk = rhs[q] / bq[q];
          } else {
            const double a = (k == nz - 1) ? 2.0 : 1.0;
            if (zero[q] && k == nz - 1) { inv = 0.0; dk = 0.0; }
            else { inv = 1.0 / (bq[q] - a * cprev[q]); dk = (rhs[q] - a * dprev[q]) * inv; }
          }
          cprev[q] = inv;
          dprev[q] = dk;
          co[q] = (float)inv;
          xo[q] = (float)dk;
        }
        c[(long long)k * ps] = make_float2(co[0], co[1]);
        x[(long long)k * ps] = make_float2(xo[0], xo[1]);
      }
    }
  }
  // back substitution, same batching (descending)
  double xn[2] = {0.0, 0.0};
  float2 xvn[8], cvn[8];
#pragma unroll
  for (int u = 0; u < 8; ++u) {
    const int k = nz - 1 - u;
    xvn[u] = (k >= 0) ? x[(long long)k * ps] : make_float2(0.f, 0.f);
    cvn[u] = (k >= 0) ? __ldcs(c + (long long)k * ps) : make_float2(0.f, 0.f);
  }
  for (int kb = nz - 1; kb >= 0; kb -= 8) {
    float2 xv[8], cv[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) { xv[u] = xvn[u]; cv[u] = cvn[u]; }
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int k = kb - 8 - u;
      xvn[u] = (k >= 0) ? x[(long long)k * ps] : make_float2(0.f, 0.f);
      cvn[u] = (k >= 0) ? __ldcs(c + (long long)k * ps) : make_float2(0.f, 0.f);
    }
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int k = kb - u;
      if (k >= 0) {
        xn[0] = (k == nz - 1) ? (double)xv[u].x : (double)xv[u].x - (double)cv[u].x * xn[0];
        xn[1] = (k == nz - 1) ? (double)xv[u].y : (double)xv[u].y - (double)cv[u].y * xn[1];
        x[(long long)k * ps] = make_float2((float)xn[0], (float)xn[1]);
      }
    }
  }
  if (zero[0] || zero[1]) {                             // singular Neumann line: remove its z-weighted mean (S7)
    float *xs = data + col + (zero[0] ? 0 : 1);
    double s = 0.0;
    for (int k = 0; k < nz; ++k) s += ((k == 0 || k == nz - 1) ? 0.5 : 1.0) * (double)xs[k * plane];
    const float mean = (float)(s / (double)(nz - 1));
    for (int k = 0; k < nz; ++k) xs[k * plane] -= mean;
  }
}

// Transform tables (fp64 trigonometry, once at create).
//   lam[q]: -c (2 - 2 cos(2 pi q/n)) periodic (Hartley index q), -c (2 - 2 cos(pi q/(n-1))) open
//   tw[m] = exp(-2 pi i m/n);  tab[m] = cas(2 pi m/n) or cos(pi m/(n-1))
__global__ void k_build_tables(float *lam, float2 *tw, double *tab, int n, int open, double c) {
  const int M = open ? 2 * (n - 1) : n;
  for (int m = blockIdx.x * blockDim.x + threadIdx.x; m < max(M, n); m += gridDim.x * blockDim.x) {
    if (m < n) {
      const double ang = open ? (double)m / (double)(n - 1) : 2.0 * (double)m / (double)n;   // in units of pi
      lam[m] = (float)(-c * (2.0 - 2.0 * cospi(ang)));
      double s, co;
      sincospi(-2.0 * (double)m / (double)n, &s, &co);
      tw[m] = make_float2((float)co, (float)s);
    }
    if (m < M) {
      double s, co;
      sincospi(open ? (double)m / (double)(n - 1) : 2.0 * (double)m / (double)n, &s, &co);
      tab[m] = open ? co : co + s;
    }
  }
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
// lengths of the shared-memory radix-4 fallback (powers of two below the register-blocked path's range)
static bool is_pow2(int n) { return n >= 4 && n < 64 && (n & (n - 1)) == 0; }

// Bluestein DCT-I fast path (dct.cu)
void launch_dct_x(float *data, int n, int LB, long long nrows, const float2 *T, const float2 *C, const float2 *H,
                  cudaStream_t st);
void launch_dct_s(float *data, int n, int LB, long long stride, long long ostride, int ncolc, int nother,
                  const float2 *T, const float2 *C, const float2 *H, cudaStream_t st);
// prime-factor DCT-I for the lengths that have a plan (dct_pfa.cu)
void launch_dct_pfa_x(int kind, float *data, long long nrows, const unsigned short *tab, cudaStream_t st);
void launch_dct_pfa_s(int kind, float *data, long long stride, long long ostride, int ncolc, int nother, const unsigned short *tab,
                      cudaStream_t st);
// register-blocked fast path (fft.cu)
bool dht_fast_supported(int n);
cudaError_t dht_fast_configure(int n);
void launch_dht_x_fast(float *data, int n, long long nrows, const float2 *tw, cudaStream_t st);
// persistent radix-8^3 kernel for n = 512 (fft_r8.cu)
cudaError_t dht_x_512_configure();
void launch_dht_x_512(float *data, long long nrows, const float2 *tw, cudaStream_t st);
void launch_dht_s_fast(float *data, int n, long long stride, long long ostride, int ncolc, int nother, const float2 *tw,
                       int divide, float scale, const float *lx, const float *ly, const float *lz, cudaStream_t st);

struct PoissonPlan {
  int nx, ny, nz, bc[3];
  float cz, scale;
  bool fast[3];
};

static size_t smem_dht_x(int n, int nfft) { return (size_t)(n + 2 * (size_t)nfft * n) * sizeof(float2); }
static size_t smem_generic(int n, int kind, int TL) {
  const int M = kind ? 2 * (n - 1) : n;
  return (size_t)M * sizeof(double) + 2 * (size_t)TL * n * sizeof(float);
}
static int nfft_x(int n) { int f = 2048 / n; return f < 1 ? 1 : (f > 32 ? 32 : f); }
static int cc_strided(int n) { return n >= 512 ? 8 : 16; }
// lines per CTA of the generic O(n^2) transform: as many as fit ~200 KB of shared memory (table + two line buffers)
static int tl_generic(int n) {
  const long long tab = 16ll * n;                       // <= 2 (n - 1) doubles
  int tl = n > 512 ? 16 : 32;
  while (tl > 1 && tab + 8ll * tl * n > 200 * 1024) tl >>= 1;
  return tl;
}

cudaError_t poisson_configure(int nx, int ny, int nz) {
  size_t a = 0, b = 0, c = 0;
  const int ns[3] = {nx, ny, nz};
  for (int ax = 0; ax < 3; ++ax) {
    const int n = ns[ax];
    if (is_pow2(n)) {
      if (ax == 0) { size_t s = smem_dht_x(n, nfft_x(n)); if (s > a) a = s; }
      else { size_t s = smem_dht_x(n, cc_strided(n)); if (s > b) b = s; }
    }
    for (int kind = 0; kind < 2; ++kind) { size_t s = smem_generic(n, kind, tl_generic(n)); if (s > c) c = s; }
  }
  cudaError_t e;
  if (nx == 512 && (e = dht_x_512_configure()) != cudaSuccess) return e;
  for (int ax = 0; ax < 3; ++ax)
    if (dht_fast_supported(ns[ax]) && (e = dht_fast_configure(ns[ax])) != cudaSuccess) return e;
  if (a && (e = cudaFuncSetAttribute(k_dht_x, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)a)) != cudaSuccess) return e;
  if (b && (e = cudaFuncSetAttribute(k_dht_strided, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)b)) != cudaSuccess) return e;
  return cudaFuncSetAttribute(k_transform_generic, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c);
}

void launch_build_tables(float *lam, float2 *tw, double *tab, int n, int open, double c, cudaStream_t st) {
  k_build_tables<<<8, 256, 0, st>>>(lam, tw, tab, n, open, c);
}

// One axis transform, in place.  axis 0 = x (contiguous), 1 = y, 2 = z.  Returns launches made.
static int transform_axis(const Dev &dv, float *data, int axis, bool divide, float scale, cudaStream_t st) {
  const int ns[3] = {dv.nx, dv.ny, dv.nz};
  const int bcs[3] = {dv.bcx, dv.bcy, dv.bcz};
  const int n = ns[axis];
  if (n == 1) return 0;                                   // a periodic axis of one point: the transform is the identity
  const bool open = bcs[axis] == 1;
  const long long plane = (long long)dv.nx * dv.ny;
  if (open && dv.pfaK[axis] >= 0 && !divide) {
    if (axis == 0) launch_dct_pfa_x(dv.pfaK[0], data, (long long)dv.ny * dv.nz, dv.pfaT[0], st);
    else launch_dct_pfa_s(dv.pfaK[axis], data, axis == 1 ? dv.nx : plane, axis == 1 ? plane : dv.nx, dv.nx / 2,
                          axis == 1 ? dv.nz : dv.ny, dv.pfaT[axis], st);
    return 1;
  }
  if (open && dv.bLB[axis] && !divide) {
    if (axis == 0) launch_dct_x(data, n, dv.bLB[0], (long long)dv.ny * dv.nz, dv.bT[0], dv.bC[0], dv.bH[0], st);
    else launch_dct_s(data, n, dv.bLB[axis], axis == 1 ? dv.nx : plane, axis == 1 ? plane : dv.nx, dv.nx / 2,
                      axis == 1 ? dv.nz : dv.ny, dv.bT[axis], dv.bC[axis], dv.bH[axis], st);
    return 1;
  }
  if (!open && dht_fast_supported(n)) {
    if (axis == 0) {
      if (n == 512) launch_dht_x_512(data, (long long)dv.ny * dv.nz, dv.tw[0], st);
      else launch_dht_x_fast(data, n, (long long)dv.ny * dv.nz, dv.tw[0], st);
    } else {
      launch_dht_s_fast(data, n, axis == 1 ? dv.nx : plane, axis == 1 ? plane : dv.nx, dv.nx / 2,
                        axis == 1 ? dv.nz : dv.ny, dv.tw[axis], divide ? 1 : 0, scale, dv.lam[0], dv.lam[1], dv.lam[2], st);
    }
    return 1;
  }
  if (!open && is_pow2(n)) {
    if (axis == 0) {
      const long long nrows = (long long)dv.ny * dv.nz;
      const int nfft = nfft_x(n);
      const long long npairs = (nrows + 1) / 2;
      const unsigned grid = (unsigned)((npairs + nfft - 1) / nfft);
      k_dht_x<<<grid, 256, smem_dht_x(n, nfft), st>>>(data, n, nrows, nfft, dv.tw[0]);
    } else {
      const int CC = cc_strided(n);
      const int ncolc = dv.nx / 2;
      dim3 grid((ncolc + CC - 1) / CC, axis == 1 ? dv.nz : dv.ny);
      const long long stride = axis == 1 ? dv.nx : plane;
      const long long ostride = axis == 1 ? plane : dv.nx;
      k_dht_strided<<<grid, 256, smem_dht_x(n, CC), st>>>(data, n, stride, ostride, ncolc, CC, dv.tw[axis],
                                                           divide ? 1 : 0, scale, dv.lam[0], dv.lam[1], dv.lam[2]);
    }
    return 1;
  }
  const int TL = tl_generic(n);
  const int kind = open ? 1 : 0;
  const double *tab = reinterpret_cast<const double *>(dv.tab[axis]);
  if (axis == 0) {
    const long long nrows = (long long)dv.ny * dv.nz;
    dim3 grid((unsigned)((nrows + TL - 1) / TL), 1);
    k_transform_generic<<<grid, 256, smem_generic(n, kind, TL), st>>>(data, n, kind, 1, nrows, 1, 0, TL, tab, 0, scale,
                                                                       dv.lam[0], dv.lam[1], dv.lam[2]);
  } else {
    dim3 grid((dv.nx + TL - 1) / TL, axis == 1 ? dv.nz : dv.ny);
    const long long stride = axis == 1 ? dv.nx : plane;
    const long long ostride = axis == 1 ? plane : dv.nx;
    k_transform_generic<<<grid, 256, smem_generic(n, kind, TL), st>>>(data, n, kind, 0, dv.nx, stride, ostride, TL, tab,
                                                                       divide ? 1 : 0, scale, dv.lam[0], dv.lam[1],
                                                                       dv.lam[2]);
  }
  return 1;
}

// mu <- Delta_h^{-1} mu (in place on `data`).  `thomas_open_z`: use the Thomas solver when z is open.
int poisson_solve(const Dev &dv, float *data, bool thomas_open_z, cudaStream_t st) {
  const double nrm[3] = {dv.bcx ? 2.0 * (dv.nx - 1) : (double)dv.nx, dv.bcy ? 2.0 * (dv.ny - 1) : (double)dv.ny,
                         dv.bcz ? 2.0 * (dv.nz - 1) : (double)dv.nz};
  int launches = 0;
  launches += transform_axis(dv, data, 0, false, 1.f, st);
  launches += transform_axis(dv, data, 1, false, 1.f, st);
  if (dv.bcz == 1 && thomas_open_z) {
    const long long plane = (long long)dv.nx * dv.ny;
    const float scale = (float)(1.0 / (nrm[0] * nrm[1]));
    k_thomas_z<<<(unsigned)((plane / 2 + 63) / 64), 64, 0, st>>>(data, dv.scratch, dv.nx, dv.ny, dv.nz, dv.cz, scale,
                                                                 dv.lam[0], dv.lam[1]);
    launches += 1;
  } else {
    const float scale = (float)(1.0 / (nrm[0] * nrm[1] * nrm[2]));
    launches += transform_axis(dv, data, 2, true, scale, st);
  }
  launches += transform_axis(dv, data, 1, false, 1.f, st);
  launches += transform_axis(dv, data, 0, false, 1.f, st);
  return launches;
}
