// Fast DCT-I for open axes of any length 3 <= n <= 1366 (a7), by Bluestein's chirp-z identity on the
// register-blocked power-of-two FFT of fft_regs.cuh.
//
// DCT-I of x_0..x_{n-1} (X_q = x_0 + (-1)^q x_{n-1} + 2 sum x_p cos(pi q p/(n-1))) is the DFT of length
// M = 2(n-1) of the even extension y (y_p = x_p, y_{M-p} = x_p).  With c_m = exp(i pi m^2/M) (period M, the
// phase is taken from m^2 mod 2M in exact integer arithmetic)
//     X_q = conj(c_q) sum_p [y_p conj(c_p)] c_{q-p},
// a linear convolution evaluated as a circular one of power-of-two length LB >= 3n-3:
//     a = y conj(c) zero-padded;  A = FFT(a);  r = IFFT(A . H),  H = FFT(chirp kernel), precomputed in fp64;
//     X_q = conj(c_q) r_q.          IFFT(B) = conj(FFT(conj(B)))/LB.
// Two real lines ride in the real and imaginary part of one complex sequence (the transform is linear and
// its matrix real).  The transform is its own inverse up to 1/(2(n-1)).
#include "fft_regs.cuh"

// tables: T[m] = exp(-2 pi i m/LB); C[m] = c_m, m < M; H = DFT_LB of h, h[d mod LB] = c_d for -(M-1) <= d <= n-1
__global__ void k_build_bluestein(float2 *T, float2 *C, float2 *H, int n, int LB) {
  const int M = 2 * (n - 1);
  for (int m = blockIdx.x * blockDim.x + threadIdx.x; m < LB; m += gridDim.x * blockDim.x) {
    double s, c;
    sincospi(-2.0 * (double)m / (double)LB, &s, &c);
    T[m] = make_float2((float)c, (float)s);
    if (m < M) {
      const long long t = ((long long)m * m) % (2LL * M);
      sincospi((double)t / (double)M, &s, &c);
      C[m] = make_float2((float)c, (float)s);
    }
    double hr = 0.0, hi = 0.0;
    for (int d = -(M - 1); d <= n - 1; ++d) {
      const long long t = ((long long)d * d) % (2LL * M);
      double sc, cc, st, ct;
      sincospi((double)t / (double)M, &sc, &cc);
      long long kd = ((long long)m * d) % LB;
      if (kd < 0) kd += LB;
      sincospi(-2.0 * (double)kd / (double)LB, &st, &ct);
      hr += cc * ct - sc * st;
      hi += cc * st + sc * ct;
    }
    H[m] = make_float2((float)hr, (float)hi);
  }
}

// shared core: v holds a_m = y_m conj(c_m) for m = j + r LB/8; on return shared memory holds
// V = FFT(conj(A . H)); the caller forms X_q = conj(c_q V_q)/LB.
template <int LB, bool XPASS, int CC>
__device__ __forceinline__ void bluestein_core(float2 *v, float2 *sm, const float2 *tw, const float2 *__restrict__ Hg,
                                               int j, int f) {
  constexpr int TPF = LB / 8;
  fft_regs<LB, XPASS, CC, false>(v, sm, tw, j, f);
#pragma unroll
  for (int r = 0; r < 8; ++r) {
    const int m = j + r * TPF;
    const float2 z = cmul(sm[saddr<LB, XPASS, CC>(f, m)], Hg[m]);
    v[r] = make_float2(z.x, -z.y);
  }
  __syncthreads();
  fft_regs<LB, XPASS, CC, false>(v, sm, tw, j, f);
}

// x pass: contiguous rows, two rows per complex sequence
template <int LB>
__global__ void __launch_bounds__((LB / 8 > 256) ? LB / 8 : 256, (LB >= 2048) ? 2 : 1)
k_dct_x(float *__restrict__ data, int n, long long nrows, const float2 *__restrict__ twg,
        const float2 *__restrict__ Cg, const float2 *__restrict__ Hg) {
  constexpr int TPF = LB / 8, F = (TPF >= 256) ? 1 : 256 / TPF, NT = F * TPF;
  extern __shared__ float4 smem4[];
  float2 *tw = reinterpret_cast<float2 *>(smem4);
  float2 *sm = tw + LB;
  const int tid = threadIdx.x;
  fill_twiddles<LB>(tw, twg, tid, NT);
  const int j = tid % TPF, f = tid / TPF;
  const int M = 2 * (n - 1);
  const long long ra = 2 * ((long long)blockIdx.x * F + f), rb = ra + 1;
  const bool va = ra < nrows, vb = rb < nrows;
  float *A = data + ra * n, *B = data + rb * n;
  float2 v[8];
#pragma unroll
  for (int r = 0; r < 8; ++r) {
    const int m = j + r * TPF;
    float2 a = make_float2(0.f, 0.f);
    if (m < M) {
      const int p = (m < n) ? m : M - m;
      const float2 z = make_float2(va ? A[p] : 0.f, vb ? B[p] : 0.f);
      a = cmulc(Cg[m], z);                          // y conj(c)
    }
    v[r] = a;
  }
  bluestein_core<LB, true, 1>(v, sm, tw, Hg, j, f);
  const float inv = 1.f / (float)LB;
#pragma unroll
  for (int r = 0; r < 8; ++r) {
    const int q = j + r * TPF;
    if (q < n) {
      const float2 w = cmul(Cg[q], sm[saddr<LB, true, 1>(f, q)]);
      if (va) A[q] = w.x * inv;
      if (vb) B[q] = -w.y * inv;
    }
  }
}

// x pass for the long transforms (LB >= 2048): CC row pairs per CTA in the [p][f] layout of the strided pass, which
// ncu shows free of bank conflicts, whereas the one-pair-per-CTA layout above had 34 % conflict wavefronts
template <int LB, int CC>
__global__ void __launch_bounds__(CC *LB / 8)
k_dct_x2(float *__restrict__ data, int n, long long nrows, const float2 *__restrict__ twg,
         const float2 *__restrict__ Cg, const float2 *__restrict__ Hg) {
  constexpr int TPF = LB / 8, NT = CC * TPF;
  extern __shared__ float4 smem4[];
  float2 *tw = reinterpret_cast<float2 *>(smem4);
  float2 *sm = tw + LB;
  const int tid = threadIdx.x;
  fill_twiddles<LB>(tw, twg, tid, NT);
  const int f = tid % CC, j = tid / CC;
  const int M = 2 * (n - 1);
  const long long ra = 2 * ((long long)blockIdx.x * CC + f), rb = ra + 1;
  const bool va = ra < nrows, vb = rb < nrows;
  float *A = data + ra * n, *B = data + rb * n;
  float2 v[8];
#pragma unroll
  for (int r = 0; r < 8; ++r) {
    const int m = j + r * TPF;
    float2 a = make_float2(0.f, 0.f);
    if (m < M) {
      const int p = (m < n) ? m : M - m;
      a = cmulc(Cg[m], make_float2(va ? A[p] : 0.f, vb ? B[p] : 0.f));
    }
    v[r] = a;
  }
  bluestein_core<LB, false, CC>(v, sm, tw, Hg, j, f);
  const float inv = 1.f / (float)LB;
#pragma unroll
  for (int r = 0; r < 8; ++r) {
    const int q = j + r * TPF;
    if (q < n) {
      const float2 w = cmul(Cg[q], sm[saddr<LB, false, CC>(f, q)]);
      if (va) A[q] = w.x * inv;
      if (vb) B[q] = -w.y * inv;
    }
  }
}

// y / z pass: float2 columns (columns 2c, 2c+1 = re, im), CC columns per CTA
template <int LB, int CC>
__global__ void __launch_bounds__(CC *LB / 8)
k_dct_s(float *__restrict__ data, int n, long long stride, long long ostride, int ncolc,
        const float2 *__restrict__ twg, const float2 *__restrict__ Cg, const float2 *__restrict__ Hg) {
  constexpr int TPF = LB / 8, NT = CC * TPF;
  extern __shared__ float4 smem4[];
  float2 *tw = reinterpret_cast<float2 *>(smem4);
  float2 *sm = tw + LB;
  const int tid = threadIdx.x;
  fill_twiddles<LB>(tw, twg, tid, NT);
  const int f = tid % CC, j = tid / CC;
  const int col = blockIdx.x * CC + f;
  const bool valid = col < ncolc;
  const int M = 2 * (n - 1);
  float *base = data + (long long)blockIdx.y * ostride + 2 * (long long)(valid ? col : 0);
  float2 v[8];
#pragma unroll
  for (int r = 0; r < 8; ++r) {
    const int m = j + r * TPF;
    float2 a = make_float2(0.f, 0.f);
    if (m < M && valid) {
      const int p = (m < n) ? m : M - m;
      a = cmulc(Cg[m], *reinterpret_cast<const float2 *>(base + p * stride));
    }
    v[r] = a;
  }
  bluestein_core<LB, false, CC>(v, sm, tw, Hg, j, f);
  const float inv = 1.f / (float)LB;
#pragma unroll
  for (int r = 0; r < 8; ++r) {
    const int q = j + r * TPF;
    if (q < n && valid) {
      const float2 w = cmul(Cg[q], sm[saddr<LB, false, CC>(f, q)]);
      *reinterpret_cast<float2 *>(base + q * stride) = make_float2(w.x * inv, -w.y * inv);
    }
  }
}

// ---- host side -----------------------------------------------------------------------------------
int dct_fast_lb(int n) {                      // 0 = not supported
  if (n < 3 || 3 * n - 3 > 4096) return 0;
  int lb = 64;
  while (lb < 3 * n - 3) lb <<= 1;
  return lb;
}
void launch_build_bluestein(float2 *T, float2 *C, float2 *H, int n, int LB, cudaStream_t st) {
  k_build_bluestein<<<(LB + 63) / 64, 64, 0, st>>>(T, C, H, n, LB);
}

template <int LB> struct DctCfg {
  static constexpr int TPF = LB / 8;
  static constexpr int F = (TPF >= 256) ? 1 : 256 / TPF;
  static constexpr int CC = (8192 / LB > 16) ? 16 : 8192 / LB;
  static size_t smem_x() { return (size_t)(LB + F * (LB + LB / 8)) * sizeof(float2); }
  static size_t smem_s() { return (size_t)(LB + sbuf_elems_s(LB, CC)) * sizeof(float2); }
};
template <int LB> static cudaError_t cfg_dct() {
  cudaError_t e = cudaFuncSetAttribute(k_dct_x<LB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)DctCfg<LB>::smem_x());
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(k_dct_x2<LB, DctCfg<LB>::CC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)DctCfg<LB>::smem_s());
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(k_dct_s<LB, DctCfg<LB>::CC>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              (int)DctCfg<LB>::smem_s());
}
cudaError_t dct_fast_configure(int LB) {
  switch (LB) {
    case 64: return cfg_dct<64>();
    case 128: return cfg_dct<128>();
    case 256: return cfg_dct<256>();
    case 512: return cfg_dct<512>();
    case 1024: return cfg_dct<1024>();
    case 2048: return cfg_dct<2048>();
    case 4096: return cfg_dct<4096>();
  }
  return cudaSuccess;
}
template <int LB>
static void run_dct_x(float *data, int n, long long nrows, const float2 *T, const float2 *C, const float2 *H, cudaStream_t st) {
  constexpr int F = DctCfg<LB>::F;
  const long long npairs = (nrows + 1) / 2;
  if (LB >= 2048) {
    constexpr int CC = DctCfg<LB>::CC;
    k_dct_x2<LB, CC><<<(unsigned)((npairs + CC - 1) / CC), CC * LB / 8, DctCfg<LB>::smem_s(), st>>>(data, n, nrows, T, C, H);
    return;
  }
  k_dct_x<LB><<<(unsigned)((npairs + F - 1) / F), F * (LB / 8), DctCfg<LB>::smem_x(), st>>>(data, n, nrows, T, C, H);
}
template <int LB>
static void run_dct_s(float *data, int n, long long stride, long long ostride, int ncolc, int nother, const float2 *T,
                      const float2 *C, const float2 *H, cudaStream_t st) {
  constexpr int CC = DctCfg<LB>::CC;
  dim3 grid((ncolc + CC - 1) / CC, nother);
  k_dct_s<LB, CC><<<grid, CC * LB / 8, DctCfg<LB>::smem_s(), st>>>(data, n, stride, ostride, ncolc, T, C, H);
}
#define DCT_SWITCH(CALL)                   \
  switch (LB) {                            \
    case 64: CALL(64); break;              \
    case 128: CALL(128); break;            \
    case 256: CALL(256); break;            \
    case 512: CALL(512); break;            \
    case 1024: CALL(1024); break;          \
    case 2048: CALL(2048); break;          \
    case 4096: CALL(4096); break;          \
  }
void launch_dct_x(float *data, int n, int LB, long long nrows, const float2 *T, const float2 *C, const float2 *H,
                  cudaStream_t st) {
#define CALLX(L) run_dct_x<L>(data, n, nrows, T, C, H, st)
  DCT_SWITCH(CALLX)
}
void launch_dct_s(float *data, int n, int LB, long long stride, long long ostride, int ncolc, int nother,
                  const float2 *T, const float2 *C, const float2 *H, cudaStream_t st) {
#define CALLS(L) run_dct_s<L>(data, n, stride, ostride, ncolc, nother, T, C, H, st)
  DCT_SWITCH(CALLS)
}
