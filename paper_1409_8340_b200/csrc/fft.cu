// Register-blocked Hartley transforms for power-of-two periodic axes (n = 64 .. 1024), the fast path of the
// Poisson solver (a7).  Two real lines are packed as one complex line (re, im); a thread holds 8 complex
// values, does radix-8 (or a final radix-4 / radix-2) Stockham butterflies in registers and exchanges
// through ONE shared buffer (read all - barrier - write all - barrier).  The first stage reads straight
// from global memory, the result is untangled into the two Hartley spectra
//   H^a_q = (Re Z_q + Re Z_{n-q} - Im Z_q + Im Z_{n-q})/2,   H^b_q = (Im Z_q + Im Z_{n-q} + Re Z_q - Re Z_{n-q})/2
// in shared memory and stored with coalesced accesses.
//   x pass : lines are contiguous rows; layout [line][p + p/8] (pitch 9/8: conflict-free for every stage),
//            threads fastest along the butterfly index.
//   y/z pass: the real array is read as float2 columns; layout [p][column], threads fastest along columns.
#include "fft_regs.cuh"

// ---- x pass: contiguous rows, two rows per complex FFT, F = 2048/N pairs per CTA (256 threads) ----------
template <int N>
__global__ void __launch_bounds__((N > 2048) ? N / 8 : 256) k_dht_x_fast(float *__restrict__ data, long long nrows,
                                                                          const float2 *__restrict__ twg) {
  constexpr int F = (N >= 2048) ? 1 : 2048 / N, TPF = N / 8, NT = F * TPF;
  extern __shared__ float4 smem4[];
  float2 *tw = reinterpret_cast<float2 *>(smem4);
  float2 *sm = tw + N;
  const int tid = threadIdx.x;
  fill_twiddles<N>(tw, twg, tid, NT);
  const int j = tid % TPF, f = tid / TPF;
  const long long ra = 2 * ((long long)blockIdx.x * F + f), rb = ra + 1;
  const bool va = ra < nrows, vb = rb < nrows;
  float *A = data + ra * N, *B = data + rb * N;
  float2 v[8];
#pragma unroll
  for (int r = 0; r < 8; ++r) {
    const int p = j + r * TPF;
    v[r] = make_float2(va ? A[p] : 0.f, vb ? B[p] : 0.f);
  }
  fft_regs<N, true, 1, false>(v, sm, tw, j, f);
  // H^a_q, H^b_q from Z_q and Z_{N-q} on the way out of shared memory (no separate untangling pass)
#pragma unroll
  for (int r = 0; r < 8; ++r) {
    const int p = j + r * TPF;
    const float2 u = sm[saddr<N, true, 1>(f, p)], w = sm[saddr<N, true, 1>(f, (N - p) & (N - 1))];
    if (va) A[p] = 0.5f * (u.x + w.x - u.y + w.y);
    if (vb) B[p] = 0.5f * (u.y + w.y + u.x - w.x);
  }
}

// ---- y / z pass: float2 columns, CC columns per CTA, CC*N/8 threads ---------------------------------
// divide != 0 (periodic z): coefficients are multiplied by scale/(lam_x[i] + lam_y[o] + lam_z[q]) (zero
// mode -> 0, S7) and transformed back inside the kernel.
template <int N, int CC>
__global__ void __launch_bounds__(CC *N / 8) k_dht_s_fast(float *__restrict__ data, long long stride, long long ostride,
                                                          int ncolc, const float2 *__restrict__ twg, int divide,
                                                          float scale, const float *__restrict__ lamx,
                                                          const float *__restrict__ lamy,
                                                          const float *__restrict__ lamz) {
  constexpr int TPF = N / 8, NT = CC * TPF;
  extern __shared__ float4 smem4[];
  float2 *tw = reinterpret_cast<float2 *>(smem4);
  float2 *sm = tw + N;
  const int tid = threadIdx.x;
  fill_twiddles<N>(tw, twg, tid, NT);
  const int f = tid % CC, j = tid / CC;
  const int col = blockIdx.x * CC + f;
  const long long o = blockIdx.y;
  const bool valid = col < ncolc;
  float *base = data + o * ostride + 2 * (long long)(valid ? col : 0);
  float2 v[8];
#pragma unroll
  for (int r = 0; r < 8; ++r) {
    const int p = j + r * TPF;
    v[r] = valid ? *reinterpret_cast<const float2 *>(base + p * stride) : make_float2(0.f, 0.f);
  }
  fft_regs<N, false, CC, false>(v, sm, tw, j, f);
  // The two Hartley spectra of the packed pair, H^a_q and H^b_q (formulas at the top of fft_regs.cuh), are formed from
  // Z_q and Z_{N-q} on the way out of shared memory (no separate untangling pass over the buffer).
  // (one column pair per CTA only: with 8 pairs per CTA the separate pass measured 4 % faster, 141 against 148 us on C4)
  constexpr bool FOLD = CC == 1;
  if (!FOLD) untangle<N, false, CC>(sm, j, f);
  auto hartley = [&](int q) -> float2 {
    const float2 u = sm[saddr<N, false, CC>(f, q)];
    if (!FOLD) return u;
    const float2 w = sm[saddr<N, false, CC>(f, (N - q) & (N - 1))];
    return make_float2(0.5f * (u.x + w.x - u.y + w.y), 0.5f * (u.y + w.y + u.x - w.x));
  };
  if (divide) {
    const float lxa = valid ? lamx[2 * col] : 1.f, lxb = valid ? lamx[2 * col + 1] : 1.f, ly = lamy[o];
#pragma unroll
    for (int r = 0; r < 8; ++r) {
      const int q = j + r * TPF;
      const float lz = lamz[q] + ly;
      const float la = lxa + lz, lb = lxb + lz;
      float2 z = hartley(q);
      z.x = (la != 0.f) ? z.x * (scale / la) : 0.f;
      z.y = (lb != 0.f) ? z.y * (scale / lb) : 0.f;
      v[r] = z;
    }
    __syncthreads();
    fft_regs<N, false, CC, false>(v, sm, tw, j, f);
    if (!FOLD) untangle<N, false, CC>(sm, j, f);
  }
  if (valid) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
      const int p = j + r * TPF;
      *reinterpret_cast<float2 *>(base + p * stride) = hartley(p);
    }
  }
}

// ---- host side ---------------------------------------------------------------------------------------
static size_t smem_x(int n) { const int f = n >= 2048 ? 1 : 2048 / n; return (size_t)(n + f * (n + n / 8)) * sizeof(float2); }
static size_t smem_s(int n, int cc) { return (size_t)(n + sbuf_elems_s(n, cc)) * sizeof(float2); }
// float2 columns per CTA of the strided pass: CC N/8 threads <= 1024
constexpr int cc_of(int n) { return n >= 8192 ? 1 : n >= 4096 ? 2 : n >= 2048 ? 4 : n >= 512 ? 8 : 16; }

bool dht_fast_supported(int n) { return n >= 64 && n <= 8192 && (n & (n - 1)) == 0; }

template <int N> static cudaError_t cfg_n() {
  constexpr int CC = cc_of(N);
  cudaError_t e = cudaFuncSetAttribute(k_dht_x_fast<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_x(N));
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(k_dht_s_fast<N, CC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_s(N, CC));
}
cudaError_t dht_fast_configure(int n) {
  switch (n) {
    case 64: return cfg_n<64>();
    case 128: return cfg_n<128>();
    case 256: return cfg_n<256>();
    case 512: return cfg_n<512>();
    case 1024: return cfg_n<1024>();
    case 2048: return cfg_n<2048>();
    case 4096: return cfg_n<4096>();
    case 8192: return cfg_n<8192>();
  }
  return cudaSuccess;
}

template <int N> static void run_x(float *data, long long nrows, const float2 *tw, cudaStream_t st) {
  constexpr int F = (N >= 2048) ? 1 : 2048 / N;
  const long long npairs = (nrows + 1) / 2;
  k_dht_x_fast<N><<<(unsigned)((npairs + F - 1) / F), F * (N / 8), smem_x(N), st>>>(data, nrows, tw);
}
void launch_dht_x_fast(float *data, int n, long long nrows, const float2 *tw, cudaStream_t st) {
  switch (n) {
    case 64: run_x<64>(data, nrows, tw, st); break;
    case 128: run_x<128>(data, nrows, tw, st); break;
    case 256: run_x<256>(data, nrows, tw, st); break;
    case 512: run_x<512>(data, nrows, tw, st); break;
    case 1024: run_x<1024>(data, nrows, tw, st); break;
    case 2048: run_x<2048>(data, nrows, tw, st); break;
    case 4096: run_x<4096>(data, nrows, tw, st); break;
    case 8192: run_x<8192>(data, nrows, tw, st); break;
  }
}

template <int N>
static void run_s(float *data, long long stride, long long ostride, int ncolc, int nother, const float2 *tw, int divide,
                  float scale, const float *lx, const float *ly, const float *lz, cudaStream_t st) {
  constexpr int CC = cc_of(N);
  dim3 grid((ncolc + CC - 1) / CC, nother);
  k_dht_s_fast<N, CC><<<grid, CC * N / 8, smem_s(N, CC), st>>>(data, stride, ostride, ncolc, tw, divide, scale, lx, ly, lz);
}
void launch_dht_s_fast(float *data, int n, long long stride, long long ostride, int ncolc, int nother, const float2 *tw,
                       int divide, float scale, const float *lx, const float *ly, const float *lz, cudaStream_t st) {
  switch (n) {
    case 64: run_s<64>(data, stride, ostride, ncolc, nother, tw, divide, scale, lx, ly, lz, st); break;
    case 128: run_s<128>(data, stride, ostride, ncolc, nother, tw, divide, scale, lx, ly, lz, st); break;
    case 256: run_s<256>(data, stride, ostride, ncolc, nother, tw, divide, scale, lx, ly, lz, st); break;
    case 512: run_s<512>(data, stride, ostride, ncolc, nother, tw, divide, scale, lx, ly, lz, st); break;
    case 1024: run_s<1024>(data, stride, ostride, ncolc, nother, tw, divide, scale, lx, ly, lz, st); break;
    case 2048: run_s<2048>(data, stride, ostride, ncolc, nother, tw, divide, scale, lx, ly, lz, st); break;
    case 4096: run_s<4096>(data, stride, ostride, ncolc, nother, tw, divide, scale, lx, ly, lz, st); break;
    case 8192: run_s<8192>(data, stride, ostride, ncolc, nother, tw, divide, scale, lx, ly, lz, st); break;
  }
}
