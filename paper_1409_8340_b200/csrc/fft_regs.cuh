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
#pragma once
#include "tdgl_dev.cuh"

__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 mul_mi(float2 a) { return make_float2(a.y, -a.x); }      // -i a

template <int R> __device__ __forceinline__ void dft(float2 *v);
template <> __device__ __forceinline__ void dft<2>(float2 *v) {
  const float2 a = v[0];
  v[0] = cadd(a, v[1]);
  v[1] = csub(a, v[1]);
}
template <> __device__ __forceinline__ void dft<4>(float2 *v) {
  const float2 a0 = cadd(v[0], v[2]), a1 = csub(v[0], v[2]), a2 = cadd(v[1], v[3]), a3 = mul_mi(csub(v[1], v[3]));
  v[0] = cadd(a0, a2); v[1] = cadd(a1, a3); v[2] = csub(a0, a2); v[3] = csub(a1, a3);
}
template <> __device__ __forceinline__ void dft<8>(float2 *v) {
  float2 e[4] = {v[0], v[2], v[4], v[6]}, o[4] = {v[1], v[3], v[5], v[7]};
  dft<4>(e);
  dft<4>(o);
  const float h = 0.70710678118654752440f;
  const float2 o1 = make_float2(h * (o[1].x + o[1].y), h * (o[1].y - o[1].x));      // o1 exp(-i pi/4)
  const float2 o2 = mul_mi(o[2]);                                                    // o2 (-i)
  const float2 o3 = make_float2(h * (o[3].y - o[3].x), -h * (o[3].x + o[3].y));     // o3 exp(-3 i pi/4)
  v[0] = cadd(e[0], o[0]); v[4] = csub(e[0], o[0]);
  v[1] = cadd(e[1], o1);   v[5] = csub(e[1], o1);
  v[2] = cadd(e[2], o2);   v[6] = csub(e[2], o2);
  v[3] = cadd(e[3], o3);   v[7] = csub(e[3], o3);
}

// shared-memory address of element p of line f.  x pass (one line per 64+ consecutive threads): p + LAY (p >> 4).
// Padding by whole groups of 16 keeps the stride-1 accesses of every stage (16 consecutive p per half-warp)
// conflict free; the strided writes need LAY = 1 after the first stage (p = 8 jj + r) and LAY = 2 after the later
// ones (p = 64 (jj >> 3) + (jj & 7) + 8 r), so each exchange has its own layout (every stage reads all, syncs, writes
// all).  The result of a transform is in the LAY = 2 layout.  [ncu: the former p + (p >> 3) padding made every
// stride-1 read of 16 lanes straddle two pad groups: 37 % of the shared wavefronts of the x pass were conflicts.]
template <int N, bool XPASS, int CC, int LAY = 2> __device__ __forceinline__ int saddr(int f, int p) {
  return (XPASS || CC == 1) ? f * (N + N / 8) + p + LAY * (p >> 4)      // (one column pair per CTA: same situation)
                            : (CC < 8 ? (p + (p >> 3)) * CC + f : p * CC + f);
}
// elements of the shared work buffer of a y/z pass (fewer than 8 columns per CTA: rows padded 9/8 like the x pass,
// otherwise the stride-8 accesses of the radix-8 stages fall into a few banks)
__host__ __device__ constexpr size_t sbuf_elems_s(int n, int cc) { return (size_t)(cc < 8 ? n + n / 8 : n) * cc; }

// Twiddles in shared memory, one compact table per (stage, r):  ct[tw_off(NS) + (r-1) NS + k] = exp(-2 pi i r k/(NS R)),
// k < NS.  Lanes with consecutive k read consecutive addresses (the plain table tw[r k N/(NS R)] put the even
// multiples of a stage into a few banks: ncu showed half of all shared wavefronts of the x pass were conflicts).
// The values are the entries of the fp64-built global table exp(-2 pi i m/N), so results are unchanged.
__host__ __device__ constexpr int tw_off(int NS) { return NS == 8 ? 0 : NS == 64 ? 56 : NS == 512 ? 504 : 4088; }
__host__ __device__ constexpr int radix_of(int N, int NS) { return (N / NS >= 8) ? 8 : N / NS; }
template <int N> __device__ __forceinline__ void fill_twiddles(float2 *ct, const float2 *__restrict__ twg, int tid, int nth) {
#pragma unroll
  for (int NS = 8; NS < N; NS *= 8) {
    const int R = radix_of(N, NS), step = N / (NS * R);
    for (int e = tid; e < (R - 1) * NS; e += nth) {
      const int r = 1 + e / NS, k = e % NS;
      ct[tw_off(NS) + e] = twg[r * k * step];
    }
  }
}

// One Stockham stage of radix R with Ns = product of the earlier radices; the thread owns 8/R butterflies.
// FIRST: inputs are already in v (read from global); otherwise they are read from shared memory.
template <int N, int R, int NS, bool XPASS, int CC, bool FIRST>
__device__ __forceinline__ void stage(float2 *v, float2 *sm, const float2 *tw, int j, int f) {
  constexpr int NB = N / R, T = 8 / R;
  if (!FIRST) {
#pragma unroll
    for (int t = 0; t < T; ++t) {
      const int jj = j + t * (N / 8);
#pragma unroll
      for (int r = 0; r < R; ++r) v[t * R + r] = sm[saddr<N, XPASS, CC, (NS == 8) ? 1 : 2>(f, jj + r * NB)];
    }
    __syncthreads();
  }
#pragma unroll
  for (int t = 0; t < T; ++t) {
    const int jj = j + t * (N / 8);
    const int k = jj & (NS - 1);
    if (NS > 1) {
#pragma unroll
      for (int r = 1; r < R; ++r) v[t * R + r] = cmul(v[t * R + r], tw[tw_off(NS) + (r - 1) * NS + k]);
    }
    dft<R>(v + t * R);
    const int base = (jj - k) * R + k;
#pragma unroll
    for (int r = 0; r < R; ++r) sm[saddr<N, XPASS, CC, (NS == 1) ? 1 : 2>(f, base + r * NS)] = v[t * R + r];
  }
  __syncthreads();
}

// Complex FFT of length N of the 8 values per thread in v (element j + r N/8 in v[r]); result in shared
// memory in natural order.
template <int N, bool XPASS, int CC, bool FROM_SMEM>
__device__ __forceinline__ void fft_regs(float2 *v, float2 *sm, const float2 *tw, int j, int f) {
  constexpr int L = (N == 64) ? 6 : (N == 128) ? 7 : (N == 256) ? 8 : (N == 512) ? 9 : (N == 1024) ? 10 : (N == 2048) ? 11 : (N == 4096) ? 12 : 13;
  if (FROM_SMEM) {
#pragma unroll
    for (int r = 0; r < 8; ++r) v[r] = sm[saddr<N, XPASS, CC>(f, j + r * (N / 8))];
    __syncthreads();
  }
  stage<N, 8, 1, XPASS, CC, true>(v, sm, tw, j, f);
  stage<N, 8, 8, XPASS, CC, false>(v, sm, tw, j, f);
  if (L == 7) stage<N, 2, 64, XPASS, CC, false>(v, sm, tw, j, f);
  if (L == 8) stage<N, 4, 64, XPASS, CC, false>(v, sm, tw, j, f);
  if (L >= 9) stage<N, 8, 64, XPASS, CC, false>(v, sm, tw, j, f);
  if (L == 10) stage<N, 2, 512, XPASS, CC, false>(v, sm, tw, j, f);
  if (L == 11) stage<N, 4, 512, XPASS, CC, false>(v, sm, tw, j, f);
  if (L >= 12) stage<N, 8, 512, XPASS, CC, false>(v, sm, tw, j, f);
  if (L == 13) stage<N, 2, 4096, XPASS, CC, false>(v, sm, tw, j, f);
}

// Untangle the spectrum of the packed pair into the two Hartley spectra, in place in shared memory.
// The thread handles q = j + s N/8, s = 0..3 (q < N/2) together with its mirror N - q.
template <int N, bool XPASS, int CC>
__device__ __forceinline__ void untangle(float2 *sm, int j, int f) {
#pragma unroll
  for (int s = 0; s < 4; ++s) {
    const int q = j + s * (N / 8);
    if (q == 0) continue;                       // q = 0 and q = N/2 are already (H^a, H^b)
    const int a = saddr<N, XPASS, CC>(f, q), b = saddr<N, XPASS, CC>(f, N - q);
    const float2 u = sm[a], w = sm[b];
    sm[a] = make_float2(0.5f * (u.x + w.x - u.y + w.y), 0.5f * (u.y + w.y + u.x - w.x));
    sm[b] = make_float2(0.5f * (w.x + u.x - w.y + u.y), 0.5f * (w.y + u.y + w.x - u.x));
  }
  __syncthreads();
}

