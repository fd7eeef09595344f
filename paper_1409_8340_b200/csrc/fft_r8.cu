// Hartley transform along x for n = 512 = 8 x 8 x 8 (the x and y extent of the headline grid), persistent version.
//
// ncu on the generic register FFT (k_dht_x_fast<512>) showed the L1/shared pipe 90 % busy: 12.5 M of 34 M shared
// wavefronts were bank conflicts of the stride-1 reads under the 9/8 padding, 14 twiddle loads per thread came from
// shared memory, and the untangle pass re-read and re-wrote the whole spectrum.  This kernel removes all three:
//  * index algebra n = 64 n1 + 8 n2 + n3, q = k1 + 8 k2 + 64 k3 (three radix-8 steps, every thread 8 values);
//    each of the three exchanges has its OWN shared layout, chosen so that the write and the read of that
//    exchange are both conflict free for 8-byte accesses (16 lanes -> 16 distinct 8-byte banks):
//       exchange 1: [k1][n2][n3]  -> k1*72 + n2*8 + n3        (written by (n2,n3), read by (k1,n3))
//       exchange 2: [k1][k2][n3]  -> k1*72 + k2*9 + n3        (written by (k1,n3), read by (k1,k2))
//       exchange 3: natural q     -> 10*(q>>3) + (q&7)        (written by (k1,k2), read as 16-byte vectors)
//  * the 15 twiddles a thread needs are loop-invariant registers (the CTA is persistent over row pairs);
//  * the Hartley untangle H_q from (Z_q, Z_{n-q}) is folded into the final read: a thread reads its 8 consecutive
//    q and the mirrored group as 16-byte vectors and stores 32 contiguous bytes per row (fully coalesced).
// The next tile's 16 global loads are in flight while the current tile is transformed.
#include "fft_regs.cuh"

namespace {
constexpr int N = 512, LP = 4, NT = 64 * LP;                  // 4 row pairs per CTA, 64 threads each
constexpr int B1 = 576, B3 = 640;                             // padded buffer lengths (float2) per row pair
constexpr size_t SMEM = (size_t)LP * (B1 + B1 + B3) * sizeof(float2);

__global__ void __launch_bounds__(NT, 2) k_dht_x_512(float *__restrict__ data, long long nrows, long long ntiles,
                                                     const float2 *__restrict__ twg) {
  extern __shared__ float4 smem4[];
  float2 *s1 = reinterpret_cast<float2 *>(smem4), *s2 = s1 + LP * B1, *s3 = s2 + LP * B1;
  const int tid = threadIdx.x, f = tid >> 6, j = tid & 63, hi = j >> 3, lo = j & 7;
  float2 *b1 = s1 + f * B1, *b2 = s2 + f * B1, *b3 = s3 + f * B3;
  // twiddles exp(-2 pi i m/512): step 1 output k1 of thread (n2,n3)=(hi,lo): w_64^{n2 k1}; step 2 output k2 of
  // thread (k1,n3)=(hi,lo): w_512^{n3 (k1 + 8 k2)}
  float2 t1[8], t2[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    t1[k] = twg[(8 * hi * k) & (N - 1)];
    t2[k] = twg[(lo * (hi + 8 * k)) & (N - 1)];
  }
  auto rows_of = [&](long long tile, float *&A, float *&Bq, bool &va, bool &vb) {
    const long long ra = 2 * (tile * LP + f);
    va = ra < nrows; vb = ra + 1 < nrows;
    A = data + ra * N; Bq = A + N;
  };
  float2 nxt[8];
  auto load = [&](long long tile) {
    float *A, *Bq; bool va, vb;
    rows_of(tile, A, Bq, va, vb);
#pragma unroll
    for (int r = 0; r < 8; ++r) nxt[r] = make_float2(va ? __ldcs(A + 64 * r + j) : 0.f, vb ? __ldcs(Bq + 64 * r + j) : 0.f);
  };
  long long tile = blockIdx.x;
  if (tile < ntiles) load(tile);
  for (; tile < ntiles; tile += gridDim.x) {
    float2 v[8];
#pragma unroll
    for (int r = 0; r < 8; ++r) v[r] = nxt[r];
    if (tile + gridDim.x < ntiles) load(tile + gridDim.x);
    // step 1: DFT over n1, twiddle, exchange 1
    dft<8>(v);
#pragma unroll
    for (int k = 1; k < 8; ++k) v[k] = cmul(v[k], t1[k]);
#pragma unroll
    for (int k = 0; k < 8; ++k) b1[k * 72 + j] = v[k];
    __syncthreads();
#pragma unroll
    for (int n2 = 0; n2 < 8; ++n2) v[n2] = b1[hi * 72 + n2 * 8 + lo];
    // step 2: DFT over n2, twiddle, exchange 2
    dft<8>(v);
#pragma unroll
    for (int k = 0; k < 8; ++k) v[k] = cmul(v[k], t2[k]);
#pragma unroll
    for (int k = 0; k < 8; ++k) b2[hi * 72 + k * 9 + lo] = v[k];
    __syncthreads();
#pragma unroll
    for (int n3 = 0; n3 < 8; ++n3) v[n3] = b2[hi * 72 + lo * 9 + n3];
    // step 3: DFT over n3 -> Z[hi + 8 lo + 64 k3], exchange 3 in natural order
    dft<8>(v);
#pragma unroll
    for (int k = 0; k < 8; ++k) b3[10 * (lo + 8 * k) + hi] = v[k];
    __syncthreads();
    // untangle folded into the read: q = 8 j + r and its mirror n - q
    float2 z[8], m[8];
    {
      const float4 *g = reinterpret_cast<const float4 *>(b3 + 10 * j), *gm = reinterpret_cast<const float4 *>(b3 + 10 * (63 - j));
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        const float4 a = g[r], c = gm[r];
        z[2 * r] = make_float2(a.x, a.y); z[2 * r + 1] = make_float2(a.z, a.w);
        m[2 * r] = make_float2(c.x, c.y); m[2 * r + 1] = make_float2(c.z, c.w);
      }
    }
    const float2 m0 = b3[10 * ((64 - j) & 63)];             // Z[(n - 8 j) mod n]
    float ha[8], hb[8];
#pragma unroll
    for (int r = 0; r < 8; ++r) {
      const float2 u = z[r], w = (r == 0) ? m0 : m[8 - r];
      ha[r] = 0.5f * (u.x + w.x - u.y + w.y);
      hb[r] = 0.5f * (u.y + w.y + u.x - w.x);
    }
    float *A, *Bq; bool va, vb;
    rows_of(tile, A, Bq, va, vb);
    if (va) {
      reinterpret_cast<float4 *>(A + 8 * j)[0] = make_float4(ha[0], ha[1], ha[2], ha[3]);
      reinterpret_cast<float4 *>(A + 8 * j)[1] = make_float4(ha[4], ha[5], ha[6], ha[7]);
    }
    if (vb) {
      reinterpret_cast<float4 *>(Bq + 8 * j)[0] = make_float4(hb[0], hb[1], hb[2], hb[3]);
      reinterpret_cast<float4 *>(Bq + 8 * j)[1] = make_float4(hb[4], hb[5], hb[6], hb[7]);
    }
  }
}
}  // namespace

cudaError_t dht_x_512_configure() {
  return cudaFuncSetAttribute(k_dht_x_512, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM);
}
void launch_dht_x_512(float *data, long long nrows, const float2 *tw, cudaStream_t st) {
  const long long npairs = (nrows + 1) / 2, ntiles = (npairs + LP - 1) / LP;
  const long long grid = ntiles < tdgl_sm_count() * 2 ? ntiles : tdgl_sm_count() * 2;
  k_dht_x_512<<<(unsigned)grid, NT, SMEM, st>>>(data, nrows, ntiles, tw);
}
