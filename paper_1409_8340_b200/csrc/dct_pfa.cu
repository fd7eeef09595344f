// Fast DCT-I for open axes whose interval count m = n - 1 is ODD and a product of up to three pairwise coprime small
// factors (n = 1024: m = 1023 = 3 x 11 x 31, the x and y axes of BASELINE config C5; n = 256: 3 x 5 x 17; n = 64: 7 x 9),
// the transform that diagonalises the mirror-ghost (Neumann) 1-D operator of the mu solve (a7).
// Replaces the Bluestein path of dct.cu for these lengths: no chirp, no padding to 4096, no twiddles at all.
//
//   X_q = x_0 + (-1)^q x_m + 2 sum_{p=1}^{m-1} x_p cos(pi p q/m),  q = 0..m   (self-inverse up to 1/(2m))
// is the DFT of length M = 2m of the even extension y.  M = 2 x m with m odd, so by the Good-Thomas (prime factor)
// map the length-2 factor splits off exactly: with
//   e_p = x_{2p} + x_{m-2p},   o_p = x_{2p} - x_{m-2p},   p = 0..h,  h = (m-1)/2
// (both are EVEN sequences of period m: e_{m-p} = e_p), the even outputs are the DFT_m of e and the odd outputs
// the DFT_m of o:
//   X_q = E_{min(q, m-q)} (q even),   X_q = O_{min(q', m-q')}, q' = q mod m (q odd),
//   E_k = e_0 + 2 sum_{p=1}^{h} e_p cos(2 pi p k/m),   k = 0..h      -- a "symmetric DFT" on h + 1 values.
// The symmetric DFT_m is done by the prime-factor algorithm on m = R0 R1 R2: the index p is the CRT image of a
// triple (i0, i1, i2), the DFT is a 3-D DFT of sizes R0 x R1 x R2 without twiddle factors, and the evenness
// T(-i0,-i1,-i2) = T(i0,i1,i2) survives every stage, so each stage only transforms ONE line of every pair of
// mirror-image lines: ((m/R) + 1)/2 small DFTs of length R instead of m/R.  Values live in an array of h + 1 unique
// entries indexed by min(l, m - l), l = CRT(i0, i1, i2); which entries a small DFT reads and writes is precomputed on
// the host (build_tables) -- the entries a butterfly writes are exactly the ones it read, so every stage is in place.
// Two real lines ride in the real and imaginary part (all coefficients are real), so nothing is untangled.
// The small DFTs of odd length R use the pairing a_j = v_j + v_{R-j}, b_j = v_j - v_{R-j}:
//   V_k = v_0 + sum_j a_j cos(2 pi j k/R) - i sum_j b_j sin(2 pi j k/R),  V_{R-k} = conj-partner: (R-1)^2 real FMAs.
// Work per line of 1024 points: 2 x (17 x 900 + 47 x 100 + 171 x 4) = 41 k FMAs (Bluestein: two 4096-point FFTs per
// line pair, about 250 k flops per line and six times the shared-memory traffic).
#include <mutex>
#include "tdgl_dev.cuh"
#include <vector>

namespace {

// (cos, cos, sin, sin)(2 pi t/R), t = 0..R-1, for the supported radices, packed: offset of radix R below.  The pairs feed
// the packed fp32x2 FMA of sm_100 (FFMA2: one instruction for the real and the imaginary part = the two lines).
__constant__ float4 c_trig[96];
__host__ __device__ constexpr int trig_off(int R) {
  return R == 3 ? 0 : R == 5 ? 3 : R == 7 ? 8 : R == 9 ? 15 : R == 11 ? 24 : R == 17 ? 35 : R == 31 ? 52 : 83;
}
const int kRadices[] = {3, 5, 7, 9, 11, 17, 31};

typedef unsigned long long u64;
__device__ __forceinline__ u64 pk(float2 a) { u64 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a.x), "f"(a.y)); return r; }
__device__ __forceinline__ float2 upk(u64 a) { float2 r; asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(a)); return r; }
__device__ __forceinline__ float2 add2(float2 a, float2 b) {
  u64 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk(a)), "l"(pk(b))); return upk(r);
}
__device__ __forceinline__ float2 sub2(float2 a, float2 b) {
  u64 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk(a)), "l"(pk(b))); return upk(r);
}
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) {       // a * b + c, component-wise
  u64 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(pk(a)), "l"(pk(b)), "l"(pk(c))); return upk(r);
}

// DFT of odd length R of v[0..R-1] (forward, e^{-2 pi i jk/R}); output k is handed to emit(k, value).  v is destroyed.
//   a_j = v_j + v_{R-j},  b'_j = -i (v_j - v_{R-j});   V_k = v_0 + sum_j a_j cos_jk + sum_j b'_j sin_jk,  V_{R-k}: minus.
template <int R, class Emit> __device__ __forceinline__ void dft_odd(float2 (&v)[R], Emit emit) {
  constexpr int H = (R - 1) / 2;
  float2 s0 = v[0];
#pragma unroll
  for (int j = 1; j <= H; ++j) {
    const float2 a = add2(v[j], v[R - j]);
    const float2 b = make_float2(v[j].y - v[R - j].y, v[R - j].x - v[j].x);      // -i (v_j - v_{R-j})
    v[j] = a; v[R - j] = b;
    s0 = add2(s0, a);
  }
  emit(0, s0);
#pragma unroll
  for (int k = 1; k <= H; ++k) {
    float2 c = v[0], s = make_float2(0.f, 0.f);
#pragma unroll
    for (int j = 1; j <= H; ++j) {
      const float4 cs = c_trig[trig_off(R) + (j * k) % R];
      c = fma2(v[j], make_float2(cs.x, cs.y), c);
      s = fma2(v[R - j], make_float2(cs.z, cs.w), s);
    }
    emit(k, add2(c, s));
    emit(R - k, sub2(c, s));
  }
}

template <int R0, int R1, int R2> struct Plan {
  static constexpr int M = R0 * R1 * R2, H = (M - 1) / 2, N = M + 1;
  static constexpr int NB0 = (M / R0 + 1) / 2, NB1 = (M / R1 + 1) / 2, NB2 = (M / R2 + 1) / 2;
  // table layout (unsigned short), per stage s: in_e, in_o, out_e, out_o, each NB_s x R_s entries (build_tables)
  static constexpr int S0 = 0, S1 = 4 * NB0 * R0, S2 = S1 + 4 * NB1 * R1, T_TOTAL = S2 + 4 * NB2 * R2;
};
constexpr unsigned short SKIP = 0xFFFFu;

// The work array of a line pair has m + 1 slots: unique value e_id sits in slot 2 id, o_id in slot m - 2 id -- which is
// where x_{2 id} and x_{m - 2 id} sit, so the e/o split is in place too.  Shared memory holds [slot][f] (f = line pair
// within the CTA, LP of them); the tables hold the element index of (slot, f = 0) with the x pass's swizzle already
// applied (below), so that the address of a thread is  entry ^ f.

// one in-place stage in shared memory: work items (butterfly, sd) strided over the NW workers of the CTA;
// `st` = tables of this stage (in_e, in_o, out_e, out_o)
template <int R>
__device__ __forceinline__ void stage_smem(float2 *sm, const unsigned short *__restrict__ st, int nb, int f, int w, int NW) {
  for (int it = w; it < 2 * nb; it += NW) {
    const int b = it >> 1, sd = it & 1;
    const unsigned short *tin = st + sd * nb * R + b * R, *tout = tin + 2 * nb * R;
    float2 v[R];
#pragma unroll
    for (int r = 0; r < R; ++r) v[r] = sm[__ldg(tin + r) ^ f];
    dft_odd<R>(v, [&](int k, float2 val) {
      const unsigned short a = __ldg(tout + k);
      if (a != SKIP) sm[a ^ f] = val;
    });
  }
}

// ---- y / z pass: the real array is read as float2 columns (columns 2c, 2c+1 = re, im); LP column pairs per CTA.
// First stage straight from global memory (fused with the e/o split), last stage straight to global memory.
template <int R0, int R1, int R2, int LP, int NW>
__global__ void __launch_bounds__(LP *NW) k_dct_pfa_s(float *__restrict__ data, long long stride, long long ostride, int ncolc,
                                                      const unsigned short *__restrict__ tab) {
  using P = Plan<R0, R1, R2>;
  constexpr int m = P::M;
  extern __shared__ float4 smem4[];
  float2 *sm = reinterpret_cast<float2 *>(smem4);                    // [slot][f]
  const int tid = threadIdx.x, f = tid % LP, w = tid / LP;
  const int col = blockIdx.x * LP + f;
  const bool valid = col < ncolc;
  float *base = data + (long long)blockIdx.y * ostride + 2 * (long long)(valid ? col : 0);
  // stage 0: R0-point DFTs of e and o, inputs from global memory (table in_e of stage 0 holds the ids).  All global
  // loads of the thread (IT0 butterflies x R0 x 2 rows) are issued before the first use: ncu showed half of the kernel's
  // stall samples on the first add after the loads when each butterfly waited for its own six.
  constexpr int IT0 = (P::NB0 + NW - 1) / NW;
  float2 ve[IT0][R0], vo[IT0][R0];
#pragma unroll
  for (int i = 0; i < IT0; ++i) {
    const unsigned short *t0 = tab + P::S0 + min(w + i * NW, P::NB0 - 1) * R0;     // clamped: the tail re-reads, never stores
#pragma unroll
    for (int r = 0; r < R0; ++r) {
      const int id = __ldg(t0 + r);
      ve[i][r] = __ldcs(reinterpret_cast<const float2 *>(base + (long long)(2 * id) * stride));
      vo[i][r] = __ldcs(reinterpret_cast<const float2 *>(base + (long long)(m - 2 * id) * stride));
    }
  }
#pragma unroll
  for (int i = 0; i < IT0; ++i) {
    const int b = w + i * NW;
    if (b < P::NB0) {
      const unsigned short *t0 = tab + P::S0 + b * R0;
#pragma unroll
      for (int r = 0; r < R0; ++r) {
        const float2 xa = ve[i][r], xb = vo[i][r];
        ve[i][r] = add2(xa, xb);
        vo[i][r] = sub2(xa, xb);
      }
      dft_odd<R0>(ve[i], [&](int k, float2 val) {
        const unsigned short a = __ldg(t0 + 2 * P::NB0 * R0 + k);
        if (a != SKIP) sm[a ^ f] = val;
      });
      dft_odd<R0>(vo[i], [&](int k, float2 val) {
        const unsigned short a = __ldg(t0 + 3 * P::NB0 * R0 + k);
        if (a != SKIP) sm[a ^ f] = val;
      });
    }
  }
  __syncthreads();
  if (R1 > 1) {
    stage_smem<R1>(sm, tab + P::S1, P::NB1, f, w, NW);
    __syncthreads();
  }
  // last stage: to global memory (tables out_e / out_o of the last stage hold the output index q)
  for (int it = w; it < 2 * P::NB2; it += NW) {
    const int b = it >> 1, sd = it & 1;
    const unsigned short *tin = tab + P::S2 + sd * P::NB2 * R2 + b * R2, *tout = tin + 2 * P::NB2 * R2;
    float2 v[R2];
#pragma unroll
    for (int r = 0; r < R2; ++r) v[r] = sm[__ldg(tin + r) ^ f];
    dft_odd<R2>(v, [&](int k, float2 val) {
      const unsigned short q = __ldg(tout + k);
      if (q != SKIP && valid) *reinterpret_cast<float2 *>(base + (long long)q * stride) = val;
    });
  }
}

// ---- x pass: contiguous rows, LP row pairs per CTA (row 2f -> re, row 2f+1 -> im).  Rows are loaded and stored with
// the lanes along x (coalesced); the stages run with the lanes along f.  Layout [slot][f ^ g(slot)],
// g(s) = (s ^ (s >> 4)) & (LP - 1): a permutation of the f for every slot (stages: conflict free), and distinct
// for LP consecutive x on load as well as for the slot pattern 4t / m - 2 - 4t of LP consecutive outputs.
template <int R0, int R1, int R2, int LP, int NW>
__global__ void __launch_bounds__(LP *NW, (LP * (R0 * R1 * R2 + 1) * 8 <= 100 * 1024) ? 2 : 1)
k_dct_pfa_x(float *__restrict__ data, long long nrows, const unsigned short *__restrict__ tab) {
  using P = Plan<R0, R1, R2>;
  constexpr int m = P::M, n = P::N, NT = LP * NW;
  extern __shared__ float4 smem4[];
  float2 *sm = reinterpret_cast<float2 *>(smem4);
  float *smf = reinterpret_cast<float *>(smem4);
  const int tid = threadIdx.x, f = tid % LP, w = tid / LP;
  const long long row0 = 2ll * blockIdx.x * LP;
  auto sw = [&](int slot, int ff) { return slot * LP + (ff ^ ((slot ^ (slot >> 4)) & (LP - 1))); };
  // load, 16 bytes per access and coalesced (a warp reads 512 contiguous bytes of one row): x_{p..p+3} of row rr ->
  // component rr & 1 of the entries (slot p + j, f = rr >> 1); four loads in flight per thread.  [Tried and dropped:
  // 4-byte cp.async copies straight to the swizzled slots (2.27 instead of 2.05 ms per pass on 1024 x 1024 x 512), and a
  // 16-rows-per-warp mapping that makes the scalar stores conflict free (more DRAM sectors: 2.66 ms).]
  constexpr int NV = n / 4, NE = 2 * LP * NV;
  for (int e0 = tid; e0 < NE; e0 += 4 * NT) {
    float4 v[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int e = e0 + u * NT, rr = e / NV, p = 4 * (e - rr * NV);
      const long long row = row0 + rr;
      v[u] = (e < NE && row < nrows) ? __ldcs(reinterpret_cast<const float4 *>(data + row * n + p)) : make_float4(0.f, 0.f, 0.f, 0.f);
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int e = e0 + u * NT, rr = e / NV, p = 4 * (e - rr * NV);
      if (e < NE) {
        const int ff = rr >> 1, c = rr & 1;
        smf[2 * sw(p, ff) + c] = v[u].x;
        smf[2 * sw(p + 1, ff) + c] = v[u].y;
        smf[2 * sw(p + 2, ff) + c] = v[u].z;
        smf[2 * sw(p + 3, ff) + c] = v[u].w;
      }
    }
  }
  __syncthreads();
  // stage 0 fused with the e/o split, in place: (x_{2 id}, x_{m - 2 id}) -> (e_id, o_id) -> two R0-point DFTs -> the same slots
  for (int b = w; b < P::NB0; b += NW) {
    const unsigned short *t0 = tab + P::S0 + b * R0;
    float2 ve[R0], vo[R0];
#pragma unroll
    for (int r = 0; r < R0; ++r) {
      const float2 xa = sm[__ldg(t0 + r) ^ f], xb = sm[__ldg(t0 + P::NB0 * R0 + r) ^ f];
      ve[r] = add2(xa, xb);
      vo[r] = sub2(xa, xb);
    }
    dft_odd<R0>(ve, [&](int k, float2 val) {
      const unsigned short a = __ldg(t0 + 2 * P::NB0 * R0 + k);
      if (a != SKIP) sm[a ^ f] = val;
    });
    dft_odd<R0>(vo, [&](int k, float2 val) {
      const unsigned short a = __ldg(t0 + 3 * P::NB0 * R0 + k);
      if (a != SKIP) sm[a ^ f] = val;
    });
  }
  __syncthreads();
  if (R1 > 1) {
    stage_smem<R1>(sm, tab + P::S1, P::NB1, f, w, NW);
    __syncthreads();
  }
  stage_smem<R2>(sm, tab + P::S2, P::NB2, f, w, NW);
  __syncthreads();
  // store, 16 bytes per access: X_q = E_{min(q, m-q)} (q even) / O_{min(q', m-q')}, q' = q mod m (q odd)
  auto outslot = [&](int q) {
    const int qq = (q == m) ? 0 : q, id = min(qq, m - qq);
    return (q & 1) ? m - 2 * id : 2 * id;
  };
  for (int e = tid; e < NE; e += NT) {
    const int rr = e / NV, q = 4 * (e - rr * NV);
    const long long row = row0 + rr;
    const int ff = rr >> 1, c = rr & 1;
    float4 v;
    v.x = smf[2 * sw(outslot(q), ff) + c];
    v.y = smf[2 * sw(outslot(q + 1), ff) + c];
    v.z = smf[2 * sw(outslot(q + 2), ff) + c];
    v.w = smf[2 * sw(outslot(q + 3), ff) + c];
    if (row < nrows) __stcs(reinterpret_cast<float4 *>(data + row * n + q), v);
  }
}

// ---- host: the supported lengths, the index tables ----------------------------------------------------------------
struct PlanDesc { int n, R[3]; };
const PlanDesc kPlans[] = {{1024, {3, 11, 31}}, {256, {3, 5, 17}}, {64, {7, 1, 9}}};
constexpr int NPLANS = 3;

long long inv_mod(long long a, long long n) {                 // a^{-1} mod n (n small, gcd = 1)
  a %= n;
  for (long long x = 1; x < n; ++x)
    if ((a * x) % n == 1) return x;
  return 1;
}

// Index tables of the symmetric prime-factor DFT_m (see the header comment).  For stage s (radix R_s) the butterflies are
// the classes {t, -t} of the other two indices; input r of a butterfly is the unique entry min(l, m - l) of the triple
// with i_s = r; output k goes to the triple with i_s = (m/R_s) k mod R_s (CRT map on both sides: the small DFT's root is
// w_R^{(m/R)^{-1}}), and the self-mirrored butterfly (other indices 0) writes each unique entry once.
// `xpass`: tables for k_dct_pfa_x (every entry a swizzled shared-memory element index); otherwise for k_dct_pfa_s
// (stage 0 reads global memory: in_e = id; the last stage writes global memory: out = output index q).
std::vector<unsigned short> build_tables(const int R[3], int LP, bool xpass) {
  const int m = R[0] * R[1] * R[2], h = (m - 1) / 2;
  long long e[3];
  for (int j = 0; j < 3; ++j) { const long long Nj = m / R[j]; e[j] = (Nj * inv_mod(Nj, R[j])) % m; }
  auto crt = [&](const int t[3]) { return (int)((t[0] * e[0] + t[1] * e[1] + t[2] * e[2]) % m); };
  auto uid = [&](int l) { return l <= h ? l : m - l; };
  auto phys = [&](int id, int sd) {                       // element index of (slot, f = 0)
    const int slot = sd ? m - 2 * id : 2 * id;
    return (unsigned short)(slot * LP + (xpass ? ((slot ^ (slot >> 4)) & (LP - 1)) : 0));
  };
  auto qout = [&](int id, int sd) { return (unsigned short)(((id & 1) == sd) ? id : m - id); };   // X_q = E_id / O_id
  std::vector<unsigned short> tab;
  for (int s = 0; s < 3; ++s) {
    const int a = (s + 1) % 3, b = (s + 2) % 3, Rs = R[s];
    std::vector<int> tin, tout;                           // unique ids; -1 = not written
    std::vector<char> seen((size_t)R[a] * R[b], 0);
    for (int ia = 0; ia < R[a]; ++ia)
      for (int ib = 0; ib < R[b]; ++ib) {
        const int na = (R[a] - ia) % R[a], nb = (R[b] - ib) % R[b];
        if (seen[(size_t)ia * R[b] + ib] || seen[(size_t)na * R[b] + nb]) continue;
        seen[(size_t)ia * R[b] + ib] = 1;
        const bool self = ia == 0 && ib == 0;
        const int perm = (m / Rs) % Rs;
        for (int r = 0; r < Rs; ++r) {
          int t[3];
          t[a] = ia; t[b] = ib; t[s] = r;
          tin.push_back(uid(crt(t)));
          t[s] = (perm * r) % Rs;
          const int l = crt(t);
          tout.push_back((!self || l <= h) ? uid(l) : -1);
        }
      }
    const bool first = s == 0, last = s == 2;
    for (int sd = 0; sd < 2; ++sd)
      for (int id : tin) tab.push_back((first && !xpass) ? (unsigned short)id : phys(id, sd));
    for (int sd = 0; sd < 2; ++sd)
      for (int id : tout) tab.push_back(id < 0 ? SKIP : ((last && !xpass) ? qout(id, sd) : phys(id, sd)));
  }
  return tab;
}

template <int R0, int R1, int R2, int LP, int NW> struct Launch {
  using P = Plan<R0, R1, R2>;
  static constexpr size_t SMEM = (size_t)(P::M + 1) * LP * sizeof(float2);
  static cudaError_t configure() {
    cudaError_t e = cudaFuncSetAttribute(k_dct_pfa_s<R0, R1, R2, LP, NW>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_dct_pfa_x<R0, R1, R2, LP, NW>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM);
  }
  static void run_x(float *data, long long nrows, const unsigned short *tab, cudaStream_t st) {
    const long long npairs = (nrows + 1) / 2;
    k_dct_pfa_x<R0, R1, R2, LP, NW><<<(unsigned)((npairs + LP - 1) / LP), LP * NW, SMEM, st>>>(data, nrows, tab);
  }
  static void run_s(float *data, long long stride, long long ostride, int ncolc, int nother, const unsigned short *tab, cudaStream_t st) {
    dim3 grid((ncolc + LP - 1) / LP, nother);
    k_dct_pfa_s<R0, R1, R2, LP, NW><<<grid, LP * NW, SMEM, st>>>(data, stride, ostride, ncolc, tab);
  }
};
using L1024 = Launch<3, 11, 31, 8, 36>;
using L256 = Launch<3, 5, 17, 16, 16>;
using L64 = Launch<7, 1, 9, 16, 8>;

}  // namespace

// index of the plan for an open axis of n points, -1 if this length has none
int dct_pfa_kind(int n) {
  for (int k = 0; k < NPLANS; ++k)
    if (kPlans[k].n == n) return k;
  return -1;
}
size_t dct_pfa_table_entries(int kind) {
  if (kind < 0 || kind >= NPLANS) return 0;
  const int *R = kPlans[kind].R;
  const int m = R[0] * R[1] * R[2];
  size_t t = 0;
  for (int s = 0; s < 3; ++s) t += 4 * (size_t)((m / R[s] + 1) / 2) * R[s];
  return t;
}
static int plan_lp(int kind) { return kind == 0 ? 8 : 16; }           // = the LP of the Launch<> instantiations above
void dct_pfa_build_table(int kind, bool xpass, unsigned short *host_out) {
  const std::vector<unsigned short> t = build_tables(kPlans[kind].R, plan_lp(kind), xpass);
  for (size_t i = 0; i < t.size(); ++i) host_out[i] = t[i];
}
// __constant__ memory and function attributes belong to a DEVICE, not to the process: the trig table is uploaded once per
// device (the current one; tdgl_create runs with the caller's device current), and the attributes are set on every call.
cudaError_t dct_pfa_configure(int kind) {
  static std::mutex lock;
  static unsigned long long trig_done = 0;                    // bit d: cos / sin of every supported radix (fp64 -> fp32) are on device d
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  {
    std::lock_guard<std::mutex> guard(lock);
    if (dev < 0 || dev >= 64 || !((trig_done >> dev) & 1ull)) {
      float4 h[96];
      for (int i = 0; i < 96; ++i) h[i] = make_float4(0.f, 0.f, 0.f, 0.f);
      for (int R : kRadices)
        for (int t = 0; t < R; ++t) {
          const double ang = 2.0 * 3.14159265358979323846 * t / R;
          h[trig_off(R) + t] = make_float4((float)cos(ang), (float)cos(ang), (float)sin(ang), (float)sin(ang));
        }
      e = cudaMemcpyToSymbol(c_trig, h, sizeof(h));
      if (e != cudaSuccess) return e;
      if (dev >= 0 && dev < 64) trig_done |= 1ull << dev;
    }
  }
  switch (kind) {
    case 0: return L1024::configure();
    case 1: return L256::configure();
    case 2: return L64::configure();
  }
  return cudaSuccess;
}
void launch_dct_pfa_x(int kind, float *data, long long nrows, const unsigned short *tab, cudaStream_t st) {
  switch (kind) {
    case 0: L1024::run_x(data, nrows, tab, st); break;
    case 1: L256::run_x(data, nrows, tab, st); break;
    case 2: L64::run_x(data, nrows, tab, st); break;
  }
}
void launch_dct_pfa_s(int kind, float *data, long long stride, long long ostride, int ncolc, int nother, const unsigned short *tab,
                      cudaStream_t st) {
  switch (kind) {
    case 0: L1024::run_s(data, stride, ostride, ncolc, nother, tab, st); break;
    case 1: L256::run_s(data, stride, ostride, ncolc, nother, tab, st); break;
    case 2: L64::run_s(data, stride, ostride, ncolc, nother, tab, st); break;
  }
}
