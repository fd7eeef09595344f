// The marching stencil for FILMS (N_z = 1: the paper's 2D workloads; reading S22: no z links):
// Jacobi sweep + max-residual (Eq. 33-34), fused init + first sweep (Eq. 39), rho = div j_s,
// with the 5-point link-variable Laplacian  c_x (U_x(j) psi_{i+1} + U_x(j)* psi_{i-1}) + c_y (psi_{j+1} + psi_{j-1}).
//
// A CTA of 8 warps owns a strip of 1024 sites in x and marches through a chunk of rows in y.  One elected
// thread per row issues 1-D bulk copies (cp.async.bulk, the TMA engine without a tensor map: a row segment is
// contiguous) that land a stage in shared memory -- row j+1 of psi framed by its two ghost sites (wrapped,
// P:427; unused when x is open), plus, for the sweep, the b and d segments of row j -- completing on the
// stage's mbarrier.  The thread keeps rows j-1 and j of its own four sites in registers (y marching), reads
// row j+1 from the newest stage; x neighbours come from shuffles, the ones across a warp seam from the
// previous stage, where the frame makes "site - 1" and "site + 1" valid addresses for every site of the strip.
// U_x(j) changes with the marching index and is read once per row (warp-uniform).  The quasi-periodic jump
// P_i acts on the rows that wrap (j = 0, ny-1); open faces mirror.
// 32 B/site/sweep of HBM traffic, as in 3D.
#include "march_common.cuh"
#include "philox.cuh"
#include "march_film.h"

namespace {

constexpr int NW = 8;                    // warps per CTA
constexpr int SW = 128 * NW;             // strip width (sites)
constexpr int NTHREADS = 32 * NW;
// stage layout (bytes): [0,16) west ghost pair, [16, 16 + 8 nvs) the row segment, then the east ghost pair
constexpr unsigned OFF_ROW = 16;
constexpr unsigned OFF_B = 8320;         // b segment (sweep only)
constexpr unsigned OFF_D = 16512;        // d segment (sweep only)
constexpr unsigned OFF_MU = 8320;        // mu segment (init only, when nx % 4 == 0: 16-byte aligned 4-byte rows)
constexpr unsigned OFF_EPS = 12416;      // eps segment (init only)
constexpr unsigned STAGE_PSI = 8320, STAGE_INIT = 16512, STAGE_SWEEP = 24704;
constexpr unsigned HDR = 256;            // mbarriers at 0, CTA residual word at 64, 8 J_av warp sums at 128

template <int MODE> struct FCfg {
  static constexpr int NS = (MODE == MODE_SWEEP) ? 4 : 6;
  static constexpr unsigned SB = (MODE == MODE_SWEEP) ? STAGE_SWEEP : (MODE == MODE_INIT ? STAGE_INIT : STAGE_PSI);
  static constexpr unsigned SMEM = HDR + NS * SB;
};

// s += f [ c_x (U_x E + U_x* W) + c_y (T + B) ]  for the two sites of a pair (Eq. 29a without the z term)
__device__ __forceinline__ void nsum_film(const float2 ux, const float cy, const float4 &C, const float2 &W,
                                          const float2 &E, const float4 &T, const float4 &B, float2 &s0, float2 &s1) {
  s0.x = fmaf(ux.x, C.z + W.x, s0.x);  s0.x = fmaf(-ux.y, C.w - W.y, s0.x);
  s0.y = fmaf(ux.x, C.w + W.y, s0.y);  s0.y = fmaf(ux.y, C.z - W.x, s0.y);
  s1.x = fmaf(ux.x, E.x + C.x, s1.x);  s1.x = fmaf(-ux.y, E.y - C.y, s1.x);
  s1.y = fmaf(ux.x, E.y + C.y, s1.y);  s1.y = fmaf(ux.y, E.x - C.x, s1.y);
  s0.x = fmaf(cy, T.x + B.x, s0.x);    s0.y = fmaf(cy, T.y + B.y, s0.y);
  s1.x = fmaf(cy, T.z + B.z, s1.x);    s1.y = fmaf(cy, T.w + B.w, s1.y);
}

template <int MODE>
__global__ void __launch_bounds__(NTHREADS, 2) k_march_film(const __grid_constant__ Dev dv) {
  constexpr int NS = FCfg<MODE>::NS;
  constexpr int DEPTH = NS - 2;
  constexpr unsigned SB = FCfg<MODE>::SB;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  Ctl *ctl = dv.ctl;
  int l = 0;
  if (MODE == MODE_SWEEP && (blockIdx.x | blockIdx.y | blockIdx.z | threadIdx.x) == 0) ctl->body_launches += 1;   // as march_tma.cu: tdgl_launch_count in graph mode
  if (MODE != MODE_RHO) {
    if (ctl->done) return;
    l = ctl->sweeps;
  }
  const int xb = ctl->xbuf;
  const float2 *__restrict__ xin = dv.psi[xb];
  float2 *__restrict__ xout = dv.psi[xb ^ 1];

  const int nx = dv.nx, ny = dv.ny;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int i0 = blockIdx.x * SW;
  const int nvs = min(SW, nx - i0);                                 // valid sites of the strip (even)
  const int j0 = blockIdx.y * dv.zc, j1 = min(ny, j0 + dv.zc);      // rows [j0, j1)
  const int nk = j1 - j0;
  const bool px = dv.bcx == 0, py = dv.bcy == 0;
  const unsigned sbase = smem_u32(smem_raw);
  const unsigned stage0 = sbase + HDR;
  const unsigned rowbytes = 8u * (unsigned)nvs;
  // init: mu, eps of the row arrive with the stage when their row segments are 16-byte aligned multiples of 16 B
  const bool me_bulk = (MODE == MODE_INIT) && (nx % 4 == 0) && (nvs % 4 == 0) &&
                       ((reinterpret_cast<unsigned long long>(dv.mu) | reinterpret_cast<unsigned long long>(dv.eps)) & 15ull) == 0ull;

  auto ywrap = [&](int jp) -> int {                                 // row index with wrap / mirror
    if (jp < 0) return py ? ny - 1 : 1;
    if (jp >= ny) return py ? 0 : ny - 2;
    return jp;
  };
  // stage t holds psi row j0 + t (the "j+1" row of iteration j = j0 + t - 1) and b, d of row j0 + t - 1
  const int gW = (i0 > 0) ? i0 - 2 : nx - 2, gE = (i0 + nvs < nx) ? i0 + nvs : 0;
  auto issue = [&](int t) {
    const unsigned slot = (unsigned)t % NS;
    const unsigned sb = stage0 + slot * SB, bar = sbase + 8u * slot;
    const float2 *src = xin + (long long)ywrap(j0 + t) * nx;
    const bool bd = (MODE == MODE_SWEEP) && t >= 1;
    const bool me = (MODE == MODE_INIT) && me_bulk && t >= 1;         // mu, eps of row j0 + t - 1
    mbar_expect_tx(bar, rowbytes + 32u + (bd ? 2u * rowbytes : 0u) + (me ? (dv.solve_mu ? rowbytes : rowbytes / 2u) : 0u));
    bulk_load_1d(sb + OFF_ROW, src + i0, rowbytes, bar);
    bulk_load_1d(sb, src + gW, 16u, bar);
    bulk_load_1d(sb + OFF_ROW + rowbytes, src + gE, 16u, bar);
    if (bd) {
      const long long o = (long long)(j0 + t - 1) * nx + i0;
      bulk_load_1d(sb + OFF_B, dv.b + o, rowbytes, bar);
      bulk_load_1d(sb + OFF_D, dv.d + o, rowbytes, bar);
    }
    if (me) {
      const long long o = (long long)(j0 + t - 1) * nx + i0;
      if (dv.solve_mu) bulk_load_1d(sb + OFF_MU, dv.mu + o, rowbytes / 2u, bar);
      bulk_load_1d(sb + OFF_EPS, dv.eps + o, rowbytes / 2u, bar);
    }
  };

  if (tid == 0) {
    for (int s = 0; s < NS; ++s) mbar_init(sbase + 8u * s, 1u);
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    *reinterpret_cast<unsigned *>(smem_raw + 64) = 0u;
  }
  __syncthreads();
  if (tid == 0)
    for (int t = 0; t <= DEPTH && t <= nk; ++t) issue(t);

  // ---- fixed per-thread geometry ---------------------------------------------------------------------
  const int sA = 128 * warp + 2 * lane, sB = sA + 64;               // strip-local site of the two pairs
  const bool actA = sA < nvs, actB = sB < nvs;
  const int e = nvs - 1;
  const unsigned oA = OFF_ROW + 8u * (unsigned)sA, oB = oA + 512u;
  const bool w_h = lane == 0;                                        // west neighbour across a warp seam / strip edge
  const bool eA_h = (lane == 31) || (sA + 1 == e), eB_h = (lane == 31) || (sB + 1 == e);
  const int iA = i0 + sA, iB = i0 + sB;
  const bool xloA = !px && iA == 0, xhiA = !px && iA + 1 == nx - 1, xhiB = !px && iB + 1 == nx - 1;
  const bool xopen = !px && (i0 == 0 || i0 + nvs == nx);
  const float f = (MODE == MODE_RHO) ? 1.f : dv.ht2;
  const float fcx = f * dv.cx, fcy = f * dv.cy;
  unsigned nstep = 0;
  if (MODE == MODE_INIT) nstep = (unsigned)ctl->n;
  float rmax = 0.f;
  const bool jact = (MODE != MODE_RHO) && dv.solve_mu && px;       // J_av: x links inside a warp segment (Eq. 35)
  const bool lkA0 = actA, lkA1 = actA && sA + 2 < nvs;
  const bool lkB0 = actB, lkB1 = actB && sB + 2 < nvs && lane < 31;
  double jacc = 0.0;

  const int icl = min(iA, nx - 2);                                  // clamped: inactive threads stay in range
  long long idx = (long long)j0 * nx + icl;
  float4 rA[3], rB[3];
  {
    const long long ob = (long long)ywrap(j0 - 1) * nx + icl;
    rA[0] = actA ? __ldg(reinterpret_cast<const float4 *>(xin + ob)) : make_float4(0, 0, 0, 0);
    rB[0] = actB ? __ldg(reinterpret_cast<const float4 *>(xin + ob + 64)) : make_float4(0, 0, 0, 0);
  }
  mbar_wait(sbase, 0u);
  rA[1] = lds128(stage0 + oA);
  rB[1] = lds128(stage0 + oB);
  float2 Uxn = dv.Ux[j0];                                           // U_x of the next row to be processed

  float2 muA = make_float2(0.f, 0.f), muB = muA, epA = make_float2(1.f, 1.f), epB = epA;
  auto load_mu_eps = [&](long long ix, float2 &ma, float2 &mb, float2 &ea, float2 &eb) {
    if (MODE == MODE_INIT) {
      if (actA) {
        if (dv.solve_mu) ma = __ldcs(reinterpret_cast<const float2 *>(dv.mu + ix));
        ea = __ldg(reinterpret_cast<const float2 *>(dv.eps + ix));
      }
      if (actB) {
        if (dv.solve_mu) mb = __ldcs(reinterpret_cast<const float2 *>(dv.mu + ix + 64));
        eb = __ldg(reinterpret_cast<const float2 *>(dv.eps + ix + 64));
      }
    }
  };
  if (!me_bulk) load_mu_eps(idx, muA, muB, epA, epB);

  // one row: Bv, Cv = this thread's values of rows j-1, j; Tv receives row j+1
  auto do_row = [&](int t, float4 &BvA, float4 &BvB, float4 &CvA, float4 &CvB, float4 &TvA, float4 &TvB) {
    const int j = j0 + t - 1;
    const unsigned slot = (unsigned)t % NS, pslot = (unsigned)(t - 1) % NS;
    __syncthreads();                                   // every warp is done with stage t - 2: its slot is free
    if (tid == ((t & (NW - 1)) << 5) && t + DEPTH <= nk) issue(t + DEPTH);
    const float2 Ux = Uxn;                             // U_x(j) = exp(i h_x (K + B_z ybar_j))  (Eq. 27)
    if (t < nk) Uxn = dv.Ux[j + 1];
    mbar_wait(sbase + 8u * slot, ((unsigned)t / NS) & 1u);
    const unsigned cur = stage0 + slot * SB, prv = stage0 + pslot * SB;

    TvA = lds128(cur + oA);
    TvB = lds128(cur + oB);
    float4 bA, bB, dA, dB;
    if (MODE == MODE_SWEEP) {
      bA = lds128(cur + OFF_B - OFF_ROW + oA); bB = lds128(cur + OFF_B - OFF_ROW + oB);
      dA = lds128(cur + OFF_D - OFF_ROW + oA); dB = lds128(cur + OFF_D - OFF_ROW + oB);
    }
    float2 nmuA, nmuB, nepA, nepB;
    if (MODE == MODE_INIT) {
      nmuA = muA; nmuB = muB; nepA = epA; nepB = epB;
      if (me_bulk) {                                   // mu, eps of THIS row arrived with the stage
        const unsigned om = 4u * (unsigned)sA;
        if (dv.solve_mu) { muA = lds64(cur + OFF_MU + om); muB = lds64(cur + OFF_MU + om + 256u); }
        epA = lds64(cur + OFF_EPS + om); epB = lds64(cur + OFF_EPS + om + 256u);
      } else if (t < nk) load_mu_eps(idx + nx, nmuA, nmuB, nepA, nepB);
    }
    float2 WA, EA, WB, EB;
    WA.x = __shfl_up_sync(0xffffffffu, CvA.z, 1);   WA.y = __shfl_up_sync(0xffffffffu, CvA.w, 1);
    EA.x = __shfl_down_sync(0xffffffffu, CvA.x, 1); EA.y = __shfl_down_sync(0xffffffffu, CvA.y, 1);
    WB.x = __shfl_up_sync(0xffffffffu, CvB.z, 1);   WB.y = __shfl_up_sync(0xffffffffu, CvB.w, 1);
    EB.x = __shfl_down_sync(0xffffffffu, CvB.x, 1); EB.y = __shfl_down_sync(0xffffffffu, CvB.y, 1);
    if (w_h) { WA = lds64(prv + oA - 8u); WB = lds64(prv + oB - 8u); }
    if (eA_h) EA = lds64(prv + oA + 16u);
    if (eB_h) EB = lds64(prv + oB + 16u);

    float4 TA = TvA, TB = TvB, BA = BvA, BB = BvB;
    if (j == 0 || j == ny - 1) {                       // the rows that wrap (uniform over the CTA)
      if (py) {                                        // quasi-periodic jump, k = 0
        const float2 Pk = dv.Pk[0];
        const float4 PiA = *reinterpret_cast<const float4 *>(dv.Pi + icl);
        const float4 PiB = *reinterpret_cast<const float4 *>(dv.Pi + min(iB, nx - 2));
        const float2 PA0 = cmulc(Pk, lo(PiA)), PA1 = cmulc(Pk, hi(PiA)), PB0 = cmulc(Pk, lo(PiB)), PB1 = cmulc(Pk, hi(PiB));
        if (j == 0) {                                  // psi_{i,-1} = P_i psi_{i,ny-1}
          const float2 a = cmul(PA0, lo(BA)), b2 = cmul(PA1, hi(BA)), c2 = cmul(PB0, lo(BB)), d2 = cmul(PB1, hi(BB));
          BA = make_float4(a.x, a.y, b2.x, b2.y);
          BB = make_float4(c2.x, c2.y, d2.x, d2.y);
        }
        if (j == ny - 1) {                             // psi_{i,ny} = P_i* psi_{i,0}
          const float2 a = cmulc(PA0, lo(TA)), b2 = cmulc(PA1, hi(TA)), c2 = cmulc(PB0, lo(TB)), d2 = cmulc(PB1, hi(TB));
          TA = make_float4(a.x, a.y, b2.x, b2.y);
          TB = make_float4(c2.x, c2.y, d2.x, d2.y);
        }
      } else {                                         // open y faces (U_y = 1): mirror
        if (j == 0) { BA = TA; BB = TB; }
        else { TA = BA; TB = BB; }
      }
    }
    if (xopen) {                                       // open x faces: W' = U^2 E, E' = U*^2 W
      const float2 U2 = cmul(Ux, Ux);
      if (xloA) WA = cmul(U2, hi(CvA));
      if (xhiA) EA = cmulc(U2, lo(CvA));
      if (xhiB) EB = cmulc(U2, lo(CvB));
    }

    const float2 ux = make_float2(fcx * Ux.x, fcx * Ux.y);
    float2 sA0 = make_float2(0.f, 0.f), sA1 = sA0, sB0 = sA0, sB1 = sA0;
    if (MODE == MODE_SWEEP) { sA0 = lo(bA); sA1 = hi(bA); sB0 = lo(bB); sB1 = hi(bB); }
    nsum_film(ux, fcy, CvA, WA, EA, TA, BA, sA0, sA1);
    nsum_film(ux, fcy, CvB, WB, EB, TB, BB, sB0, sB1);

    if (MODE == MODE_RHO) {
      if (actA) *reinterpret_cast<float2 *>(dv.mu + idx) =
          make_float2(CvA.x * sA0.y - CvA.y * sA0.x, CvA.z * sA1.y - CvA.w * sA1.x);
      if (actB) *reinterpret_cast<float2 *>(dv.mu + idx + 64) =
          make_float2(CvB.x * sB0.y - CvB.y * sB0.x, CvB.z * sB1.y - CvB.w * sB1.x);
    } else {
      float2 nA0 = sA0, nA1 = sA1, nB0 = sB0, nB1 = sB1;
      if (MODE == MODE_INIT) {
        // d_m = 1 + (h_t/2)[|psi|^2 + 2 (c_x + c_y) - eps + i u mu]   (2D)
        // b_m = psi (2 - d) + (h_t/2)(nsum + 2 zeta)                   (Eq. 31, rearranged)
        const float ht2 = dv.ht2;
        auto init_pair = [&](const float4 &C, float2 mu, float2 ep, long long ix, bool act, float2 &s0, float2 &s1,
                             float2 &n0, float2 &n1, float4 &dout) {
          const float a0 = C.x * C.x + C.y * C.y, a1 = C.z * C.z + C.w * C.w;
          const float2 d0 = make_float2(1.f + ht2 * (a0 + dv.csum2 - ep.x), ht2 * dv.u * mu.x);
          const float2 d1 = make_float2(1.f + ht2 * (a1 + dv.csum2 - ep.y), ht2 * dv.u * mu.y);
          float2 z0 = make_float2(0.f, 0.f), z1 = z0;
          if (dv.zeta_max > 0.f) {                     // Langevin term, Eq. (39) with d = 2 (S22), S11
            const unsigned long long m = (unsigned long long)ix;
            const PhiloxOut p0 = philox4x32_10((uint32_t)m, (uint32_t)(m >> 32), nstep, 0u, dv.seed_lo, dv.seed_hi);   // m is even:
            const float zs = 2.f * ht2 * dv.zeta_max;                                     // one call per site pair (S11')
            z0 = make_float2(zs * u32_to_pm1(p0.x0), zs * u32_to_pm1(p0.x1));
            z1 = make_float2(zs * u32_to_pm1(p0.x2), zs * u32_to_pm1(p0.x3));
          }
          const float2 q0 = cmul(lo(C), make_float2(2.f - d0.x, -d0.y)), q1 = cmul(hi(C), make_float2(2.f - d1.x, -d1.y));
          const float2 b0 = make_float2(q0.x + s0.x + z0.x, q0.y + s0.y + z0.y);
          const float2 b1 = make_float2(q1.x + s1.x + z1.x, q1.y + s1.y + z1.y);
          n0 = make_float2(b0.x + s0.x, b0.y + s0.y);
          n1 = make_float2(b1.x + s1.x, b1.y + s1.y);
          dout = make_float4(d0.x, d0.y, d1.x, d1.y);
          if (act) {
            *reinterpret_cast<float4 *>(dv.b + ix) = make_float4(b0.x, b0.y, b1.x, b1.y);
            *reinterpret_cast<float4 *>(dv.d + ix) = dout;
          }
        };
        init_pair(CvA, muA, epA, idx, actA, sA0, sA1, nA0, nA1, dA);
        init_pair(CvB, muB, epB, idx + 64, actB, sB0, sB1, nB0, nB1, dB);
        if (!me_bulk) { muA = nmuA; muB = nmuB; epA = nepA; epB = nepB; }
      }
      float rloc = 0.f;
      const float4 outA = divide_pair(nA0, nA1, dA, CvA, rloc);
      if (actA) { *reinterpret_cast<float4 *>(xout + idx) = outA; rmax = fmaxf(rmax, rloc); }
      rloc = 0.f;
      const float4 outB = divide_pair(nB0, nB1, dB, CvB, rloc);
      if (actB) { *reinterpret_cast<float4 *>(xout + idx + 64) = outB; rmax = fmaxf(rmax, rloc); }
      if (jact) {                                      // Im[x*_m U_x x_{m+1}] on the links inside the warp segment
        const float nAx = __shfl_down_sync(0xffffffffu, outA.x, 1), nAy = __shfl_down_sync(0xffffffffu, outA.y, 1);
        const float rBx = __shfl_sync(0xffffffffu, outB.x, (lane + 1) & 31), rBy = __shfl_sync(0xffffffffu, outB.y, (lane + 1) & 31);
        const float2 nxA = (lane == 31) ? make_float2(rBx, rBy) : make_float2(nAx, nAy);
        auto link = [&](float ar, float ai, float br, float bi) {
          return ar * (Ux.x * bi + Ux.y * br) - ai * (Ux.x * br - Ux.y * bi);
        };
        float tsum = 0.f;
        if (lkA0) tsum += link(outA.x, outA.y, outA.z, outA.w);
        if (lkA1) tsum += link(outA.z, outA.w, nxA.x, nxA.y);
        if (lkB0) tsum += link(outB.x, outB.y, outB.z, outB.w);
        if (lkB1) tsum += link(outB.z, outB.w, rBx, rBy);
        jacc += (double)tsum;
      }
    }
    idx += nx;
  };

  for (int t = 1; t <= nk; t += 3) {
    do_row(t, rA[0], rB[0], rA[1], rB[1], rA[2], rB[2]);
    if (t + 1 <= nk) do_row(t + 1, rA[1], rB[1], rA[2], rB[2], rA[0], rB[0]);
    if (t + 2 <= nk) do_row(t + 2, rA[2], rB[2], rA[0], rB[0], rA[1], rB[1]);
  }

  if (MODE != MODE_RHO) {
    unsigned *s_max = reinterpret_cast<unsigned *>(smem_raw + 64);
    double *s_j = reinterpret_cast<double *>(smem_raw + 128);
    const unsigned w = __reduce_max_sync(0xffffffffu, __float_as_uint(rmax));
    if (lane == 0) atomicMax(s_max, w);
    if (jact) {
      for (int o = 16; o > 0; o >>= 1) jacc += __shfl_down_sync(0xffffffffu, jacc, o);
      if (lane == 0) s_j[warp] = jacc;
    }
    __syncthreads();
    if (tid == 0) {
      if (jact) {
        double sj = 0.0;
        for (int q = 0; q < NW; ++q) sj += s_j[q];
        dv.jpart[blockIdx.x + gridDim.x * blockIdx.y] = sj;
      }
      atomicMax(&ctl->resid_bits[l], *s_max);
      __threadfence();
      const unsigned nb = gridDim.x * gridDim.y * gridDim.z;
      const unsigned tk = atomicAdd(&ctl->ticket, 1u);
      if (tk == nb - 1) {
        ctl->ticket = 0u;
        sweep_decide(dv, l);
      }
    }
  }
}

}  // namespace

cudaError_t march_film_configure() {
  cudaError_t e = cudaFuncSetAttribute(k_march_film<MODE_SWEEP>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       (int)FCfg<MODE_SWEEP>::SMEM);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(k_march_film<MODE_INIT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FCfg<MODE_INIT>::SMEM);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(k_march_film<MODE_RHO>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FCfg<MODE_RHO>::SMEM);
}

int march_film_strips(int nx) { return (nx + SW - 1) / SW; }

void launch_march_film(int mode, const Dev &dv, dim3 grid, cudaStream_t st) {
  if (mode == MODE_SWEEP) k_march_film<MODE_SWEEP><<<grid, NTHREADS, FCfg<MODE_SWEEP>::SMEM, st>>>(dv);
  else if (mode == MODE_INIT) k_march_film<MODE_INIT><<<grid, NTHREADS, FCfg<MODE_INIT>::SMEM, st>>>(dv);
  else k_march_film<MODE_RHO><<<grid, NTHREADS, FCfg<MODE_RHO>::SMEM, st>>>(dv);
}
