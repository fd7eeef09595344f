// The z-marching 7-point link-variable stencil, TMA edition (sm_100a): Jacobi sweep + max-residual (a4,
// Eq. 33-34), fused init + first sweep (a3, with the Philox Langevin term a2,
// Eq. 39), rho = div j_s (a6).
//
// A CTA of 8 warps owns a 128 x 8 tile of the xy plane and marches through a chunk of z planes.  One
// elected thread per plane issues bulk tensor copies (cp.async.bulk.tensor, TMA) that land a whole
// stage in shared memory -- the psi plane k+1 of the tile (centre 128 x 8, the two ghost rows, the two
// ghost columns; wrapped or mirrored coordinates chosen by the issuing thread) plus, for
// the sweep, the b and d tiles of plane k -- and completes on the stage's mbarrier.  Stages form a ring;
// two are being read while the others are in flight, so a CTA keeps 2 x 26 KB outstanding and the
// arithmetic warps never compute a global address for a load.
// A warp owns one row; lane l owns the site pairs (2l, 2l+1) and (64+2l, 64+2l+1): every shared-memory
// access is a conflict-free 16-byte vector.  The thread keeps its values of planes k-1 and k in
// registers (z marching), reads plane k+1 (own sites) from the newest stage and the y neighbours and
// tile-edge x neighbours of plane k from the previous stage; x neighbours inside the warp come from
// shuffles.  32 B/site/sweep of HBM traffic: x^l 8, b 8, d 8 read, x^{l+1} 8 written.
#include "march_common.cuh"
#include "philox.cuh"
#include "march_tma.h"

namespace {

constexpr int TW = 128;                 // tile width (sites)
constexpr int TH = 8;                   // tile height (rows) = warps per CTA
constexpr int NTHREADS = 32 * TH;
// stage layout (bytes); every block is a TMA destination (128-byte aligned)
constexpr unsigned OFF_C = 0;           // psi centre: TH rows, pitch = 8 * min(TW, nx) bytes
constexpr unsigned OFF_RLO = 8192;      // ghost row j0 - 1
constexpr unsigned OFF_RHI = 9216;      // ghost row j0 + nvy
constexpr unsigned OFF_XW = 10240;      // ghost column pair (i0-2, i0-1): TH x 16 B
constexpr unsigned OFF_XE = 10368;      // ghost column pair (i0+nv, i0+nv+1)
constexpr unsigned OFF_B = 10496;       // b tile (sweep only)
constexpr unsigned OFF_D = 18688;       // d tile (sweep only)
constexpr unsigned OFF_MU = 10496;      // mu tile (init only, when the row pitch 4 nx is a multiple of 16 B): TH rows x 4 min(TW, nx) bytes
constexpr unsigned OFF_EPS = 14592;     // eps tile (init only)
constexpr unsigned STAGE_PSI = 10496, STAGE_INIT = 18688, STAGE_SWEEP = 26880;
constexpr unsigned HDR = 256;           // mbarriers (8 B each) at 0, the CTA residual word at 64, 8 J_av warp sums at 128

template <int MODE> struct Cfg {
  static constexpr int NS = (MODE == MODE_SWEEP) ? 4 : 6;                       // stages in the ring
  static constexpr unsigned SB = (MODE == MODE_SWEEP) ? STAGE_SWEEP : (MODE == MODE_INIT ? STAGE_INIT : STAGE_PSI); // bytes per stage
  static constexpr unsigned SMEM = HDR + NS * SB;
};

// yz Landau gauge (Eq. 24b, 29b): U_x = exp(i h_x K) is uniform, U_y(i) and U_z(i) vary along x
// (per-site constants uy, uz = both sites of a pair, already scaled by f c_y, f c_z)
__device__ __forceinline__ void nsum_pair_yz(const float2 ux, const float4 &uy, const float4 &uz, const float4 &C,
                                             const float2 &W, const float2 &E, const float4 &Nn, const float4 &Ss,
                                             const float4 &T, const float4 &B, float2 &s0, float2 &s1) {
  s0.x = fmaf(ux.x, C.z + W.x, s0.x);  s0.x = fmaf(-ux.y, C.w - W.y, s0.x);
  s0.y = fmaf(ux.x, C.w + W.y, s0.y);  s0.y = fmaf(ux.y, C.z - W.x, s0.y);
  s1.x = fmaf(ux.x, E.x + C.x, s1.x);  s1.x = fmaf(-ux.y, E.y - C.y, s1.x);
  s1.y = fmaf(ux.x, E.y + C.y, s1.y);  s1.y = fmaf(ux.y, E.x - C.x, s1.y);
  s0.x = fmaf(uy.x, Nn.x + Ss.x, s0.x);  s0.x = fmaf(-uy.y, Nn.y - Ss.y, s0.x);
  s0.y = fmaf(uy.x, Nn.y + Ss.y, s0.y);  s0.y = fmaf(uy.y, Nn.x - Ss.x, s0.y);
  s1.x = fmaf(uy.z, Nn.z + Ss.z, s1.x);  s1.x = fmaf(-uy.w, Nn.w - Ss.w, s1.x);
  s1.y = fmaf(uy.z, Nn.w + Ss.w, s1.y);  s1.y = fmaf(uy.w, Nn.z - Ss.z, s1.y);
  s0.x = fmaf(uz.x, T.x + B.x, s0.x);  s0.x = fmaf(-uz.y, T.y - B.y, s0.x);
  s0.y = fmaf(uz.x, T.y + B.y, s0.y);  s0.y = fmaf(uz.y, T.x - B.x, s0.y);
  s1.x = fmaf(uz.z, T.z + B.z, s1.x);  s1.x = fmaf(-uz.w, T.w - B.w, s1.x);
  s1.y = fmaf(uz.z, T.w + B.w, s1.y);  s1.y = fmaf(uz.w, T.z - B.z, s1.y);
}
// both sites of v times the squares of their own link variables u = (u0, u1) (open faces: ghost = U^2 neighbour)
__device__ __forceinline__ float4 sq_mul4(const float4 &u, const float4 &v, bool conj_) {
  const float2 a = cmul(lo(u), lo(u)), b = cmul(hi(u), hi(u));
  const float2 p = conj_ ? cmulc(a, lo(v)) : cmul(a, lo(v)), q = conj_ ? cmulc(b, hi(v)) : cmul(b, hi(v));
  return make_float4(p.x, p.y, q.x, q.y);
}

template <int MODE, bool YZ>
__global__ void __launch_bounds__(NTHREADS, 2) k_march_tma(const __grid_constant__ Dev dv,
                                                           const __grid_constant__ MarchMaps mm) {
  constexpr int NS = Cfg<MODE>::NS;
  constexpr int DEPTH = NS - 2;                       // stages in flight beyond the two being read
  constexpr unsigned SB = Cfg<MODE>::SB;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  Ctl *ctl = dv.ctl;
  int l = 0;
  if (MODE == MODE_SWEEP && (blockIdx.x | blockIdx.y | blockIdx.z | threadIdx.x) == 0) ctl->body_launches += 1;
  if (MODE != MODE_RHO) {
    if (ctl->done) return;
    if (MODE == MODE_SWEEP && ctl->use_pair) return;   // this iteration belongs to the fused pair kernel (march_pair.cu)
    l = ctl->sweeps;
  }
  const int xb = ctl->xbuf;

  const int nx = dv.nx, ny = dv.ny, nz = dv.nz;
  const int tid = threadIdx.x, lane = tid & 31, row = tid >> 5;
  const int i0 = blockIdx.x * TW, j0 = blockIdx.y * TH;
  const int nv = min(TW, nx - i0), nvy = min(TH, ny - j0);          // valid sites per row, valid rows
  const int k0 = blockIdx.z * dv.zc, k1 = min(nz, k0 + dv.zc);      // planes [k0, k1)
  const int nk = k1 - k0;
  const bool px = dv.bcx == 0, py = dv.bcy == 0, pz = dv.bcz == 0;
  const long long plane = (long long)nx * ny;
  const unsigned pitch = 8u * (unsigned)min(TW, nx);                // bytes per row of a tile in smem
  const unsigned bh = (unsigned)min(TH, ny);
  const unsigned sbase = smem_u32(smem_raw);
  const unsigned stage0 = sbase + HDR;

  auto zwrap = [&](int kp) -> int {                                 // plane index with wrap / mirror
    if (kp < 0) return pz ? nz - 1 : 1;
    if (kp >= nz) return pz ? 0 : nz - 2;
    return kp;
  };

  // ---- producer side: coordinates of the five psi boxes of this tile (floats in x) ----------------
  const int cx0 = 2 * i0;
  const int yLo = (j0 > 0) ? j0 - 1 : (py ? ny - 1 : 1);
  const int yHi = (j0 + nvy < ny) ? j0 + nvy : (py ? 0 : ny - 2);
  const int xW = 2 * ((i0 > 0) ? i0 - 2 : nx - 2);
  const int xE = 2 * ((i0 + nv < nx) ? i0 + nv : 0);
  const unsigned tx_psi = pitch * bh + 2u * pitch + 2u * 16u * bh;
  const unsigned tx_bd = 2u * pitch * bh;
  const bool me_tma = (MODE == MODE_INIT) && mm.me_tma;             // mu, eps through the stage (else plain loads)
  const unsigned tx_me = (pitch / 2u) * bh * (dv.solve_mu ? 2u : 1u);
  const CUtensorMap *mC = &mm.psiC[xb], *mR = &mm.psiR[xb], *mX = &mm.psiX[xb];
  // stage t holds psi plane k0 + t (the "k+1" plane of iteration k = k0 + t - 1) and b, d of plane k0 + t - 1
  auto issue = [&](int t) {
    const unsigned slot = (unsigned)t % NS;
    const unsigned sb = stage0 + slot * SB, bar = sbase + 8u * slot;
    const int kz = zwrap(k0 + t);
    const bool bd = (MODE == MODE_SWEEP) && t >= 1;
    const bool me = (MODE == MODE_INIT) && me_tma && t >= 1;          // mu, eps of plane k0 + t - 1
    mbar_expect_tx(bar, tx_psi + (bd ? tx_bd : 0u) + (me ? tx_me : 0u));
    tma_load_3d(sb + OFF_C, mC, cx0, j0, kz, bar);
    tma_load_3d(sb + OFF_RLO, mR, cx0, yLo, kz, bar);
    tma_load_3d(sb + OFF_RHI, mR, cx0, yHi, kz, bar);
    tma_load_3d(sb + OFF_XW, mX, xW, j0, kz, bar);
    tma_load_3d(sb + OFF_XE, mX, xE, j0, kz, bar);
    if (bd) {
      tma_load_3d(sb + OFF_B, &mm.bC, cx0, j0, k0 + t - 1, bar);
      tma_load_3d(sb + OFF_D, &mm.dC, cx0, j0, k0 + t - 1, bar);
    }
    if (me) {
      if (dv.solve_mu) tma_load_3d(sb + OFF_MU, &mm.muC, i0, j0, k0 + t - 1, bar);
      tma_load_3d(sb + OFF_EPS, &mm.epsC, i0, j0, k0 + t - 1, bar);
    }
  };

  if (tid == 0) {
    for (int s = 0; s < NS; ++s) mbar_init(sbase + 8u * s, 1u);
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    *reinterpret_cast<unsigned *>(smem_raw + 64) = 0u;              // CTA max-residual word
  }
  __syncthreads();
  if (tid == 0)
    for (int t = 0; t <= DEPTH && t <= nk; ++t) issue(t);

  // ---- consumer side: fixed per-thread geometry ----------------------------------------------------
  const int j = j0 + row;
  const int jc = min(j, ny - 1);
  const int iA = i0 + 2 * lane, iB = iA + 64;
  const bool rowact = row < nvy;
  const bool actA = rowact && 2 * lane < nv, actB = rowact && 64 + 2 * lane < nv;
  const int e = nv - 1;                                              // last valid site of the tile row (odd)
  // shared-memory offsets relative to a stage base
  const unsigned oA = OFF_C + (unsigned)row * pitch + 16u * lane, oB = oA + 512u;
  const unsigned oNA = (row == nvy - 1) ? OFF_RHI + 16u * lane : oA + pitch, oNB = oNA + 512u;
  const unsigned oSA = (row == 0) ? OFF_RLO + 16u * lane : oA - pitch, oSB = oSA + 512u;
  // x neighbours that do not come from the shuffle: tile edges, the seam between the two halves
  const bool wA_h = lane == 0, wB_h = lane == 0;
  const bool eA_h = (lane == 31) || (2 * lane + 1 == e), eB_h = (lane == 31) || (64 + 2 * lane + 1 == e);
  const unsigned oWA = OFF_XW + 16u * row + 8u;                                      // site i0 - 1
  const unsigned oWB = OFF_C + (unsigned)row * pitch + 8u * 63u;                    // site i0 + 63
  const unsigned oEA = (2 * lane + 1 == e) ? OFF_XE + 16u * row : OFF_C + (unsigned)row * pitch + 8u * 64u;
  const unsigned oEB = OFF_XE + 16u * row;                                           // site i0 + nv
  // boundary roles
  const bool ylo = py && j == 0, yhi = py && j == ny - 1;           // quasi-periodic jump rows (warp-uniform)
  const bool xloA = !px && iA == 0, xhiA = !px && iA + 1 == nx - 1;
  const bool xhiB = !px && iB + 1 == nx - 1;                        // (iB == 0 never happens)
  const bool xopen = !px && (i0 == 0 || i0 + nv == nx);             // CTA-uniform

  const float f = (MODE == MODE_RHO) ? 1.f : dv.ht2;
  const float2 Uxj = dv.Ux[jc], Uzj = dv.Uz[jc];
  const float2 Lux = make_float2(f * dv.cx * Uxj.x, f * dv.cx * Uxj.y);
  const Links L = make_links(Lux, make_float2(f * dv.cz * Uzj.x, f * dv.cz * Uzj.y), f * dv.cy);
  const int icA = min(iA, nx - 2), icB = min(iB, nx - 2);
  float4 uyA, uyB, uzA, uzB;                                         // yz gauge: scaled U_y(i), U_z(i) of the four sites
  if (YZ) {
    const float sy = f * dv.cy, sz = f * dv.cz;
    const float4 a = *reinterpret_cast<const float4 *>(dv.Uy + icA), b = *reinterpret_cast<const float4 *>(dv.Uy + icB);
    const float4 c = *reinterpret_cast<const float4 *>(dv.Uzx + icA), d = *reinterpret_cast<const float4 *>(dv.Uzx + icB);
    uyA = make_float4(sy * a.x, sy * a.y, sy * a.z, sy * a.w); uyB = make_float4(sy * b.x, sy * b.y, sy * b.z, sy * b.w);
    uzA = make_float4(sz * c.x, sz * c.y, sz * c.z, sz * c.w); uzB = make_float4(sz * d.x, sz * d.y, sz * d.z, sz * d.w);
  }
  const bool xedge = px && (i0 == 0 || i0 + nv == nx);              // yz: the CTA touches the quasi-periodic seam in x
  unsigned nstep = 0;
  if (MODE == MODE_INIT) nstep = (unsigned)ctl->n;
  float rmax = 0.f;
  // J_av (Eq. 35): x links of the NEW iterate that lie inside this tile row (step_ctl.cu, k_jav_edges
  // adds the links that cross a tile edge); only with x periodic and the mu / K part active
  const bool jact = (MODE != MODE_RHO) && dv.solve_mu && px;
  const bool lkA0 = actA, lkA1 = actA && 2 * lane + 2 < nv;
  const bool lkB0 = actB, lkB1 = actB && 64 + 2 * lane + 2 < nv && lane < 31;
  double jacc = 0.0;

  // element index of pair A in plane k0 (float2 units); clamped so that inactive threads stay in range
  const long long rowoff = (long long)jc * nx + min(iA, nx - 2);
  long long idx = (long long)k0 * plane + rowoff;
  const float2 *__restrict__ xin = dv.psi[xb];
  float2 *__restrict__ xout = dv.psi[xb ^ 1];

  // planes k0 - 1 (global load, wrapped / mirrored) and k0 (stage 0) of this thread's sites
  float4 rA[3], rB[3];
  {
    const long long ob = (long long)zwrap(k0 - 1) * plane + rowoff;
    rA[0] = actA ? __ldg(reinterpret_cast<const float4 *>(xin + ob)) : make_float4(0, 0, 0, 0);
    rB[0] = actB ? __ldg(reinterpret_cast<const float4 *>(xin + ob + 64)) : make_float4(0, 0, 0, 0);
  }
  const bool ztop = !pz && k1 == nz;                  // this chunk ends at the open top face
  if (!pz && k0 == 0) {                               // open bottom face: psi_{-1} = U_z^2 psi_1 (plane 1 is what was loaded)
    if (YZ) {
      const float4 ua = *reinterpret_cast<const float4 *>(dv.Uzx + icA), ub = *reinterpret_cast<const float4 *>(dv.Uzx + icB);
      rA[0] = sq_mul4(ua, rA[0], false); rB[0] = sq_mul4(ub, rB[0], false);
    } else {
      const float2 U2 = cmul(Uzj, Uzj);
      rA[0] = cmul4(U2, rA[0]); rB[0] = cmul4(U2, rB[0]);
    }
  }
  mbar_wait(sbase, 0u);
  rA[1] = lds128(stage0 + oA);
  rB[1] = lds128(stage0 + oB);

  // INIT: mu and eps of plane k arrive with the stage when nx % 4 == 0 (me_tma); otherwise their row stride is not a
  // multiple of 16 B, which rules out TMA, and they are prefetched one plane ahead with plain loads
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
  if (!me_tma) load_mu_eps(idx, muA, muB, epA, epB);
  const unsigned oME = (unsigned)row * (pitch / 2u) + 8u * lane;   // this thread's pair A in a mu / eps tile (pair B: + 256)

  // one plane: Bv, Cv = this thread's values of planes k-1, k; Tv receives plane k+1
  auto do_plane = [&](int t, float4 &BvA, float4 &BvB, float4 &CvA, float4 &CvB, float4 &TvA, float4 &TvB) {
    const int k = k0 + t - 1;
    const unsigned slot = (unsigned)t % NS, pslot = (unsigned)(t - 1) % NS;
    __syncthreads();                                   // every warp is done with stage t - 2: its slot is free
    if (tid == ((t & (TH - 1)) << 5) && t + DEPTH <= nk) issue(t + DEPTH);
    mbar_wait(sbase + 8u * slot, ((unsigned)t / NS) & 1u);
    const unsigned cur = stage0 + slot * SB, prv = stage0 + pslot * SB;

    TvA = lds128(cur + oA);
    TvB = lds128(cur + oB);
    float4 NA = lds128(prv + oNA), NB = lds128(prv + oNB);
    float4 SA = lds128(prv + oSA), SB_ = lds128(prv + oSB);
    float4 bA, bB, dA, dB;
    if (MODE == MODE_SWEEP) {
      bA = lds128(cur + OFF_B + oA); bB = lds128(cur + OFF_B + oB);
      dA = lds128(cur + OFF_D + oA); dB = lds128(cur + OFF_D + oB);
    }
    float2 nmuA, nmuB, nepA, nepB;
    if (MODE == MODE_INIT) {
      nmuA = muA; nmuB = muB; nepA = epA; nepB = epB;
      if (me_tma) {                                    // mu, eps of THIS plane arrived with the stage
        if (dv.solve_mu) { muA = lds64(cur + OFF_MU + oME); muB = lds64(cur + OFF_MU + oME + 256u); }
        epA = lds64(cur + OFF_EPS + oME); epB = lds64(cur + OFF_EPS + oME + 256u);
      } else if (t < nk) load_mu_eps(idx + plane, nmuA, nmuB, nepA, nepB);
    }
    float2 WA, EA, WB, EB;
    WA.x = __shfl_up_sync(0xffffffffu, CvA.z, 1);   WA.y = __shfl_up_sync(0xffffffffu, CvA.w, 1);
    EA.x = __shfl_down_sync(0xffffffffu, CvA.x, 1); EA.y = __shfl_down_sync(0xffffffffu, CvA.y, 1);
    WB.x = __shfl_up_sync(0xffffffffu, CvB.z, 1);   WB.y = __shfl_up_sync(0xffffffffu, CvB.w, 1);
    EB.x = __shfl_down_sync(0xffffffffu, CvB.x, 1); EB.y = __shfl_down_sync(0xffffffffu, CvB.y, 1);
    if (wA_h) WA = lds64(prv + oWA);
    if (wB_h) WB = lds64(prv + oWB);
    if (eA_h) EA = lds64(prv + oEA);
    if (eB_h) EB = lds64(prv + oEB);

    if (YZ) {
      if (xedge) {                                     // quasi-periodic jump in x: psi_{-1} = P_{j,k} psi_{nx-1}
        const float2 P = cmul(dv.Pj[jc], dv.Pk[k]);
        if (iA == 0) WA = cmul(P, WA);
        if (iA + 1 == nx - 1) EA = cmulc(P, EA);       // psi_{nx} = P*_{j,k} psi_0
        if (iB + 1 == nx - 1) EB = cmulc(P, EB);
      }
      if (!py && (j == 0 || j == ny - 1)) {            // open y faces with U_y != 1: ghost = U_y^2 neighbour
        const float4 ua = *reinterpret_cast<const float4 *>(dv.Uy + icA), ub = *reinterpret_cast<const float4 *>(dv.Uy + icB);
        if (j == 0) { SA = sq_mul4(ua, NA, false); SB_ = sq_mul4(ub, NB, false); }
        else { NA = sq_mul4(ua, SA, true); NB = sq_mul4(ub, SB_, true); }
      }
    }
    if (!YZ && (ylo || yhi)) {                         // quasi-periodic jump in y, rows 0 and ny-1 only
      const float2 Pk = dv.Pk[k];
      const float4 PiA = *reinterpret_cast<const float4 *>(dv.Pi + min(iA, nx - 2));
      const float4 PiB = *reinterpret_cast<const float4 *>(dv.Pi + min(iB, nx - 2));
      const float2 PA0 = cmulc(Pk, lo(PiA)), PA1 = cmulc(Pk, hi(PiA));     // P_{i,k} = Pi[i] conj(Pk[k])
      const float2 PB0 = cmulc(Pk, lo(PiB)), PB1 = cmulc(Pk, hi(PiB));
      if (ylo) {                                       // psi_{i,-1,k} = P psi_{i,ny-1,k}
        const float2 a = cmul(PA0, lo(SA)), b2 = cmul(PA1, hi(SA)), c2 = cmul(PB0, lo(SB_)), d2 = cmul(PB1, hi(SB_));
        SA = make_float4(a.x, a.y, b2.x, b2.y);
        SB_ = make_float4(c2.x, c2.y, d2.x, d2.y);
      }
      if (yhi) {                                       // psi_{i,ny,k} = P* psi_{i,0,k}
        const float2 a = cmulc(PA0, lo(NA)), b2 = cmulc(PA1, hi(NA)), c2 = cmulc(PB0, lo(NB)), d2 = cmulc(PB1, hi(NB));
        NA = make_float4(a.x, a.y, b2.x, b2.y);
        NB = make_float4(c2.x, c2.y, d2.x, d2.y);
      }
    }
    if (xopen) {                                       // open x faces: W' = U^2 E, E' = U*^2 W
      const float2 U2 = cmul(Uxj, Uxj);
      if (xloA) WA = cmul(U2, hi(CvA));
      if (xhiA) EA = cmulc(U2, lo(CvA));
      if (xhiB) EB = cmulc(U2, lo(CvB));
    }
    if (ztop && t == nk) {                             // open top face: psi_{nz} = U_z*^2 psi_{nz-2}; the stage
      if (YZ) {                                        // holds plane nz - 2 (mirror), nobody reads Tv after this plane
        const float4 ua = *reinterpret_cast<const float4 *>(dv.Uzx + icA), ub = *reinterpret_cast<const float4 *>(dv.Uzx + icB);
        TvA = sq_mul4(ua, TvA, true); TvB = sq_mul4(ub, TvB, true);
      } else {
        const float2 U2 = cmul(Uzj, Uzj);
        TvA = cmulc4(U2, TvA); TvB = cmulc4(U2, TvB);
      }
    }

    float2 sA0 = make_float2(0.f, 0.f), sA1 = sA0, sB0 = sA0, sB1 = sA0;
    if (MODE == MODE_SWEEP) { sA0 = lo(bA); sA1 = hi(bA); sB0 = lo(bB); sB1 = hi(bB); }
    if (YZ) {
      nsum_pair_yz(Lux, uyA, uzA, CvA, WA, EA, NA, SA, TvA, BvA, sA0, sA1);
      nsum_pair_yz(Lux, uyB, uzB, CvB, WB, EB, NB, SB_, TvB, BvB, sB0, sB1);
    } else {
      nsum_pair(L, CvA, WA, EA, NA, SA, TvA, BvA, sA0, sA1);
      nsum_pair(L, CvB, WB, EB, NB, SB_, TvB, BvB, sB0, sB1);
    }

    if (MODE == MODE_RHO) {
      // rho_m = sum_alpha c_alpha Im[psi*_m (S+ psi + S- psi)_m]
      if (actA) *reinterpret_cast<float2 *>(dv.mu + idx) =
          make_float2(CvA.x * sA0.y - CvA.y * sA0.x, CvA.z * sA1.y - CvA.w * sA1.x);
      if (actB) *reinterpret_cast<float2 *>(dv.mu + idx + 64) =
          make_float2(CvB.x * sB0.y - CvB.y * sB0.x, CvB.z * sB1.y - CvB.w * sB1.x);
    } else {
      float2 nA0 = sA0, nA1 = sA1, nB0 = sB0, nB1 = sB1;       // numerators b + (h_t/2) nsum
      if (MODE == MODE_INIT) {
        // d_m = 1 + (h_t/2)[|psi|^2 + 2 sum c - eps + i u mu]
        // b_m = psi (2 - d) + (h_t/2)(nsum + 2 zeta)             (Eq. 31, rearranged)
        const float ht2 = dv.ht2;
        auto init_pair = [&](const float4 &C, float2 mu, float2 ep, long long ix, bool act, float2 &s0, float2 &s1,
                             float2 &n0, float2 &n1, float4 &dout) {
          const float a0 = C.x * C.x + C.y * C.y, a1 = C.z * C.z + C.w * C.w;
          const float2 d0 = make_float2(1.f + ht2 * (a0 + dv.csum2 - ep.x), ht2 * dv.u * mu.x);
          const float2 d1 = make_float2(1.f + ht2 * (a1 + dv.csum2 - ep.y), ht2 * dv.u * mu.y);
          float2 z0 = make_float2(0.f, 0.f), z1 = z0;
          if (dv.zeta_max > 0.f) {                     // Langevin term, Eq. (39), S11
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
        if (!me_tma) { muA = nmuA; muB = nmuB; epA = nepA; epB = nepB; }
      }
      float rloc = 0.f;
      const float4 outA = divide_pair(nA0, nA1, dA, CvA, rloc);
      if (actA) { *reinterpret_cast<float4 *>(xout + idx) = outA; rmax = fmaxf(rmax, rloc); }
      rloc = 0.f;
      const float4 outB = divide_pair(nB0, nB1, dB, CvB, rloc);
      if (actB) { *reinterpret_cast<float4 *>(xout + idx + 64) = outB; rmax = fmaxf(rmax, rloc); }
      if (jact) {
        // Im[x*_m U x_{m+1}] on the links (2l,2l+1), (2l+1,2l+2), (64+2l,65+2l), (65+2l,66+2l); the east
        // end of the second comes from lane l+1, for lane 31 it is site 64 = lane 0's second pair
        const float nAx = __shfl_down_sync(0xffffffffu, outA.x, 1), nAy = __shfl_down_sync(0xffffffffu, outA.y, 1);
        const float rBx = __shfl_sync(0xffffffffu, outB.x, (lane + 1) & 31), rBy = __shfl_sync(0xffffffffu, outB.y, (lane + 1) & 31);
        const float2 nxA = (lane == 31) ? make_float2(rBx, rBy) : make_float2(nAx, nAy);
        auto link = [&](float ar, float ai, float br, float bi) { return jlink(Uxj, ar, ai, br, bi); };
        float tsum = 0.f;
        if (lkA0) tsum += link(outA.x, outA.y, outA.z, outA.w);
        if (lkA1) tsum += link(outA.z, outA.w, nxA.x, nxA.y);
        if (lkB0) tsum += link(outB.x, outB.y, outB.z, outB.w);
        if (lkB1) tsum += link(outB.z, outB.w, rBx, rBy);
        jacc += (double)tsum;
      }
    }
    idx += plane;
  };

  // z march; the register ring (planes k-1, k, k+1) rotates by renaming over three unrolled planes
  for (int t = 1; t <= nk; t += 3) {
    do_plane(t, rA[0], rB[0], rA[1], rB[1], rA[2], rB[2]);
    if (t + 1 <= nk) do_plane(t + 1, rA[1], rB[1], rA[2], rB[2], rA[0], rB[0]);
    if (t + 2 <= nk) do_plane(t + 2, rA[2], rB[2], rA[0], rB[0], rA[1], rB[1]);
  }

  if (MODE != MODE_RHO) {
    // max-residual reduction: redux over the warp on the uint pattern (non-negative floats order like
    // uints), one shared atomic per warp, one global atomic per CTA; the last CTA decides (Eq. 34).
    unsigned *s_max = reinterpret_cast<unsigned *>(smem_raw + 64);
    double *s_j = reinterpret_cast<double *>(smem_raw + 128);
    const unsigned w = __reduce_max_sync(0xffffffffu, __float_as_uint(rmax));
    if (lane == 0) atomicMax(s_max, w);
    if (jact) {
      for (int o = 16; o > 0; o >>= 1) jacc += __shfl_down_sync(0xffffffffu, jacc, o);
      if (lane == 0) s_j[row] = jacc;
    }
    __syncthreads();
    if (tid == 0) {
      if (jact) {                                        // fixed order => bit-reproducible
        double sj = 0.0;
        for (int q = 0; q < TH; ++q) sj += s_j[q];
        dv.jpart[blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z)] = sj;
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

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

}  // namespace

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
// Tensor maps of an interleaved complex fp32 field seen as floats [nz][ny][2 nx] with the three box
// shapes of a stage.  Returns 0, or a negative CUresult / -1000 if the driver entry point is missing.
int march_tma_build_maps(const Dev &dv, MarchMaps *mm) {
  void *fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
      qres != cudaDriverEntryPointSuccess)
    return -1000;
  EncodeTiledFn enc = (EncodeTiledFn)fn;
  const cuuint64_t gdim[3] = {2ull * dv.nx, (cuuint64_t)dv.ny, (cuuint64_t)dv.nz};
  const cuuint64_t gstr[2] = {8ull * dv.nx, 8ull * dv.nx * dv.ny};
  const cuuint32_t es[3] = {1, 1, 1};
  const cuuint32_t bw = (cuuint32_t)(2 * (dv.nx < TW ? dv.nx : TW)), bh = (cuuint32_t)(dv.ny < TH ? dv.ny : TH);
  const cuuint32_t boxC[3] = {bw, bh, 1}, boxR[3] = {bw, 1, 1}, boxX[3] = {4, bh, 1};
  auto mk = [&](CUtensorMap *m, void *base, const cuuint32_t *box) -> int {
    const CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, base, gdim, gstr, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                           CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? 0 : -(int)r;
  };
  int rc = 0;
  for (int s = 0; s < 2 && !rc; ++s) {
    if (!rc) rc = mk(&mm->psiC[s], dv.psi[s], boxC);
    if (!rc) rc = mk(&mm->psiR[s], dv.psi[s], boxR);
    if (!rc) rc = mk(&mm->psiX[s], dv.psi[s], boxX);
  }
  if (!rc) rc = mk(&mm->bC, dv.b, boxC);
  if (!rc) rc = mk(&mm->dC, dv.d, boxC);
  mm->me_tma = 0;
  if (!rc && dv.nx % 4 == 0) {                                      // row pitch of a 4-byte field: a multiple of 16 B
    const cuuint64_t gdim1[3] = {(cuuint64_t)dv.nx, (cuuint64_t)dv.ny, (cuuint64_t)dv.nz};
    const cuuint64_t gstr1[2] = {4ull * dv.nx, 4ull * dv.nx * dv.ny};
    const cuuint32_t box1[3] = {(cuuint32_t)(dv.nx < TW ? dv.nx : TW), bh, 1};
    auto mk1 = [&](CUtensorMap *m, void *base) -> int {
      const CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, base, gdim1, gstr1, box1, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                             CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
      return r == CUDA_SUCCESS ? 0 : -(int)r;
    };
    rc = mk1(&mm->muC, dv.mu);
    if (!rc) rc = mk1(&mm->epsC, dv.eps);
    if (!rc) mm->me_tma = 1;
  }
  return rc;
}

template <int MODE, bool YZ> static cudaError_t cfg_one() {
  return cudaFuncSetAttribute(k_march_tma<MODE, YZ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg<MODE>::SMEM);
}
cudaError_t march_tma_configure() {
  cudaError_t e;
  if ((e = cfg_one<MODE_SWEEP, false>()) != cudaSuccess) return e;
  if ((e = cfg_one<MODE_INIT, false>()) != cudaSuccess) return e;
  if ((e = cfg_one<MODE_RHO, false>()) != cudaSuccess) return e;
  if ((e = cfg_one<MODE_SWEEP, true>()) != cudaSuccess) return e;
  if ((e = cfg_one<MODE_INIT, true>()) != cudaSuccess) return e;
  return cfg_one<MODE_RHO, true>();
}

int march_tma_tile_w() { return TW; }

void march_tma_grid(int nx, int ny, int *gx, int *gy) {
  *gx = (nx + TW - 1) / TW;
  *gy = (ny + TH - 1) / TH;
}

template <bool YZ> static void launch_g(int mode, const Dev &dv, const MarchMaps &mm, dim3 grid, cudaStream_t st) {
  if (mode == MODE_SWEEP) k_march_tma<MODE_SWEEP, YZ><<<grid, NTHREADS, Cfg<MODE_SWEEP>::SMEM, st>>>(dv, mm);
  else if (mode == MODE_INIT) k_march_tma<MODE_INIT, YZ><<<grid, NTHREADS, Cfg<MODE_INIT>::SMEM, st>>>(dv, mm);
  else k_march_tma<MODE_RHO, YZ><<<grid, NTHREADS, Cfg<MODE_RHO>::SMEM, st>>>(dv, mm);
}
void launch_march_tma(int mode, const Dev &dv, const MarchMaps &mm, dim3 grid, cudaStream_t st) {
  if (dv.gauge_yz) launch_g<true>(mode, dv, mm, grid, st);
  else launch_g<false>(mode, dv, mm, grid, st);
}
