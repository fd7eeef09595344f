// Two Jacobi sweeps in one pass over HBM (temporal blocking of Eq. 33): the plain sweep
// (march_tma.cu) is at the HBM roofline with 32 B/site, so the next factor can only come from not writing x^{l+1}
// and not re-reading b, d for sweep l+2.  Per site this kernel reads x^l, b, d once (plus the halo of its tile) and
// writes x^{l+2}: 32 B instead of 64 B for the two sweeps.
//
// A CTA of 19 warps owns a 128 x 16 tile of the xy plane and marches through a chunk of z planes, two pipeline
// stages per iteration t:
//   stage 1  x^{l+1} of plane p1 = k0 - 1 + t on the tile grown by one site (rows -1 .. 16: warps 0 .. 17, one row
//            each; columns -1 and 128: the column warp, 18), from x^l planes p1 - 1, p1 (registers) and p1 + 1 (TMA
//            stage), written to a three-plane shared-memory ring Y;
//   stage 2  x^{l+2} of plane p2 = p1 - 1 on the tile itself (warps 1 .. 16) from x^{l+1} planes p2 - 1, p2 and the
//            in-plane neighbours (all in Y) and p2 + 1 (just computed, registers), written to HBM.
// Both stages use the arithmetic of the plain sweep (nsum_pair / divide_pair, same operand order, contractions
// spelled out), so x^{l+1}, x^{l+2}, both residuals and the J_av partial sums are bit-identical to two plain sweeps.
// Criterion (34) stays exact: the residuals of BOTH sweeps are reduced; if the first one already meets it, the pair
// is discarded (x^l is intact in its buffer) and the plain sweep recomputes x^{l+1} (pair_decide, march_common.cuh).
//
// TMA: one stage = x^l rows -2 .. 17 of plane p1 + 1 (three boxes: centre 16 rows, two rows below, two above;
// wrapped rows for tiles at a periodic seam) and the b, d rows -1 .. 16 of plane p1; ring of 3 stages (56 KB each).
// The column warp feeds itself with plain 16-byte loads one plane ahead and hands the x^l halo columns to the row
// warps through a small shared array; it also issues the TMA copies.
// Eligible meshes: xz gauge, nx % 128 == 0, ny % 16 == 0, ny >= 32, nz >= 4 (march_pair_ok); everything else runs
// plain sweeps only.
#include "march_common.cuh"
#include "march_pair.h"

namespace {

constexpr int TW = 128;                              // tile width (sites)
constexpr int PH = 16;                               // tile height (rows)
constexpr int NROWW = PH + 2;                        // row warps: tile rows -1 .. PH
constexpr int CW = NROWW;                            // index of the column warp
constexpr int NT = 32 * (NROWW + 1);                 // 608 threads
constexpr unsigned ROWB = 8u * TW;                   // bytes per tile row
constexpr unsigned OFF_X = 0;                        // x^l: row slots for rows -2 .. PH+1
constexpr unsigned OFF_B = (PH + 4) * ROWB;          // b: row slots for rows -1 .. PH
constexpr unsigned OFF_D = OFF_B + (PH + 2) * ROWB;
constexpr unsigned SB = OFF_D + (PH + 2) * ROWB;     // 57344 bytes per stage
constexpr int NS = 3;
constexpr unsigned YPITCH = 8u * (TW + 4);           // Y row: columns -2 .. TW+1, column c at (c + 2) * 8
constexpr unsigned YPLANE = NROWW * YPITCH;          // rows -1 .. PH
constexpr unsigned HDR = 256;                        // mbarriers at 0, residual words at 64, J_av row sums at 128
constexpr unsigned OFF_Y = HDR + NS * SB;
constexpr unsigned XHPLANE = 2u * NROWW * 8u;        // x^l halo columns of one plane: [side][row] float2
constexpr int NY = 3;                                // Y ring: x^{l+1} planes p1 - 2, p1 - 1, p1
constexpr unsigned OFF_XH = OFF_Y + NY * YPLANE;
constexpr unsigned SMEM = OFF_XH + 2 * XHPLANE;

__device__ __forceinline__ void sts128(unsigned a, const float4 &v) {
  asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};\n" ::"r"(a), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}
__device__ __forceinline__ void sts64(unsigned a, const float2 &v) {
  asm volatile("st.shared.v2.f32 [%0], {%1, %2};\n" ::"r"(a), "f"(v.x), "f"(v.y) : "memory");
}

__global__ void __launch_bounds__(NT, 1) k_march_pair(const __grid_constant__ Dev dv, const __grid_constant__ PairMaps pm) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  Ctl *ctl = dv.ctl;
  if ((blockIdx.x | blockIdx.y | blockIdx.z | threadIdx.x) == 0) ctl->body_launches += 1;
  if (ctl->done || !ctl->use_pair) return;
  const int l = ctl->sweeps;
  const int xb = ctl->xbuf;

  const int nx = dv.nx, ny = dv.ny, nz = dv.nz;
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const int i0 = blockIdx.x * TW, j0 = blockIdx.y * PH;
  const int k0 = blockIdx.z * dv.zc, k1 = min(nz, k0 + dv.zc);
  const int nk = k1 - k0;
  const bool px = dv.bcx == 0, py = dv.bcy == 0, pz = dv.bcz == 0;
  const long long plane = (long long)nx * ny;
  const unsigned sbase = smem_u32(smem_raw);
  const unsigned stage0 = sbase + HDR;
  const unsigned ybase = sbase + OFF_Y, xhbase = sbase + OFF_XH;

  // planes: stage 1 runs for t in [tb, te], stage 2 for t in [2, nk + 1]; open z faces have no plane beyond them
  const bool lo_ghost = !pz && k0 == 0, hi_ghost = !pz && k1 == nz;
  const int tb = lo_ghost ? 1 : 0, te = hi_ghost ? nk : nk + 1;
  auto zw = [&](int kp) -> int {                       // plane index with wrap / mirror
    if (kp < 0) return pz ? kp + nz : -kp;
    if (kp >= nz) return pz ? kp - nz : 2 * (nz - 1) - kp;
    return kp;
  };
  // rows: the halo rows exist unless the tile touches an open y face (there the ghost row is the mirror image of a
  // row of the tile itself)
  const bool loRow = j0 > 0 || py, hiRow = j0 + PH < ny || py;
  const int jlo = j0 > 0 ? j0 - 1 : ny - 1, jhi = j0 + PH < ny ? j0 + PH : 0;
  // columns: likewise
  const bool wCol = i0 > 0 || px, eCol = i0 + TW < nx || px;
  const int xWp = i0 > 0 ? i0 - 2 : nx - 2, xEp = i0 + TW < nx ? i0 + TW : 0;     // first site of the halo column pair

  // ---- producer: stage s holds x^l plane zw(k0 - 1 + s) and (s > tb) b, d of plane zw(k0 - 2 + s) --------------
  const CUtensorMap *mC = &pm.psiC[xb], *mR = &pm.psiR2[xb];
  auto issue = [&](int s) {
    const unsigned slot = (unsigned)(s - tb) % NS;
    const unsigned sb = stage0 + slot * SB, bar = sbase + 8u * slot;
    const int kz = zw(k0 - 1 + s), kb = zw(k0 - 2 + s);
    const bool bd = s > tb;
    const unsigned rows_x = PH + (loRow ? 2u : 0u) + (hiRow ? 2u : 0u), rows_b = PH + (loRow ? 1u : 0u) + (hiRow ? 1u : 0u);
    mbar_expect_tx(bar, ROWB * (rows_x + (bd ? 2u * rows_b : 0u)));
    tma_load_3d(sb + OFF_X + 2 * ROWB, mC, 2 * i0, j0, kz, bar);
    if (loRow) tma_load_3d(sb + OFF_X, mR, 2 * i0, jlo - 1, kz, bar);
    if (hiRow) tma_load_3d(sb + OFF_X + (PH + 2) * ROWB, mR, 2 * i0, jhi, kz, bar);
    if (bd) {
      tma_load_3d(sb + OFF_B + ROWB, &pm.bC, 2 * i0, j0, kb, bar);
      tma_load_3d(sb + OFF_D + ROWB, &pm.dC, 2 * i0, j0, kb, bar);
      if (loRow) {
        tma_load_3d(sb + OFF_B, &pm.bR, 2 * i0, jlo, kb, bar);
        tma_load_3d(sb + OFF_D, &pm.dR, 2 * i0, jlo, kb, bar);
      }
      if (hiRow) {
        tma_load_3d(sb + OFF_B + (PH + 1) * ROWB, &pm.bR, 2 * i0, jhi, kb, bar);
        tma_load_3d(sb + OFF_D + (PH + 1) * ROWB, &pm.dR, 2 * i0, jhi, kb, bar);
      }
    }
  };
  auto stage_of = [&](int s) -> unsigned { return stage0 + ((unsigned)(s - tb) % NS) * SB; };
  auto wait_stage = [&](int s) { mbar_wait(sbase + 8u * ((unsigned)(s - tb) % NS), ((unsigned)(s - tb) / NS) & 1u); };

  if (tid == 0) {
    for (int s = 0; s < NS; ++s) mbar_init(sbase + 8u * s, 1u);
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    *reinterpret_cast<unsigned *>(smem_raw + 64) = 0u;              // CTA max-residual words of the two sweeps
    *reinterpret_cast<unsigned *>(smem_raw + 68) = 0u;
  }
  __syncthreads();
  if (tid == CW * 32) { issue(tb); issue(tb + 1); }

  const float2 *__restrict__ xin = dv.psi[xb];
  float2 *__restrict__ xout = dv.psi[xb ^ 1];
  const float f = dv.ht2;
  float rmax1 = 0.f, rmax2 = 0.f;
  double jacc = 0.0;
  const bool jact = dv.solve_mu && px;

  if (w < NROWW) {
    // ======================================= row warps ===========================================================
    const int rr = w - 1;                                            // tile row -1 .. PH
    const bool centre = rr >= 0 && rr < PH;
    const bool act1 = centre || (rr < 0 ? loRow : hiRow);            // this row takes part in stage 1
    const int jr = centre ? j0 + rr : (rr < 0 ? jlo : jhi);          // its row of the mesh
    const bool ylo = py && jr == 0, yhi = py && jr == ny - 1;        // quasi-periodic jump rows
    const bool mlo = !py && jr == 0, mhi = !py && jr == ny - 1;      // open y faces: mirror (U_y = 1)
    const unsigned oX = OFF_X + (unsigned)(rr + 2) * ROWB + 16u * lane;          // own sites, pair A (B: + 512)
    const unsigned oN = mhi ? oX - ROWB : oX + ROWB, oS = mlo ? oX + ROWB : oX - ROWB;
    const unsigned oBD = (unsigned)(rr + 1) * ROWB + 16u * lane;                 // within the b / d block
    const unsigned oY = (unsigned)(rr + 1) * YPITCH + 16u + 16u * lane;          // own sites in a Y plane
    const unsigned oYN = mhi ? oY - YPITCH : oY + YPITCH, oYS = mlo ? oY + YPITCH : oY - YPITCH;
    const unsigned oXrow = OFF_X + (unsigned)(rr + 2) * ROWB, oYrow = (unsigned)(rr + 1) * YPITCH;
    const unsigned oXH = (unsigned)(rr + 1) * 8u;                                // + side * NROWW * 8
    const int iA = i0 + 2 * lane, iB = iA + 64;
    const bool xloA = !px && iA == 0, xhiB = !px && iB + 1 == nx - 1;            // open x faces
    const float2 Uxj = dv.Ux[jr], Uzj = dv.Uz[jr];
    const Links L = make_links(make_float2(f * dv.cx * Uxj.x, f * dv.cx * Uxj.y),
                               make_float2(f * dv.cz * Uzj.x, f * dv.cz * Uzj.y), f * dv.cy);
    const float2 U2z = cmul(Uzj, Uzj);
    const long long rowoff = (long long)jr * nx + iA;
    long long idx2 = (long long)k0 * plane + rowoff;                 // stage 2 output index of pair A

    // The Jacobi update of this thread's four sites of plane `kp`; shared by both stages.  C = own values of that
    // plane, T / B = own values of the planes above / below (registers); the in-plane neighbours and b, d are read
    // from shared memory at the given addresses (x^l from a TMA stage or x^{l+1} from a Y plane; pair B at + 512):
    // aN, aS = rows above / below, aW / aE = the sites left of site 0 / right of site 127 (lanes 0 / 31 only),
    // aM = site 63 of the own row (sites 63 | 64 are the seam between the pairs of lanes 31 and 0).
    // One half (pair) at a time keeps the live registers under the 96 of a 608-thread CTA.
    auto update = [&](int kp, const float4 &CA, const float4 &CB, const float4 &TA, const float4 &TB, const float4 &BA,
                      const float4 &BB, unsigned aN, unsigned aS, unsigned aW, unsigned aE, unsigned aM, unsigned ab,
                      unsigned ad, float &rmax, float4 &outA, float4 &outB) {
      float2 WA, EA, WB, EB;
      WA.x = __shfl_up_sync(0xffffffffu, CA.z, 1);   WA.y = __shfl_up_sync(0xffffffffu, CA.w, 1);
      EA.x = __shfl_down_sync(0xffffffffu, CA.x, 1); EA.y = __shfl_down_sync(0xffffffffu, CA.y, 1);
      WB.x = __shfl_up_sync(0xffffffffu, CB.z, 1);   WB.y = __shfl_up_sync(0xffffffffu, CB.w, 1);
      EB.x = __shfl_down_sync(0xffffffffu, CB.x, 1); EB.y = __shfl_down_sync(0xffffffffu, CB.y, 1);
      if (lane == 0) { WA = lds64(aW); WB = lds64(aM); }
      if (lane == 31) { EA = lds64(aM + 8u); EB = lds64(aE); }
      if (xloA) WA = cmul(cmul(Uxj, Uxj), hi(CA));       // open x faces: W' = U^2 E, E' = U*^2 W
      if (xhiB) EB = cmulc(cmul(Uxj, Uxj), lo(CB));
      float rloc = 0.f;
      auto half = [&](const float4 &C, const float4 &T, const float4 &B, float2 W, float2 E, unsigned o, int i, float4 &out) {
        float4 Nn = lds128(aN + o), Ss = lds128(aS + o);
        if (ylo || yhi) {                                // quasi-periodic jump in y, P_{i,k} = Pi[i] conj(Pk[k])
          const float2 Pk = dv.Pk[kp];
          const float4 Pi = *reinterpret_cast<const float4 *>(dv.Pi + i);
          const float2 P0 = cmulc(Pk, lo(Pi)), P1 = cmulc(Pk, hi(Pi));
          if (ylo) {                                     // psi_{i,-1,k} = P psi_{i,ny-1,k}
            const float2 a = cmul(P0, lo(Ss)), b2 = cmul(P1, hi(Ss));
            Ss = make_float4(a.x, a.y, b2.x, b2.y);
          }
          if (yhi) {                                     // psi_{i,ny,k} = P* psi_{i,0,k}
            const float2 a = cmulc(P0, lo(Nn)), b2 = cmulc(P1, hi(Nn));
            Nn = make_float4(a.x, a.y, b2.x, b2.y);
          }
        }
        const float4 b = lds128(ab + o);
        float2 s0 = lo(b), s1 = hi(b);
        nsum_pair(L, C, W, E, Nn, Ss, T, B, s0, s1);
        out = divide_pair(s0, s1, lds128(ad + o), C, rloc);
      };
      half(CA, TA, BA, WA, EA, 0u, iA, outA);
      half(CB, TB, BB, WB, EB, 512u, iB, outB);
      rmax = fmaxf(rmax, rloc);
    };

    // x^l ring: this thread's values of planes p1 - 1, p1 stay in registers while plane p1 + 1 arrives
    float4 xA[3], xB[3];
    for (int q = 0; q < 3; ++q) xA[q] = xB[q] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (act1) {
      const long long ob = (long long)zw(k0 - 2 + tb) * plane + rowoff;          // plane below the first stage-1 plane
      xA[0] = __ldg(reinterpret_cast<const float4 *>(xin + ob));
      xB[0] = __ldg(reinterpret_cast<const float4 *>(xin + ob + 64));
      if (lo_ghost) { xA[0] = cmul4(U2z, xA[0]); xB[0] = cmul4(U2z, xB[0]); }   // psi_{-1} = U_z^2 psi_1
    }
    wait_stage(tb);
    if (act1) {
      xA[1] = lds128(stage_of(tb) + oX);
      xB[1] = lds128(stage_of(tb) + oX + 512u);
    }

    float rdummy = 0.f;                                              // residuals of the halo rows belong to other tiles
    auto iter = [&](int t, float4 &B1A, float4 &B1B, float4 &C1A, float4 &C1B, float4 &T1A, float4 &T1B) {
      __syncthreads();
      const bool do1 = t <= te;
      const unsigned prv = stage_of(t);
      const unsigned ym = (unsigned)t % NY;
      float4 T2A, T2B;                                               // x^{l+1} of plane p1: stage 1 -> stage 2
      if (do1) {
        const int p1 = k0 - 1 + t;
        const unsigned cur = stage_of(t + 1);
        wait_stage(t + 1);
        if (act1) {
          T1A = lds128(cur + oX);
          T1B = lds128(cur + oX + 512u);
          if (hi_ghost && t == nk) { T1A = cmulc4(U2z, T1A); T1B = cmulc4(U2z, T1B); }   // psi_{nz} = U_z*^2 psi_{nz-2}
          const unsigned xh = xhbase + (unsigned)(t & 1) * XHPLANE + oXH;
          update(zw(p1), C1A, C1B, T1A, T1B, B1A, B1B, prv + oN, prv + oS, xh, xh + NROWW * 8u, prv + oXrow + 8u * 63u,
                 cur + OFF_B + oBD, cur + OFF_D + oBD, centre ? rmax1 : rdummy, T2A, T2B);
          const unsigned yw = ybase + ym * YPLANE + oY;
          sts128(yw, T2A);
          sts128(yw + 512u, T2B);
        }
      }
      if (centre && t >= 2) {
        const int p2 = k0 - 2 + t;
        const unsigned yr = ybase + ((ym + NY - 1) % NY) * YPLANE;     // plane p2
        const unsigned yb = ybase + ((ym + NY - 2) % NY) * YPLANE;     // plane p2 - 1
        const float4 C2A = lds128(yr + oY), C2B = lds128(yr + oY + 512u);
        float4 B2A, B2B;
        if (lo_ghost && t == 2) { B2A = cmul4(U2z, T2A); B2B = cmul4(U2z, T2B); }   // open bottom face
        else { B2A = lds128(yb + oY); B2B = lds128(yb + oY + 512u); }
        if (!do1) { T2A = cmulc4(U2z, B2A); T2B = cmulc4(U2z, B2B); }               // open top face, sweep l + 2
        float4 outA, outB;
        update(p2, C2A, C2B, T2A, T2B, B2A, B2B, yr + oYN, yr + oYS, yr + oYrow + 8u, yr + oYrow + 8u * (TW + 2),
               yr + oYrow + 8u * 65u, prv + OFF_B + oBD, prv + OFF_D + oBD, rmax2, outA, outB);
        *reinterpret_cast<float4 *>(xout + idx2) = outA;
        *reinterpret_cast<float4 *>(xout + idx2 + 64) = outB;
        idx2 += plane;
        if (jact) {
          // J_av (Eq. 35): x links of x^{l+2} inside the tile row, exactly as the plain sweep sums them
          const float nAx = __shfl_down_sync(0xffffffffu, outA.x, 1), nAy = __shfl_down_sync(0xffffffffu, outA.y, 1);
          const float rBx = __shfl_sync(0xffffffffu, outB.x, (lane + 1) & 31), rBy = __shfl_sync(0xffffffffu, outB.y, (lane + 1) & 31);
          const float2 nxA = (lane == 31) ? make_float2(rBx, rBy) : make_float2(nAx, nAy);
          float tsum = 0.f;
          tsum += jlink(Uxj, outA.x, outA.y, outA.z, outA.w);
          tsum += jlink(Uxj, outA.z, outA.w, nxA.x, nxA.y);
          tsum += jlink(Uxj, outB.x, outB.y, outB.z, outB.w);
          if (lane < 31) tsum += jlink(Uxj, outB.z, outB.w, rBx, rBy);
          jacc += (double)tsum;
        }
      }
    };

    // z march; the register ring rotates by renaming over three unrolled iterations
    for (int t = tb; t <= nk + 1; t += 3) {
      iter(t, xA[0], xB[0], xA[1], xB[1], xA[2], xB[2]);
      if (t + 1 <= nk + 1) iter(t + 1, xA[1], xB[1], xA[2], xB[2], xA[0], xB[0]);
      if (t + 2 <= nk + 1) iter(t + 2, xA[2], xB[2], xA[0], xB[0], xA[1], xB[1]);
    }
  } else {
    // ======================================= column warp =========================================================
    // lane q < 18 owns the halo sites of tile row q - 1: (row, i0 - 1) on the west side (second site of the pair
    // loaded from xWp) and (row, i0 + 128) on the east side (first site of the pair loaded from xEp); rows -1 and 16
    // only supply their x^l values (corners of the halo).
    const int rr = lane - 1;
    const bool rowok = lane < NROWW && ((rr >= 0 && rr < PH) || (rr < 0 ? loRow : hiRow));
    const bool comp = lane < NROWW && rr >= 0 && rr < PH;
    const int jr = (rr >= 0 && rr < PH) ? j0 + rr : (rr < 0 ? jlo : jhi);
    const bool ylo = py && jr == 0, yhi = py && jr == ny - 1, mlo = !py && jr == 0, mhi = !py && jr == ny - 1;
    const bool ldW = rowok && wCol, ldE = rowok && eCol;
    const int jc = min(max(jr, 0), ny - 1);
    const float2 Uxj = dv.Ux[jc], Uzj = dv.Uz[jc];
    const Links L = make_links(make_float2(f * dv.cx * Uxj.x, f * dv.cx * Uxj.y),
                               make_float2(f * dv.cz * Uzj.x, f * dv.cz * Uzj.y), f * dv.cy);
    const float2 U2z = cmul(Uzj, Uzj);
    const float2 PiW = dv.Pi[xWp + 1], PiE = dv.Pi[xEp];
    const long long offW = (long long)jc * nx + xWp, offE = (long long)jc * nx + xEp;
    const unsigned oXrow = OFF_X + (unsigned)(rr + 2) * ROWB;
    const unsigned oXH = (unsigned)(rr + 1) * 8u, oYrow = (unsigned)(rr + 1) * YPITCH;
    const float4 z4 = make_float4(0.f, 0.f, 0.f, 0.f);
    const float2 z2 = make_float2(0.f, 0.f);
    auto ldx = [&](int kp, bool on, long long off) -> float4 {
      return on ? __ldg(reinterpret_cast<const float4 *>(xin + (long long)kp * plane + off)) : z4;
    };
    // rings of the two halo columns (pairs), planes p1 - 1, p1, p1 + 1
    float4 cW[3], cE[3];
    cW[0] = ldx(zw(k0 - 2 + tb), ldW, offW); cE[0] = ldx(zw(k0 - 2 + tb), ldE, offE);
    if (lo_ghost) { cW[0] = cmul4(U2z, cW[0]); cE[0] = cmul4(U2z, cE[0]); }
    cW[1] = ldx(zw(k0 - 1 + tb), ldW, offW); cE[1] = ldx(zw(k0 - 1 + tb), ldE, offE);
    // the x^l halo columns of the first stage-1 plane for the row warps
    if (ldW) sts64(xhbase + (unsigned)(tb & 1) * XHPLANE + oXH, hi(cW[1]));
    if (ldE) sts64(xhbase + (unsigned)(tb & 1) * XHPLANE + NROWW * 8u + oXH, lo(cE[1]));
    // prefetch: plane p1 + 1 of the first iteration and its b, d
    float4 nW = ldx(zw(k0 + tb), ldW, offW), nE = ldx(zw(k0 + tb), ldE, offE);
    auto ldbd = [&](const float2 *arr, int kp, bool on, long long off) -> float2 {
      return on ? __ldg(arr + (long long)kp * plane + off) : z2;
    };
    const bool cpW = comp && wCol, cpE = comp && eCol;
    float2 bW = ldbd(dv.b, zw(k0 - 1 + tb), cpW, offW + 1), dW = ldbd(dv.d, zw(k0 - 1 + tb), cpW, offW + 1);
    float2 bE = ldbd(dv.b, zw(k0 - 1 + tb), cpE, offE), dE = ldbd(dv.d, zw(k0 - 1 + tb), cpE, offE);

    auto site = [&](int kp, float2 C, float2 Wn, float2 En, float2 T, float2 B, float2 Pi, float2 b, float2 d) -> float2 {
      float2 Nn = make_float2(__shfl_down_sync(0xffffffffu, C.x, 1), __shfl_down_sync(0xffffffffu, C.y, 1));
      float2 Sn = make_float2(__shfl_up_sync(0xffffffffu, C.x, 1), __shfl_up_sync(0xffffffffu, C.y, 1));
      if (mlo) Sn = Nn;
      if (mhi) Nn = Sn;
      if (ylo || yhi) {
        const float2 P = cmulc(dv.Pk[kp], Pi);
        if (ylo) Sn = cmul(P, Sn);
        if (yhi) Nn = cmulc(P, Nn);
      }
      const float2 s = nsum_site(L, b, Wn, En, Nn, Sn, T, B);
      float r = 0.f;
      const float4 o = divide_pair(s, s, make_float4(d.x, d.y, d.x, d.y), make_float4(C.x, C.y, C.x, C.y), r);
      return lo(o);
    };

    auto iter = [&](int t, float4 &BW, float4 &BE, float4 &CWv, float4 &CEv, float4 &TW_, float4 &TE_) {
      __syncthreads();
      if (lane == 0 && t + 2 <= te + 1) issue(t + 2);
      if (t <= te) {
        const int p1 = k0 - 1 + t;
        const unsigned prv = stage_of(t);
        wait_stage(t);                                                  // (complete since the last iteration: visibility only)
        TW_ = nW; TE_ = nE;
        const float2 b_w = bW, d_w = dW, b_e = bE, d_e = dE;
        if (t + 1 <= te) {                                              // next plane's loads in flight during this one
          nW = ldx(zw(p1 + 2), ldW, offW); nE = ldx(zw(p1 + 2), ldE, offE);
          bW = ldbd(dv.b, zw(p1 + 1), cpW, offW + 1); dW = ldbd(dv.d, zw(p1 + 1), cpW, offW + 1);
          bE = ldbd(dv.b, zw(p1 + 1), cpE, offE); dE = ldbd(dv.d, zw(p1 + 1), cpE, offE);
        }
        if (hi_ghost && t == nk) { TW_ = cmulc4(U2z, TW_); TE_ = cmulc4(U2z, TE_); }
        // hand the x^l halo columns of plane p1 + 1 to the row warps of the next iteration
        const unsigned xh = xhbase + (unsigned)((t + 1) & 1) * XHPLANE + oXH;
        if (ldW) sts64(xh, hi(TW_));
        if (ldE) sts64(xh + NROWW * 8u, lo(TE_));
        // stage 1 on the halo sites (tile rows 0 .. PH-1); neighbours inside the tile come from the TMA stage
        const unsigned yw = ybase + ((unsigned)t % NY) * YPLANE + oYrow;
        if (wCol) {                                                     // warp-uniform
          const float2 En = comp ? lds64(prv + oXrow) : z2;
          const float2 o = site(zw(p1), hi(CWv), lo(CWv), En, hi(TW_), hi(BW), PiW, b_w, d_w);
          if (comp) sts64(yw + 8u, o);
        }
        if (eCol) {
          const float2 Wn = comp ? lds64(prv + oXrow + 8u * (TW - 1)) : z2;
          const float2 o = site(zw(p1), lo(CEv), Wn, hi(CEv), lo(TE_), lo(BE), PiE, b_e, d_e);
          if (comp) sts64(yw + 8u * (TW + 2), o);
        }
      }
    };
    for (int t = tb; t <= nk + 1; t += 3) {
      iter(t, cW[0], cE[0], cW[1], cE[1], cW[2], cE[2]);
      if (t + 1 <= nk + 1) iter(t + 1, cW[1], cE[1], cW[2], cE[2], cW[0], cE[0]);
      if (t + 2 <= nk + 1) iter(t + 2, cW[2], cE[2], cW[0], cE[0], cW[1], cE[1]);
    }
  }

  // ---- residuals of both sweeps, J_av partial sums, the decision of the last CTA ---------------------------------
  unsigned *s_max = reinterpret_cast<unsigned *>(smem_raw + 64);
  double *s_j = reinterpret_cast<double *>(smem_raw + 128);
  const bool crow = w >= 1 && w <= PH;
  if (crow) {
    const unsigned m1 = __reduce_max_sync(0xffffffffu, __float_as_uint(rmax1));
    const unsigned m2 = __reduce_max_sync(0xffffffffu, __float_as_uint(rmax2));
    if (lane == 0) { atomicMax(s_max, m1); atomicMax(s_max + 1, m2); }
    if (jact) {
      for (int o = 16; o > 0; o >>= 1) jacc += __shfl_down_sync(0xffffffffu, jacc, o);
      if (lane == 0) s_j[w - 1] = jacc;
    }
  }
  __syncthreads();
  if (tid == 0) {
    if (jact) {                                          // one partial per 128 x 8 tile of the plain sweep's grid, same order
      const unsigned gy8 = 2u * gridDim.y;
      for (int hlf = 0; hlf < 2; ++hlf) {
        double sj = 0.0;
        for (int q = 0; q < 8; ++q) sj += s_j[8 * hlf + q];
        dv.jpart[blockIdx.x + gridDim.x * ((2u * blockIdx.y + hlf) + gy8 * blockIdx.z)] = sj;
      }
    }
    atomicMax(&ctl->resid_bits[l], s_max[0]);
    atomicMax(&ctl->resid_bits[l + 1], s_max[1]);
    __threadfence();
    const unsigned nb = gridDim.x * gridDim.y * gridDim.z;
    const unsigned tk = atomicAdd(&ctl->ticket, 1u);
    if (tk == nb - 1) {
      ctl->ticket = 0u;
      pair_decide(dv, l);
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
bool march_pair_ok(int nx, int ny, int nz, bool gauge_yz) {
  return !gauge_yz && nx % TW == 0 && ny % PH == 0 && ny >= 2 * PH && nz >= 4;
}

int march_pair_build_maps(const Dev &dv, PairMaps *pm) {
  void *fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
      qres != cudaDriverEntryPointSuccess)
    return -1000;
  EncodeTiledFn enc = (EncodeTiledFn)fn;
  const cuuint64_t gdim[3] = {2ull * dv.nx, (cuuint64_t)dv.ny, (cuuint64_t)dv.nz};
  const cuuint64_t gstr[2] = {8ull * dv.nx, 8ull * dv.nx * dv.ny};
  const cuuint32_t es[3] = {1, 1, 1};
  const cuuint32_t boxC[3] = {2 * TW, PH, 1}, boxR2[3] = {2 * TW, 2, 1}, boxR1[3] = {2 * TW, 1, 1};
  auto mk = [&](CUtensorMap *m, void *base, const cuuint32_t *box) -> int {
    const CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, base, gdim, gstr, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                           CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? 0 : -(int)r;
  };
  int rc = 0;
  for (int s = 0; s < 2 && !rc; ++s) {
    if (!rc) rc = mk(&pm->psiC[s], dv.psi[s], boxC);
    if (!rc) rc = mk(&pm->psiR2[s], dv.psi[s], boxR2);
  }
  if (!rc) rc = mk(&pm->bC, dv.b, boxC);
  if (!rc) rc = mk(&pm->dC, dv.d, boxC);
  if (!rc) rc = mk(&pm->bR, dv.b, boxR1);
  if (!rc) rc = mk(&pm->dR, dv.d, boxR1);
  return rc;
}

cudaError_t march_pair_configure() {
  return cudaFuncSetAttribute(k_march_pair, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM);
}

// grid: the plain sweep's z chunks (dv.zc) so that both kernels fill the same J_av partial sums
void launch_march_pair(const Dev &dv, const PairMaps &pm, cudaStream_t st) {
  const dim3 grid((unsigned)(dv.nx / TW), (unsigned)(dv.ny / PH), (unsigned)((dv.nz + dv.zc - 1) / dv.zc));
  k_march_pair<<<grid, NT, SMEM, st>>>(dv, pm);
}
