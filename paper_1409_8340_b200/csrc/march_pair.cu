// Two Jacobi sweeps in one pass over HBM (temporal blocking of Eq. 33): the plain sweep
// (march_tma.cu) is at the HBM roofline with 32 B/site, so the next factor can only come from not writing x^{l+1}
// and not re-reading b, d for sweep l+2.  Per site this kernel reads x^l, b, d once (plus the halo of its tile) and
// writes x^{l+2}: 32 B instead of 64 B for the two sweeps.
//
// A CTA of 20 warps owns a 128 x 16 tile of the xy plane and marches through a chunk of z planes, two pipeline
// stages per iteration t:
//   stage 1  x^{l+1} of plane p1 = k0 - 1 + t on the tile grown by one site (rows -1 .. 16: warps 0 .. 17, one row
//            each; columns -1 and 128: one warp each, 18 and 19), from x^l planes p1 - 1 (registers), p1 and p1 + 1 (the
//            two resident TMA stages), written to a three-plane shared-memory ring Y;
//   stage 2  x^{l+2} of plane p2 = p1 - 1 on the tile itself (warps 1 .. 16) from x^{l+1} planes p2 - 1, p2 and the
//            in-plane neighbours (all in Y) and p2 + 1 (just computed, registers), written to HBM.
// Both stages use the arithmetic of the plain sweep (nsum_pair / divide_pair, same operand order, contractions
// spelled out), so x^{l+1}, x^{l+2}, both residuals and the J_av partial sums are bit-identical to two plain sweeps.
// Criterion (34) stays exact: the residuals of BOTH sweeps are reduced; if the first one already meets it, the pair
// is discarded (x^l is intact in its buffer) and the plain sweep recomputes x^{l+1} (pair_decide, march_common.cuh).
// The J_av link sums of x^{l+2} are formed only if this pair may end the step (choose_next); k_jav_tiles below supplies
// them, bit-identically, in the rare case that a pair that skipped them did end it.
//
// TMA: one stage = x^l rows -2 .. 17 of plane p1 + 1 (three boxes: centre 16 rows, two rows below, two above;
// wrapped rows for tiles at a periodic seam) and the b, d rows -1 .. 16 of plane p1; ring of 3 stages (56 KB each).
// The column warps feed themselves with plain 16-byte loads one plane ahead and hand the x^l halo columns to the row
// warps through a small shared array; warp 0 (a halo row: half the work of a centre row) issues the TMA copies.
// Eligible meshes: xz gauge, nx % 128 == 0, ny % 16 == 0, ny >= 32, nz >= 4 (march_pair_ok); everything else runs
// plain sweeps only.
#include "march_common.cuh"
#include "march_pair.h"
#include <type_traits>

namespace {

constexpr int TW = 128;                              // tile width (sites)
constexpr int PH = 16;                               // tile height (rows)
constexpr int NROWW = PH + 2;                        // row warps: tile rows -1 .. PH
constexpr int NT = 32 * (NROWW + 2);                 // + two column warps: 640 threads (17 .. 20 warps leave 96 registers each)
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
    const unsigned rows_x = PH + 4u, rows_b = PH + (loRow ? 1u : 0u) + (hiRow ? 1u : 0u);
    mbar_expect_tx(bar, ROWB * (rows_x + (bd ? 2u * rows_b : 0u)));
    tma_load_3d(sb + OFF_X + 2 * ROWB, mC, 2 * i0, j0, kz, bar);
    // the two rows below / above the tile: real or wrapped rows, or -- at an open y face -- the rows whose mirror
    // images they are (P:483 with U_y = 1: row -1 = row 1, row ny = row ny - 2), so that "row +- 1" is always one slot away
    tma_load_3d(sb + OFF_X, mR, 2 * i0, loRow ? jlo - 1 : 0, kz, bar);
    tma_load_3d(sb + OFF_X + (PH + 2) * ROWB, mR, 2 * i0, hiRow ? jhi : ny - 2, kz, bar);
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
  if (tid == 0) { issue(tb); issue(tb + 1); }

  const float2 *__restrict__ xin = dv.psi[xb];
  float2 *__restrict__ xout = dv.psi[xb ^ 1];
  const float f = dv.ht2;
  float rmax1 = 0.f, rmax2 = 0.f;
  double jacc = 0.0;
  const bool jact = dv.solve_mu && px && ctl->pair_jav;   // J_av link sums only if this pair may end the step (choose_next)

  if (w < NROWW) {
    // ======================================= row warps ===========================================================
    const int rr = w - 1;                                            // tile row -1 .. PH
    const bool centre = rr >= 0 && rr < PH;
    const bool act1 = centre || (rr < 0 ? loRow : hiRow);            // this row takes part in stage 1
    const int jr = centre ? j0 + rr : (rr < 0 ? jlo : jhi);          // its row of the mesh
    const bool ylo = py && jr == 0, yhi = py && jr == ny - 1;        // quasi-periodic jump rows
    // open y faces: the x^{l+1} ghost rows of stage 2 are the mirror images of rows 1 and ny - 2, stored twice
    const bool dupLo = !py && jr == 1, dupHi = !py && jr == ny - 2;
    const unsigned oX = OFF_X + (unsigned)(rr + 2) * ROWB + 16u * lane;          // own sites in a stage, pair A (B: + 512);
    constexpr unsigned DB = OFF_B - ROWB, DD = OFF_D - ROWB;                     //   b, d of the same sites at oX + DB, + DD
    const unsigned oY = (unsigned)(rr + 1) * YPITCH + 16u + 16u * lane;          // own sites in a Y plane
    const unsigned oXH = (unsigned)(rr + 1) * 8u;                                // + side * NROWW * 8
    const bool xloA = !px && i0 + 2 * lane == 0, xhiB = !px && i0 + 64 + 2 * lane + 1 == nx - 1;   // open x faces
    const float2 Uxj = dv.Ux[jr], Uzj = dv.Uz[jr];
    const Links L = make_links(make_float2(f * dv.cx * Uxj.x, f * dv.cx * Uxj.y),
                               make_float2(f * dv.cz * Uzj.x, f * dv.cz * Uzj.y), f * dv.cy);
    const float2 U2z = cmul(Uzj, Uzj);
    const long long rowoff = (long long)jr * nx + i0 + 2 * lane;
    float4 *out2 = reinterpret_cast<float4 *>(xout + (long long)k0 * plane + rowoff);   // stage 2 output, pair A

    // The Jacobi update of ONE pair (two sites) of this thread in plane `kp`; shared by both stages.  C = own values
    // of that plane, T / B = own values of the planes above / below; the in-plane neighbours are read from shared
    // memory: aC = address of the own pair in that plane's buffer (x^l: TMA stage, row pitch ROWB; x^{l+1}: Y plane, row
    // pitch YPITCH), W / E = the x neighbours of the pair's outer sites, ab / ad = b, d of the pair.  One pair at a
    // time keeps the live registers under the 96 of a 608-thread CTA.
    auto half = [&](auto fast_tag, int kp, const unsigned pitch, int col, const float4 &C, const float4 &T, const float4 &B,
                    float2 W, float2 E, unsigned aC, unsigned ab, unsigned ad, float &rmax) -> float4 {
      constexpr bool FAST = decltype(fast_tag)::value;      // no boundary role in this warp and plane: the checks vanish
      float4 Nn = lds128(aC + pitch), Ss = lds128(aC - pitch);
      if (!FAST && (ylo || yhi)) {                       // quasi-periodic jump in y, P_{i,k} = Pi[i] conj(Pk[k])
        const float2 Pk = dv.Pk[kp];
        const float4 Pi = *reinterpret_cast<const float4 *>(dv.Pi + col);
        const float2 P0 = cmulc(Pk, lo(Pi)), P1 = cmulc(Pk, hi(Pi));
        if (ylo) {                                       // psi_{i,-1,k} = P psi_{i,ny-1,k}
          const float2 a = cmul(P0, lo(Ss)), b2 = cmul(P1, hi(Ss));
          Ss = make_float4(a.x, a.y, b2.x, b2.y);
        }
        if (yhi) {                                       // psi_{i,ny,k} = P* psi_{i,0,k}
          const float2 a = cmulc(P0, lo(Nn)), b2 = cmulc(P1, hi(Nn));
          Nn = make_float4(a.x, a.y, b2.x, b2.y);
        }
      }
      const float4 b = lds128(ab);
      float2 s0 = lo(b), s1 = hi(b);
      nsum_pair(L, C, W, E, Nn, Ss, T, B, s0, s1);
      float rloc = 0.f;
      const float4 out = divide_pair(s0, s1, lds128(ad), C, rloc);
      rmax = fmaxf(rmax, rloc);
      return out;
    };
    // x neighbours of pair A (sites 2 lane, 2 lane + 1) and pair B (64 + 2 lane, ...): shuffles, and for lanes 0 / 31
    // the sites left of site 0 (aW) / right of site 127 (aE) and the seam 63 | 64 between the pairs of lanes 31 and 0
    auto xnbA = [&](auto fast_tag, const float4 &CA, unsigned aC, unsigned aW, float2 &W, float2 &E) {
      constexpr bool FAST = decltype(fast_tag)::value;
      W.x = __shfl_up_sync(0xffffffffu, CA.z, 1);   W.y = __shfl_up_sync(0xffffffffu, CA.w, 1);
      E.x = __shfl_down_sync(0xffffffffu, CA.x, 1); E.y = __shfl_down_sync(0xffffffffu, CA.y, 1);
      const float2 e = lds64(lane == 0 ? aW : (lane == 31 ? aC + 16u : xhbase));   // every lane loads (branch-free); the
                                                                                    // idle lanes share one address (broadcast)
      if (lane == 0) W = e;
      if (lane == 31) E = e;
      if (!FAST && xloA) W = cmul(cmul(Uxj, Uxj), hi(CA));          // open x face: W' = U^2 E
    };
    auto xnbB = [&](auto fast_tag, const float4 &CB, unsigned aC, unsigned aE, float2 &W, float2 &E) {
      constexpr bool FAST = decltype(fast_tag)::value;
      W.x = __shfl_up_sync(0xffffffffu, CB.z, 1);   W.y = __shfl_up_sync(0xffffffffu, CB.w, 1);
      E.x = __shfl_down_sync(0xffffffffu, CB.x, 1); E.y = __shfl_down_sync(0xffffffffu, CB.y, 1);
      const float2 e = lds64(lane == 31 ? aE : (lane == 0 ? aC + 8u * 63u : xhbase));   // aC = pair A's address
      if (lane == 0) W = e;
      if (lane == 31) E = e;
      if (!FAST && xhiB) E = cmulc(cmul(Uxj, Uxj), lo(CB));         // open x face: E' = U*^2 W
    };

    // x^l: this thread's values of plane p1 - 1 stay in registers (the stage that held them is being refilled);
    // planes p1 and p1 + 1 are read from the two resident stages
    float4 pA = make_float4(0.f, 0.f, 0.f, 0.f), pB = pA;
    if (act1) {
      const long long ob = (long long)zw(k0 - 2 + tb) * plane + rowoff;          // plane below the first stage-1 plane
      pA = __ldg(reinterpret_cast<const float4 *>(xin + ob));
      pB = __ldg(reinterpret_cast<const float4 *>(xin + ob + 64));
      if (lo_ghost) { pA = cmul4(U2z, pA); pB = cmul4(U2z, pB); }               // psi_{-1} = U_z^2 psi_1
    }
    wait_stage(tb);

    float rdummy = 0.f;                                              // residuals of the halo rows belong to other tiles
    // B1 = plane p1 - 1 on entry, plane p1 on exit.
    // FAST: a warp without boundary role (no jump / mirror row, no open x face) on a plane away from the z faces of the
    // chunk runs a copy of the iteration from which every boundary check is compiled out.
    auto iter = [&](auto fast_tag, int t, float4 &B1A, float4 &B1B) {
      constexpr bool FAST = decltype(fast_tag)::value;
      __syncthreads();
      if (!FAST && tid == 0 && t + 2 <= te + 1) issue(t + 2);        // warp 0 (a halo row: half the work) is the producer
      const bool do1 = FAST || t <= te;
      const unsigned prv = stage_of(t);
      const unsigned ym = (unsigned)t % NY;
      float4 T2A, T2B;                                               // x^{l+1} of plane p1: stage 1 -> stage 2
      if (do1) {
        const int p1 = k0 - 1 + t, kp = FAST ? p1 : zw(p1);
        const unsigned cur = stage_of(t + 1);
        wait_stage(t + 1);
        if (FAST || act1) {
          const unsigned xh = xhbase + (unsigned)(t & 1) * XHPLANE + oXH;
          const bool top = !FAST && hi_ghost && t == nk;             // psi_{nz} = U_z*^2 psi_{nz-2}
          float &r1 = centre ? rmax1 : rdummy;
          float2 W, E;
          {
            const float4 C = lds128(prv + oX);
            float4 T = lds128(cur + oX);
            if (top) T = cmulc4(U2z, T);
            xnbA(fast_tag, C, prv + oX, xh, W, E);
            T2A = half(fast_tag, kp, ROWB, i0 + 2 * lane, C, T, B1A, W, E, prv + oX, cur + oX + DB, cur + oX + DD, r1);
            B1A = C;
          }
          {
            const float4 C = lds128(prv + oX + 512u);
            float4 T = lds128(cur + oX + 512u);
            if (top) T = cmulc4(U2z, T);
            xnbB(fast_tag, C, prv + oX, xh + NROWW * 8u, W, E);
            T2B = half(fast_tag, kp, ROWB, i0 + 64 + 2 * lane, C, T, B1B, W, E, prv + oX + 512u, cur + oX + DB + 512u,
                       cur + oX + DD + 512u, r1);
            B1B = C;
          }
          const unsigned yw = ybase + ym * YPLANE + oY;
          sts128(yw, T2A);
          sts128(yw + 512u, T2B);
          if (!FAST) {
            if (dupLo) { sts128(yw - 2u * YPITCH, T2A); sts128(yw - 2u * YPITCH + 512u, T2B); }
            if (dupHi) { sts128(yw + 2u * YPITCH, T2A); sts128(yw + 2u * YPITCH + 512u, T2B); }
          }
        }
      }
      if (centre && (FAST || t >= 2)) {
        const int p2 = k0 - 2 + t;
        const unsigned yr = ybase + ((ym + NY - 1) % NY) * YPLANE + oY;     // own sites in plane p2
        const unsigned yb = ybase + ((ym + NY - 2) % NY) * YPLANE + oY;     // ... in plane p2 - 1
        const bool bot = !FAST && lo_ghost && t == 2, top = !FAST && !do1;  // open z faces, sweep l + 2
        float4 outA, outB;
        float2 W, E;
        {
          const float4 C = lds128(yr);
          float4 B = bot ? cmul4(U2z, T2A) : lds128(yb);
          if (top) T2A = cmulc4(U2z, B);
          xnbA(fast_tag, C, yr, yr - 8u, W, E);
          outA = half(fast_tag, p2, YPITCH, i0 + 2 * lane, C, T2A, B, W, E, yr, prv + oX + DB, prv + oX + DD, rmax2);
        }
        {
          const float4 C = lds128(yr + 512u);
          float4 B = bot ? cmul4(U2z, T2B) : lds128(yb + 512u);
          if (top) T2B = cmulc4(U2z, B);
          xnbB(fast_tag, C, yr, yr + 512u + 16u, W, E);
          outB = half(fast_tag, p2, YPITCH, i0 + 64 + 2 * lane, C, T2B, B, W, E, yr + 512u, prv + oX + DB + 512u,
                      prv + oX + DD + 512u, rmax2);
        }
        out2[0] = outA;
        out2[32] = outB;                                             // + 64 sites
        out2 += plane / 2;
        if (jact) {
          // J_av (Eq. 35): x links of x^{l+2} inside the tile row, exactly as the plain sweep sums them
          const float nAx = __shfl_down_sync(0xffffffffu, outA.x, 1), nAy = __shfl_down_sync(0xffffffffu, outA.y, 1);
          const float rBx = __shfl_sync(0xffffffffu, outB.x, (lane + 1) & 31), rBy = __shfl_sync(0xffffffffu, outB.y, (lane + 1) & 31);
          const float2 nxA = (lane == 31) ? make_float2(rBx, rBy) : make_float2(nAx, nAy);
          float tsum = 0.f;
          tsum += jlink(Uxj, outA.x, outA.y, outA.z, outA.w);
          tsum += jlink(Uxj, outA.z, outA.w, nxA.x, nxA.y);
          tsum += jlink(Uxj, outB.x, outB.y, outB.z, outB.w);
          const float last = jlink(Uxj, outB.z, outB.w, rBx, rBy);
          tsum += (lane < 31) ? last : 0.f;                          // (adding +0 leaves the sum as it is)
          jacc += (double)tsum;
        }
      }
    };
    // warps that may take the fast copy, and the iterations on which every warp may: both stages active, no z face
    const bool xface = __any_sync(0xffffffffu, xloA || xhiB);
    const bool wfast = w != 0 && act1 && !(ylo || yhi || dupLo || dupHi || xface);
    const int tf0 = 3, tf1 = nk - 1;                                 // 3 <= t <= nk - 1
    // z march
    for (int t = tb; t <= nk + 1; ++t) {
      if (wfast && t >= tf0 && t <= tf1) iter(std::true_type{}, t, pA, pB);
      else iter(std::false_type{}, t, pA, pB);
    }
  } else {
    // ======================================= column warps ========================================================
    // Warp 18 owns the halo column i0 - 1, warp 19 the column i0 + 128.  Lane q < 18 owns the halo site of tile row
    // q - 1; rows -1 and 16 only supply their x^l values (corners of the halo).  The site is one of a 16-byte pair in
    // HBM: (i0 - 2, i0 - 1) on the west side, (i0 + 128, i0 + 129) on the east side; the other site of the pair is its
    // outer x neighbour, the inner one is in the TMA stage.  Plain 16-byte loads one plane ahead; the x^l values are
    // handed to the row warps through the shared array XH.
    const bool east = w != NROWW;                                    // warp-uniform
    const bool sideon = east ? eCol : wCol;                          // no halo column beyond an open x face
    const int rr = lane - 1;
    const bool rowok = lane < NROWW && ((rr >= 0 && rr < PH) || (rr < 0 ? loRow : hiRow));
    const bool comp = lane < NROWW && rr >= 0 && rr < PH;
    const int jr = min(max((rr >= 0 && rr < PH) ? j0 + rr : (rr < 0 ? jlo : jhi), 0), ny - 1);
    const bool ld = sideon && rowok, cp = sideon && comp;
    const bool ylo = py && jr == 0, yhi = py && jr == ny - 1, mlo = !py && jr == 0, mhi = !py && jr == ny - 1;
    const float2 *xpair = xin + (long long)jr * nx + (east ? xEp : xWp);          // the pair, plane 0
    const long long bdoff = (long long)jr * nx + (east ? xEp : xWp + 1);         // the halo site itself
    const unsigned oXin = OFF_X + (unsigned)(rr + 2) * ROWB + (east ? 8u * (TW - 1) : 0u);   // inner neighbour in a stage
    const unsigned oYc = (unsigned)(rr + 1) * YPITCH + (east ? 8u * (TW + 2) : 8u);
    const unsigned oXHc = (east ? NROWW * 8u : 0u) + (unsigned)(rr + 1) * 8u;
    const float2 Uxj = dv.Ux[jr], Uzj = dv.Uz[jr];
    const Links L = make_links(make_float2(f * dv.cx * Uxj.x, f * dv.cx * Uxj.y),
                               make_float2(f * dv.cz * Uzj.x, f * dv.cz * Uzj.y), f * dv.cy);
    const float2 U2z = cmul(Uzj, Uzj);
    const float2 Pic = dv.Pi[east ? xEp : xWp + 1];
    const float4 z4 = make_float4(0.f, 0.f, 0.f, 0.f);
    const float2 z2 = make_float2(0.f, 0.f);
    auto ldx = [&](int kp) -> float4 { return ld ? __ldg(reinterpret_cast<const float4 *>(xpair + (long long)kp * plane)) : z4; };
    auto ldbd = [&](const float2 *arr, int kp) -> float2 { return cp ? __ldg(arr + (long long)kp * plane + bdoff) : z2; };
    auto own = [&](const float4 &v) -> float2 { return east ? lo(v) : hi(v); };
    auto outer = [&](const float4 &v) -> float2 { return east ? hi(v) : lo(v); };
    float4 cB = ldx(zw(k0 - 2 + tb));                                // planes p1 - 1, p1 and (prefetched) p1 + 1
    if (lo_ghost) cB = cmul4(U2z, cB);
    float4 cC = ldx(zw(k0 - 1 + tb));
    if (ld) sts64(xhbase + (unsigned)(tb & 1) * XHPLANE + oXHc, own(cC));       // x^l halo column of the first plane
    float4 cN = ldx(zw(k0 + tb));
    float2 cb = ldbd(dv.b, zw(k0 - 1 + tb)), cd = ldbd(dv.d, zw(k0 - 1 + tb)); // b, d of plane p1 (prefetched)
    for (int t = tb; t <= nk + 1; ++t) {
      __syncthreads();
      if (t > te) continue;
      const int p1 = k0 - 1 + t;
      const unsigned prv = stage_of(t);
      wait_stage(t);                                                  // (complete since the last iteration: visibility only)
      float4 cT = cN;
      const float2 b_ = cb, d_ = cd;
      if (t + 1 <= te) {                                              // next plane's loads in flight during this one
        cN = ldx(zw(p1 + 2));
        cb = ldbd(dv.b, zw(p1 + 1));
        cd = ldbd(dv.d, zw(p1 + 1));
      }
      if (hi_ghost && t == nk) cT = cmulc4(U2z, cT);
      if (ld) sts64(xhbase + (unsigned)((t + 1) & 1) * XHPLANE + oXHc, own(cT));   // for the row warps' next iteration
      if (sideon) {
        // stage 1 on the halo sites; N / S neighbours are the lanes above / below
        const float2 C = own(cC);
        float2 Nn = make_float2(__shfl_down_sync(0xffffffffu, C.x, 1), __shfl_down_sync(0xffffffffu, C.y, 1));
        float2 Sn = make_float2(__shfl_up_sync(0xffffffffu, C.x, 1), __shfl_up_sync(0xffffffffu, C.y, 1));
        if (mlo) Sn = Nn;                                              // open y faces: mirror (U_y = 1)
        if (mhi) Nn = Sn;
        if (ylo || yhi) {
          const float2 P = cmulc(dv.Pk[zw(p1)], Pic);
          if (ylo) Sn = cmul(P, Sn);
          if (yhi) Nn = cmulc(P, Nn);
        }
        const float2 inner = comp ? lds64(prv + oXin) : z2;
        const float2 sm = nsum_site(L, b_, east ? inner : outer(cC), east ? outer(cC) : inner, Nn, Sn, own(cT), own(cB));
        float r = 0.f;
        const float4 o = divide_pair(sm, sm, make_float4(d_.x, d_.y, d_.x, d_.y), make_float4(C.x, C.y, C.x, C.y), r);
        if (comp) sts64(ybase + ((unsigned)t % NY) * YPLANE + oYc, lo(o));
      }
      cB = cC;
      cC = cT;
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

// J_av link sums of the current iterate per 128 x 8 tile and z chunk of the plain sweep's grid, exactly as the sweep
// kernels form them on their own output (same lane layout, same order: bit-identical partial sums).  Acts only when the
// step ended with a fused pair that had been told to skip them (ctl->need_jav, choose_next): one 8 B/site pass.
__global__ void __launch_bounds__(256) k_jav_tiles(const __grid_constant__ Dev dv) {
  Ctl *ctl = dv.ctl;
  if (!ctl->need_jav) return;
  __shared__ double s_j[8];
  const int lane = threadIdx.x & 31, row = threadIdx.x >> 5;
  const int j = blockIdx.y * 8 + row;
  const int k0 = blockIdx.z * dv.zc, k1 = min(dv.nz, k0 + dv.zc);
  const long long plane = (long long)dv.nx * dv.ny;
  const float4 *x = reinterpret_cast<const float4 *>(dv.psi[ctl->xbuf] + (long long)k0 * plane + (long long)j * dv.nx +
                                                      blockIdx.x * TW + 2 * lane);
  const float2 Uxj = dv.Ux[j];
  double jacc = 0.0;
  for (int k = k0; k < k1; ++k, x += plane / 2) {
    const float4 outA = __ldcs(x), outB = __ldcs(x + 32);
    const float nAx = __shfl_down_sync(0xffffffffu, outA.x, 1), nAy = __shfl_down_sync(0xffffffffu, outA.y, 1);
    const float rBx = __shfl_sync(0xffffffffu, outB.x, (lane + 1) & 31), rBy = __shfl_sync(0xffffffffu, outB.y, (lane + 1) & 31);
    const float2 nxA = (lane == 31) ? make_float2(rBx, rBy) : make_float2(nAx, nAy);
    float tsum = 0.f;
    tsum += jlink(Uxj, outA.x, outA.y, outA.z, outA.w);
    tsum += jlink(Uxj, outA.z, outA.w, nxA.x, nxA.y);
    tsum += jlink(Uxj, outB.x, outB.y, outB.z, outB.w);
    const float last = jlink(Uxj, outB.z, outB.w, rBx, rBy);
    tsum += (lane < 31) ? last : 0.f;
    jacc += (double)tsum;
  }
  for (int o = 16; o > 0; o >>= 1) jacc += __shfl_down_sync(0xffffffffu, jacc, o);
  if (lane == 0) s_j[row] = jacc;
  __syncthreads();
  if (threadIdx.x == 0) {
    double sj = 0.0;
    for (int q = 0; q < 8; ++q) sj += s_j[q];
    dv.jpart[blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z)] = sj;
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

// grid of the plain sweep (128 x 8 tiles, dv.zc planes): one partial sum per CTA, where k_step_finish expects it
void launch_jav_tiles(const Dev &dv, cudaStream_t st) {
  const dim3 grid((unsigned)(dv.nx / TW), (unsigned)(dv.ny / 8), (unsigned)((dv.nz + dv.zc - 1) / dv.zc));
  k_jav_tiles<<<grid, 256, 0, st>>>(dv);
}
