// Device helpers shared by the marching kernels (march_tma.cu: 3D, z marching; march_film.cu: films, y
// marching): mbarrier / bulk-copy PTX wrappers, the link-variable neighbour sum, the Jacobi division with
// the residual, and the convergence decision of the last CTA.
#pragma once
#include "tdgl_dev.cuh"
#include <cuda.h>
#include <cuda_device_runtime_api.h>

#define MODE_SWEEP 0
#define MODE_INIT  1
#define MODE_RHO   2

namespace {

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "LAB_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra DONE;\n"
      "bra LAB_WAIT;\n"
      "DONE:\n"
      "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_3d(unsigned dst, const CUtensorMap *map, int c0, int c1, int c2, unsigned bar) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];\n"
               ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
// 1-D bulk copy global -> shared (bytes: multiple of 16; both addresses 16-byte aligned), completing on an mbarrier
__device__ __forceinline__ void bulk_load_1d(unsigned dst, const void *src, unsigned bytes, unsigned bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ float4 lds128(unsigned a) {
  float4 v;
  asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];\n" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
  return v;
}
__device__ __forceinline__ float2 lds64(unsigned a) {
  float2 v;
  asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];\n" : "=f"(v.x), "=f"(v.y) : "r"(a));
  return v;
}
__device__ __forceinline__ float rcp_approx(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;\n" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float2 lo(const float4 &v) { return make_float2(v.x, v.y); }
__device__ __forceinline__ float2 hi(const float4 &v) { return make_float2(v.z, v.w); }
__device__ __forceinline__ float4 cmul4(float2 a, const float4 &v) {      // a * both sites
  const float2 p = cmul(a, lo(v)), q = cmul(a, hi(v));
  return make_float4(p.x, p.y, q.x, q.y);
}
__device__ __forceinline__ float4 cmulc4(float2 a, const float4 &v) {     // conj(a) * both sites
  const float2 p = cmulc(a, lo(v)), q = cmulc(a, hi(v));
  return make_float4(p.x, p.y, q.x, q.y);
}

// packed fp32x2 arithmetic of sm_100 (one instruction for the (re, im) pair of a site: FADD2 / FMUL2 / FFMA2)
typedef unsigned long long u64;
__device__ __forceinline__ u64 pk2(float a, float b) { u64 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ u64 pk2(float2 a) { return pk2(a.x, a.y); }
__device__ __forceinline__ float2 upk2(u64 a) { float2 r; asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(a)); return r; }
__device__ __forceinline__ u64 add2(u64 a, u64 b) { u64 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 sub2(u64 a, u64 b) { u64 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 mul2(u64 a, u64 b) { u64 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) { u64 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }

// per-thread link constants, already scaled:  f c_x U_x(j),  f c_z U_z(j),  f c_y   (f = h_t/2 or 1), each component
// broadcast to both halves of a packed pair
struct Links { u64 uxr, uxi, uzr, uzi, cy; };
__device__ __forceinline__ Links make_links(float2 ux, float2 uz, float cy) {
  Links L;
  L.uxr = pk2(ux.x, ux.x); L.uxi = pk2(ux.y, ux.y);
  L.uzr = pk2(uz.x, uz.x); L.uzi = pk2(uz.y, uz.y);
  L.cy = pk2(cy, cy);
  return L;
}

// s += f [ c_x (U_x E + U_x* W) + c_y (N + S) + c_z (U_z T + U_z* B) ]  for one site (Eq. 29a):
//   U E + U* W = U.re (E + W) + i U.im (E - W);  the real multiples are gathered in a1 (which starts from s), the
//   multiples of i in a2, on (re, im) pairs: 5 packed adds, 1 packed product, 4 packed FMAs and the final
//   s = a1 + i a2 (2 scalar adds) per site
__device__ __forceinline__ float2 nsum_site(const Links &L, float2 s, float2 W, float2 E, float2 N, float2 S, float2 T,
                                            float2 B) {
  const u64 e = pk2(E), w = pk2(W), t = pk2(T), b = pk2(B);
  u64 a1 = fma2(L.uxr, add2(e, w), pk2(s));
  u64 a2 = mul2(L.uxi, sub2(e, w));
  a1 = fma2(L.cy, add2(pk2(N), pk2(S)), a1);
  a1 = fma2(L.uzr, add2(t, b), a1);
  a2 = fma2(L.uzi, sub2(t, b), a2);
  const float2 r = upk2(a1), q = upk2(a2);
  return make_float2(r.x - q.y, r.y + q.x);
}
__device__ __forceinline__ void nsum_pair(const Links &L, const float4 &C, const float2 &W, const float2 &E,
                                          const float4 &Nn, const float4 &Ss, const float4 &T, const float4 &B,
                                          float2 &s0, float2 &s1) {
  // site 0: west W, east C.hi;  site 1: west C.lo, east E
  s0 = nsum_site(L, s0, W, hi(C), lo(Nn), lo(Ss), lo(T), lo(B));
  s1 = nsum_site(L, s1, lo(C), E, hi(Nn), hi(Ss), hi(T), hi(B));
}

// x^{l+1} = n / d for both sites of a pair (Eq. 33) and |r^l|^2 = |d|^2 |x^{l+1} - x^l|^2 (S8)
__device__ __forceinline__ float4 divide_pair(const float2 &n0, const float2 &n1, const float4 &d, const float4 &C,
                                              float &rmax) {
  const float m0 = __fmaf_rn(d.x, d.x, __fmul_rn(d.y, d.y)), m1 = __fmaf_rn(d.z, d.z, __fmul_rn(d.w, d.w));
  const float i0 = rcp_approx(m0), i1 = rcp_approx(m1);
  const float2 y0 = cmulc(lo(d), n0), y1 = cmulc(hi(d), n1);
  const u64 o0 = mul2(pk2(y0), pk2(i0, i0)), o1 = mul2(pk2(y1), pk2(i1, i1));
  const float2 e0 = upk2(sub2(o0, pk2(lo(C)))), e1 = upk2(sub2(o1, pk2(hi(C))));
  const float q0 = __fmul_rn(__fmaf_rn(e0.x, e0.x, __fmul_rn(e0.y, e0.y)), m0);
  const float q1 = __fmul_rn(__fmaf_rn(e1.x, e1.x, __fmul_rn(e1.y, e1.y)), m1);
  rmax = fmaxf(rmax, fmaxf(q0, q1));
  const float2 a = upk2(o0), b = upk2(o1);
  return make_float4(a.x, a.y, b.x, b.y);
}

// Im[a* U b] of one x link (Eq. 35), contraction spelled out (the plain sweep and the fused pair must agree)
__device__ __forceinline__ float jlink(float2 U, float ar, float ai, float br, float bi) {
  const float p = __fmaf_rn(U.x, bi, __fmul_rn(U.y, br)), q = __fmaf_rn(U.x, br, -__fmul_rn(U.y, bi));
  return __fmaf_rn(ar, p, -__fmul_rn(ai, q));
}

// The decision taken by the last CTA of a sweep (Eq. 34; S8: residual of the input iterate,
// keep the new one; S9/S10: prescribed counts, cap).
// Which kernel of the loop body acts next: the fused pair (march_pair.cu) only when two more sweeps are certain
// (prescribed counts) or predicted from the residual history (criterion (34) stays exact either way: a pair whose
// FIRST sweep already met it is discarded and redone as a plain sweep, see pair_decide).
__device__ __forceinline__ void choose_next(const Dev &dv, Ctl *c, int sweeps, int target, float r_last, float r_prev) {
  int up = 0, jav = 1;
  if (dv.pair_ok && c->pair_mode > 0) {
    if (target > 0) {
      up = target - sweeps >= 2;
      jav = sweeps + 2 >= target;                          // only the last sweep's J_av is used
    } else if (sweeps + 2 <= c->max_sweeps) {
      // Two more sweeps are needed iff the NEXT residual is still >= eps.  Two predictors: geometric decay of the last two
      // residuals (trusted alone when it says "far above eps"), and the previous time step, whose sweep count the
      // present one rarely undercuts (a pair that ends at or before that count is taken unless the decay says the next
      // sweep converges).  A wrong guess costs one discarded pair, never a wrong result.
      const float q = r_prev > 0.f ? fminf(1.f, r_last / r_prev) : 1.f;
      const float next = r_last * q, next2 = next * q;
      up = next >= 10.f * c->eps_tol || (sweeps + 2 <= c->sweeps_last && next >= c->eps_tol);
      // The J_av link sums of a pair's output (17 % of its time on C4) are needed only if its second sweep ends the
      // step: skipped when the residual after the pair is predicted far above eps, or when the previous step needed
      // more sweeps than the pair reaches.  A wrong guess costs one pass of k_jav_tiles.
      jav = !(r_prev > 0.f ? (next2 >= 10.f * c->eps_tol || (sweeps + 2 < c->sweeps_last && next2 >= c->eps_tol))
                           : sweeps + 2 < c->sweeps_last);
      if (sweeps + 2 >= c->max_sweeps) jav = 1;          // the cap would end the step with this pair
      if (c->pair_mode >= 2) up = 1;
      if (c->pair_mode == 3) jav = 0;
    }
  }
  c->use_pair = up;
  c->pair_jav = jav;
}

__device__ __noinline__ void sweep_decide(const Dev &dv, int l) {
  Ctl *c = dv.ctl;
  const float r2 = __uint_as_float(atomicMax(&c->resid_bits[l], 0u));
  const int sweeps = l + 1;
  c->sweeps = sweeps;
  c->xbuf ^= 1;
  int target = c->fixed_sweeps;
  if (c->sched_pos < c->sched_n) target = dv.sched[c->sched_pos];
  bool done;
  if (target > 0) {
    done = sweeps >= target;
  } else {
    done = (r2 < c->eps_tol) || sweeps >= c->max_sweeps;
    if (!(r2 < c->eps_tol) && sweeps >= c->max_sweeps) c->status |= 1;
  }
  choose_next(dv, c, sweeps, target, r2, l > 0 ? c->r_hist : 0.f);
  c->r_hist = r2;
  if (done) {
    c->done = 1;
    c->use_pair = 0;
    c->need_jav = 0;                                    // a plain sweep always sums its J_av links
    c->sweeps_last = sweeps;
    c->resid_last = r2;
  }
  if (dv.use_cond) cudaGraphSetConditional((cudaGraphConditionalHandle)dv.cond_handle, done ? 0u : 1u);
  __threadfence();
}

// The decision after a fused pair of sweeps l+1, l+2 (residuals r^l, r^{l+1} of their input iterates, S8).  If r^l
// already meets criterion (34) the answer is x^{l+1}, which the pair did not keep: nothing is committed (x^l is
// intact in its buffer) and the next kernel is the plain sweep, which recomputes x^{l+1} and stops.
__device__ __noinline__ void pair_decide(const Dev &dv, int l) {
  Ctl *c = dv.ctl;
  const float r1 = __uint_as_float(atomicMax(&c->resid_bits[l], 0u));
  const float r2 = __uint_as_float(atomicMax(&c->resid_bits[l + 1], 0u));
  int target = c->fixed_sweeps;
  if (c->sched_pos < c->sched_n) target = dv.sched[c->sched_pos];
  c->pair_launches += 1;
  bool done = false;
  if (target <= 0 && r1 < c->eps_tol) {
    c->use_pair = 0;
    c->pair_redone += 1;
  } else {
    const int sweeps = l + 2;
    c->sweeps = sweeps;
    c->xbuf ^= 1;
    if (target > 0) {
      done = sweeps >= target;
    } else {
      done = (r2 < c->eps_tol) || sweeps >= c->max_sweeps;
      if (!(r2 < c->eps_tol) && sweeps >= c->max_sweeps) c->status |= 1;
    }
    const int had_jav = c->pair_jav;                    // (read before choose_next overwrites it)
    choose_next(dv, c, sweeps, target, r2, r1);
    c->r_hist = r2;
    if (done) {
      c->done = 1;
      c->use_pair = 0;
      c->sweeps_last = sweeps;
      c->resid_last = r2;
      c->need_jav = !had_jav;                           // the last sweep did not sum its J_av links: k_jav_tiles will
    }
  }
  if (dv.use_cond) cudaGraphSetConditional((cudaGraphConditionalHandle)dv.cond_handle, done ? 0u : 1u);
  __threadfence();
}

}  // namespace
