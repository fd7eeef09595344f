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

// per-thread link constants, already scaled:  f c_x U_x(j),  f c_z U_z(j),  f c_y   (f = h_t/2 or 1)
struct Links { float2 ux, uz; float cy; };

// s += f [ c_x (U_x E + U_x* W) + c_y (N + S) + c_z (U_z T + U_z* B) ]  for the two sites of a pair:
//   U E + U* W = U.re (E + W) + i U.im (E - W): 10 adds and 10 FMAs per site (Eq. 29a)
__device__ __forceinline__ void nsum_pair(const Links &L, const float4 &C, const float2 &W, const float2 &E,
                                          const float4 &Nn, const float4 &Ss, const float4 &T, const float4 &B,
                                          float2 &s0, float2 &s1) {
  // site 0: west W, east C.hi;  site 1: west C.lo, east E
  s0.x = fmaf(L.ux.x, C.z + W.x, s0.x);  s0.x = fmaf(-L.ux.y, C.w - W.y, s0.x);
  s0.y = fmaf(L.ux.x, C.w + W.y, s0.y);  s0.y = fmaf(L.ux.y, C.z - W.x, s0.y);
  s1.x = fmaf(L.ux.x, E.x + C.x, s1.x);  s1.x = fmaf(-L.ux.y, E.y - C.y, s1.x);
  s1.y = fmaf(L.ux.x, E.y + C.y, s1.y);  s1.y = fmaf(L.ux.y, E.x - C.x, s1.y);
  s0.x = fmaf(L.cy, Nn.x + Ss.x, s0.x);  s0.y = fmaf(L.cy, Nn.y + Ss.y, s0.y);
  s1.x = fmaf(L.cy, Nn.z + Ss.z, s1.x);  s1.y = fmaf(L.cy, Nn.w + Ss.w, s1.y);
  s0.x = fmaf(L.uz.x, T.x + B.x, s0.x);  s0.x = fmaf(-L.uz.y, T.y - B.y, s0.x);
  s0.y = fmaf(L.uz.x, T.y + B.y, s0.y);  s0.y = fmaf(L.uz.y, T.x - B.x, s0.y);
  s1.x = fmaf(L.uz.x, T.z + B.z, s1.x);  s1.x = fmaf(-L.uz.y, T.w - B.w, s1.x);
  s1.y = fmaf(L.uz.x, T.w + B.w, s1.y);  s1.y = fmaf(L.uz.y, T.z - B.z, s1.y);
}

// x^{l+1} = n / d for both sites of a pair (Eq. 33) and |r^l|^2 = |d|^2 |x^{l+1} - x^l|^2 (S8)
__device__ __forceinline__ float4 divide_pair(const float2 &n0, const float2 &n1, const float4 &d, const float4 &C,
                                              float &rmax) {
  const float m0 = d.x * d.x + d.y * d.y, m1 = d.z * d.z + d.w * d.w;
  const float i0 = rcp_approx(m0), i1 = rcp_approx(m1);
  const float2 y0 = cmulc(lo(d), n0), y1 = cmulc(hi(d), n1);
  const float4 out = make_float4(y0.x * i0, y0.y * i0, y1.x * i1, y1.y * i1);
  const float e0x = out.x - C.x, e0y = out.y - C.y, e1x = out.z - C.z, e1y = out.w - C.w;
  rmax = fmaxf(rmax, fmaxf((e0x * e0x + e0y * e0y) * m0, (e1x * e1x + e1y * e1y) * m1));
  return out;
}

// The decision taken by the last CTA of a sweep (Eq. 34; S8: residual of the input iterate,
// keep the new one; S9/S10: prescribed counts, cap).
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
    if (!(r2 < c->eps_tol) && sweeps >= c->max_sweeps) c->status = 1;
  }
  if (done) {
    c->done = 1;
    c->sweeps_last = sweeps;
    c->resid_last = r2;
  }
  if (dv.use_cond) cudaGraphSetConditional((cudaGraphConditionalHandle)dv.cond_handle, done ? 0u : 1u);
  __threadfence();
}

}  // namespace
