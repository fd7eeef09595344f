// tdgl_mean_abs2_static: <|psi|^2> for callers that have no way to obtain device memory.
//
// Everything else in libtdgl works out of a workspace the caller allocates (44 B/site, handed over at tdgl_create) --
// the two-stage reduction behind tdgl_observables keeps its per-CTA partial sums there (Dev::part).  That is fine
// for the program that owns the simulation, and useless for code that sits NEXT to it and was only given a device
// pointer to psi: an in-situ monitor or a logging thread watching a running solver, a plug-in inside a host
// application whose own pool has reserved the whole of HBM at start-up (the 1024 x 1024 x 512 mesh is sized against
// the 180 GB of the device, so a cudaMalloc there may simply fail), or a component that must not call cudaMalloc /
// cudaFree at all because they synchronise the whole device and would stall the time-stepping stream.  Such a caller
// has no workspace and no handle.  For them this one entry point carries its scratch memory inside the library
// image: a file-scope __device__ array of fixed size, so the call allocates nothing, neither here nor through any
// library routine.
//
// Costs and rules that follow from that choice (also in include/tdgl.h):
//  * the array (TDGL_STATIC_SCRATCH_BYTES, 64.25 KiB) is part of the module: every GPU on which the library's kernels are
//    loaded keeps it until the process exits, whether or not this entry point is ever called;
//  * its size fixes the largest input: one fp64 partial sum per 65 536 sites, 8192 of them, i.e. 2^29 sites
//    (TDGL_STATIC_MAX_SITES = 1024 x 1024 x 512, the largest BASELINE mesh); more is refused with TDGL_ESCRATCH;
//  * there is ONE array per device and every call uses it, so two calls that may overlap on the GPU (different
//    streams, no dependency between them) race on the partial sums and on the election counter.  Order them;
//  * the array keeps what the last call left.  The partial sums are overwritten before they are read, the election
//    counter must start at zero and is cleared on the stream ahead of every launch (so a call that was cut short --
//    a failed launch, a device reset by someone else -- cannot poison the next one);
//  * the first call on each device looks up the array's device address (cudaGetSymbolAddress, which also makes the
//    runtime load the module there).  That is set-up work outside the stream: make that first call at start-up, before
//    any stream capture begins on that device.  Later calls only enqueue a 4-byte memset and one kernel.
//
// The arithmetic is the one of k_obs_partial (aux.cu; observable a8): |psi_m|^2 formed in fp32 per site,
// summed in fp64.  The summation ORDER differs (fixed 65 536-site chunks here, so the result does not depend on the
// number of SMs), hence the two agree to fp64 rounding of the sum, not bit for bit.
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>

#include "../../include/tdgl.h"

#define SS_CHUNK 65536                                    // sites per CTA = per partial sum
#define SS_NPART (TDGL_STATIC_MAX_SITES / SS_CHUNK)       // 8192
#define SS_THREADS 256
#define SS_TICKET_OFFSET (SS_NPART * sizeof(double))      // the election counter sits behind the partial sums
static_assert((long long)SS_NPART * SS_CHUNK == TDGL_STATIC_MAX_SITES, "the maximum is a whole number of chunks");
static_assert(SS_TICKET_OFFSET + 256 == TDGL_STATIC_SCRATCH_BYTES, "header and array size disagree");

// The scratch itself.  In HOST code this name is only a stand-in the runtime uses to find the symbol: it is not a
// device address and must never be handed to a kernel.  Host code below goes through cudaGetSymbolAddress.
static __device__ __align__(256) unsigned char g_static_scratch[TDGL_STATIC_SCRATCH_BYTES];

__device__ __forceinline__ double ss_abs2(float2 v) { return (double)(v.x * v.x + v.y * v.y); }

// One CTA per chunk of SS_CHUNK consecutive sites.  `part` and `ticket` point into g_static_scratch (resolved on the
// host, once per device).  The CTA that draws the last ticket adds the partial sums in index order and writes the mean.
__global__ void __launch_bounds__(SS_THREADS) k_mean_abs2_static(const float2 *__restrict__ psi, long long n, int vec16,
                                                                 double *part, unsigned int *ticket, double *mean_out) {
  const long long lo = (long long)blockIdx.x * SS_CHUNK;
  const long long hi = (lo + SS_CHUNK < n) ? lo + SS_CHUNK : n;
  double a = 0.0, b = 0.0;
  if (vec16) {                                            // psi is 16-byte aligned: two sites per load
    const float4 *p4 = reinterpret_cast<const float4 *>(psi + lo);
    const long long npair = (hi - lo) >> 1;
    long long q = threadIdx.x;
    for (; q + 3 * SS_THREADS < npair; q += 4 * SS_THREADS) {
      const float4 v0 = __ldg(p4 + q), v1 = __ldg(p4 + q + SS_THREADS), v2 = __ldg(p4 + q + 2 * SS_THREADS), v3 = __ldg(p4 + q + 3 * SS_THREADS);
      a += ss_abs2(make_float2(v0.x, v0.y)); b += ss_abs2(make_float2(v0.z, v0.w));
      a += ss_abs2(make_float2(v1.x, v1.y)); b += ss_abs2(make_float2(v1.z, v1.w));
      a += ss_abs2(make_float2(v2.x, v2.y)); b += ss_abs2(make_float2(v2.z, v2.w));
      a += ss_abs2(make_float2(v3.x, v3.y)); b += ss_abs2(make_float2(v3.z, v3.w));
    }
    for (; q < npair; q += SS_THREADS) {
      const float4 v = __ldg(p4 + q);
      a += ss_abs2(make_float2(v.x, v.y)); b += ss_abs2(make_float2(v.z, v.w));
    }
    if (((hi - lo) & 1) && threadIdx.x == 0) a += ss_abs2(__ldg(psi + hi - 1));     // odd tail of the last chunk
  } else {
    for (long long m = lo + threadIdx.x; m < hi; m += SS_THREADS) a += ss_abs2(__ldg(psi + m));
  }
  a += b;
  __shared__ double sh[SS_THREADS / 32];
  __shared__ bool last;
  for (int o = 16; o > 0; o >>= 1) a += __shfl_down_sync(0xffffffffu, a, o);
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = a;
  __syncthreads();
  if (threadIdx.x == 0) {
    double s = 0.0;
    for (int w = 0; w < SS_THREADS / 32; ++w) s += sh[w];
    part[blockIdx.x] = s;
    __threadfence();                                      // the partial sum is visible before the ticket is drawn
    last = atomicAdd(ticket, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!last) return;
  __threadfence();
  double s = 0.0;
  for (int p = threadIdx.x; p < (int)gridDim.x; p += SS_THREADS) s += __ldcg(part + p);
  __shared__ double fin[SS_THREADS];
  fin[threadIdx.x] = s;
  __syncthreads();
  for (int o = SS_THREADS / 2; o > 0; o >>= 1) {
    if (threadIdx.x < o) fin[threadIdx.x] += fin[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) mean_out[0] = fin[0] / (double)n;
}

// Device address of g_static_scratch on the CURRENT device, looked up once per device and remembered.
#define SS_MAX_DEVICES 64
static std::mutex g_ss_lock;
static unsigned char *g_ss_addr[SS_MAX_DEVICES];

static int static_scratch_of_current_device(unsigned char **out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= SS_MAX_DEVICES) return TDGL_ECUDA;
  std::lock_guard<std::mutex> guard(g_ss_lock);
  if (!g_ss_addr[dev]) {
    void *p = nullptr;
    if (cudaGetSymbolAddress(&p, g_static_scratch) != cudaSuccess || !p) return TDGL_ECUDA;
    g_ss_addr[dev] = static_cast<unsigned char *>(p);
  }
  *out = g_ss_addr[dev];
  return TDGL_OK;
}

extern "C" int tdgl_mean_abs2_static(const void *psi_dev, int64_t n_sites, double *mean_dev, void *stream) {
  if (!psi_dev || !mean_dev || n_sites < 1) return TDGL_EINVAL;
  if ((reinterpret_cast<uintptr_t>(psi_dev) & 7u) || (reinterpret_cast<uintptr_t>(mean_dev) & 7u)) return TDGL_EINVAL;
  if (n_sites > (int64_t)TDGL_STATIC_MAX_SITES) return TDGL_ESCRATCH;      // the built-in array has no room for the partial sums
  unsigned char *scratch = nullptr;
  const int rc = static_scratch_of_current_device(&scratch);
  if (rc != TDGL_OK) return rc;
  double *part = reinterpret_cast<double *>(scratch);
  unsigned int *ticket = reinterpret_cast<unsigned int *>(scratch + SS_TICKET_OFFSET);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  if (cudaMemsetAsync(ticket, 0, sizeof(unsigned int), st) != cudaSuccess) return TDGL_ECUDA;
  const unsigned grid = (unsigned)((n_sites + SS_CHUNK - 1) / SS_CHUNK);
  const int vec16 = (reinterpret_cast<uintptr_t>(psi_dev) & 15u) == 0;
  k_mean_abs2_static<<<grid, SS_THREADS, 0, st>>>(static_cast<const float2 *>(psi_dev), (long long)n_sites, vec16, part, ticket, mean_dev);
  return cudaPeekAtLastError() == cudaSuccess ? TDGL_OK : TDGL_ECUDA;
}
