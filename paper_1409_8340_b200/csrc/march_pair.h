// Host/device interface of the fused two-sweep kernel (march_pair.cu).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include "tdgl_dev.cuh"

// Tensor maps of the complex fields seen as fp32 [nz][ny][2 nx]: C = tile centre box (2*128 x 16 x 1),
// R2 = two halo rows (2*128 x 2 x 1), R = one halo row of b / d (2*128 x 1 x 1)
struct PairMaps {
  CUtensorMap psiC[2], psiR2[2];
  CUtensorMap bC, dC, bR, dR;
};

bool march_pair_ok(int nx, int ny, int nz, bool gauge_yz);
int march_pair_build_maps(const Dev &dv, PairMaps *pm);
cudaError_t march_pair_configure();
void launch_march_pair(const Dev &dv, const PairMaps &pm, cudaStream_t st);
void launch_jav_tiles(const Dev &dv, cudaStream_t st);
