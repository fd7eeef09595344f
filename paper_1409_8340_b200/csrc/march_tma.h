// Host/device interface of the TMA marching kernels (march_tma.cu).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include "tdgl_dev.cuh"

// Tensor maps (cuTensorMapEncodeTiled) of the complex fields seen as fp32 [nz][ny][2 nx]:
//   C = tile centre box (2*128 x 8 x 1), R = one ghost row (2*128 x 1 x 1), X = ghost column pair (4 x 8 x 1)
struct MarchMaps {
  CUtensorMap psiC[2], psiR[2], psiX[2];   // the two ping-pong psi buffers
  CUtensorMap bC, dC;                       // right side b and diagonal d of the linear system (Eq. 30-31)
  CUtensorMap muC, epsC;                    // mu and eps as fp32 [nz][ny][nx], box 128 x 8 x 1 (init kernel; only if nx % 4 == 0)
  int me_tma;                               // 1: the init kernel takes mu, eps through the TMA stage, 0: plain loads
};

int march_tma_build_maps(const Dev &dv, MarchMaps *mm);
cudaError_t march_tma_configure();
void march_tma_grid(int nx, int ny, int *gx, int *gy);
int march_tma_tile_w();
void launch_march_tma(int mode, const Dev &dv, const MarchMaps &mm, dim3 grid, cudaStream_t st);
