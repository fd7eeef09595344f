// Host interface of the film (N_z = 1) marching kernels (march_film.cu).
#pragma once
#include <cuda_runtime.h>
#include "tdgl_dev.cuh"

cudaError_t march_film_configure();
int march_film_strips(int nx);            // CTAs along x: strips of 1024 sites
void launch_march_film(int mode, const Dev &dv, dim3 grid, cudaStream_t st);   // grid = (strips, row chunks, 1); dv.zc = rows per chunk
