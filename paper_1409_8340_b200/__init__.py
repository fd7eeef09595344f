"""B200-native hot path of the large-lambda TDGL solver of arXiv:1409.8340.

The product is the C-ABI library `libtdgl.so` (include/tdgl.h; CUDA for sm_100a).  This package is its
thin ctypes binding: argument marshalling only, every step of the path runs in the library's kernels.
torch is used for device memory and streams.  There is no CPU path: loading fails loudly if the
library has not been built (`python -m paper_1409_8340_b200.build`).
"""
from .binding import (  # noqa: F401
    TDGL_BC_OPEN, TDGL_BC_PERIODIC, TDGL_FLAG_FP64, TDGL_FLAG_GAUGE_YZ, TDGL_FLAG_HOST_LOOP, TDGL_FLAG_INSULATORS, TDGL_FLAG_MU_ITERATIVE, TDGL_FLAG_SOLVE_MU, TdglError, TdglObs, TdglParams,
    TdglSphere, Solver, lib, tdgl_create, tdgl_destroy, tdgl_get_psi_mu, tdgl_observables, tdgl_set_field_current,
    tdgl_set_pinning, tdgl_step, tdgl_strerror, tdgl_workspace_bytes,
    TDGL_ESCRATCH, TDGL_STATIC_MAX_SITES, tdgl_mean_abs2_static,
    TDGL_FLAG_MU_DIRECT, TDGL_FLAG_MU_REFINE, TDGL_FLAG_MU_NOREFINE, TDGL_WMAXSWEEPS, TDGL_WMUCAP,
)
