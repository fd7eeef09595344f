"""ctypes binding of include/tdgl.h.  Same names, same arguments; no arithmetic of the method here."""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.environ.get("TDGL_LIB") or os.path.join(_HERE, "libtdgl.so")     # TDGL_LIB: another build of the same ABI

TDGL_OK, TDGL_EINVAL, TDGL_ENOMEM, TDGL_EINCOMPAT, TDGL_ECUDA, TDGL_WMAXSWEEPS = 0, -1, -2, -3, -4, 1
TDGL_ESCRATCH = -5
TDGL_WMUCAP = 2
TDGL_STATIC_MAX_SITES, TDGL_STATIC_SCRATCH_BYTES = 536870912, 65792
TDGL_BC_PERIODIC, TDGL_BC_OPEN = 0, 1
TDGL_FLAG_SOLVE_MU, TDGL_FLAG_HOST_LOOP, TDGL_FLAG_GAUGE_YZ, TDGL_FLAG_MU_REFINE, TDGL_FLAG_MU_NOREFINE = 1, 2, 4, 8, 16
TDGL_FLAG_MU_ITERATIVE, TDGL_FLAG_FP64, TDGL_FLAG_INSULATORS, TDGL_FLAG_MU_DIRECT = 32, 64, 128, 256

EXPORTS = (
    "tdgl_workspace_bytes", "tdgl_create", "tdgl_destroy", "tdgl_set_pinning", "tdgl_set_field_current", "tdgl_step",
    "tdgl_get_psi_mu", "tdgl_observables", "tdgl_strerror", "tdgl_last_cuda_error", "tdgl_set_state", "tdgl_set_solver",
    "tdgl_set_sweep_schedule", "tdgl_get_sweep_log", "tdgl_get_eps", "tdgl_debug_noise", "tdgl_debug_poisson",
    "tdgl_debug_rho", "tdgl_launch_count", "tdgl_sweep_timing", "tdgl_mu_gain", "tdgl_mu_refine_enabled",
    "tdgl_set_mu_solver", "tdgl_get_mu_log", "tdgl_set_insulators", "tdgl_set_pinning_shapes", "tdgl_set_insulator_shapes", "tdgl_set_pair_mode", "tdgl_get_pair_stats", "tdgl_get_mu_direct_stats",
    "tdgl_mean_abs2_static",
)


class TdglParams(C.Structure):
    _fields_ = [
        ("struct_size", C.c_uint32), ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
        ("hx", C.c_float), ("hy", C.c_float), ("hz", C.c_float), ("dt", C.c_float), ("u", C.c_float), ("g", C.c_float),
        ("bc", C.c_int32 * 3), ("eps_tol", C.c_float), ("max_sweeps", C.c_int32), ("fixed_sweeps", C.c_int32),
        ("temperature", C.c_float), ("seed", C.c_uint64), ("init_amp", C.c_float), ("flags", C.c_uint32),
        ("workspace_dev", C.c_void_p), ("workspace_bytes", C.c_uint64), ("stream", C.c_void_p),
    ]


class TdglSphere(C.Structure):
    _fields_ = [("cx", C.c_float), ("cy", C.c_float), ("cz", C.c_float), ("r", C.c_float)]


class TdglObs(C.Structure):
    _fields_ = [
        ("t", C.c_double), ("K", C.c_double), ("Ex", C.c_double), ("Jav", C.c_double), ("Ex_mean", C.c_double),
        ("free_energy", C.c_double), ("mean_abs2", C.c_double), ("vortices_per_slice", C.c_double),
        ("max_resid2", C.c_double), ("Bx_eff", C.c_float), ("Bz_eff", C.c_float), ("steps", C.c_int64),
        ("sweeps_total", C.c_int64), ("sweeps_last", C.c_int32), ("status", C.c_int32),
    ]


class TdglError(RuntimeError):
    def __init__(self, code: int, what: str, cuda: int = 0):
        super().__init__(f"{what}: {tdgl_strerror(code)} (code {code}" + (f", cudaError {cuda})" if cuda else ")"))
        self.code = code
        self.cuda = cuda


_lib = None


def lib() -> C.CDLL:
    """Loads libtdgl.so.  Fails loudly when it is missing: there is no other implementation."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise ImportError(f"{_LIB_PATH} is missing: build it with `python -m paper_1409_8340_b200.build` "
                          "(nvcc, sm_100a).  There is no CPU fallback.")
    L = C.CDLL(_LIB_PATH)
    vp, i32, i64, f32, f64 = C.c_void_p, C.c_int32, C.c_int64, C.c_float, C.c_double
    L.tdgl_workspace_bytes.restype = C.c_uint64
    L.tdgl_workspace_bytes.argtypes = [C.POINTER(TdglParams)]
    L.tdgl_create.argtypes = [C.POINTER(TdglParams), C.POINTER(vp)]
    L.tdgl_destroy.argtypes = [vp]
    L.tdgl_set_pinning.argtypes = [vp, C.POINTER(TdglSphere), i64, f32, f32]
    L.tdgl_set_field_current.argtypes = [vp, f32, f32, f32, f32]
    L.tdgl_step.argtypes = [vp, i32]
    L.tdgl_get_psi_mu.argtypes = [vp, vp, vp]
    L.tdgl_observables.argtypes = [vp, C.POINTER(TdglObs)]
    L.tdgl_strerror.restype = C.c_char_p
    L.tdgl_strerror.argtypes = [C.c_int]
    L.tdgl_last_cuda_error.argtypes = [vp]
    L.tdgl_set_state.argtypes = [vp, vp, vp, f64]
    L.tdgl_set_solver.argtypes = [vp, f32, i32, i32]
    L.tdgl_set_sweep_schedule.argtypes = [vp, C.POINTER(i32), i32]
    L.tdgl_get_sweep_log.argtypes = [vp, C.POINTER(i32), C.POINTER(f32), i32]
    L.tdgl_get_eps.argtypes = [vp, vp]
    L.tdgl_debug_noise.argtypes = [vp, i64, vp]
    L.tdgl_debug_poisson.argtypes = [vp, vp, vp]
    L.tdgl_debug_rho.argtypes = [vp, vp]
    L.tdgl_launch_count.restype = i64
    L.tdgl_launch_count.argtypes = [vp]
    L.tdgl_sweep_timing.argtypes = [vp, i32, C.POINTER(f64), C.POINTER(i64)]
    L.tdgl_mu_gain.restype = f64
    L.tdgl_mu_gain.argtypes = [C.POINTER(TdglParams)]
    L.tdgl_mu_refine_enabled.argtypes = [vp]
    L.tdgl_set_mu_solver.argtypes = [vp, f32, f32, f32, i32, i32]
    L.tdgl_set_insulators.argtypes = [vp, C.POINTER(TdglSphere), i64]
    L.tdgl_set_pinning_shapes.argtypes = [vp, vp, i64, f32, f32]
    L.tdgl_set_insulator_shapes.argtypes = [vp, vp, i64]
    L.tdgl_get_mu_direct_stats.argtypes = [vp, C.POINTER(i64), C.POINTER(i64), C.POINTER(f64)]
    L.tdgl_set_pair_mode.argtypes = [vp, i32]
    L.tdgl_get_pair_stats.argtypes = [vp, C.POINTER(i32), C.POINTER(i64), C.POINTER(i64)]
    L.tdgl_get_mu_log.argtypes = [vp, i32, C.POINTER(i32), C.POINTER(i32), i32, C.POINTER(i32)]
    L.tdgl_mean_abs2_static.argtypes = [vp, i64, vp, vp]
    _lib = L
    return L


def tdgl_strerror(code: int) -> str:
    return lib().tdgl_strerror(int(code)).decode()


def _check(code: int, what: str, handle=None, allow_warning: bool = True) -> int:
    if code < 0 or (code > 0 and not allow_warning):
        cuda = lib().tdgl_last_cuda_error(handle) if handle else 0
        raise TdglError(code, what, cuda)
    return code


# ---- the six calls of the boundary, same names as in include/tdgl.h -------------------------------
def tdgl_workspace_bytes(params: TdglParams) -> int:
    params.struct_size = C.sizeof(TdglParams)
    return int(lib().tdgl_workspace_bytes(C.byref(params)))


def tdgl_create(params: TdglParams) -> C.c_void_p:
    params.struct_size = C.sizeof(TdglParams)
    h = C.c_void_p()
    _check(lib().tdgl_create(C.byref(params), C.byref(h)), "tdgl_create")
    return h


def tdgl_destroy(h) -> None:
    _check(lib().tdgl_destroy(h), "tdgl_destroy")


def tdgl_set_pinning(h, spheres: np.ndarray, eps_in: float, eps_out: float) -> None:
    """spheres: float32 array (n, 4) = (cx, cy, cz, r), HOST memory."""
    s = np.ascontiguousarray(spheres, dtype=np.float32).reshape(-1, 4)
    ptr = s.ctypes.data_as(C.POINTER(TdglSphere)) if len(s) else None
    _check(lib().tdgl_set_pinning(h, ptr, len(s), eps_in, eps_out), "tdgl_set_pinning", h)


def tdgl_set_pinning_shapes(h, shapes: np.ndarray, eps_in: float, eps_out: float) -> None:
    """shapes: float32 array (n, 10) = (kind, c[3], a[3], n[3]) (tdgl_shape), HOST memory."""
    s = np.ascontiguousarray(shapes, dtype=np.float32).reshape(-1, 10)
    _check(lib().tdgl_set_pinning_shapes(h, s.ctypes.data if len(s) else None, len(s), eps_in, eps_out), "tdgl_set_pinning_shapes", h)


def tdgl_set_insulator_shapes(h, shapes: np.ndarray) -> None:
    s = np.ascontiguousarray(shapes, dtype=np.float32).reshape(-1, 10)
    _check(lib().tdgl_set_insulator_shapes(h, s.ctypes.data if len(s) else None, len(s)), "tdgl_set_insulator_shapes", h)


def tdgl_set_field_current(h, Bx: float, By: float, Bz: float, Jx: float) -> None:
    _check(lib().tdgl_set_field_current(h, Bx, By, Bz, Jx), "tdgl_set_field_current", h)


def tdgl_step(h, nsteps: int) -> None:
    _check(lib().tdgl_step(h, int(nsteps)), "tdgl_step", h)


def tdgl_get_psi_mu(h, psi_dev_ptr: Optional[int], mu_dev_ptr: Optional[int]) -> None:
    _check(lib().tdgl_get_psi_mu(h, psi_dev_ptr, mu_dev_ptr), "tdgl_get_psi_mu", h)


def tdgl_observables(h) -> TdglObs:
    o = TdglObs()
    _check(lib().tdgl_observables(h, C.byref(o)), "tdgl_observables", h)
    return o


def tdgl_mean_abs2_static(psi_dev_ptr: Optional[int], n_sites: int, mean_dev_ptr: Optional[int], stream_ptr: Optional[int] = None) -> None:
    """<|psi|^2> of n_sites (re, im) fp32 pairs at DEVICE address psi_dev_ptr into the double at DEVICE address
    mean_dev_ptr, enqueued on the CUDA stream stream_ptr -- for callers that hold a pointer to psi but cannot allocate
    device memory (no handle, no workspace: the scratch is a fixed array inside libtdgl.so).  At most
    TDGL_STATIC_MAX_SITES sites (TdglError with code TDGL_ESCRATCH beyond); one call at a time per device; make the
    first call on a device at start-up.  See include/tdgl.h."""
    _check(lib().tdgl_mean_abs2_static(psi_dev_ptr, int(n_sites), mean_dev_ptr, stream_ptr), "tdgl_mean_abs2_static")


# ---- convenience wrapper: torch owns the device memory and the stream ------------------------------
class Solver:
    """One TDGL problem on the current CUDA device.  Allocates the workspace as a torch tensor, passes
    torch's current stream, and forwards every call to libtdgl.  Holds no arithmetic."""

    def __init__(self, nx: int, ny: int, nz: int, bc: Sequence[int] = (0, 0, 0), h: float = 0.5, dt: float = 0.1,
                 u: float = 1.0, g: float = 1.0, eps_tol: float = 1e-6, max_sweeps: int = 100, fixed_sweeps: int = 0,
                 temperature: float = 0.0, seed: int = 0, init_amp: float = 0.01, solve_mu: bool = True,
                 host_loop: bool = False, hxyz: Optional[Sequence[float]] = None, device: Optional[str] = None,
                 gauge_yz: bool = False, mu_refine: Optional[bool] = None, mu_iterative: bool = False, fp64: bool = False, insulators: bool = False,
                 mu_direct: bool = False):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1409_8340_b200 needs a CUDA device (sm_100a); there is no CPU path")
        self.torch = torch
        # the CURRENT device unless one is named (one process per GPU: bench.py sets it from LOCAL_RANK)
        self.device = torch.device(device) if device is not None else torch.device("cuda", torch.cuda.current_device())
        torch.cuda.set_device(self.device)
        hx, hy, hz = (hxyz if hxyz is not None else (h, h, h))
        p = TdglParams()
        p.nx, p.ny, p.nz = nx, ny, nz
        p.hx, p.hy, p.hz, p.dt, p.u, p.g = hx, hy, hz, dt, u, g
        p.bc[0], p.bc[1], p.bc[2] = bc
        p.eps_tol, p.max_sweeps, p.fixed_sweeps = eps_tol, max_sweeps, fixed_sweeps
        p.temperature, p.seed, p.init_amp = temperature, seed, init_amp
        p.flags = ((TDGL_FLAG_SOLVE_MU if solve_mu else 0) | (TDGL_FLAG_HOST_LOOP if host_loop else 0)
                   | (TDGL_FLAG_GAUGE_YZ if gauge_yz else 0)
                   | (0 if mu_refine is None else (TDGL_FLAG_MU_REFINE if mu_refine else TDGL_FLAG_MU_NOREFINE))
                   | (TDGL_FLAG_MU_ITERATIVE if mu_iterative else 0) | (TDGL_FLAG_FP64 if fp64 else 0)
                   | (TDGL_FLAG_INSULATORS if insulators else 0) | (TDGL_FLAG_MU_DIRECT if mu_direct else 0))
        self.fp64 = bool(fp64)
        nbytes = tdgl_workspace_bytes(p)
        if nbytes == 0:
            raise TdglError(TDGL_EINVAL, "tdgl_workspace_bytes")
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = (self.workspace.data_ptr() + 255) // 256 * 256
        self.stream = torch.cuda.current_stream(self.device)
        p.workspace_dev, p.workspace_bytes, p.stream = base, nbytes, self.stream.cuda_stream
        self.params = p
        self.shape = (nz, ny, nx)
        self.n_sites = nx * ny * nz
        self.h = tdgl_create(p)

    def close(self):
        if getattr(self, "h", None):
            tdgl_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # the boundary
    def set_pinning(self, spheres, eps_in=-1.0, eps_out=1.0):
        tdgl_set_pinning(self.h, np.asarray(spheres, dtype=np.float32), eps_in, eps_out)

    def set_insulators(self, spheres):
        """spheres: float32 array (n, 4) = (cx, cy, cz, r), HOST memory (TDGL_FLAG_INSULATORS)."""
        s = np.ascontiguousarray(spheres, dtype=np.float32).reshape(-1, 4)
        ptr = s.ctypes.data_as(C.POINTER(TdglSphere)) if len(s) else None
        _check(lib().tdgl_set_insulators(self.h, ptr, len(s)), "tdgl_set_insulators", self.h)

    def set_pinning_shapes(self, shapes, eps_in=-1.0, eps_out=1.0):
        tdgl_set_pinning_shapes(self.h, shapes, eps_in, eps_out)

    def set_insulator_shapes(self, shapes):
        tdgl_set_insulator_shapes(self.h, shapes)

    def set_field_current(self, Bx=0.0, By=0.0, Bz=0.0, Jx=0.0):
        tdgl_set_field_current(self.h, Bx, By, Bz, Jx)

    def step(self, n=1):
        tdgl_step(self.h, n)

    @property
    def real_dtype(self):
        """torch dtype of the state the library holds: float32, or float64 with TDGL_FLAG_FP64."""
        return self.torch.float64 if self.fp64 else self.torch.float32

    def get_psi_mu(self):
        t = self.torch
        psi = t.empty(self.shape + (2,), dtype=self.real_dtype, device=self.device)
        mu = t.empty(self.shape, dtype=self.real_dtype, device=self.device)
        tdgl_get_psi_mu(self.h, psi.data_ptr(), mu.data_ptr())
        return t.view_as_complex(psi), mu

    def observables(self) -> TdglObs:
        return tdgl_observables(self.h)

    # extensions
    def set_state(self, psi, mu=None, K: float = 0.0):
        t = self.torch
        psi = t.view_as_real(psi.to(self.device, t.complex128 if self.fp64 else t.complex64).contiguous())
        assert psi.numel() == 2 * self.n_sites
        mu_ptr = None
        if mu is not None:
            mu = mu.to(self.device, self.real_dtype).contiguous()
            assert mu.numel() == self.n_sites
            mu_ptr = mu.data_ptr()
        _check(lib().tdgl_set_state(self.h, psi.data_ptr(), mu_ptr, float(K)), "tdgl_set_state", self.h)
        self.stream.synchronize()     # psi / mu may be temporaries

    def set_solver(self, eps_tol: float, max_sweeps: int, fixed_sweeps: int = 0):
        _check(lib().tdgl_set_solver(self.h, eps_tol, max_sweeps, fixed_sweeps), "tdgl_set_solver", self.h)

    def set_sweep_schedule(self, counts):
        c = np.ascontiguousarray(counts, dtype=np.int32)
        ptr = c.ctypes.data_as(C.POINTER(C.c_int32)) if len(c) else None
        _check(lib().tdgl_set_sweep_schedule(self.h, ptr, len(c)), "tdgl_set_sweep_schedule", self.h)

    def sweep_log(self, n: int):
        c = np.zeros(n, dtype=np.int32)
        r = np.zeros(n, dtype=np.float32)
        _check(lib().tdgl_get_sweep_log(self.h, c.ctypes.data_as(C.POINTER(C.c_int32)),
                                        r.ctypes.data_as(C.POINTER(C.c_float)), n), "tdgl_get_sweep_log", self.h)
        return c, r

    def get_eps(self):
        t = self.torch
        e = t.empty(self.shape, dtype=t.float32, device=self.device)
        _check(lib().tdgl_get_eps(self.h, e.data_ptr()), "tdgl_get_eps", self.h)
        return e

    def debug_noise(self, step: int):
        t = self.torch
        z = t.empty(self.shape + (2,), dtype=self.real_dtype, device=self.device)
        _check(lib().tdgl_debug_noise(self.h, step, z.data_ptr()), "tdgl_debug_noise", self.h)
        return t.view_as_complex(z)

    def debug_poisson(self, rho):
        t = self.torch
        mu = rho.to(self.device, self.real_dtype).contiguous().clone()
        _check(lib().tdgl_debug_poisson(self.h, mu.data_ptr(), mu.data_ptr()), "tdgl_debug_poisson", self.h)
        return mu

    def debug_rho(self):
        t = self.torch
        rho = t.empty(self.shape, dtype=self.real_dtype, device=self.device)
        _check(lib().tdgl_debug_rho(self.h, rho.data_ptr()), "tdgl_debug_rho", self.h)
        return rho

    def set_mu_solver(self, h_tau: float = 0.1, eps_mu: float = 1e-6, eps_in: float = 1e-6, max_outer: int = 1000,
                      max_inner: int = 100):
        _check(lib().tdgl_set_mu_solver(self.h, h_tau, eps_mu, eps_in, max_outer, max_inner), "tdgl_set_mu_solver", self.h)

    def mu_log(self, nsolves: int):
        """(outer iterations per solve, list of per-solve lists of inner sweep counts) of the last nsolves mu solves."""
        outer = np.zeros(nsolves, dtype=np.int32)
        n_in = C.c_int32()
        _check(lib().tdgl_get_mu_log(self.h, nsolves, outer.ctypes.data_as(C.POINTER(C.c_int32)), None, 0, C.byref(n_in)),
               "tdgl_get_mu_log", self.h)
        inner = np.zeros(max(1, n_in.value), dtype=np.int32)
        _check(lib().tdgl_get_mu_log(self.h, nsolves, outer.ctypes.data_as(C.POINTER(C.c_int32)),
                                     inner.ctypes.data_as(C.POINTER(C.c_int32)), len(inner), C.byref(n_in)),
               "tdgl_get_mu_log", self.h)
        out, pos = [], 0
        for o in outer:
            out.append([int(v) for v in inner[pos:pos + o]])
            pos += o
        return outer, out

    def mu_gain(self) -> float:
        return float(lib().tdgl_mu_gain(C.byref(self.params)))

    def mu_refine_enabled(self) -> bool:
        return bool(lib().tdgl_mu_refine_enabled(self.h))

    def launch_count(self) -> int:
        return int(lib().tdgl_launch_count(self.h))

    def mu_direct_stats(self):
        """TDGL_FLAG_MU_DIRECT: (solves, refinement passes, max |rho - Delta_h mu| of the last solve)."""
        a, b, r = C.c_int64(), C.c_int64(), C.c_double()
        _check(lib().tdgl_get_mu_direct_stats(self.h, C.byref(a), C.byref(b), C.byref(r)), "tdgl_get_mu_direct_stats", self.h)
        return a.value, b.value, r.value

    def set_pair_mode(self, mode: int):
        """Fused sweep pairs: 0 never, 1 automatic (default), 2 whenever the cap allows (forces the redo path)."""
        _check(lib().tdgl_set_pair_mode(self.h, int(mode)), "tdgl_set_pair_mode", self.h)

    def pair_stats(self):
        """(mesh eligible, pairs launched, pairs discarded and redone as plain sweeps)."""
        e, a, b = C.c_int32(), C.c_int64(), C.c_int64()
        _check(lib().tdgl_get_pair_stats(self.h, C.byref(e), C.byref(a), C.byref(b)), "tdgl_get_pair_stats", self.h)
        return bool(e.value), a.value, b.value

    def sweep_timing(self, enable):
        """enable: 0 / False off, 1 / True plain sweeps, 2 fused pairs."""
        ms, n = C.c_double(), C.c_int64()
        _check(lib().tdgl_sweep_timing(self.h, int(enable), C.byref(ms), C.byref(n)), "tdgl_sweep_timing", self.h)
        return ms.value, n.value
