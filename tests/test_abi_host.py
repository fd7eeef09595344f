"""CPU-side checks of the boundary: libtdgl.so loads and exports every symbol include/tdgl.h declares,
the binding's structs match the header, and the host-only logic (parameter validation, workspace
size, error strings) behaves as the header states.  No kernel is launched here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "tdgl.h")


@pytest.fixture(scope="module")
def L():
    from paper_1409_8340_b200 import build as B
    B.build()
    from paper_1409_8340_b200 import binding
    return binding.lib()


def declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(tdgl_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_six_calls_of_the_north_star():
    names = declared_functions()
    for n in ("tdgl_create", "tdgl_set_pinning", "tdgl_set_field_current", "tdgl_step", "tdgl_get_psi_mu",
              "tdgl_observables", "tdgl_destroy", "tdgl_workspace_bytes", "tdgl_strerror"):
        assert n in names


def test_library_exports_every_declared_symbol(L):
    from paper_1409_8340_b200.binding import EXPORTS
    names = declared_functions()
    assert names, "no declarations parsed"
    for n in names:
        assert hasattr(L, n), f"libtdgl.so does not export {n}"
    assert sorted(EXPORTS) == names, "binding.EXPORTS and include/tdgl.h disagree"


def test_no_torch_types_in_the_header():
    src = open(HEADER).read()
    assert 'extern "C"' in src
    for bad in ("torch", "at::", "Tensor", "std::"):
        assert bad not in src


def _params(**kw):
    from paper_1409_8340_b200.binding import TdglParams
    p = TdglParams()
    p.struct_size = C.sizeof(TdglParams)
    p.nx, p.ny, p.nz = 32, 32, 32
    p.hx = p.hy = p.hz = 0.5
    p.dt, p.u, p.g = 0.1, 1.0, 1.0
    p.bc[0] = p.bc[1] = p.bc[2] = 0
    p.eps_tol, p.max_sweeps, p.fixed_sweeps = 1e-6, 100, 0
    p.temperature, p.seed, p.init_amp, p.flags = 0.0, 0, 0.01, 1
    for k, v in kw.items():
        if k == "bc":
            for a in range(3):
                p.bc[a] = v[a]
        else:
            setattr(p, k, v)
    return p


def test_struct_layout_matches_the_header(L):
    """struct_size is the version check of the ABI: a mismatch makes every call return EINVAL / 0."""
    from paper_1409_8340_b200.binding import TdglObs, TdglParams, TdglSphere
    assert L.tdgl_workspace_bytes(C.byref(_params())) > 0
    bad = _params()
    bad.struct_size = C.sizeof(TdglParams) - 4
    assert L.tdgl_workspace_bytes(C.byref(bad)) == 0
    assert C.sizeof(TdglSphere) == 16
    assert C.sizeof(TdglObs) == 9 * 8 + 2 * 4 + 2 * 8 + 2 * 4


def test_workspace_bytes_scales_with_sites(L):
    # psi x2, b, d (8 B each) + mu, eps, scratch (4 B each) = 44 B per site + small tables
    for (nx, ny, nz) in ((32, 32, 32), (64, 64, 64), (512, 512, 256), (1024, 1024, 512), (34, 13, 11)):
        w = L.tdgl_workspace_bytes(C.byref(_params(nx=nx, ny=ny, nz=nz)))
        n = nx * ny * nz
        assert 44 * n <= w <= 44 * n + (4 << 20), (nx, ny, nz, w)
    assert L.tdgl_workspace_bytes(C.byref(_params(nx=1024, ny=1024, nz=512))) < 30e9     # C5 fits 180 GB many times


@pytest.mark.parametrize("kw", [
    dict(nx=33), dict(nx=0), dict(ny=1), dict(nz=-4), dict(hx=0.0), dict(hy=-1.0), dict(dt=0.0), dict(u=0.0),
    dict(g=0.0), dict(bc=(0, 2, 0)), dict(bc=(-1, 0, 0)), dict(eps_tol=-1.0), dict(max_sweeps=0),
    dict(max_sweeps=100000), dict(fixed_sweeps=-1), dict(temperature=-1.0), dict(hz=float("nan")),
])
def test_invalid_params_are_rejected_on_the_host(L, kw):
    from paper_1409_8340_b200.binding import TDGL_EINVAL
    p = _params(**kw)
    assert L.tdgl_workspace_bytes(C.byref(p)) == 0
    h = C.c_void_p()
    assert L.tdgl_create(C.byref(p), C.byref(h)) == TDGL_EINVAL
    assert not h.value


def test_create_rejects_missing_or_misaligned_workspace(L):
    from paper_1409_8340_b200.binding import TDGL_EINVAL, TDGL_ENOMEM
    p = _params()
    h = C.c_void_p()
    assert L.tdgl_create(C.byref(p), C.byref(h)) == TDGL_ENOMEM          # workspace_dev == NULL
    p.workspace_dev, p.workspace_bytes = 0x10000100, 16                   # too small (never dereferenced)
    assert L.tdgl_create(C.byref(p), C.byref(h)) == TDGL_ENOMEM
    p.workspace_dev, p.workspace_bytes = 0x10000101, 1 << 40              # misaligned
    assert L.tdgl_create(C.byref(p), C.byref(h)) == TDGL_ENOMEM
    assert L.tdgl_create(C.byref(p), None) == TDGL_EINVAL


def test_null_handles_are_rejected(L):
    from paper_1409_8340_b200.binding import TDGL_EINVAL, TdglObs
    assert L.tdgl_destroy(None) == TDGL_EINVAL
    assert L.tdgl_step(None, 1) == TDGL_EINVAL
    assert L.tdgl_set_field_current(None, 0.0, 0.0, 0.0, 0.0) == TDGL_EINVAL
    assert L.tdgl_set_pinning(None, None, 0, -1.0, 1.0) == TDGL_EINVAL
    assert L.tdgl_get_psi_mu(None, None, None) == TDGL_EINVAL
    ob = TdglObs()
    assert L.tdgl_observables(None, C.byref(ob)) == TDGL_EINVAL
    assert L.tdgl_launch_count(None) == 0


def test_strerror_covers_every_code(L):
    from paper_1409_8340_b200 import binding as Bd
    seen = set()
    for code in (Bd.TDGL_OK, Bd.TDGL_EINVAL, Bd.TDGL_ENOMEM, Bd.TDGL_EINCOMPAT, Bd.TDGL_ECUDA, Bd.TDGL_ESCRATCH, Bd.TDGL_WMAXSWEEPS, Bd.TDGL_WMUCAP):
        s = Bd.tdgl_strerror(code)
        assert s and s != "unknown code"
        seen.add(s)
    assert len(seen) == 8
    assert Bd.tdgl_strerror(12345) == "unknown code"
    # the header's numeric values
    src = open(HEADER).read()
    for name in ("TDGL_OK", "TDGL_EINVAL", "TDGL_ENOMEM", "TDGL_EINCOMPAT", "TDGL_ECUDA", "TDGL_ESCRATCH", "TDGL_WMAXSWEEPS", "TDGL_WMUCAP"):
        m = re.search(r"#define\s+%s\s+\(?(-?\d+)\)?" % name, src)
        assert m and int(m.group(1)) == getattr(Bd, name), name


def test_solver_wrapper_fails_loudly_without_cuda():
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    from paper_1409_8340_b200 import Solver
    with pytest.raises(Exception):
        Solver(32, 32, 32)


def test_product_path_does_not_import_the_oracle():
    """The oracle is test infrastructure: nothing under the package (or bench.py's GPU arm) may route through it."""
    pkg = os.path.join(ROOT, "paper_1409_8340_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), f
                assert "tdgl_oracle" not in txt, f
    otxt = open(os.path.join(ROOT, "oracle", "tdgl_oracle.py")).read()
    assert "paper_1409_8340_b200" not in otxt and "ctypes" not in otxt


def test_input_recipes_match_the_baseline_configs():
    import tdgl_inputs as I
    shapes = {"C1": (32, 32, 32), "C2": (64, 64, 64), "C3": (256, 256, 128), "C4": (512, 512, 256),
              "C5a": (1024, 1024, 512), "C5b": (1024, 1024, 512)}
    for k, s in shapes.items():
        c = I.CONFIGS[k]
        assert (c.nx, c.ny, c.nz) == s and c.h == 0.5 and c.dt == 0.1
    assert tuple(I.CONFIGS["C4"].bc) == (0, 0, 1) and tuple(I.CONFIGS["C5a"].bc) == (1, 1, 1)
    assert tuple(I.CONFIGS["C5b"].bc) == (0, 1, 1) and I.CONFIGS["C5a"].Jx == 0.0
    # S19: n_s = round(-ln(1 - f) V / vbar), seeded and reproducible
    c = I.CONFIGS["C2"]
    a, b = I.sphere_list(c), I.sphere_list(c)
    assert a.dtype == np.float32 and a.shape[1] == 4 and np.array_equal(a, b)
    V = (c.nx * c.h) * (c.ny * c.h) * (c.nz * c.h)
    assert len(a) == round(-np.log(1 - 0.10) * V / (4 / 3 * np.pi * 2.0 ** 3))
    assert len(I.sphere_list(I.CONFIGS["C1"])) == 0


def test_mu_gain_is_the_white_noise_gain_of_the_inverse_laplacian(L):
    """tdgl_mu_gain (host arithmetic only): G = ((1/N) sum_{q != 0} 1/lambda_q^2)^{1/2} against the exact sum over the
    oracle's eigenvalue table on small meshes; the automatic refinement rule G > TDGL_MU_REFINE_GAIN = 200 leaves the
    3D BASELINE grids alone and catches long thin meshes."""
    import math
    from oracle import tdgl_oracle as O
    L.tdgl_mu_gain.restype = C.c_double

    def gain_c(nx, ny, nz, bc, h=(0.5, 0.5, 0.5), g=1.0):
        p = _params(nx=nx, ny=ny, nz=nz, hx=h[0], hy=h[1], hz=h[2], g=g)
        p.bc[0], p.bc[1], p.bc[2] = bc
        return L.tdgl_mu_gain(C.byref(p))

    for (nx, ny, nz), bc, h, g in [((34, 13, 11), (0, 1, 1), (0.5, 0.4, 0.7), 1.3), ((200, 6, 1), (1, 0, 0), (0.5, 0.5, 0.5), 1.0),
                                   ((64, 64, 32), (0, 0, 1), (0.5, 0.5, 0.5), 1.0), ((30, 30, 30), (1, 1, 1), (0.5, 0.5, 0.5), 1.0)]:
        f32 = lambda v: float(np.float32(v))
        p = O.Params(nx, ny, nz, hx=f32(h[0]), hy=f32(h[1]), hz=f32(h[2]), g=f32(g), bc=(bc[0], bc[1], 0 if nz == 1 else bc[2]))
        lam = O.laplacian_eigenvalues(p).ravel()
        lam = lam[np.abs(lam) > 1e-12]
        exact = math.sqrt(np.sum(1.0 / lam ** 2) / p.n_sites)
        assert abs(gain_c(nx, ny, nz, bc, h, g) - exact) < 1e-2 * exact, (nx, ny, nz, bc)   # 48 lowest modes per axis carry the sum
    assert gain_c(512, 512, 256, (0, 0, 1)) < 1.0 and gain_c(1024, 1024, 512, (1, 1, 1)) < 3.0
    assert gain_c(256, 256, 128, (0, 0, 1)) < 1.0 and gain_c(64, 64, 64, (0, 0, 0)) < 1.0
    assert gain_c(1026, 4, 1, (1, 1, 0)) > 400.0 and gain_c(2050, 10, 1, (1, 0, 0)) > 700.0
    bad = _params(nx=31)
    assert L.tdgl_mu_gain(C.byref(bad)) == -1.0
