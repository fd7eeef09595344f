"""Seeded synthetic inputs shared by the oracle tests, the GPU tests and bench.py.

This module holds NONE of the method's arithmetic (no stencil, no Philox, no
Poisson, no epsilon inside-test): it only fixes the *workloads* -- grid sizes,
boundary types, field / current / temperature values, initial order parameter
and sphere lists -- so that the CUDA path and the fp64 oracle are fed the
very same numbers.  Neither `oracle/` nor `paper_1409_8340_b200/` is imported
here.

The five configurations are the ones `BASELINE.json: configs[0..4]` names
(C1..C5); the recipe is restated in DESIGN.md ("Synthetic input recipe").  The
paper used no public data set: its workloads were its own seeded runs
(PAPER.md:571 "randomly initialized", :513 "random lattices").
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import Optional, Tuple

import numpy as np

PERIODIC = 0
OPEN = 1


@dataclass(frozen=True)
class Config:
    name: str
    nx: int
    ny: int
    nz: int
    bc: Tuple[int, int, int]            # per axis: PERIODIC / OPEN
    h: float = 0.5                      # mesh size in xi_0 (all configs)
    dt: float = 0.1
    Bx: float = 0.0                     # requested field (H_c2 units), before snapping
    Bz: float = 0.0
    Jx: float = 0.0
    temperature: float = 0.0            # reduced T-bar of PAPER.md Eq.(39)
    incl_fraction: float = 0.0          # target covered volume fraction
    incl_rmin: float = 0.0              # sphere radii uniform in [rmin, rmax] (xi_0)
    incl_rmax: float = 0.0
    eps_in: float = -1.0
    eps_out: float = 1.0
    steps: int = 100
    init_amp: float = 0.01              # psi0 = 1 + init_amp * (N(0,1) + i N(0,1))
    seed: int = 0
    nz_flux: Optional[int] = None       # if set: Bz = 2 pi nz_flux / (Lx Ly) exactly

    @property
    def n_sites(self) -> int:
        return self.nx * self.ny * self.nz

    def lengths(self) -> Tuple[float, float, float]:
        """L_a = N_a h (periodic) or (N_a - 1) h (open)  -- PAPER.md:243."""
        n = (self.nx, self.ny, self.nz)
        return tuple((n[a] - (1 if self.bc[a] == OPEN else 0)) * self.h for a in range(3))

    def requested_field(self) -> Tuple[float, float]:
        """(Bx, Bz) handed to set_field_current (the solver snaps to flux quanta)."""
        if self.nz_flux is not None:
            lx, ly, _ = self.lengths()
            return self.Bx, 2.0 * math.pi * self.nz_flux / (lx * ly)
        return self.Bx, self.Bz

    def scaled(self, nx: int, ny: int, nz: int, name: Optional[str] = None) -> "Config":
        """Same physics on a smaller grid (replica used where the oracle must finish in seconds)."""
        return replace(self, nx=nx, ny=ny, nz=nz, name=name or f"{self.name}@{nx}x{ny}x{nz}")


def _tilt(b: float, deg: float) -> Tuple[float, float]:
    return b * math.sin(math.radians(deg)), b * math.cos(math.radians(deg))


_c3bx, _c3bz = _tilt(0.2, 30.0)

CONFIGS = {
    # C1: 32^3, quasi-periodic all axes, 4 flux quanta through xy, no pinning/current/noise.
    "C1": Config("C1", 32, 32, 32, (PERIODIC,) * 3, nz_flux=4, steps=100),
    # C2: 64^3 periodic, Bz = 0.1 Hc2, 10 % spheres r=2, Jx=0.01, T=1e-3, 1000 steps.
    "C2": Config("C2", 64, 64, 64, (PERIODIC,) * 3, Bz=0.1, Jx=0.01, temperature=1e-3,
                 incl_fraction=0.10, incl_rmin=2.0, incl_rmax=2.0, steps=1000),
    # C3: 256x256x128, periodic x,y / open z, 0.2 Hc2 tilted 30 deg from z in the xz plane,
    #     15 % spheres r in [1.5,3]; I-V sweep is harness level (10 currents x 2000 steps).
    "C3": Config("C3", 256, 256, 128, (PERIODIC, PERIODIC, OPEN), Bx=_c3bx, Bz=_c3bz, Jx=0.005,
                 temperature=1e-3, incl_fraction=0.15, incl_rmin=1.5, incl_rmax=3.0, steps=2000),
    # C4: 512x512x256 headline, periodic x,y / open z, Bz=0.3, 20 % spheres r=2, Jx=0.02, T=1e-3.
    "C4": Config("C4", 512, 512, 256, (PERIODIC, PERIODIC, OPEN), Bz=0.3, Jx=0.02,
                 temperature=1e-3, incl_fraction=0.20, incl_rmin=2.0, incl_rmax=2.0, steps=5000),
    # C5a: 1024x1024x512 open on all faces, Jx=0 (PAPER.md:481 forbids a current with open x).
    "C5a": Config("C5a", 1024, 1024, 512, (OPEN,) * 3, Bz=0.2, Jx=0.0, temperature=1e-3,
                  incl_fraction=0.10, incl_rmin=1.0, incl_rmax=4.0, steps=500),
    # C5b: same grid, x periodic so that the transport current Jx=0.01 of BASELINE.json can flow.
    "C5b": Config("C5b", 1024, 1024, 512, (PERIODIC, OPEN, OPEN), Bz=0.2, Jx=0.01,
                  temperature=1e-3, incl_fraction=0.10, incl_rmin=1.0, incl_rmax=4.0, steps=500),
    # The paper's own timed workloads ("disorder-free system with periodic boundary conditions
    # with a magnetic field applied in z direction and an external current in x direction", eps_tol 1e-6), as
    # context beside its K20Xm numbers.  The paper gives neither B nor J for them; B_z = 0.1 puts ~267 000 vortices
    # on the 8192^2 film, the ">250 000" of its Fig. 4; J_x = 0.02 and T = 0 are ours.
    "F2D": Config("F2D", 8192, 8192, 1, (PERIODIC, PERIODIC, PERIODIC), Bz=0.1, Jx=0.02, steps=1000),
    # 3D counterpart of its 406^3 run (66.9e6 sites): 512 x 512 x 256 (67.1e6 sites), all periodic, eps = 1.
    "P3D": Config("P3D", 512, 512, 256, (PERIODIC, PERIODIC, PERIODIC), Bz=0.1, Jx=0.02, steps=1000),
}
C3_CURRENTS = tuple(round(0.005 * (i + 1), 6) for i in range(10))   # 0.005 .. 0.05


def initial_psi(cfg: Config, seed: Optional[int] = None) -> np.ndarray:
    """psi0[k, j, i] = 1 + init_amp * (N(0,1) + i N(0,1)), complex64, seeded (BASELINE.json C1).

    Returned in the storage order m = i + nx*(j + ny*k), i.e. shape (nz, ny, nx).
    The values are rounded to fp32 ONCE here, so the oracle (which widens them to fp64) and the
    CUDA path start from bit-identical numbers.
    """
    rng = np.random.default_rng(cfg.seed if seed is None else seed)
    shape = (cfg.nz, cfg.ny, cfg.nx)
    re = rng.standard_normal(shape, dtype=np.float32)
    im = rng.standard_normal(shape, dtype=np.float32)
    out = np.empty(shape, dtype=np.complex64)
    out.real = np.float32(1.0) + np.float32(cfg.init_amp) * re
    out.imag = np.float32(cfg.init_amp) * im
    return out


def random_state(cfg: Config, seed: int, amp: float = 1.0) -> Tuple[np.ndarray, np.ndarray]:
    """A rough (psi, mu) pair for single-kernel parity tests: psi complex64 with |psi|~amp and random
    phase structure, mu float32 ~ U(-0.1, 0.1)."""
    rng = np.random.default_rng(seed)
    shape = (cfg.nz, cfg.ny, cfg.nx)
    psi = np.empty(shape, dtype=np.complex64)
    psi.real = (amp * rng.uniform(-1, 1, shape)).astype(np.float32)
    psi.imag = (amp * rng.uniform(-1, 1, shape)).astype(np.float32)
    mu = rng.uniform(-0.1, 0.1, shape).astype(np.float32)
    return psi, mu


def sphere_list(cfg: Config, seed: Optional[int] = None) -> np.ndarray:
    """Seeded inclusion list, float32 array (n_s, 4) = (cx, cy, cz, r) in xi_0, domain coords [0, L).

    Placement law (the paper only says "random lattices"): centres uniform in the
    box, overlaps allowed, radius uniform in [rmin, rmax]; the count is chosen so that the EXPECTED
    covered fraction is f for Poisson-placed overlapping spheres:
        n_s = round( -ln(1 - f) * V / E[4/3 pi r^3] ).
    """
    if cfg.incl_fraction <= 0.0:
        return np.zeros((0, 4), dtype=np.float32)
    lx, ly, lz = cfg.lengths()
    vol = lx * ly * lz
    a, b = cfg.incl_rmin, cfg.incl_rmax
    mean_r3 = a ** 3 if a == b else (b ** 4 - a ** 4) / (4.0 * (b - a))
    n_s = int(round(-math.log(1.0 - cfg.incl_fraction) * vol / (4.0 / 3.0 * math.pi * mean_r3)))
    rng = np.random.default_rng((cfg.seed if seed is None else seed) + 7919)
    out = np.empty((n_s, 4), dtype=np.float32)
    out[:, 0] = rng.uniform(0.0, lx, n_s)
    out[:, 1] = rng.uniform(0.0, ly, n_s)
    out[:, 2] = rng.uniform(0.0, lz, n_s)
    out[:, 3] = rng.uniform(a, b, n_s) if b > a else a
    return out


def shape_list(cfg: Config, n_ellipsoids: int, n_columns: int, seed: Optional[int] = None) -> np.ndarray:
    """Seeded list of the further generator shapes (Fig. 2d/e), float32 array (n, 10) =
    (kind, c_x, c_y, c_z, a_0, a_1, a_2, n_x, n_y, n_z): `n_ellipsoids` axis-aligned ellipsoids (kind 1) with semi-axes
    uniform in [rmin, 2 rmax] at uniform random centres, then `n_columns` columnar defects (kind 2) of radius uniform
    in [rmin, rmax] through the whole thickness, tilted by +45 or -45 degrees from z in the xz plane with equal
    probability (Fig. 2e)."""
    lx, ly, lz = cfg.lengths()
    a, b = max(cfg.incl_rmin, 0.5), max(cfg.incl_rmax, 1.0)
    rng = np.random.default_rng((cfg.seed if seed is None else seed) + 104729)
    n = n_ellipsoids + n_columns
    out = np.zeros((n, 10), dtype=np.float32)
    out[:, 1] = rng.uniform(0.0, lx, n)
    out[:, 2] = rng.uniform(0.0, ly, n)
    out[:, 3] = rng.uniform(0.0, lz, n)
    out[:n_ellipsoids, 0] = 1
    out[:n_ellipsoids, 4:7] = rng.uniform(a, 2.0 * b, (n_ellipsoids, 3))
    out[n_ellipsoids:, 0] = 2
    out[n_ellipsoids:, 4] = rng.uniform(a, b, n_columns)
    out[n_ellipsoids:, 5] = 2.0 * (lx + ly + lz)                    # half-length: beyond the box
    out[n_ellipsoids:, 7] = rng.choice([-1.0, 1.0], n_columns)
    out[n_ellipsoids:, 9] = 1.0
    return out
