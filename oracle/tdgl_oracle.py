"""Plain fp64 CPU oracle of the per-time-step hot path of arXiv:1409.8340 (Sadovskyy et al.).

ORACLE / TEST INFRASTRUCTURE -- see oracle/__init__.py.  Shares no code with the CUDA path.

`P:NNN` cites /root/reference/PAPER.md line NNN.  `Sxx` cites a reading listed in DESIGN.md
("Readings of the paper"), taken from SURVEY.md section 8(c).

What is computed.  The psi update is an *iteration stopped by a tolerance*, so it follows the paper's
algorithm step by step, in the paper's order and notation (Eqs. 26-35).  The scalar potential is *the
solution of a linear elliptic problem* (Eq. 18 discretised), so it is that definition:
Delta_h mu = rho with sum_m w_m mu_m = 0 (S5-S7), obtained with library transforms (FFT on periodic axes,
DCT-I on open axes, which diagonalise the 7-point operator exactly).

Array convention: every field is a numpy array of shape (nz, ny, nx), i.e. f[k, j, i], which is the
paper's multi-index m = i + nx*(j + ny*k) in C order.  Axis numbers: x -> 2, y -> 1, z -> 0.

All link phases are kept as general per-link arrays th_x, th_y, th_z (phase of the link that leaves site
m in direction +alpha), filled by `paper_links` from the paper's Landau gauge (Eq. 24a, 27) and its
quasi-periodic jump P_{i,k}.  Every operator below only uses those arrays, which is what allows
the gauge-invariance pin (psi -> psi e^{i chi}, th_alpha(m) -> th_alpha(m) + chi(m+alpha) - chi(m)).

Parity pins (tests/test_oracle_*.py, all `-m "not gpu"`):
  reaction+CN closed form, uniform fixed point, plane-wave growth factor, J_av closed form, Ohmic normal
  state, flux quantisation (integer plaquette windings summing to n_z), current conservation, gauge
  invariance, dense LU of M Psi = b on 8^3 built from the printed matrix entries, dense bordered
  solve of the Poisson problem on 8^3, zero normal current at open faces, free-energy descent and its
  finite-difference gradient, Philox known-answer vectors, noise amplitude zeta_max of Eq. (39); the initial
  condition (S13) by its distribution (moments, Kolmogorov-Smirnov distance, independence); the paper's pseudo-time
  mu iteration (Eq. 40) by its fixed point (= the direct solve) and a dense solve of N mu = c from the printed entries.
Single-precision replay: every function below keeps the dtype of the state it is given; a complex64 / float32
state runs the same formulas in fp32 (link variables rounded to fp32 after fp64 trigonometry, scalars K, J_av in
fp64, as the CUDA library does).  Used only to show what fp32 does to the paper's rule without the CUDA path (R3).
Parity unpinned: none of the functions below; the paper's Fig. 5/6 curves are image-only and pin nothing.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import List, Optional, Sequence, Tuple

import numpy as np
import scipy.fft

from . import philox

PERIODIC = 0
OPEN = 1
_AXIS = {"x": 2, "y": 1, "z": 0}


# --------------------------------------------------------------------------------------------------
# parameters and state
# --------------------------------------------------------------------------------------------------
@dataclass
class Params:
    nx: int
    ny: int
    nz: int
    hx: float = 0.5
    hy: float = 0.5
    hz: float = 0.5
    dt: float = 0.1                 # real time step; h_t = dt / u (P:257 footnote 3, S1)
    u: float = 1.0                  # S1
    g: float = 1.0                  # anisotropy
    bc: Tuple[int, int, int] = (PERIODIC, PERIODIC, PERIODIC)   # (x, y, z)
    eps_tol: float = 1e-6           # Eq. (34) threshold on max |r|^2
    max_sweeps: int = 100           # S10
    temperature: float = 0.0        # reduced T-bar of Eq. (39); 0 = no noise
    seed: int = 0                   # Philox key
    solve_mu: bool = True           # S15
    # mu solver: "direct" = the definition Delta_h mu = rho (solve_poisson); "pseudotime" = the paper's own iteration
    # (Eq. 40, solve_poisson_pseudotime) warm-started from the previous step's mu, with the controls below (S20)
    mu_solver: str = "direct"
    h_tau: float = 0.1
    eps_mu: float = 1e-6
    eps_mu_in: float = 1e-6
    mu_max_outer: int = 1000
    mu_max_inner: int = 100
    # S25: insulating inclusions (P:511 (ii): "no-current (open) boundary conditions across internal grid edges").
    # Boolean array of the grid shape, True = superconductor, False = a site inside an insulating inclusion (removed:
    # psi = 0, mu = 0).  Every link ("grid edge") between a superconducting and a removed site is CUT: it carries no
    # current and drops out of the covariant Laplacian, of rho = div j_s and of Delta_h mu.  None = no such inclusions.
    sc_mask: Optional[np.ndarray] = None

    @property
    def shape(self):
        return (self.nz, self.ny, self.nx)

    @property
    def n_sites(self):
        return self.nx * self.ny * self.nz

    def length(self, a: str) -> float:
        """L_a = N_a h_a (periodic) or (N_a - 1) h_a (open)  (typo G: h_z = L_z/(N_z-1))."""
        n = {"x": self.nx, "y": self.ny, "z": self.nz}[a]
        h = {"x": self.hx, "y": self.hy, "z": self.hz}[a]
        o = self.bc["xyz".index(a)] == OPEN
        return (n - 1) * h if o else n * h

    @property
    def ht(self):
        return self.dt / self.u

    @property
    def cx(self):
        return 1.0 / self.hx ** 2

    @property
    def cy(self):
        return 1.0 / self.hy ** 2

    @property
    def cz(self):
        """1/(g h_z)^2; a film (N_z = 1: the paper's 2D mode) has no z links at all: c_z = 0 (S22)."""
        if self.nz == 1:
            return 0.0
        return 1.0 / (self.g ** 2 * self.hz ** 2)

    @property
    def cell(self):
        """Volume of a mesh cell, h_x h_y h_z; area h_x h_y for a film (d = 2 in Eq. 38-39; S22)."""
        return self.hx * self.hy * (self.hz if self.nz > 1 else 1.0)

    def __post_init__(self):
        if self.nz == 1 and self.bc[2] != PERIODIC:
            raise ValueError("a film (nz = 1) has no z faces: bc[2] must be PERIODIC")


@dataclass
class State:
    psi: np.ndarray                 # complex128 (nz, ny, nx)
    mu: np.ndarray                  # float64
    K: float = 0.0
    n: int = 0                      # step index (Philox counter word 2)
    # bookkeeping written by step()
    Ex: float = 0.0
    Jav: float = 0.0
    sweeps_last: int = 0
    sweeps_total: int = 0
    max_resid2: float = 0.0
    sweep_log: List[int] = field(default_factory=list)
    resid_log: List[float] = field(default_factory=list)   # max|r|^2 at the deciding sweep of each step
    resid_trace: List[List[float]] = field(default_factory=list)   # max|r|^2 of every sweep of each step (S9 check)
    mu_log: List[list] = field(default_factory=list)       # pseudo-time solver: per step, [(inner sweeps, max|d_tau mu|^2), ...]
    hit_max_sweeps: bool = False


# --------------------------------------------------------------------------------------------------
# field, links
# --------------------------------------------------------------------------------------------------
def snap_field(p: Params, Bx: float, Bz: float) -> Tuple[float, float, Optional[int], Optional[int]]:
    """Flux quantisation: B_z = 2 pi n_z/(L_x L_y) iff x and y are periodic,
    B_x = 2 pi n_x/(L_y L_z) iff y and z are periodic; otherwise the component is left as given."""
    nzq = nxq = None
    if p.bc[0] == PERIODIC and p.bc[1] == PERIODIC:
        a = p.length("x") * p.length("y")
        nzq = int(np.rint(Bz * a / (2.0 * math.pi)))
        Bz = 2.0 * math.pi * nzq / a
    if p.bc[1] == PERIODIC and p.bc[2] == PERIODIC:
        a = p.length("y") * p.length("z")
        nxq = int(np.rint(Bx * a / (2.0 * math.pi)))
        Bx = 2.0 * math.pi * nxq / a
    return Bx, Bz, nxq, nzq


def paper_links(p: Params, K: float, Bx: float, Bz: float):
    """Link phases of the xz Landau gauge.  U_{alpha,j} = exp(-i h_alpha A~_alpha), A~ = A - K e_x,
    A^{xz} = ybar [-B_z, 0, B_x], ybar = j h_y - L_y/2  (Eq. 24a, Eq. 27-28):
        th_x(j) = h_x (K + B_z ybar_j),   th_y = 0,   th_z(j) = -h_z B_x ybar_j
    (signs agree with the paper's own U_{x,j=-1}, U_{z,j=-1} at P:441, 447).
    Quasi-periodic jump in y: psi_{i,-1,k} = P_{i,k} psi_{i,Ny-1,k},
        P_{i,k} = exp(i (i h_x L_y B_z - k h_z L_y B_x)),
    i.e. the wrap link that leaves row Ny-1 in +y carries exp(i th_y) = P*_{i,k}.
    """
    return paper_links_at(p, K, Bx, Bz, np.arange(p.nx), np.arange(p.ny), np.arange(p.nz))


def paper_links_at(p: Params, K: float, Bx: float, Bz: float, ii, jj, kk):
    """The link phases of `paper_links` on the sub-lattice of global indices ii x jj x kk (1-D integer
    arrays, x, y, z): arrays of shape (len(kk), len(jj), len(ii)).  `paper_links` is this function on the
    full index ranges; the windowed form lets a test evaluate the same formulas on samples of a grid that
    is too large for a whole oracle step."""
    ii, jj, kk = (np.asarray(a, dtype=np.int64) for a in (ii, jj, kk))
    shape = (len(kk), len(jj), len(ii))
    ybar = (jj * p.hy - p.length("y") / 2.0)[None, :, None]
    thx = np.broadcast_to(p.hx * (K + Bz * ybar), shape).copy()
    thz = np.broadcast_to(-p.hz * Bx * ybar, shape).copy()
    thy = np.zeros(shape)
    if p.bc[1] == PERIODIC:
        i = ii[None, :]
        k = kk[:, None]
        wrap = -(i * p.hx * p.length("y") * Bz - k * p.hz * p.length("y") * Bx)
        for w in np.nonzero(jj == p.ny - 1)[0]:
            thy[:, w, :] = wrap
    return thx, thy, thz


def snap_field_yz(p: Params, By: float, Bz: float) -> Tuple[float, float, Optional[int], Optional[int]]:
    """Flux quantisation for a field in the yz plane (P:467 applied to the jump P_{j,k} of P:459):
    B_z = 2 pi n_z/(L_x L_y) iff x and y are periodic, B_y = 2 pi n_y/(L_x L_z) iff x and z are periodic."""
    nzq = nyq = None
    if p.bc[0] == PERIODIC and p.bc[1] == PERIODIC:
        a = p.length("x") * p.length("y")
        nzq = int(np.rint(Bz * a / (2.0 * math.pi)))
        Bz = 2.0 * math.pi * nzq / a
    if p.bc[0] == PERIODIC and p.bc[2] == PERIODIC:
        a = p.length("x") * p.length("z")
        nyq = int(np.rint(By * a / (2.0 * math.pi)))
        By = 2.0 * math.pi * nyq / a
    return By, Bz, nyq, nzq


def paper_links_yz(p: Params, K: float, By: float, Bz: float):
    """Link phases of the yz Landau gauge, A^{yz} = xbar [0, B_z, -B_y], xbar = i h_x - L_x/2 (Eq. 24b with
    the typo "B_u" -> B_y; Eq. 25b; discretised as Eq. 29b):
        th_x = h_x K,   th_y(i) = -h_y B_z xbar_i,   th_z(i) = +h_z B_y xbar_i        (U = exp(-i h A~))
    Quasi-periodic jump in x: psi_{-1,j,k} = P_{j,k} psi_{Nx-1,j,k},
        P_{j,k} = exp(i (-j h_y L_x B_z + k h_z L_x B_y)),
    i.e. the wrap link that leaves column Nx-1 in +x carries exp(i th_x) P*_{j,k}."""
    return paper_links_yz_at(p, K, By, Bz, np.arange(p.nx), np.arange(p.ny), np.arange(p.nz))


def paper_links_yz_at(p: Params, K: float, By: float, Bz: float, ii, jj, kk):
    """`paper_links_yz` on the sub-lattice of global indices ii x jj x kk (see `paper_links_at`)."""
    ii, jj, kk = (np.asarray(a, dtype=np.int64) for a in (ii, jj, kk))
    shape = (len(kk), len(jj), len(ii))
    xbar = (ii * p.hx - p.length("x") / 2.0)[None, None, :]
    thx = np.full(shape, p.hx * K)
    thy = np.broadcast_to(-p.hy * Bz * xbar, shape).copy()
    thz = np.broadcast_to(p.hz * By * xbar, shape).copy()
    if p.bc[0] == PERIODIC:
        j = jj[None, :]
        k = kk[:, None]
        wrap = -(-j * p.hy * p.length("x") * Bz + k * p.hz * p.length("x") * By)
        for w in np.nonzero(ii == p.nx - 1)[0]:
            thx[:, :, w] += wrap
    return thx, thy, thz


# --------------------------------------------------------------------------------------------------
# neighbour operators
# --------------------------------------------------------------------------------------------------
def _S(f, th, axis, bc):
    """(S+ f)_m = e^{i th(m)} f(m+alpha),  (S- f)_m = e^{-i th(m-alpha)} f(m-alpha).
    Periodic: indices wrap.  Open: the ghost value follows from n.(grad - iA~)psi = 0, i.e.
    U* f_{-1} = U f_{1} and U f_{N} = U* f_{N-2}: at the first site S- := S+, at the last S+ := S-."""
    e = np.exp(1j * th)
    if f.dtype == np.complex64:          # single-precision replay (reading R3): fp64 phases, fp32 link variables
        e = e.astype(np.complex64)
    sp = e * np.roll(f, -1, axis)
    sm = np.roll(np.conj(e) * f, 1, axis)
    if bc == OPEN:
        first = [slice(None)] * 3
        last = [slice(None)] * 3
        first[axis] = 0
        last[axis] = -1
        first, last = tuple(first), tuple(last)
        sm[first] = sp[first]
        sp[last] = sm[last]
    return sp, sm


def _link_exists(p: Params, axis, bc):
    """S25: (e+, e-), 1 where the forward / backward link of site m along `axis` exists: both ends are superconducting
    sites.  On an EXTERNAL open face the paper's rule stands (S- := S+ at the first site, S+ := S- at the last,
    P:471): the mirrored term exists iff the link it mirrors does."""
    m = p.sc_mask
    fw = np.roll(m, -1, axis)
    bw = np.roll(m, 1, axis)
    if bc == OPEN:
        first = [slice(None)] * 3
        last = [slice(None)] * 3
        first[axis] = 0
        last[axis] = -1
        first, last = tuple(first), tuple(last)
        bw = bw.copy()
        fw = fw.copy()
        bw[first] = np.roll(m, -1, axis)[first]
        fw[last] = np.roll(m, 1, axis)[last]
    return (m & fw).astype(np.float64), (m & bw).astype(np.float64)


def neighbour_sum(p: Params, f, links):
    """sum_alpha c_alpha (S+_alpha f + S-_alpha f)_m, c_x = 1/h_x^2, c_y = 1/h_y^2, c_z = 1/(g h_z)^2; with insulating
    inclusions (S25) only over the links that exist."""
    thx, thy, thz = links
    xp, xm = _S(f, thx, 2, p.bc[0])
    yp, ym = _S(f, thy, 1, p.bc[1])
    zp, zm = _S(f, thz, 0, p.bc[2])
    if p.sc_mask is None:
        return p.cx * (xp + xm) + p.cy * (yp + ym) + p.cz * (zp + zm)
    ex, ey, ez = (_link_exists(p, 2, p.bc[0]), _link_exists(p, 1, p.bc[1]), _link_exists(p, 0, p.bc[2]))
    return (p.cx * (ex[0] * xp + ex[1] * xm) + p.cy * (ey[0] * yp + ey[1] * ym) + p.cz * (ez[0] * zp + ez[1] * zm))


def link_diagonal(p: Params):
    """sum over the links of site m of c_alpha: 2 (c_x + c_y + c_z) (the "2 sum c" of M_mm), or, with insulating
    inclusions (S25), the sum over the links that exist (an array)."""
    if p.sc_mask is None:
        return 2.0 * (p.cx + p.cy + p.cz)
    ex, ey, ez = (_link_exists(p, 2, p.bc[0]), _link_exists(p, 1, p.bc[1]), _link_exists(p, 0, p.bc[2]))
    return p.cx * (ex[0] + ex[1]) + p.cy * (ey[0] + ey[1]) + p.cz * (ez[0] + ez[1])


def covariant_laplacian(p: Params, f, links):
    """Eq. (29a): (L f)_m = sum_alpha c_alpha (S+ f + S- f - 2 f)_m.  On open faces this is
    the printed 2 (U f_1 - f_0)/h^2 form; a cut link (S25) contributes nothing."""
    return neighbour_sum(p, f, links) - link_diagonal(p) * f


def _zero_links(p: Params):
    z = np.zeros(p.shape)
    return z, z, z


def laplacian_real(p: Params, m):
    """Left side of the discretised Poisson equation: the same 7-point operator with U = 1, P = 1;
    periodic wrap (mu is continuous) or mirror ghost on open faces (S6)."""
    return covariant_laplacian(p, m.astype(np.complex128), _zero_links(p)).real


def site_weights(p: Params):
    """w_m = prod_alpha w_alpha, w_alpha = 1/2 on an open face of axis alpha, else 1 (S7)."""
    w = np.ones(p.shape)
    for a, axis in ((0, 2), (1, 1), (2, 0)):
        if p.bc[a] == OPEN:
            sl = [slice(None)] * 3
            sl[axis] = 0
            w[tuple(sl)] *= 0.5
            sl[axis] = -1
            w[tuple(sl)] *= 0.5
    if p.sc_mask is not None:                       # removed sites carry no weight (S25)
        w = w * p.sc_mask
    return w


# --------------------------------------------------------------------------------------------------
# noise and initial condition
# --------------------------------------------------------------------------------------------------
def zeta_max(p: Params) -> float:
    """Eq. (39): zeta_max = (3 T u / (2 h_t h_x h_y h_z))^{1/2}; per S1/S12 the time step in it is
    the real step dt and T is the reduced T-bar.  In d = 2 (film, N_z = 1) the delta function of Eq. (38)
    discretises as delta_ij/(h_x h_y) ("d = 2, 3"), so h_z drops out (S22)."""
    return math.sqrt(3.0 * p.temperature * p.u / (2.0 * p.dt * p.cell))


def langevin_noise(p: Params, step: int):
    """zeta_m = zeta_max (r1 + i r2), r uniform in (-1, 1), independent per site and step;
    Philox stream 0, one call per site PAIR (reading S11'; see langevin_noise_at)."""
    return langevin_noise_at(p, step, np.arange(p.n_sites, dtype=np.uint64)).reshape(p.shape)


def langevin_noise_at(p: Params, step: int, m):
    """The Langevin term of `langevin_noise` at the global site indices m = i + nx (j + ny k) (any shape).
    Reading S11': the four words of ONE Philox4x32-10 call serve the two sites of a pair -- key = seed,
    counter = (m_e lo, m_e hi, step, stream 0) with m_e = m - (m mod 2) the even site of the pair; site m_e takes
    the words (x0, x1) as (re, im), site m_e + 1 the words (x2, x3).  nx is even, so a pair never straddles a row.
    The four output words of a Philox call are as independent as the words of different calls (Salmon et al., SC'11)."""
    m = np.asarray(m, dtype=np.uint64)
    me = m & ~np.uint64(1)
    x0, x1, x2, x3 = philox.philox4x32_10(me & np.uint64(0xFFFFFFFF), me >> np.uint64(32), step, 0,
                                          p.seed & 0xFFFFFFFF, (p.seed >> 32) & 0xFFFFFFFF)
    odd = (m & np.uint64(1)) == np.uint64(1)
    re, im = np.where(odd, x2, x0), np.where(odd, x3, x1)
    return zeta_max(p) * (philox.uniform_pm1(re) + 1j * philox.uniform_pm1(im))


def box_muller(x0, x1):
    """Two independent N(0,1) deviates per pair of Philox words (S13): u1, u2 uniform in (0, 1) from x0, x1,
    g1 + i g2 = sqrt(-2 ln u1) exp(2 pi i u2)  (Box and Muller, 1958)."""
    u1, u2 = philox.uniform_01(x0), philox.uniform_01(x1)
    rad = np.sqrt(-2.0 * np.log(u1))
    return rad * np.cos(2.0 * math.pi * u2) + 1j * rad * np.sin(2.0 * math.pi * u2)


def initial_state(p: Params, init_amp: float) -> State:
    """psi0 = 1 + init_amp (N(0,1) + i N(0,1)), Box-Muller on Philox stream 1; mu = 0, K = 0 (S13)."""
    x0, x1 = philox.site_words(p.n_sites, 0, 1, p.seed)
    psi = 1.0 + init_amp * box_muller(x0, x1)
    return State(psi=psi.reshape(p.shape), mu=np.zeros(p.shape))


# --------------------------------------------------------------------------------------------------
# inclusion pattern (a0)
# --------------------------------------------------------------------------------------------------
def epsilon_from_spheres(p: Params, spheres, eps_in: float, eps_out: float):
    """eps_m = eps_in if site m lies within radius r_s of any sphere centre, else eps_out (P:245, 511 (i),
    S19).  Distance uses the minimum image on periodic axes.  Site coordinates are (i h_x, j h_y, k h_z)
    (P:243).  The test is d_x^2 + d_y^2 + d_z^2 <= r^2 in fp64, each product and sum rounded
    separately in that order (the CUDA path evaluates the same expression without contraction, so the
    mask is bit-identical)."""
    eps = np.full(p.shape, float(eps_out))
    n = (p.nx, p.ny, p.nz)
    h = (float(np.float32(p.hx)), float(np.float32(p.hy)), float(np.float32(p.hz)))
    L = tuple(n[a] * h[a] for a in range(3))        # periodic image distance
    for s in np.asarray(spheres, dtype=np.float32).reshape(-1, 4):
        c = [float(s[0]), float(s[1]), float(s[2])]
        r = float(s[3])
        idx, d2 = [], []
        for a in range(3):
            lo = int(math.floor((c[a] - r) / h[a])) - 1
            hi = int(math.ceil((c[a] + r) / h[a])) + 1
            if p.bc[a] == OPEN:
                lo, hi = max(lo, 0), min(hi, n[a] - 1)
            elif hi - lo + 1 >= n[a]:
                lo, hi = 0, n[a] - 1
            q = np.arange(lo, hi + 1)
            ii = np.mod(q, n[a])
            d = ii.astype(np.float64) * h[a] - c[a]
            if p.bc[a] == PERIODIC:
                d = d - L[a] * np.rint(d / L[a])
            idx.append(ii)
            d2.append(d * d)
        dist2 = (d2[0][None, None, :] + d2[1][None, :, None]) + d2[2][:, None, None]
        inside = dist2 <= r * r
        sub = eps[np.ix_(idx[2], idx[1], idx[0])]
        sub[inside] = float(eps_in)
        eps[np.ix_(idx[2], idx[1], idx[0])] = sub
    return eps


def epsilon_brute_force(p: Params, spheres, eps_in: float, eps_out: float):
    """The same definition as an N x n_s loop over every site and every sphere (tiny inputs only)."""
    h = (float(np.float32(p.hx)), float(np.float32(p.hy)), float(np.float32(p.hz)))
    n = (p.nx, p.ny, p.nz)
    kk, jj, ii = np.meshgrid(np.arange(p.nz), np.arange(p.ny), np.arange(p.nx), indexing="ij")
    pos = (ii * h[0], jj * h[1], kk * h[2])
    eps = np.full(p.shape, float(eps_out))
    for s in np.asarray(spheres, dtype=np.float32).reshape(-1, 4):
        d2 = []
        for a in range(3):
            d = pos[a] - float(s[a])
            if p.bc[a] == PERIODIC:
                La = n[a] * h[a]
                d = d - La * np.rint(d / La)
            d2.append(d * d)
        eps[(d2[0] + d2[1]) + d2[2] <= float(s[3]) * float(s[3])] = float(eps_in)
    return eps


# Further generator shapes ("ellipsoids ... cylinders", Fig. 2(d) elliptical inclusions, Fig. 2(e) +-45 degree
# columnar defects; reading S26).  A shape is a row of 10 float32 numbers
#     (kind, c_x, c_y, c_z, a_0, a_1, a_2, n_x, n_y, n_z)
# kind 0 SPHERE    radius a_0                              : d_x^2 + d_y^2 + d_z^2 <= a_0^2
# kind 1 ELLIPSOID semi-axes (a_0, a_1, a_2) along x, y, z : (d_x/a_0)^2 + (d_y/a_1)^2 + (d_z/a_2)^2 <= 1
# kind 2 CYLINDER  radius a_0, half-length a_1, axis n (any non-zero vector, normalised in fp64):
#                  t = d.n_hat, |t| <= a_1 and |d|^2 - t^2 <= a_0^2
# d = site position minus centre, minimum image on periodic axes, exactly as for spheres; every product, quotient and
# sum is a separately rounded fp64 operation in the order written (no contraction), so that a mask is reproducible.
SHAPE_SPHERE, SHAPE_ELLIPSOID, SHAPE_CYLINDER = 0, 1, 2


def _shape_inside(kind: int, a, nhat, dx, dy, dz):
    """The inside test of one shape on broadcastable fp64 displacement arrays."""
    if kind == SHAPE_SPHERE:
        return (dx * dx + dy * dy) + dz * dz <= a[0] * a[0]
    if kind == SHAPE_ELLIPSOID:
        ex, ey, ez = dx / a[0], dy / a[1], dz / a[2]
        return (ex * ex + ey * ey) + ez * ez <= 1.0
    if kind == SHAPE_CYLINDER:
        t = (dx * nhat[0] + dy * nhat[1]) + dz * nhat[2]
        q = ((dx * dx + dy * dy) + dz * dz) - t * t
        return (np.abs(t) <= a[1]) & (q <= a[0] * a[0])
    raise ValueError(f"unknown shape kind {kind}")


def _shape_unpack(row):
    row = np.asarray(row, dtype=np.float32)
    kind = int(row[0])
    c = [float(row[1]), float(row[2]), float(row[3])]
    a = [float(row[4]), float(row[5]), float(row[6])]
    n = [float(row[7]), float(row[8]), float(row[9])]
    nhat = [0.0, 0.0, 0.0]
    if kind == SHAPE_CYLINDER:
        nn = math.sqrt((n[0] * n[0] + n[1] * n[1]) + n[2] * n[2])
        nhat = [n[0] / nn, n[1] / nn, n[2] / nn]
    return kind, c, a, nhat


def shape_half_extent(kind: int, a, nhat):
    """Half-width of the axis-aligned bounding box of a shape along x, y, z."""
    if kind == SHAPE_SPHERE:
        return [a[0], a[0], a[0]]
    if kind == SHAPE_ELLIPSOID:
        return [a[0], a[1], a[2]]
    # capped cylinder: |n_a| * half-length + r sqrt(1 - n_a^2)
    return [abs(nhat[q]) * a[1] + a[0] * math.sqrt(max(0.0, 1.0 - nhat[q] * nhat[q])) for q in range(3)]


def epsilon_from_shapes(p: Params, shapes, eps_in: float, eps_out: float):
    """eps_m = eps_in if site m lies inside any shape of the list, else eps_out (P:511 (i), 513; S26).  Each shape is
    tested on the sites of its bounding box only."""
    eps = np.full(p.shape, float(eps_out))
    n = (p.nx, p.ny, p.nz)
    h = (float(np.float32(p.hx)), float(np.float32(p.hy)), float(np.float32(p.hz)))
    L = tuple(n[q] * h[q] for q in range(3))
    for row in np.asarray(shapes, dtype=np.float32).reshape(-1, 10):
        kind, c, a, nhat = _shape_unpack(row)
        ext = shape_half_extent(kind, a, nhat)
        idx, dd = [], []
        for q in range(3):
            lo = int(math.floor((c[q] - ext[q]) / h[q])) - 1
            hi = int(math.ceil((c[q] + ext[q]) / h[q])) + 1
            if p.bc[q] == OPEN:
                lo, hi = max(lo, 0), min(hi, n[q] - 1)
            elif hi - lo + 1 >= n[q]:
                lo, hi = 0, n[q] - 1
            r = np.arange(lo, hi + 1)
            ii = np.mod(r, n[q])
            d = ii.astype(np.float64) * h[q] - c[q]
            if p.bc[q] == PERIODIC:
                d = d - L[q] * np.rint(d / L[q])
            idx.append(ii)
            dd.append(d)
        if min(len(i) for i in idx) == 0:
            continue
        inside = _shape_inside(kind, a, nhat, dd[0][None, None, :], dd[1][None, :, None], dd[2][:, None, None])
        sub = eps[np.ix_(idx[2], idx[1], idx[0])]
        sub[inside] = float(eps_in)
        eps[np.ix_(idx[2], idx[1], idx[0])] = sub
    return eps


def epsilon_shapes_brute_force(p: Params, shapes, eps_in: float, eps_out: float):
    """The same definition as a loop over every site and every shape (tiny inputs only)."""
    h = (float(np.float32(p.hx)), float(np.float32(p.hy)), float(np.float32(p.hz)))
    n = (p.nx, p.ny, p.nz)
    kk, jj, ii = np.meshgrid(np.arange(p.nz), np.arange(p.ny), np.arange(p.nx), indexing="ij")
    pos = (ii * h[0], jj * h[1], kk * h[2])
    eps = np.full(p.shape, float(eps_out))
    for row in np.asarray(shapes, dtype=np.float32).reshape(-1, 10):
        kind, c, a, nhat = _shape_unpack(row)
        d = []
        for q in range(3):
            dq = pos[q] - c[q]
            if p.bc[q] == PERIODIC:
                Lq = n[q] * h[q]
                dq = dq - Lq * np.rint(dq / Lq)
            d.append(dq)
        eps[_shape_inside(kind, a, nhat, d[0], d[1], d[2])] = float(eps_in)
    return eps


# --------------------------------------------------------------------------------------------------
# the psi solve
# --------------------------------------------------------------------------------------------------
def build_system(p: Params, psi, mu, eps, links, zeta=None):
    """Right-hand side b (Eq. 31) and diagonal d = M_mm of the linearised Crank-Nicolson
    system, with psi^est = psi^- (P:255):
        c_m = |psi_m|^2
        b_m = psi_m + (h_t/2) [ (eps_m - i u mu_m) psi_m - c_m psi_m + (L psi)_m + 2 zeta_m ]
        d_m = 1 + (h_t/2) [ c_m + 2 (c_x + c_y + c_z) - eps_m + i u mu_m ]
    """
    ht2 = p.ht / 2.0
    c = np.abs(psi) ** 2
    if zeta is None:
        zeta = 0.0
    elif p.sc_mask is not None:
        zeta = zeta * p.sc_mask                     # no order parameter, hence no Langevin term, on a removed site (S25)
    b = psi + ht2 * ((eps - 1j * p.u * mu) * psi - c * psi + covariant_laplacian(p, psi, links) + 2.0 * zeta)
    d = 1.0 + ht2 * (c + link_diagonal(p) - eps + 1j * p.u * mu)
    return b, d


def jacobi_sweep(p: Params, x, b, d, links):
    """Eq. (33).  The off-diagonal entries are M_{m,m+-alpha} = -(h_t/2) c_alpha U (on open
    faces the single neighbour's entry doubles, S21), so
        x^{l+1}_m = ( b_m + (h_t/2) sum_alpha c_alpha (S+ x^l + S- x^l)_m ) / d_m.
    Also returns the residual of the INPUT iterate, r^l = b - M x^l = d (x^{l+1} - x^l) (S8)."""
    xn = (b + (p.ht / 2.0) * neighbour_sum(p, x, links)) / d
    r = d * (xn - x)
    return xn, r


def solve_psi(p: Params, psi, b, d, links, fixed_sweeps: Optional[int] = None, trace: Optional[list] = None):
    """Jacobi iteration from x^0 = psi^- until max_m |r^l_m|^2 < eps_tol (Eq. 34) or the cap (S10);
    keeps x^{l+1}; sweeps = l + 1 (S8).  `fixed_sweeps`: run exactly that many sweeps, no test (S9 replay)."""
    x = psi
    sweeps = 0
    r2 = 0.0
    while True:
        x, r = jacobi_sweep(p, x, b, d, links)
        sweeps += 1
        r2 = float(np.max(r.real ** 2 + r.imag ** 2))
        if trace is not None:
            trace.append(r2)          # logging only
        if fixed_sweeps is not None:
            if sweeps >= fixed_sweeps:
                break
        elif r2 < p.eps_tol or sweeps >= p.max_sweeps:
            break
    return x, sweeps, r2


# --------------------------------------------------------------------------------------------------
# current, K, rho, mu
# --------------------------------------------------------------------------------------------------
def average_supercurrent(p: Params, psi, links):
    """Eq. (35): J_av = 1/(2 N h_x) sum_m Im[ psi*_m (U_x psi_{i+1} - U_x* psi_{i-1}) ]  (plain 1/N
    mean, S18)."""
    xp, xm = _S(psi, links[0], 2, p.bc[0])
    if p.sc_mask is not None:                       # only links that exist carry a current (S25); still the plain 1/N mean
        ex = _link_exists(p, 2, p.bc[0])
        xp, xm = ex[0] * xp, ex[1] * xm
    return float(np.sum(np.imag(np.conj(psi) * (xp - xm))) / (2.0 * p.n_sites * p.hx))


def rewind(p: Params, K: float) -> float:
    """K -> K - (2 pi/h_x) floor(K h_x / 2 pi)."""
    return K - (2.0 * math.pi / p.hx) * math.floor(K * p.hx / (2.0 * math.pi))


def supercurrent_divergence(p: Params, psi, links):
    """Right side of the discretised Poisson equation:
    rho_m = sum_alpha c_alpha Im[ psi*_m (S+ psi + S- psi)_m ]  ( = Im[psi*_m (L psi)_m] )."""
    return np.imag(np.conj(psi) * neighbour_sum(p, psi, links))


def laplacian_eigenvalues(p: Params):
    """Eigenvalues of the real 7-point operator in the transform basis: per axis
    -c (2 - 2 cos(2 pi q/N)) (periodic, Fourier) or -c (2 - 2 cos(pi q/(N-1))) (open, cosine / DCT-I)."""
    lam = np.zeros(p.shape)
    for a, axis, n, c in ((0, 2, p.nx, p.cx), (1, 1, p.ny, p.cy), (2, 0, p.nz, p.cz)):
        q = np.arange(n)
        if p.bc[a] == PERIODIC:
            la = -c * (2.0 - 2.0 * np.cos(2.0 * math.pi * q / n))
        else:
            la = -c * (2.0 - 2.0 * np.cos(math.pi * q / (n - 1)))
        sh = [1, 1, 1]
        sh[axis] = n
        lam = lam + la.reshape(sh)
    return lam


def solve_poisson(p: Params, rho):
    """mu = the solution of (Delta_h mu)_m = rho_m with sum_m w_m mu_m = 0 (Eq. 18 as discretised at
    P:379-383; S5: the fixed point of the paper's pseudo-time iteration IS this equation; S6: Neumann
    mirror ghost on open faces; S7: weighted zero mode removed).
    FFT along periodic axes and DCT-I along open axes diagonalise Delta_h; the zero mode (whose DCT-I/FFT
    coefficient is 2^{#open} sum_m w_m f_m) is set to zero."""
    if p.sc_mask is not None:
        raise ValueError("the transform solver does not apply with insulating inclusions (S25): use mu_solver='pseudotime'")
    f = rho.astype(np.complex128)
    for a, axis in ((0, 2), (1, 1), (2, 0)):
        if p.bc[a] == PERIODIC:
            f = np.fft.fft(f, axis=axis)
        else:
            f = scipy.fft.dct(f.real, type=1, axis=axis) + 1j * scipy.fft.dct(f.imag, type=1, axis=axis)
    lam = laplacian_eigenvalues(p)
    lam[0, 0, 0] = 1.0
    f = f / lam
    f[0, 0, 0] = 0.0
    for a, axis in ((0, 2), (1, 1), (2, 0)):
        if p.bc[a] == PERIODIC:
            f = np.fft.ifft(f, axis=axis)
        else:
            f = scipy.fft.idct(f.real, type=1, axis=axis) + 1j * scipy.fft.idct(f.imag, type=1, axis=axis)
    return f.real


def solve_poisson_pseudotime(p: Params, rho, mu0, h_tau: float = 0.1, eps_mu: float = 1e-6, eps_in: float = 1e-6,
                             max_outer: int = 10000, max_inner: int = 1000, inner_counts: Optional[Sequence[int]] = None):
    """The paper's OWN mu solver, step by step (Eq. 40; readings S5, S20): pseudo-time relaxation
    d_tau mu = Delta_h mu - rho  (the STABLE sign: as printed at P:387 the flow is anti-diffusive and the printed
    N mu = c, whose matrix N at P:399-405 is the diagonally dominant one of the stable flow, has no fixed point unless
    rho = 0 -- S5), one Crank-Nicolson step of size h_tau per outer iteration,
        N mu = c,   N_mm = 1 + h_tau (c_x + c_y + c_z),  N_{m,m+-alpha} = -h_tau c_alpha / 2   (
                    on an open face the single neighbour's entry doubles: mirror ghost, S6/S21)
        c_m = mu^-_m + h_tau [ (Delta_h mu^-)_m / 2 - rho_m ]                                   (P:409-419 with S5)
    solved by Jacobi sweeps "like Eq. (33)" from x^0 = mu^-:  x^{l+1}_m = (c_m + (h_tau/2) sum_alpha c_alpha (x^l_{+alpha}
    + x^l_{-alpha})) / N_mm, stopped at the first l with max_m |N_mm (x^{l+1} - x^l)_m|^2 < eps_in (residual of the input
    iterate, keep x^{l+1}: the rule S8 of the psi solve; eps_in is not given by the paper, S20), and outer iterations
    until max_m |(mu - mu^-)_m / h_tau|^2 < eps_mu.  h_tau is not given either; the default 0.1 is the value of
    the real time step h_t, for which N is as diagonally dominant as M (a handful of sweeps per solve).  The fixed point is Delta_h mu = rho; the weighted mean
    sum_m w_m mu_m of the start value is conserved (S7: start from a mean-free mu).
    `inner_counts` (optional): replay exactly len(inner_counts) outer iterations with these sweep counts (S9).
    Returns (mu, log) with log = list of (inner sweeps, max|d_tau mu|^2) per outer iteration."""
    mu = np.array(mu0, dtype=np.float64)
    rho = np.asarray(rho, dtype=np.float64)
    zl = _zero_links(p)
    d = 1.0 + 0.5 * h_tau * link_diagonal(p)        # N_mm = 1 + h_tau sum c; with S25 over the existing links
    log = []
    n_out = 0
    while True:
        c = mu + h_tau * (0.5 * laplacian_real(p, mu) - rho)
        x = mu
        sweeps = 0
        target = None if inner_counts is None else int(inner_counts[n_out])
        while True:
            xn = (c + 0.5 * h_tau * neighbour_sum(p, x.astype(np.complex128), zl).real) / d
            r2 = float(np.max((d * (xn - x)) ** 2))
            x = xn
            sweeps += 1
            if target is not None:
                if sweeps >= target:
                    break
            elif r2 < eps_in or sweeps >= max_inner:
                break
        dt2 = float(np.max(((x - mu) / h_tau) ** 2))
        mu = x
        log.append((sweeps, dt2))
        n_out += 1
        if inner_counts is not None:
            if n_out >= len(inner_counts):
                break
        elif dt2 < eps_mu or n_out >= max_outer:
            break
    return mu, log


# --------------------------------------------------------------------------------------------------
# one time step
# --------------------------------------------------------------------------------------------------
def step(p: Params, st: State, eps, Bx: float, Bz: float, Jext: float,
         fixed_sweeps: Optional[int] = None, links_fn=None, mu_inner_counts: Optional[Sequence[int]] = None) -> State:
    """One time step in the paper's order "psi, then E, then mu".  mu and K inside the psi
    solve are the values left by the previous step (S2).
    `links_fn(K)` (optional) replaces `paper_links(p, K, Bx, Bz)`: any gauge-equivalent set of link
    phases must give the same physics (used by the gauge-invariance pin only)."""
    if links_fn is None:
        def links_fn(K):
            return paper_links(p, K, Bx, Bz)
    links = links_fn(st.K)
    zeta = langevin_noise(p, st.n) if p.temperature > 0.0 else None          # step 1
    b, d = build_system(p, st.psi, st.mu, eps, links, zeta)                   # steps 2, 3
    trace: List[float] = []
    psi, sweeps, r2 = solve_psi(p, st.psi, b, d, links, fixed_sweeps, trace)  # step 4
    K, Ex, Jav = st.K, 0.0, 0.0
    if p.solve_mu and p.bc[0] == PERIODIC:                                    # step 5 (S3)
        Jav = average_supercurrent(p, psi, links)      # new psi, old K
        Ex = Jext - Jav                                # Eq. (21) with d_t A = 0, Eq. (15)
        K = rewind(p, st.K + p.dt * Ex)                # forward Euler, then rewinding
    mu = st.mu
    if p.solve_mu:                                                            # step 6 (S4: updated K)
        links = links_fn(K)
        rho = supercurrent_divergence(p, psi, links)
        if p.mu_solver == "pseudotime":                # the paper's iteration, warm start = last step's mu
            mu, mlog = solve_poisson_pseudotime(p, rho, st.mu, p.h_tau, p.eps_mu, p.eps_mu_in, p.mu_max_outer,
                                                p.mu_max_inner, mu_inner_counts)
            st.mu_log.append(mlog)
        else:
            mu = solve_poisson(p, rho)
        if psi.dtype == np.complex64:    # single-precision replay (R3): mu is stored in fp32 like psi
            mu = mu.astype(np.float32)
    st.psi, st.mu, st.K, st.n = psi, mu, K, st.n + 1
    st.Ex, st.Jav = Ex, Jav
    st.sweeps_last, st.max_resid2 = sweeps, r2
    st.sweeps_total += sweeps
    st.sweep_log.append(sweeps)
    st.resid_log.append(r2)
    st.resid_trace.append(trace)
    if fixed_sweeps is None and sweeps >= p.max_sweeps and not r2 < p.eps_tol:
        st.hit_max_sweeps = True
    return st


def run(p: Params, st: State, eps, Bx, Bz, Jext, nsteps: int,
        sweep_counts: Optional[Sequence[int]] = None, links_fn=None, mu_schedule: Optional[Sequence[Sequence[int]]] = None) -> State:
    """nsteps steps; `sweep_counts[n]` (optional) replays prescribed per-step sweep counts (S9); `mu_schedule[n]`
    (optional, pseudo-time mu solver) the inner sweep counts of every outer iteration of step n."""
    for s in range(nsteps):
        step(p, st, eps, Bx, Bz, Jext, None if sweep_counts is None else int(sweep_counts[s]), links_fn,
             None if mu_schedule is None else mu_schedule[s])
    return st


# --------------------------------------------------------------------------------------------------
# observables (a8)
# --------------------------------------------------------------------------------------------------
def mean_abs2(psi) -> float:
    return float(np.mean(np.abs(psi) ** 2))


def free_energy(p: Params, psi, eps, links) -> float:
    """Discrete GL free energy (the paper only names F_GL; form chosen so that
    -dF/dpsi*_m / (w_m h_x h_y h_z) is the right side of Eq. (16) as discretised, open faces included):
        F = h_x h_y h_z { sum_m w_m [ -eps_m |psi_m|^2 + |psi_m|^4 / 2 ]
                          + sum_alpha c_alpha sum_links w_link |S+_alpha psi_m - psi_m|^2 },
    links = all sites on a periodic axis, i = 0..N-2 on an open axis; w_link = product of the two
    transverse face weights."""
    w = site_weights(p)
    a2 = np.abs(psi) ** 2
    F = np.sum(w * (-eps * a2 + 0.5 * a2 * a2))
    for a, axis, c, th in ((0, 2, p.cx, links[0]), (1, 1, p.cy, links[1]), (2, 0, p.cz, links[2])):
        sp = np.exp(1j * th) * np.roll(psi, -1, axis)
        g2 = np.abs(sp - psi) ** 2
        wl = np.ones(p.shape)
        for a2_, axis2 in ((0, 2), (1, 1), (2, 0)):
            if a2_ != a and p.bc[a2_] == OPEN:
                sl = [slice(None)] * 3
                sl[axis2] = 0
                wl[tuple(sl)] *= 0.5
                sl[axis2] = -1
                wl[tuple(sl)] *= 0.5
        if p.bc[a] == OPEN:
            sl = [slice(None)] * 3
            sl[axis] = -1
            wl[tuple(sl)] = 0.0
        if p.sc_mask is not None:                   # a cut link stores no gradient energy (S25)
            wl = wl * (p.sc_mask & np.roll(p.sc_mask, -1, axis))
        F += c * np.sum(wl * g2)
    return float(F * p.cell)


def plaquette_windings(p: Params, psi, links, Bz: float):
    """Winding of every z-plaquette: n_p = (g_x(i,j) + g_y(i+1,j) - g_x(i,j+1) - g_y(i,j) + B_z h_x h_y)/2 pi,
    g_alpha(m) = arg(psi*_m S+_alpha psi_m) in (-pi, pi].  On an open axis the last row/column of
    plaquettes does not exist (returned as 0)."""
    gx = np.angle(np.conj(psi) * np.exp(1j * links[0]) * np.roll(psi, -1, 2))
    gy = np.angle(np.conj(psi) * np.exp(1j * links[1]) * np.roll(psi, -1, 1))
    circ = gx + np.roll(gy, -1, 2) - np.roll(gx, -1, 1) - gy
    n = (circ + Bz * p.hx * p.hy) / (2.0 * math.pi)
    if p.bc[0] == OPEN:
        n[:, :, -1] = 0.0
    if p.bc[1] == OPEN:
        n[:, -1, :] = 0.0
    if p.sc_mask is not None:                       # a plaquette with a removed corner has no winding (S25)
        m = p.sc_mask
        n = np.where(m & np.roll(m, -1, 2) & np.roll(m, -1, 1) & np.roll(np.roll(m, -1, 1), -1, 2), n, 0.0)
    return n


def vortices_per_slice(p: Params, psi, links, Bz: float) -> float:
    """Signed winding summed over all z-plaquettes, divided by N_z."""
    n = np.rint(plaquette_windings(p, psi, links, Bz))
    return float(np.sum(n) / p.nz)


def link_supercurrents(p: Params, psi, links):
    """j_s on forward links, Im[psi*_m S+_alpha psi_m]/h_alpha (z component / g^2), zero on the
    non-existent last link of an open axis."""
    out = []
    for a, axis, h, th, gg in ((0, 2, p.hx, links[0], 1.0), (1, 1, p.hy, links[1], 1.0),
                               (2, 0, p.hz, links[2], p.g ** 2)):
        j = np.imag(np.conj(psi) * np.exp(1j * th) * np.roll(psi, -1, axis)) / (h * gg)
        if p.bc[a] == OPEN:
            sl = [slice(None)] * 3
            sl[axis] = -1
            j[tuple(sl)] = 0.0
        if p.sc_mask is not None:                   # no current across a cut link (S25)
            j = j * (p.sc_mask & np.roll(p.sc_mask, -1, axis))
        out.append(j)
    return out
