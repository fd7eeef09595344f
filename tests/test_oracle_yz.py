"""Pins of the oracle's yz Landau gauge (Eq. 24b/29b, jump P_{j,k}: P:205, 278-283, 457-465), CPU only.
What fixes it: the magnetic field a set of link phases describes is the lattice curl of the phases -- every
plaquette, the ones across the quasi-periodic seam included -- and must be the requested B in the convention that
the xz gauge (itself pinned by P6/P13) uses; flux quantisation; exact gauge equivalence with the xz gauge where
the topology allows it (open x, y)."""
import math

import numpy as np
import pytest

from oracle import tdgl_oracle as O

P_, O_ = O.PERIODIC, O.OPEN


def circulation(th_a, th_b, axis_a, axis_b):
    """Sum of link phases around the plaquette spanned by +a then +b at every site (wrapping)."""
    return th_a + np.roll(th_b, -1, axis_a) - np.roll(th_a, -1, axis_b) - th_b


def mod2pi(x):
    return np.angle(np.exp(1j * x))


def test_both_gauges_describe_the_same_field():
    """theta = -h A  =>  circulation around an (a, b) plaquette = -B_c h_a h_b (mod 2 pi), seams included."""
    p = O.Params(12, 10, 8, hx=0.5, hy=0.6, hz=0.4)
    Bx, Bz, _, _ = O.snap_field(p, 0.31, 0.27)
    thx, thy, thz = O.paper_links(p, 0.3, Bx, Bz)                       # xz gauge: B = (Bx, 0, Bz)
    assert np.max(np.abs(mod2pi(circulation(thx, thy, 2, 1) + Bz * p.hx * p.hy))) < 1e-12
    assert np.max(np.abs(mod2pi(circulation(thy, thz, 1, 0) + Bx * p.hy * p.hz))) < 1e-12
    assert np.max(np.abs(mod2pi(circulation(thz, thx, 0, 2)))) < 1e-12
    By, Bz2, nyq, nzq = O.snap_field_yz(p, 0.22, 0.27)
    assert nyq is not None and nzq is not None and abs(Bz2 - Bz) < 1e-15
    thx, thy, thz = O.paper_links_yz(p, 0.3, By, Bz2)                   # yz gauge: B = (0, By, Bz)
    assert np.max(np.abs(mod2pi(circulation(thx, thy, 2, 1) + Bz2 * p.hx * p.hy))) < 1e-12
    assert np.max(np.abs(mod2pi(circulation(thz, thx, 0, 2) + By * p.hz * p.hx))) < 1e-12
    assert np.max(np.abs(mod2pi(circulation(thy, thz, 1, 0)))) < 1e-12
    # the uniform part of th_x is the gauge variable K
    assert abs(thx[0, 0, 0] - p.hx * 0.3) < 1e-15


def test_unsnapped_field_breaks_the_seam_plaquettes():
    p = O.Params(12, 10, 8)
    thx, thy, thz = O.paper_links_yz(p, 0.0, 0.0, 0.3)                  # not a multiple of 2 pi/(Lx Ly)
    c = mod2pi(circulation(thx, thy, 2, 1) + 0.3 * p.hx * p.hy)
    assert np.max(np.abs(c[:, :, :-1])) < 1e-12 and np.max(np.abs(c[:, :, -1])) > 1e-3


@pytest.mark.parametrize("nzq,nyq", [(3, 0), (-2, 1)])
def test_flux_quantisation_yz(nzq, nyq):
    p = O.Params(12, 10, 6, hx=0.5, hy=0.6, hz=0.4)
    Bz = 2 * math.pi * nzq / (p.length("x") * p.length("y"))
    By = 2 * math.pi * nyq / (p.length("x") * p.length("z"))
    rng = np.random.default_rng(1)
    psi = (1 + 0.5 * rng.uniform(-1, 1, p.shape)) * np.exp(1j * rng.uniform(-math.pi, math.pi, p.shape))
    links = O.paper_links_yz(p, 0.2, By, Bz)
    n = O.plaquette_windings(p, psi, links, Bz)
    assert np.max(np.abs(n - np.rint(n))) < 1e-12
    assert O.vortices_per_slice(p, psi, links, Bz) == float(nzq)


@pytest.mark.parametrize("bcz", [P_, O_])
def test_gauge_equivalence_with_the_xz_gauge(bcz):
    """B || z, x and y open (no holonomy): A^{yz} - A^{xz} = grad(B_z xbar ybar), so psi^{yz} = psi^{xz} e^{i chi}
    with chi = B_z xbar ybar at every step; |psi|, mu, the free energy and the windings coincide."""
    p = O.Params(10, 9, 4, hx=0.5, hy=0.45, hz=0.5, bc=(O_, O_, bcz), eps_tol=1e-24, max_sweeps=3000)
    Bz = 0.4
    xbar = (np.arange(p.nx) * p.hx - p.length("x") / 2)[None, None, :]
    ybar = (np.arange(p.ny) * p.hy - p.length("y") / 2)[None, :, None]
    chi = np.broadcast_to(Bz * xbar * ybar, p.shape)
    rng = np.random.default_rng(7)
    psi0 = (0.8 + 0.2 * rng.uniform(-1, 1, p.shape)) * np.exp(1j * rng.uniform(-1, 1, p.shape))
    eps = np.where(rng.uniform(size=p.shape) < 0.2, -1.0, 1.0)
    a = O.State(psi=psi0.copy(), mu=np.zeros(p.shape))
    b = O.State(psi=psi0 * np.exp(1j * chi), mu=np.zeros(p.shape))
    for _ in range(5):
        O.step(p, a, eps, 0.0, Bz, 0.0)
        O.step(p, b, eps, 0.0, Bz, 0.0, links_fn=lambda K: O.paper_links_yz(p, K, 0.0, Bz))
    assert np.max(np.abs(b.psi - a.psi * np.exp(1j * chi))) < 1e-10
    assert np.max(np.abs(b.mu - a.mu)) < 1e-10
    la, lb = O.paper_links(p, 0.0, 0.0, Bz), O.paper_links_yz(p, 0.0, 0.0, Bz)
    assert abs(O.free_energy(p, a.psi, eps, la) - O.free_energy(p, b.psi, eps, lb)) < 1e-9


def test_windowed_yz_links_match_full_arrays():
    p = O.Params(12, 10, 6)
    full = O.paper_links_yz(p, 0.2, 0.1, 0.3)
    ii, jj, kk = np.array([11, 0, 3]), np.array([9, 0]), np.array([5, 2])
    win = O.paper_links_yz_at(p, 0.2, 0.1, 0.3, ii, jj, kk)
    sel = np.ix_(kk, jj, ii)
    for f, w in zip(full, win):
        assert np.array_equal(w, f[sel])
