"""Pins of the oracle's film mode (N_z = 1: the paper's 2D workloads; reading S22: no z links at
all, d = 2 in Eq. 38-39), CPU only.  Expected values are closed forms, invariants and dense two-dimensional
assemblies written here from the printed entries -- none uses the oracle's own c_z or cell."""
import math

import numpy as np
import pytest

from oracle import tdgl_oracle as O

P_, O_ = O.PERIODIC, O.OPEN
BC2 = [(a, b, P_) for a in (P_, O_) for b in (P_, O_)]


def rand_psi(p, seed):
    rng = np.random.default_rng(seed)
    return rng.uniform(-1, 1, p.shape) + 1j * rng.uniform(-1, 1, p.shape)


def test_film_has_no_z_faces():
    with pytest.raises(ValueError):
        O.Params(8, 8, 1, bc=(P_, P_, O_))


@pytest.mark.parametrize("a,eps0", [(0.3, 1.0), (1.2, 0.5)])
def test_single_sweep_uniform_closed_form(a, eps0):
    """One Jacobi sweep (Eq. 33) from a uniform real psi = a at B = 0 in 2D:
    x^1 = [a + (h_t/2)(eps a - a^3 + 2 (c_x + c_y) a)] / [1 + (h_t/2)(a^2 + 2 (c_x + c_y) - eps)].
    A z contribution 2 c_z in the diagonal and in the neighbour sum would change x^1 (not the fixed point)."""
    p = O.Params(8, 6, 1, hx=0.5, hy=0.4, hz=0.3, solve_mu=False)
    st = O.State(psi=np.full(p.shape, a, dtype=np.complex128), mu=np.zeros(p.shape))
    O.step(p, st, np.full(p.shape, eps0), 0.0, 0.0, 0.0, fixed_sweeps=1)
    ht2, cs = 0.05, 2.0 * (1 / 0.25 + 1 / 0.16)
    expect = (a + ht2 * (eps0 * a - a ** 3 + cs * a)) / (1 + ht2 * (a * a + cs - eps0))
    assert np.max(np.abs(st.psi - expect)) < 1e-14
    # converged: the closed form of Eq. (26) with psi_est = psi^-
    st = O.State(psi=np.full(p.shape, a, dtype=np.complex128), mu=np.zeros(p.shape))
    p2 = O.Params(8, 6, 1, hx=0.5, hy=0.4, hz=0.3, solve_mu=False, eps_tol=1e-30, max_sweeps=4000)
    O.step(p2, st, np.full(p.shape, eps0), 0.0, 0.0, 0.0)
    q = 0.05 * (eps0 - a * a)
    assert np.max(np.abs(st.psi - a * (1 + q) / (1 - q))) < 1e-13


@pytest.mark.parametrize("K", [0.0, 0.41])
def test_plane_wave_growth_factor_2d(K):
    """Small plane wave at B = 0: factor (1 + (h_t/2)(eps - lam)) / (1 - (h_t/2)(eps - lam)) with the 2D symbol
    lam = c_x (2 - 2 cos((k_x + K) h_x)) + c_y (2 - 2 cos(k_y h_y))  (Eq. 26, 29a without the z term)."""
    p = O.Params(16, 8, 1, hx=0.5, hy=0.4, eps_tol=1e-30, max_sweeps=5000, solve_mu=False)
    kx, ky = 2 * math.pi * 3 / (16 * 0.5), 2 * math.pi * 1 / (8 * 0.4)
    j, i = np.meshgrid(np.arange(8), np.arange(16), indexing="ij")
    delta = 1e-4
    psi = (delta * np.exp(1j * (kx * i * 0.5 + ky * j * 0.4)))[None]
    st = O.State(psi=psi.copy(), mu=np.zeros(p.shape), K=K)
    O.step(p, st, np.ones(p.shape), 0.0, 0.0, 0.0)
    lam = (2 - 2 * math.cos((kx + K) * 0.5)) / 0.25 + (2 - 2 * math.cos(ky * 0.4)) / 0.16
    fac = (1 + 0.05 * (1.0 - lam)) / (1 - 0.05 * (1.0 - lam))
    assert np.max(np.abs(st.psi / psi - fac)) < 1e-8                  # O(delta^2) from the cubic term


def test_noise_amplitude_in_two_dimensions():
    """Eq. (39) with delta(r - r') = delta_ij / (h_x h_y) (d = 2): zeta_max^2 = 3 T u / (2 dt h_x h_y),
    i.e. T_zeta = dt h_x h_y zeta_max^2 is grid independent."""
    for hx, hy, dt in ((0.5, 0.5, 0.1), (0.25, 0.4, 0.05)):
        p = O.Params(8, 8, 1, hx=hx, hy=hy, hz=0.123, dt=dt, temperature=2e-3)
        assert abs(dt * hx * hy * O.zeta_max(p) ** 2 - 1.5 * 2e-3) < 1e-15
    z = O.langevin_noise(O.Params(64, 64, 1, temperature=1e-3, seed=3), 5)
    zm = O.zeta_max(O.Params(64, 64, 1, temperature=1e-3))
    assert np.max(np.abs(z.real)) < zm and abs(np.mean(np.abs(z) ** 2) / (2 * zm * zm / 3) - 1) < 0.05


@pytest.mark.parametrize("nzq", [3, -2])
def test_flux_quantisation_2d(nzq):
    p = O.Params(12, 10, 1, hx=0.5, hy=0.6)
    Bz = 2 * math.pi * nzq / (p.length("x") * p.length("y"))
    _, Bzs, _, q = O.snap_field(p, 0.0, Bz)
    assert q == nzq
    rng = np.random.default_rng(1)
    psi = (1 + 0.5 * rng.uniform(-1, 1, p.shape)) * np.exp(1j * rng.uniform(-math.pi, math.pi, p.shape))
    links = O.paper_links(p, 0.3, 0.0, Bzs)
    n = O.plaquette_windings(p, psi, links, Bzs)
    assert np.max(np.abs(n - np.rint(n))) < 1e-12
    assert O.vortices_per_slice(p, psi, links, Bzs) == float(nzq)


def dense_laplacian_2d(p):
    """(nx ny) x (nx ny) matrix of the 5-point operator, wrap or mirror ghost per axis."""
    n, c = (p.nx, p.ny), (1 / p.hx ** 2, 1 / p.hy ** 2)
    A = np.zeros((p.nx * p.ny, p.nx * p.ny))
    for j in range(p.ny):
        for i in range(p.nx):
            m = i + p.nx * j
            for a in range(2):
                A[m, m] -= 2 * c[a]
                for s in (1, -1):
                    r = [i, j]
                    r[a] += s
                    if p.bc[a] == P_:
                        r[a] %= n[a]
                    elif r[a] < 0:
                        r[a] = 1
                    elif r[a] >= n[a]:
                        r[a] = n[a] - 2
                    A[m, r[0] + p.nx * r[1]] += c[a]
    return A


@pytest.mark.parametrize("bc", BC2)
def test_poisson_2d_dense_bordered_solve(bc):
    p = O.Params(9, 8, 1, hx=0.5, hy=0.4, hz=0.7, bc=bc)
    A = dense_laplacian_2d(p)
    w = O.site_weights(p).ravel()
    rng = np.random.default_rng(8)
    f = rng.uniform(-1, 1, p.shape)
    assert np.max(np.abs(O.laplacian_real(p, f).ravel() - A @ f.ravel())) < 1e-12
    rho = rng.uniform(-1, 1, p.shape)
    rho -= np.sum(w * rho.ravel()) / np.sum(w)
    N = p.n_sites
    B = np.zeros((N + 1, N + 1))
    B[:N, :N], B[:N, N], B[N, :N] = A, 1.0, w
    sol = np.linalg.solve(B, np.append(rho.ravel(), 0.0))
    mu = O.solve_poisson(p, rho)
    assert np.max(np.abs(mu.ravel() - sol[:N])) < 1e-11


@pytest.mark.parametrize("bc", BC2)
def test_implicit_step_2d_dense_solve(bc):
    """M Psi = b assembled from the printed entries in 2D (diagonal 1 + (h_t/2)[|psi|^2 + 2/h_x^2 + 2/h_y^2 -
    eps + i u mu], off-diagonals -(h_t/2) c U; S21 on open faces; Eq. 31 for b) against the converged Jacobi solve."""
    p = O.Params(8, 7, 1, hx=0.5, hy=0.55, u=1.7, bc=bc, eps_tol=1e-28, max_sweeps=6000, solve_mu=False)
    _, Bz, _, _ = O.snap_field(p, 0.0, 0.3)
    K = 0.2 if bc[0] == P_ else 0.0
    thx, thy, _ = O.paper_links(p, K, 0.0, Bz)
    psi = rand_psi(p, 4)
    rng = np.random.default_rng(5)
    mu, eps = 0.1 * rng.standard_normal(p.shape), rng.choice([-1.0, 1.0], p.shape)
    ht2, c, n = 0.5 * p.dt / p.u, (1 / p.hx ** 2, 1 / p.hy ** 2), (p.nx, p.ny)
    N = p.n_sites
    M, L = np.zeros((N, N), complex), np.zeros((N, N), complex)       # L = covariant Laplacian
    th = (thx[0], thy[0])
    for j in range(p.ny):
        for i in range(p.nx):
            m, q = i + p.nx * j, (i, j)
            for a in range(2):
                L[m, m] -= 2 * c[a]
                rp, rm = list(q), list(q)
                rp[a] += 1
                rm[a] -= 1
                lo, hi = q[a] == 0, q[a] == n[a] - 1
                if p.bc[a] == P_:
                    rp[a] %= n[a]
                    rm[a] %= n[a]
                    L[m, rp[0] + p.nx * rp[1]] += c[a] * np.exp(1j * th[a][j, i])
                    L[m, rm[0] + p.nx * rm[1]] += c[a] * np.exp(-1j * th[a][rm[1], rm[0]])
                else:                                                   # single neighbour's entry doubles (S21)
                    if lo:
                        L[m, rp[0] + p.nx * rp[1]] += 2 * c[a] * np.exp(1j * th[a][j, i])
                    elif hi:
                        L[m, rm[0] + p.nx * rm[1]] += 2 * c[a] * np.exp(-1j * th[a][rm[1], rm[0]])
                    else:
                        L[m, rp[0] + p.nx * rp[1]] += c[a] * np.exp(1j * th[a][j, i])
                        L[m, rm[0] + p.nx * rm[1]] += c[a] * np.exp(-1j * th[a][rm[1], rm[0]])
    pv, mv, ev = psi.ravel(), mu.ravel(), eps.ravel()
    cabs = np.abs(pv) ** 2
    M = np.diag(1 + ht2 * (cabs - ev + 1j * p.u * mv)) - ht2 * L
    b = pv + ht2 * ((ev - 1j * p.u * mv) * pv - cabs * pv + L @ pv)
    x = np.linalg.solve(M, b)
    st = O.State(psi=psi.copy(), mu=mu.copy(), K=K)
    O.step(p, st, eps, 0.0, Bz, 0.0)
    assert np.max(np.abs(st.psi.ravel() - x)) < 1e-12


@pytest.mark.parametrize("bc", BC2)
def test_current_conservation_2d(bc):
    p = O.Params(10, 8, 1, hx=0.5, hy=0.45, bc=bc)
    _, Bz, _, _ = O.snap_field(p, 0.0, 0.25)
    links = O.paper_links(p, 0.3 if bc[0] == P_ else 0.0, 0.0, Bz)
    psi = rand_psi(p, 2)
    rho = O.supercurrent_divergence(p, psi, links)
    mu = O.solve_poisson(p, rho)
    assert np.max(np.abs(O.laplacian_real(p, mu) - rho)) < 1e-11       # div (j_s + j_n) = rho - Delta_h mu = 0
    assert abs(np.sum(O.site_weights(p) * mu)) < 1e-11
    # rho is the lattice divergence of the two in-plane link currents
    jx, jy, _ = O.link_supercurrents(p, psi, links)
    div = np.zeros(p.shape)
    for a, axis, h, j in ((0, 2, p.hx, jx), (1, 1, p.hy, jy)):
        d = (j - np.roll(j, 1, axis)) / h
        if p.bc[a] == O_:
            first, last = [slice(None)] * 3, [slice(None)] * 3
            first[axis], last[axis] = 0, -1
            d[tuple(first)] = 2.0 * j[tuple(first)] / h
            d[tuple(last)] = -2.0 * np.take(j, -2, axis=axis) / h
        div += d
    assert np.max(np.abs(div - rho)) < 1e-12
