"""Pins of the fp64 oracle against what the paper and the mathematics fix (CPU only).

Each test names the pin (P1..P15 of SURVEY.md 8(c)-P / DESIGN.md "Oracle pins") and the passage it rests on.
None of the expected values comes from the oracle itself or from the CUDA path: they are closed forms,
invariants, dense direct solves assembled from the paper's printed matrix entries, or brute force.
"""
import math

import numpy as np
import pytest

from oracle import tdgl_oracle as O

P_, O_ = O.PERIODIC, O.OPEN
ALL_BC = [(a, b, c) for a in (P_, O_) for b in (P_, O_) for c in (P_, O_)]


def rand_psi(p, seed, amp=1.0):
    rng = np.random.default_rng(seed)
    return amp * (rng.uniform(-1, 1, p.shape) + 1j * rng.uniform(-1, 1, p.shape))


def nonzero_psi(p, seed):
    """Zero-free field with a rough phase (modulus in [0.5, 1.5])."""
    rng = np.random.default_rng(seed)
    return (1.0 + 0.5 * rng.uniform(-1, 1, p.shape)) * np.exp(1j * rng.uniform(-math.pi, math.pi, p.shape))


# ------------------------------------------------------------------------------------------------
# P1 / P2: reaction term + Crank-Nicolson linearisation (Eq. 26 with psi_est = psi^-)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("a,eps0", [(0.3, 1.0), (1.2, 1.0), (0.7, 0.5), (0.4, -1.0)])
def test_P1_uniform_reaction_closed_form(a, eps0):
    # Eq. (26), B = 0, uniform real psi = a:  psi+ (1 - q) = psi- (1 + q),  q = h_t (eps - a^2)/2
    p = O.Params(8, 6, 4, eps_tol=1e-28, max_sweeps=2000, solve_mu=False)
    st = O.State(psi=np.full(p.shape, a, dtype=np.complex128), mu=np.zeros(p.shape))
    O.step(p, st, np.full(p.shape, eps0), 0.0, 0.0, 0.0)
    q = p.ht * (eps0 - a * a) / 2.0
    assert np.max(np.abs(st.psi - a * (1 + q) / (1 - q))) < 1e-13


@pytest.mark.parametrize("bc", [(P_, P_, P_), (P_, P_, O_), (O_, O_, O_)])
def test_P2_uniform_fixed_point(bc):
    # psi = sqrt(eps) at zero field is stationary (BASELINE.json north_star); residual 0, one sweep.
    p = O.Params(8, 8, 8, bc=bc, solve_mu=True)
    eps0 = 0.64
    st = O.State(psi=np.full(p.shape, math.sqrt(eps0), dtype=np.complex128), mu=np.zeros(p.shape))
    for _ in range(3):
        O.step(p, st, np.full(p.shape, eps0), 0.0, 0.0, 0.0)
        assert st.sweeps_last == 1
    assert np.max(np.abs(st.psi - math.sqrt(eps0))) < 1e-15
    assert np.max(np.abs(st.mu)) < 1e-15 and st.K == 0.0


# ------------------------------------------------------------------------------------------------
# P3: plane wave -> Laplacian, sign of U, CN factor (Eqs. 26, 27, 29a)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("K", [0.0, 0.37, -1.1])
def test_P3_plane_wave_growth_factor(K):
    p = O.Params(16, 8, 4, hx=0.5, hy=0.4, hz=0.7, g=1.3, eps_tol=1e-30, max_sweeps=5000, solve_mu=False)
    eps0, delta = 0.8, 1e-7
    mx, my, mz = 3, 1, 1
    kx, ky, kz = (2 * math.pi * mx / p.length("x"), 2 * math.pi * my / p.length("y"),
                  2 * math.pi * mz / p.length("z"))
    k_, j_, i_ = np.meshgrid(np.arange(p.nz), np.arange(p.ny), np.arange(p.nx), indexing="ij")
    wave = np.exp(1j * (kx * i_ * p.hx + ky * j_ * p.hy + kz * k_ * p.hz))
    st = O.State(psi=delta * wave, mu=np.zeros(p.shape), K=K)
    O.step(p, st, np.full(p.shape, eps0), 0.0, 0.0, 0.0, fixed_sweeps=200)   # |r| is O(delta): iterate to rounding
    # (grad - iA~)^2 with A~ = -K e_x acts on e^{ikx} as -(k+K)^2; lattice version 2 - 2cos((k+K)h)
    lam = ((2 - 2 * math.cos((kx + K) * p.hx)) / p.hx ** 2 + (2 - 2 * math.cos(ky * p.hy)) / p.hy ** 2
           + (2 - 2 * math.cos(kz * p.hz)) / (p.g * p.hz) ** 2)
    q = p.ht * (eps0 - lam) / 2.0
    fac = (1 + q) / (1 - q)
    assert np.max(np.abs(st.psi / (delta * wave) - fac)) < 1e-12   # nonlinearity is O(delta^2)


# ------------------------------------------------------------------------------------------------
# P4: J_av (Eq. 35)
# ------------------------------------------------------------------------------------------------
def test_P4_average_supercurrent_closed_form():
    # psi = a e^{ikx}: continuum J = a^2 (k + K); Eq. (35) central difference gives a^2 sin((k+K)h)/h
    p = O.Params(16, 4, 4)
    a, K, mx = 0.9, 0.23, 2
    kx = 2 * math.pi * mx / p.length("x")
    i_ = np.arange(p.nx)[None, None, :]
    psi = a * np.exp(1j * kx * i_ * p.hx) * np.ones(p.shape)
    J = O.average_supercurrent(p, psi, O.paper_links(p, K, 0.0, 0.0))
    assert abs(J - a * a * math.sin((kx + K) * p.hx) / p.hx) < 1e-14


# ------------------------------------------------------------------------------------------------
# P5: Ohmic normal state (Eq. 21 with psi = 0: d_t K = J_ext, E = J)
# ------------------------------------------------------------------------------------------------
def test_P5_ohmic_normal_state():
    p = O.Params(8, 8, 4)
    st = O.State(psi=np.zeros(p.shape, dtype=np.complex128), mu=np.zeros(p.shape))
    Jext = 0.7
    for n in range(1, 400):
        O.step(p, st, np.full(p.shape, -1.0), 0.0, 0.0, Jext)
        assert abs(st.Ex - Jext) < 1e-15
        expect = math.fmod(n * p.dt * Jext, 2 * math.pi / p.hx)      # rewinding
        assert abs(st.K - expect) < 1e-9
    assert n * p.dt * Jext > 2 * math.pi / p.hx                        # the run did wrap at least once
    assert np.max(np.abs(st.mu)) == 0.0 and np.max(np.abs(st.psi)) == 0.0


# ------------------------------------------------------------------------------------------------
# P6: quasi-periodic boundary, P_{i,k}, flux quantisation
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("nzq,nxq", [(4, 0), (1, 2), (-3, 1)])
def test_P6_flux_quantisation_topological(nzq, nxq):
    p = O.Params(12, 10, 6, hx=0.5, hy=0.6, hz=0.4)
    Bz_req = 2 * math.pi * nzq / (p.length("x") * p.length("y")) * 1.0004   # slightly off: must snap
    Bx_req = 2 * math.pi * nxq / (p.length("y") * p.length("z")) + 1e-4
    Bx, Bz, nx_, nz_ = O.snap_field(p, Bx_req, Bz_req)
    assert (nx_, nz_) == (nxq, nzq)
    psi = nonzero_psi(p, 5)
    links = O.paper_links(p, 0.31, Bx, Bz)
    n = O.plaquette_windings(p, psi, links, Bz)
    assert np.max(np.abs(n - np.rint(n))) < 1e-12          # every winding is an integer ...
    per_slice = np.rint(n).sum(axis=(1, 2))
    assert np.all(per_slice == nzq)                          # ... and each z-slice holds exactly n_z quanta
    assert abs(O.vortices_per_slice(p, psi, links, Bz) - nzq) < 1e-12


def test_P6_unsnapped_field_breaks_the_identity():
    # negative control: without the flux constraint the phase jump is discontinuous and the count is not n_z
    p = O.Params(12, 10, 4)
    Bz = 2 * math.pi * 3.5 / (p.length("x") * p.length("y"))
    psi = nonzero_psi(p, 6)
    n = O.plaquette_windings(p, psi, O.paper_links(p, 0.0, 0.0, Bz), Bz)
    assert np.max(np.abs(n - np.rint(n))) > 1e-3


# ------------------------------------------------------------------------------------------------
# P7: current conservation after the mu solve (Eqs. 17, 18)
# ------------------------------------------------------------------------------------------------
def _divergence(p, jx, jy, jz):
    """Lattice divergence of link currents; at an open face the ghost link carries minus the first link
    (mirror), so the boundary divergence is 2 j / h."""
    out = np.zeros(p.shape)
    for a, axis, h, j in ((0, 2, p.hx, jx), (1, 1, p.hy, jy), (2, 0, p.hz, jz)):
        d = (j - np.roll(j, 1, axis)) / h
        if p.bc[a] == O_:
            first = [slice(None)] * 3
            last = [slice(None)] * 3
            first[axis], last[axis] = 0, -1
            first, last = tuple(first), tuple(last)
            jm1 = np.take(j, -2, axis=axis)
            d[first] = 2.0 * j[first] / h
            d[last] = -2.0 * jm1 / h
        out += d
    return out


@pytest.mark.parametrize("bc", ALL_BC)
def test_P7_current_conservation(bc):
    p = O.Params(8, 6, 7, hx=0.5, hy=0.45, hz=0.6, g=1.2, bc=bc)
    Bx, Bz, _, _ = O.snap_field(p, 0.07, 0.21)
    links = O.paper_links(p, 0.4 if bc[0] == P_ else 0.0, Bx, Bz)
    psi = rand_psi(p, 11)
    rho = O.supercurrent_divergence(p, psi, links)
    js = O.link_supercurrents(p, psi, links)
    assert np.max(np.abs(_divergence(p, *js) - rho)) < 1e-12           # rho IS div j_s
    assert abs(np.sum(O.site_weights(p) * rho)) < 1e-11                 # solvability (S6)
    mu = O.solve_poisson(p, rho)
    jn = []
    for a, axis, h, gg in ((0, 2, p.hx, 1.0), (1, 1, p.hy, 1.0), (2, 0, p.hz, p.g ** 2)):
        j = -(np.roll(mu, -1, axis) - mu) / (h * gg)
        if bc[a] == O_:
            sl = [slice(None)] * 3
            sl[axis] = -1
            j[tuple(sl)] = 0.0
        jn.append(j)
    total = [js[a] + jn[a] for a in range(3)]
    assert np.max(np.abs(_divergence(p, *total))) < 1e-11              # div (j_s + j_n) = 0
    assert abs(np.sum(O.site_weights(p) * mu)) < 1e-11                  # gauge S7


# ------------------------------------------------------------------------------------------------
# P8: gauge invariance
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc", [(P_, P_, P_), (P_, P_, O_), (P_, O_, O_), (O_, O_, O_)])
def test_P8_gauge_invariance(bc):
    p = O.Params(8, 8, 6, bc=bc, eps_tol=1e-6)
    Jext = 0.05 if bc[0] == P_ else 0.0
    Bx, Bz, _, _ = O.snap_field(p, 0.1, 0.4)
    rng = np.random.default_rng(3)
    chi = rng.uniform(-3, 3, p.shape)
    eps = np.where(rng.uniform(size=p.shape) < 0.2, -1.0, 1.0)

    def links_fn(K):
        return O.paper_links(p, K, Bx, Bz)

    def links_fn_g(K):
        # psi' = psi e^{i chi};  S'+ f' = e^{i chi} S+ f  <=>  th'(m) = th(m) + chi(m) - chi(m + alpha)
        thx, thy, thz = O.paper_links(p, K, Bx, Bz)
        return (thx + chi - np.roll(chi, -1, 2), thy + chi - np.roll(chi, -1, 1), thz + chi - np.roll(chi, -1, 0))

    psi0 = 1.0 + 0.3 * rand_psi(p, 2)
    a = O.State(psi=psi0.copy(), mu=np.zeros(p.shape))
    b = O.State(psi=psi0 * np.exp(1j * chi), mu=np.zeros(p.shape))
    for n in range(12):
        O.step(p, a, eps, Bx, Bz, Jext, links_fn=links_fn)
        O.step(p, b, eps, Bx, Bz, Jext, links_fn=links_fn_g)
        assert a.sweeps_last == b.sweeps_last
        assert np.max(np.abs(b.psi - a.psi * np.exp(1j * chi))) < 1e-12
        assert np.max(np.abs(a.mu - b.mu)) < 1e-12
        assert abs(a.K - b.K) < 1e-12 and abs(a.Jav - b.Jav) < 1e-13
    la, lb = links_fn(a.K), links_fn_g(b.K)
    assert abs(O.free_energy(p, a.psi, eps, la) - O.free_energy(p, b.psi, eps, lb)) < 1e-10
    ja, jb = O.link_supercurrents(p, a.psi, la), O.link_supercurrents(p, b.psi, lb)
    assert max(np.max(np.abs(x - y)) for x, y in zip(ja, jb)) < 1e-12
    assert np.max(np.abs(O.supercurrent_divergence(p, a.psi, la) - O.supercurrent_divergence(p, b.psi, lb))) < 1e-11


# ------------------------------------------------------------------------------------------------
# P9: the implicit step against a dense direct solve (BASELINE.json north_star)
# ------------------------------------------------------------------------------------------------
def dense_M(p, psi_prev, mu, eps, K, Bx, Bz):
    """Assemble the N x N matrix of Eq. (30) entry by entry from the printed list, the
    quasi-periodic rows and the open-face second derivatives."""
    N = p.n_sites
    M = np.zeros((N, N), dtype=np.complex128)
    ht = p.ht
    Ly = p.length("y")

    def idx(i, j, k):
        return i + p.nx * (j + p.ny * k)

    for k in range(p.nz):
        for j in range(p.ny):
            ybar = j * p.hy - Ly / 2
            Ux = np.exp(1j * p.hx * (K + Bz * ybar))           # U = exp(-i h A~), A~_x = -B_z ybar - K
            Uz = np.exp(-1j * p.hz * Bx * ybar)                 # A~_z = +B_x ybar
            for i in range(p.nx):
                m = idx(i, j, k)
                Pik = np.exp(1j * (i * p.hx * Ly * Bz - k * p.hz * Ly * Bx))
                M[m, m] = 1 + (ht / 2) * (abs(psi_prev[k, j, i]) ** 2
                                          + 2 * (1 / p.hx ** 2 + 1 / p.hy ** 2 + 1 / (p.g * p.hz) ** 2)
                                          + 1j * p.u * mu[k, j, i] - eps[k, j, i])
                # x
                ax = -ht / (2 * p.hx ** 2)
                if p.bc[0] == P_:
                    M[m, idx((i + 1) % p.nx, j, k)] += ax * Ux
                    M[m, idx((i - 1) % p.nx, j, k)] += ax * np.conj(Ux)
                elif i == 0:
                    M[m, idx(1, j, k)] += 2 * ax * Ux                       # 2(U psi_1 - psi_0)/h^2
                elif i == p.nx - 1:
                    M[m, idx(p.nx - 2, j, k)] += 2 * ax * np.conj(Ux)        # 2(U* psi_{N-2} - psi_{N-1})/h^2
                else:
                    M[m, idx(i + 1, j, k)] += ax * Ux
                    M[m, idx(i - 1, j, k)] += ax * np.conj(Ux)
                # y
                ay = -ht / (2 * p.hy ** 2)
                if p.bc[1] == P_:
                    if j == 0:
                        M[m, idx(i, 1 % p.ny, k)] += ay
                        M[m, idx(i, p.ny - 1, k)] += ay * Pik
                    elif j == p.ny - 1:
                        M[m, idx(i, 0, k)] += ay * np.conj(Pik)
                        M[m, idx(i, p.ny - 2, k)] += ay
                    else:
                        M[m, idx(i, j + 1, k)] += ay
                        M[m, idx(i, j - 1, k)] += ay
                elif j == 0:
                    M[m, idx(i, 1, k)] += 2 * ay
                elif j == p.ny - 1:
                    M[m, idx(i, p.ny - 2, k)] += 2 * ay
                else:
                    M[m, idx(i, j + 1, k)] += ay
                    M[m, idx(i, j - 1, k)] += ay
                # z
                az = -ht / (2 * (p.g * p.hz) ** 2)
                if p.bc[2] == P_:
                    M[m, idx(i, j, (k + 1) % p.nz)] += az * Uz
                    M[m, idx(i, j, (k - 1) % p.nz)] += az * np.conj(Uz)
                elif k == 0:
                    M[m, idx(i, j, 1)] += 2 * az * Uz
                elif k == p.nz - 1:
                    M[m, idx(i, j, p.nz - 2)] += 2 * az * np.conj(Uz)
                else:
                    M[m, idx(i, j, k + 1)] += az * Uz
                    M[m, idx(i, j, k - 1)] += az * np.conj(Uz)
    return M


@pytest.mark.parametrize("bc", [(P_, P_, P_), (P_, P_, O_), (P_, O_, P_), (O_, O_, O_)])
def test_P9_implicit_step_dense_solve(bc):
    p = O.Params(8, 8, 8, hx=0.5, hy=0.55, hz=0.45, g=1.1, u=1.7, bc=bc, eps_tol=1e-28, max_sweeps=5000,
                 solve_mu=False)
    Bx, Bz, _, _ = O.snap_field(p, 0.12, 0.35)
    K = 0.21 if bc[0] == P_ else 0.0
    rng = np.random.default_rng(4)
    psi0 = 1.0 + 0.4 * rand_psi(p, 7)
    mu0 = rng.uniform(-0.2, 0.2, p.shape)
    eps = np.where(rng.uniform(size=p.shape) < 0.3, -1.0, 1.0)
    M = dense_M(p, psi0, mu0, eps, K, Bx, Bz)
    # Crank-Nicolson: M = I - (h_t/2) Lin, b = (I + (h_t/2) Lin) psi^-  =>  b = 2 psi^- - M psi^-  (Eq. 26, 31)
    b_dense = 2 * psi0.ravel() - M @ psi0.ravel()
    links = O.paper_links(p, K, Bx, Bz)
    b, d = O.build_system(p, psi0, mu0, eps, links)
    assert np.max(np.abs(b.ravel() - b_dense)) < 1e-13
    assert np.max(np.abs(d.ravel() - np.diag(M))) < 1e-15
    # diagonal dominance margin the paper relies on
    off = np.sum(np.abs(M), axis=1) - np.abs(np.diag(M))
    assert np.all(np.abs(np.diag(M)) > off)
    x_dense = np.linalg.solve(M, b_dense)
    st = O.State(psi=psi0.copy(), mu=mu0.copy(), K=K)
    O.step(p, st, eps, Bx, Bz, 0.0)
    assert np.max(np.abs(st.psi.ravel() - x_dense)) < 1e-12
    # residual bookkeeping (S8): r^l = b - M x^l
    x1, r0 = O.jacobi_sweep(p, psi0, b, d, links)
    assert np.max(np.abs(r0.ravel() - (b_dense - M @ psi0.ravel()))) < 1e-13


def test_P9_noise_enters_as_ht_zeta():
    # Eq. (26): the Langevin term contributes h_t zeta_m to psi - psi^-  =>  M (psi_T - psi_0) = h_t zeta
    p0 = O.Params(8, 8, 8, eps_tol=1e-28, max_sweeps=5000, solve_mu=False)
    pT = O.Params(8, 8, 8, eps_tol=1e-28, max_sweeps=5000, solve_mu=False, temperature=1e-3, seed=99)
    Bx, Bz, _, _ = O.snap_field(p0, 0.0, 0.4)
    psi0 = 1.0 + 0.2 * rand_psi(p0, 1)
    eps = np.ones(p0.shape)
    a = O.State(psi=psi0.copy(), mu=np.zeros(p0.shape), n=5)
    b = O.State(psi=psi0.copy(), mu=np.zeros(p0.shape), n=5)
    O.step(p0, a, eps, Bx, Bz, 0.0)
    O.step(pT, b, eps, Bx, Bz, 0.0)
    M = dense_M(p0, psi0, np.zeros(p0.shape), eps, 0.0, Bx, Bz)
    zeta = (M @ (b.psi - a.psi).ravel()) / pT.ht
    zmax = O.zeta_max(pT)
    assert abs(zmax - math.sqrt(0.12)) < 1e-15          # Eq. (39) at h = 0.5, dt = 0.1, T = 1e-3, u = 1
    assert np.max(np.abs(zeta.real)) < zmax and np.max(np.abs(zeta.imag)) < zmax
    # <|zeta|^2> = (2/3) zeta_max^2; 512 samples -> ~4 % statistical error
    assert abs(np.mean(np.abs(zeta) ** 2) / (2.0 / 3.0 * zmax ** 2) - 1.0) < 0.15
    # and it is exactly the generator's stream for (seed, step 5)
    assert np.max(np.abs(zeta - O.langevin_noise(pT, 5).ravel())) < 1e-12


# ------------------------------------------------------------------------------------------------
# P10: Poisson problem against a dense bordered solve and eigen-checks (PAPER.md:379, S5-S7)
# ------------------------------------------------------------------------------------------------
def dense_laplacian(p):
    N = p.n_sites
    A = np.zeros((N, N))
    n = (p.nx, p.ny, p.nz)
    c = (1 / p.hx ** 2, 1 / p.hy ** 2, 1 / (p.g * p.hz) ** 2)

    def idx(q):
        return q[0] + p.nx * (q[1] + p.ny * q[2])

    for k in range(p.nz):
        for j in range(p.ny):
            for i in range(p.nx):
                q = [i, j, k]
                m = idx(q)
                for a in range(3):
                    A[m, m] -= 2 * c[a]
                    for s in (+1, -1):
                        r = list(q)
                        r[a] += s
                        if p.bc[a] == P_:
                            r[a] %= n[a]
                        elif r[a] < 0:
                            r[a] = 1                      # mirror ghost mu_{-1} = mu_{1} (S6)
                        elif r[a] >= n[a]:
                            r[a] = n[a] - 2
                        A[m, idx(r)] += c[a]
    return A


@pytest.mark.parametrize("bc", ALL_BC)
def test_P10_poisson_dense_bordered_solve(bc):
    p = O.Params(8, 7, 6, hx=0.5, hy=0.4, hz=0.65, g=1.25, bc=bc)
    A = dense_laplacian(p)
    w = O.site_weights(p).ravel()
    rng = np.random.default_rng(8)
    rho = rng.uniform(-1, 1, p.shape)
    rho -= np.sum(w * rho.ravel()) / np.sum(w)                    # compatible right side
    # the stencil operator is that matrix
    f = rng.uniform(-1, 1, p.shape)
    assert np.max(np.abs(O.laplacian_real(p, f).ravel() - A @ f.ravel())) < 1e-12
    N = p.n_sites
    B = np.zeros((N + 1, N + 1))
    B[:N, :N] = A
    B[:N, N] = 1.0
    B[N, :N] = w
    sol = np.linalg.solve(B, np.append(rho.ravel(), 0.0))
    mu = O.solve_poisson(p, rho)
    assert abs(sol[N]) < 1e-12
    assert np.max(np.abs(mu.ravel() - sol[:N])) < 1e-11
    assert np.max(np.abs(O.laplacian_real(p, mu) - rho)) < 1e-11


@pytest.mark.parametrize("bc", [(P_, P_, O_), (O_, P_, P_)])
def test_P10_eigenvectors(bc):
    p = O.Params(8, 8, 9, bc=bc)
    k_, j_, i_ = np.meshgrid(np.arange(p.nz), np.arange(p.ny), np.arange(p.nx), indexing="ij")
    for axis_name, idx, n, c in (("x", i_, p.nx, p.cx), ("z", k_, p.nz, p.cz)):
        a = "xyz".index(axis_name)
        for q in (1, 3):
            if bc[a] == P_:
                v, lam = np.cos(2 * math.pi * q * idx / n), -c * (2 - 2 * math.cos(2 * math.pi * q / n))
            else:
                v, lam = np.cos(math.pi * q * idx / (n - 1)), -c * (2 - 2 * math.cos(math.pi * q / (n - 1)))
            assert np.max(np.abs(O.laplacian_real(p, v) - lam * v)) < 1e-12


# ------------------------------------------------------------------------------------------------
# P11: open faces carry no normal supercurrent
# ------------------------------------------------------------------------------------------------
def test_P11_open_face_normal_current_vanishes():
    p = O.Params(6, 7, 5, bc=(O_, O_, O_))
    links = O.paper_links(p, 0.0, 0.13, 0.29)
    psi = rand_psi(p, 12)
    for th, axis in ((links[0], 2), (links[1], 1), (links[2], 0)):
        sp, sm = O._S(psi, th, axis, O_)
        jn = np.imag(np.conj(psi) * (sp - sm))                 # 2 h x central-difference normal current
        first = [slice(None)] * 3
        last = [slice(None)] * 3
        first[axis], last[axis] = 0, -1
        assert np.max(np.abs(jn[tuple(first)])) == 0.0 and np.max(np.abs(jn[tuple(last)])) == 0.0
    # and the Laplacian there is the printed form 2 (U psi_1 - psi_0)/h^2
    L = O.covariant_laplacian(p, psi, links)
    j = 3
    Ux = np.exp(1j * p.hx * 0.29 * (j * p.hy - p.length("y") / 2))
    Uz = np.exp(-1j * p.hz * 0.13 * (j * p.hy - p.length("y") / 2))
    k, i = 2, 0
    expect = (2 * (Ux * psi[k, j, 1] - psi[k, j, 0]) / p.hx ** 2
              + (psi[k, j + 1, 0] + psi[k, j - 1, 0] - 2 * psi[k, j, 0]) / p.hy ** 2
              + (Uz * psi[k + 1, j, 0] + np.conj(Uz) * psi[k - 1, j, 0] - 2 * psi[k, j, 0]) / p.hz ** 2)
    assert abs(L[k, j, i] - expect) < 1e-13


# ------------------------------------------------------------------------------------------------
# P12: free energy -- gradient by finite differences, and descent
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc", [(P_, P_, P_), (P_, P_, O_), (O_, P_, O_), (O_, O_, O_)])
def test_P12_free_energy_gradient(bc):
    # -dF/dpsi*_m / (w_m h^3) = eps psi - |psi|^2 psi + (grad - iA~)^2 psi  (right side of Eq. 16, zeta = 0)
    p = O.Params(4, 5, 4, hx=0.5, hy=0.6, hz=0.45, g=1.15, bc=bc)
    Bx, Bz, _, _ = O.snap_field(p, 0.2, 0.5)
    links = O.paper_links(p, 0.3 if bc[0] == P_ else 0.0, Bx, Bz)
    rng = np.random.default_rng(21)
    eps = rng.uniform(-1, 1, p.shape)
    psi = rand_psi(p, 22)
    rhs = eps * psi - np.abs(psi) ** 2 * psi + O.covariant_laplacian(p, psi, links)
    w = O.site_weights(p)
    vol = p.hx * p.hy * p.hz
    dlt = 1e-6
    for m in rng.choice(p.n_sites, size=12, replace=False):
        k, j, i = np.unravel_index(m, p.shape)
        g = 0.0
        for dz, fac in ((dlt, 1.0), (1j * dlt, 1j)):
            a, b = psi.copy(), psi.copy()
            a[k, j, i] += dz
            b[k, j, i] -= dz
            dF = (O.free_energy(p, a, eps, links) - O.free_energy(p, b, eps, links)) / (2 * dlt)
            g = g + 0.5 * fac * dF                 # dF/dpsi* = (dF/dRe + i dF/dIm)/2
        assert abs(-g / (w[k, j, i] * vol) - rhs[k, j, i]) < 1e-6      # FD round-off ~1e-7; a wrong term is O(1)


def test_P12_free_energy_decreases():
    p = O.Params(16, 16, 4, solve_mu=False, eps_tol=1e-12)
    Bx, Bz, _, _ = O.snap_field(p, 0.0, 0.2)
    st = O.State(psi=1.0 + 0.3 * rand_psi(p, 30), mu=np.zeros(p.shape))
    eps = np.ones(p.shape)
    links = O.paper_links(p, 0.0, Bx, Bz)
    F = [O.free_energy(p, st.psi, eps, links)]
    for _ in range(60):
        O.step(p, st, eps, Bx, Bz, 0.0)
        F.append(O.free_energy(p, st.psi, eps, links))
    assert all(F[n + 1] <= F[n] + 1e-12 for n in range(60))
    assert F[-1] < F[0] - 1.0


# ------------------------------------------------------------------------------------------------
# P13: physics sanity -- lowest-Landau-level growth rate (H_c2 = 1 in these units)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("eps0,grows", [(1.0, True), (0.05, False)])
def test_P13_landau_level_growth_rate(eps0, grows):
    p = O.Params(16, 16, 2, solve_mu=False, eps_tol=1e-30, max_sweeps=3000)
    Bx, Bz, _, nzq = O.snap_field(p, 0.0, 0.1)
    assert nzq == 1
    st = O.State(psi=1e-12 * rand_psi(p, 40), mu=np.zeros(p.shape))
    eps = np.full(p.shape, eps0)
    norms = []
    for _ in range(160):
        O.step(p, st, eps, Bx, Bz, 0.0, fixed_sweeps=80)      # |psi| ~ 1e-12: an absolute tolerance is useless
        norms.append(np.linalg.norm(st.psi))
    rate = math.log(norms[-1] / norms[-11]) / (10 * p.dt)
    # linearised Eq. (16): d_t psi = (eps - E) psi, lowest eigenvalue of -(grad - iA)^2 is E = B_z (+O(B^2 h^2))
    assert abs(rate - (eps0 - Bz)) < 5e-3
    assert (rate > 0) == grows


# ------------------------------------------------------------------------------------------------
# P15 (soft): sweep counts the paper quotes ("about 4-6 iterations", tests/golden/paper_values.txt)
# ------------------------------------------------------------------------------------------------
def test_P15_sweep_counts_are_in_the_quoted_range():
    lo, hi = None, None
    for line in open(__file__.rsplit("/", 1)[0] + "/golden/paper_values.txt"):
        if line.startswith("jacobi_sweeps_steady_flow"):
            lo, hi = (int(v) for v in line.split()[1:3])
    p = O.Params(32, 32, 8, eps_tol=1e-6)
    Bx, Bz, _, _ = O.snap_field(p, 0.0, 0.1)
    st = O.State(psi=1.0 + 0.01 * rand_psi(p, 50), mu=np.zeros(p.shape))
    O.run(p, st, np.ones(p.shape), Bx, Bz, 0.05, 250)
    late = st.sweep_log[150:]
    assert lo - 1 <= np.mean(late) <= hi + 1, np.mean(late)
    assert not st.hit_max_sweeps


# ------------------------------------------------------------------------------------------------
# a0: inclusion pattern
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc", [(P_, P_, P_), (P_, P_, O_), (O_, O_, O_)])
def test_epsilon_bounding_box_equals_brute_force(bc):
    p = O.Params(16, 12, 10, bc=bc)
    rng = np.random.default_rng(60)
    sph = np.stack([rng.uniform(0, 8, 9), rng.uniform(0, 6, 9), rng.uniform(0, 5, 9), rng.uniform(0.4, 2.5, 9)], 1)
    sph[0] = (0.1, 0.2, 0.1, 2.0)          # straddles the corner: exercises the minimum image
    sph[1] = (4.0, 3.0, 2.5, 30.0)         # larger than the box
    a = O.epsilon_from_spheres(p, sph[:1], -1.0, 1.0)
    assert (a[0, 0, -1] == -1.0) == (bc[0] == P_)          # image across the periodic x face only
    e1 = O.epsilon_from_spheres(p, sph[[0, 2, 3, 4, 5, 6, 7, 8]], -1.0, 1.0)
    e2 = O.epsilon_brute_force(p, sph[[0, 2, 3, 4, 5, 6, 7, 8]], -1.0, 1.0)
    assert np.array_equal(e1, e2)
    assert 0.0 < np.mean(e1 < 0) < 1.0
    assert np.all(O.epsilon_from_spheres(p, sph[1:2], -1.0, 1.0) == -1.0)
    # a sphere of radius r centred on a site covers exactly the lattice points with d^2 <= r^2
    one = O.epsilon_from_spheres(p, np.array([[4.0, 3.0, 2.5, 1.0]]), -1.0, 1.0)
    assert int(np.sum(one < 0)) == 33          # |n|^2 <= 4 on the cubic lattice h = 0.5: 1+6+12+8+6


def _mixed_shapes(rng, n, box):
    sh = np.zeros((n, 10), dtype=np.float32)
    sh[:, 0] = rng.integers(0, 3, n)
    for q in range(3):
        sh[:, 1 + q] = rng.uniform(0, box[q], n)
        sh[:, 4 + q] = rng.uniform(0.4, 2.2, n)
        sh[:, 7 + q] = rng.normal(size=n)
    return sh


@pytest.mark.parametrize("bc", [(P_, P_, P_), (P_, P_, O_), (O_, P_, O_), (O_, O_, O_)])
def test_shapes_bounding_box_equals_brute_force(bc):
    # S26 (Fig. 2d/e): spheres, axis-aligned ellipsoids, capped cylinders with any axis
    p = O.Params(18, 14, 12, bc=bc)
    sh = _mixed_shapes(np.random.default_rng(61), 14, (9.0, 7.0, 6.0))
    sh[0, :7] = (2, 0.1, 0.2, 0.1, 0.8, 3.0, 0.0)          # a cylinder through the corner: minimum image
    sh[1, :7] = (1, 8.9, 0.1, 5.9, 2.0, 1.0, 1.5)          # an ellipsoid through the opposite corner
    e1 = O.epsilon_from_shapes(p, sh, -1.0, 1.0)
    e2 = O.epsilon_shapes_brute_force(p, sh, -1.0, 1.0)
    assert np.array_equal(e1, e2)
    assert 0.05 < np.mean(e1 < 0) < 0.95
    for kind in (0, 1, 2):                                  # and each kind on its own
        one = sh[sh[:, 0] == kind]
        assert len(one) > 0
        assert np.array_equal(O.epsilon_from_shapes(p, one, -1.0, 1.0), O.epsilon_shapes_brute_force(p, one, -1.0, 1.0))


def test_shapes_reduce_to_spheres_and_lattice_counts():
    p = O.Params(20, 16, 14, bc=(P_, P_, O_))
    rng = np.random.default_rng(62)
    sph = np.stack([rng.uniform(0, 10, 7), rng.uniform(0, 8, 7), rng.uniform(0, 7, 7), rng.uniform(0.45, 2.3, 7)], 1).astype(np.float32)
    sh = np.zeros((7, 10), dtype=np.float32)
    sh[:, 1:5] = sph
    ref = O.epsilon_from_spheres(p, sph, -1.0, 1.0)
    assert np.array_equal(O.epsilon_from_shapes(p, sh, -1.0, 1.0), ref)         # kind 0 = the sphere generator
    el = sh.copy()
    el[:, 0] = 1
    el[:, 5] = el[:, 4]
    el[:, 6] = el[:, 4]
    assert np.array_equal(O.epsilon_from_shapes(p, el, -1.0, 1.0), ref)         # equal semi-axes = a sphere
    # ellipsoid centred on a site, semi-axes (1, 0.5, 1.5), h = 0.5: lattice points with 9 i^2 + 36 j^2 + 4 k^2 <= 36
    want = sum(1 for i in range(-3, 4) for j in range(-3, 4) for k in range(-4, 5) if 9 * i * i + 36 * j * j + 4 * k * k <= 36)
    one = O.epsilon_from_shapes(p, np.array([[1, 5.0, 4.0, 3.5, 1.0, 0.5, 1.5, 0, 0, 0]]), -1.0, 1.0)
    assert int(np.sum(one < 0)) == want == 21
    # cylinder along z through the whole (open) thickness: every slice is the disc i^2 + j^2 <= 4 (13 lattice points)
    col = O.epsilon_from_shapes(p, np.array([[2, 5.0, 4.0, 3.0, 1.0, 50.0, 0.0, 0, 0, 2.5]]), -1.0, 1.0)
    assert np.all(np.sum(col < 0, axis=(1, 2)) == 13)
    assert np.all(col == col[0][None])
    # capped: half-length 1.0 keeps the slices |k h - 3.0| <= 1.0 only
    cap = O.epsilon_from_shapes(p, np.array([[2, 5.0, 4.0, 3.0, 1.0, 1.0, 0.0, 0, 0, 1.0]]), -1.0, 1.0)
    assert [int(v) for v in np.sum(cap < 0, axis=(1, 2))] == [13 if abs(k * 0.5 - 3.0) <= 1.0 else 0 for k in range(14)]


def test_shapes_cylinder_axis_covariance_and_volume():
    # the same cylinder with its axis along x, y: the masks are transposes of each other
    p = O.Params(24, 24, 10, bc=(P_, P_, P_))
    cx = O.epsilon_from_shapes(p, np.array([[2, 6.0, 5.0, 2.0, 1.3, 3.1, 0, 1, 0, 0]]), -1.0, 1.0)
    cy = O.epsilon_from_shapes(p, np.array([[2, 5.0, 6.0, 2.0, 1.3, 3.1, 0, 0, 1, 0]]), -1.0, 1.0)
    assert np.array_equal(cx, np.swapaxes(cy, 1, 2))
    # +-45 degree columns (Fig. 2e): a column along (1, 0, 1) is invariant under the lattice shift (i, k) -> (i+1, k+1)
    # (x periodic, half-length far beyond the box); the -45 degree column is its mirror image i -> -i
    p = O.Params(32, 12, 16, bc=(P_, P_, O_))
    a = O.epsilon_from_shapes(p, np.array([[2, 8.0, 3.0, 4.0, 1.3, 100.0, 0, 1, 0, 1]]), -1.0, 1.0) < 0
    assert 0 < a.sum()
    assert np.array_equal(a[1:], np.roll(a, 1, axis=2)[:-1])
    b = O.epsilon_from_shapes(p, np.array([[2, 8.0, 3.0, 4.0, 1.3, 100.0, 0, -1, 0, 1]]), -1.0, 1.0) < 0
    assert np.array_equal(b, np.roll(a[:, :, ::-1], 2 * 16 + 1, axis=2))
    # each slice of a 45 degree column is an ellipse of area pi r^2 sqrt(2): site count within 5 %
    assert abs(a[8].sum() * 0.25 / (math.pi * 1.3 ** 2 * math.sqrt(2.0)) - 1.0) < 0.05
    # volume of a tilted capped cylinder / of an ellipsoid on a fine mesh
    pf = O.Params(64, 64, 64, hx=0.125, hy=0.125, hz=0.125, bc=(O_, O_, O_))
    cyl = O.epsilon_from_shapes(pf, np.array([[2, 4.0, 4.0, 4.0, 1.5, 2.0, 0, 1.0, 2.0, -0.5]]), -1.0, 1.0) < 0
    assert abs(cyl.sum() * 0.125 ** 3 / (math.pi * 1.5 ** 2 * 4.0) - 1.0) < 0.01
    ell = O.epsilon_from_shapes(pf, np.array([[1, 4.0, 4.0, 4.0, 3.0, 1.5, 2.5, 0, 0, 0]]), -1.0, 1.0) < 0
    assert abs(ell.sum() * 0.125 ** 3 / (4.0 / 3.0 * math.pi * 3.0 * 1.5 * 2.5) - 1.0) < 0.01
    # point symmetry about a centre that sits on a site
    c = O.epsilon_from_shapes(pf, np.array([[2, 4.0, 4.0, 4.0, 1.1, 1.7, 0, 0.3, -1.0, 0.8]]), -1.0, 1.0) < 0
    assert np.array_equal(c[1:, 1:, 1:], c[1:, 1:, 1:][::-1, ::-1, ::-1])


# ------------------------------------------------------------------------------------------------
# single-sweep amplification of the checkerboard mode
# ------------------------------------------------------------------------------------------------
def test_single_sweep_checkerboard_amplification_factor():
    # Eq. (33) with x^0 = psi^-: one sweep gives x^1 = [psi (2 - d) + h_t nsum(psi)]/d.  For a small
    # checkerboard psi = delta (-1)^(i+j+k): nsum = -2 (c_x + c_y + c_z) psi and d = 1 + (h_t/2)(2 sum c - eps),
    # so the per-step factor is [(2 - d) - 2 h_t sum c]/d = -1.186 at h = 0.5, h_t = 0.1, eps = 1, although
    # the exact Crank-Nicolson factor (1 + q)/(1 - q), q = (h_t/2)(eps - 4 sum c) = -2.35, is -0.403.
    p = O.Params(8, 8, 8, solve_mu=False)
    k_, j_, i_ = np.meshgrid(np.arange(8), np.arange(8), np.arange(8), indexing="ij")
    cb = (-1.0) ** (i_ + j_ + k_)
    eps = np.ones(p.shape)
    sc = p.cx + p.cy + p.cz
    d = 1 + p.ht / 2 * (2 * sc - 1.0)
    one_sweep = ((2 - d) - 2 * p.ht * sc) / d
    assert abs(one_sweep + 1.186) < 1e-3
    st = O.State(psi=1e-9 * cb.astype(np.complex128), mu=np.zeros(p.shape))
    O.step(p, st, eps, 0.0, 0.0, 0.0, fixed_sweeps=1)
    assert np.max(np.abs(st.psi / (1e-9 * cb) - one_sweep)) < 1e-9
    q = p.ht / 2 * (1.0 - 4 * sc)
    st = O.State(psi=1e-9 * cb.astype(np.complex128), mu=np.zeros(p.shape))
    O.step(p, st, eps, 0.0, 0.0, 0.0, fixed_sweeps=400)
    assert np.max(np.abs(st.psi / (1e-9 * cb) - (1 + q) / (1 - q))) < 1e-9


# ------------------------------------------------------------------------------------------------
# S13: the initial condition psi0 = 1 + a (N(0,1) + i N(0,1)) by Box-Muller on Philox stream 1.
# What the mathematics fixes: Re(psi0) - 1 and Im(psi0) are independent N(0, a^2) deviates, independent
# from site to site.  A dropped factor 2 in -2 ln u1 halves the variance, cos/cos makes the two parts
# identical, the wrong word or stream correlates them with the Langevin stream, a wrong uniform map
# (u1 = 0 reachable, or [0, 1) instead of (0, 1)) breaks finiteness or the tail.
# ------------------------------------------------------------------------------------------------
def _ks_distance_to_normal(x):
    """sup_x |F_n(x) - Phi(x)| of the sample against the standard normal distribution."""
    from scipy.special import ndtr
    xs = np.sort(x)
    n = len(xs)
    cdf = ndtr(xs)
    return float(max(np.max(np.arange(1, n + 1) / n - cdf), np.max(cdf - np.arange(0, n) / n)))


@pytest.mark.parametrize("seed", [0, 12345, (1 << 40) + 99])
def test_S13_initial_state_is_one_plus_complex_gaussian(seed):
    amp = 0.01
    p = O.Params(64, 64, 64, seed=seed)                      # 2^18 sites
    st = O.initial_state(p, amp)
    n = p.n_sites
    assert st.psi.shape == p.shape and st.psi.dtype == np.complex128
    assert np.all(st.mu == 0.0) and st.K == 0.0 and st.n == 0
    g1 = (st.psi.real.ravel() - 1.0) / amp
    g2 = st.psi.imag.ravel() / amp
    assert np.all(np.isfinite(g1)) and np.all(np.isfinite(g2))
    for g in (g1, g2):
        assert abs(np.mean(g)) < 5.0 / math.sqrt(n)                        # mean 0 +- 5 sigma/sqrt(n)
        assert abs(np.var(g) - 1.0) < 0.01                                 # variance a^2 within 1 %
        assert abs(np.mean(g ** 3)) < 5.0 * math.sqrt(15.0 / n)            # skewness 0 (Var g^3 = 15)
        assert abs(np.mean(g ** 4) - 3.0) < 5.0 * math.sqrt(96.0 / n)      # kurtosis 3 (Var g^4 = 96)
        assert _ks_distance_to_normal(g) < 2.5 / math.sqrt(n)              # P(sqrt(n) D > 2.5) = 7e-6
    assert abs(np.mean(g1 * g2)) < 5.0 / math.sqrt(n)                      # the two parts are uncorrelated
    assert abs(np.mean(g1 * g1 * g2 * g2) - 1.0) < 5.0 * math.sqrt(8.0 / n)   # ... and independent (E = 1, Var = 8)
    for g in (g1, g2):                                                     # neighbouring sites are uncorrelated
        assert abs(np.mean(g[:-1] * g[1:])) < 5.0 / math.sqrt(n)
    # radius and angle separately: |g|^2 = -2 ln u1 is chi^2 with 2 degrees of freedom (mean 2, variance 4),
    # the angle is uniform on the circle
    r2 = g1 * g1 + g2 * g2
    assert abs(np.mean(r2) - 2.0) < 5.0 * 2.0 / math.sqrt(n)
    ang = np.arctan2(g2, g1)
    assert abs(np.mean(np.cos(ang))) < 5.0 / math.sqrt(2 * n) and abs(np.mean(np.sin(2 * ang))) < 5.0 / math.sqrt(2 * n)
    # the largest radius 23 random bits allow: u1 >= 2^-24  =>  |g| <= sqrt(48 ln 2) = 5.77
    assert 3.5 < np.max(np.sqrt(r2)) <= math.sqrt(48.0 * math.log(2.0))
    # a different key gives a different field; the Langevin stream (stream 0) is not reused (S11: stream 1)
    other = O.initial_state(O.Params(64, 64, 64, seed=seed + 1), amp).psi
    assert abs(np.mean(((other.real.ravel() - 1.0) / amp) * g1)) < 5.0 / math.sqrt(n)
    pn = O.Params(64, 64, 64, seed=seed, temperature=1e-3)
    z = O.langevin_noise(pn, 0).ravel() / O.zeta_max(pn)
    assert abs(np.mean(z.real * g1)) < 5.0 / math.sqrt(3 * n) * 1.2 and abs(np.mean(z.imag * g2)) < 5.0 / math.sqrt(3 * n) * 1.2


def test_S11_langevin_pair_by_hand_from_the_known_answer_vector():
    """Reading S11': one Philox call per site pair.  Seed 0, step 0, pair (0, 1): counter (0, 0, 0, 0), key (0, 0) is the
    first published known-answer vector (tests/golden/philox4x32_10_kat.txt): 6627e8d5 e169c58d bc57ac4c 9b00dbd8.
    Site 0 takes the first two words, site 1 the last two; r = ((x >> 9) + 1/2) 2^-22 - 1."""
    p = O.Params(4, 2, 2, seed=0, temperature=1e-3)
    z = O.langevin_noise(p, 0).ravel() / O.zeta_max(p)
    r = [((w >> 9) + 0.5) / 4194304.0 - 1.0 for w in (0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8)]
    assert abs(z[0] - complex(r[0], r[1])) < 1e-15 and abs(z[1] - complex(r[2], r[3])) < 1e-15   # (one product, one quotient)
    # the next pair is another counter: sites 2, 3 come from the call with counter word 0 = 2
    from oracle import philox
    w = [int(v) for v in philox.philox4x32_10(2, 0, 0, 0, 0, 0)]
    r = [((v >> 9) + 0.5) / 4194304.0 - 1.0 for v in w]
    assert abs(z[2] - complex(r[0], r[1])) < 1e-15 and abs(z[3] - complex(r[2], r[3])) < 1e-15
    # step and seed enter as counter word 2 and as the key
    w = [int(v) for v in philox.philox4x32_10(6, 0, 9, 0, 77, 1)]
    p2 = O.Params(4, 2, 2, seed=(1 << 32) + 77, temperature=1e-3)
    z2 = O.langevin_noise(p2, 9).ravel() / O.zeta_max(p2)
    assert abs(z2[7] - complex(((w[2] >> 9) + 0.5) / 4194304.0 - 1.0, ((w[3] >> 9) + 0.5) / 4194304.0 - 1.0)) < 1e-15


def test_S11_langevin_field_is_white():
    """Eq. (38)-(39): <zeta> = 0, <zeta_m zeta*_m'> = (2/3) zeta_max^2 delta_mm' delta_tt'; both components uniform in
    (-zeta_max, zeta_max); nothing correlates -- not the two components of a site, not the two sites of a Philox pair,
    not neighbouring pairs, rows, or steps."""
    p = O.Params(64, 64, 64, seed=7, temperature=1e-3)
    n = p.n_sites
    z = O.langevin_noise(p, 3).ravel() / O.zeta_max(p)
    a, b = z.real, z.imag
    tol = 5.0 / 3.0 / math.sqrt(n)                                         # 5 sigma of a mean of products of U(-1,1) pairs
    for c in (a, b):
        assert abs(c.mean()) < 5.0 / math.sqrt(3 * n)
        assert abs((c ** 2).mean() - 1.0 / 3.0) < 5.0 * math.sqrt(4.0 / 45.0 / n)
        assert abs((c ** 4).mean() - 0.2) < 5.0 * math.sqrt((1.0 / 9.0 - 1.0 / 25.0) / n)
        assert np.max(np.abs(c)) < 1.0
        assert abs(np.mean(c[0::2] * c[1::2])) < tol * math.sqrt(2)     # the two sites of a pair
        assert abs(np.mean(c[1:-1:2] * c[2::2])) < tol * math.sqrt(2)   # neighbouring pairs
        assert abs(np.mean(c[:-64] * c[64:])) < tol                        # neighbouring rows
        hist = np.histogram(c, bins=32, range=(-1, 1))[0]
        assert np.max(np.abs(hist - n / 32)) < 5.0 * math.sqrt(n / 32)
    assert abs(np.mean(a * b)) < tol
    assert abs(np.mean(a[0::2] * b[1::2])) < tol * math.sqrt(2) and abs(np.mean(b[0::2] * a[1::2])) < tol * math.sqrt(2)
    assert abs(np.mean(a[0::2] ** 2 * a[1::2] ** 2) - 1.0 / 9.0) < 5.0 * math.sqrt(2.0 / n) * 0.2   # independence, not just no correlation
    z4 = O.langevin_noise(p, 4).ravel() / O.zeta_max(p)
    assert abs(np.mean(z.real * z4.real)) < tol and abs(np.mean(z.imag * z4.imag)) < tol
    assert abs(np.mean(np.abs(z) ** 2) - 2.0 / 3.0) < 5.0 * math.sqrt(2 * 4.0 / 45.0 / n)


def test_S13_box_muller_two_sites_by_hand():
    """Sites m = 0, 1 of seed 0, evaluated by hand from the Philox words (whose generator is pinned by the
    published known-answer vectors): u = ((x >> 9) + 1/2) 2^-23, g1 + i g2 = sqrt(-2 ln u1) e^{2 pi i u2}."""
    from oracle import philox
    p = O.Params(2, 2, 2, seed=0)
    psi = O.initial_state(p, 0.01).psi.ravel()
    for m in (0, 1):
        x0, x1, _, _ = (int(w) for w in philox.philox4x32_10(m, 0, 0, 1, 0, 0))     # counter (m_lo, m_hi, step 0, stream 1)
        u1 = ((x0 >> 9) + 0.5) / 8388608.0
        u2 = ((x1 >> 9) + 0.5) / 8388608.0
        assert 0.0 < u1 < 1.0 and 0.0 < u2 < 1.0
        rad = math.sqrt(-2.0 * math.log(u1))
        want = complex(1.0 + 0.01 * rad * math.cos(2.0 * math.pi * u2), 0.01 * rad * math.sin(2.0 * math.pi * u2))
        assert abs(psi[m] - want) < 1e-15
    # the known-answer words themselves through the same map: counter 0, key 0 -> 6627e8d5 e169c58d (golden file)
    g = O.box_muller(np.array([0x6627e8d5], np.uint32), np.array([0xe169c58d], np.uint32))[0]
    u1, u2 = ((0x6627e8d5 >> 9) + 0.5) / 8388608.0, ((0xe169c58d >> 9) + 0.5) / 8388608.0
    assert abs(abs(g) ** 2 + 2.0 * math.log(u1)) < 1e-14                 # |g|^2 = -2 ln u1
    assert abs(math.atan2(g.imag, g.real) % (2 * math.pi) - 2 * math.pi * u2) < 1e-14


# ------------------------------------------------------------------------------------------------
# R3: what single precision does to the paper's rule on C1 (BASELINE.json configs[0]), WITHOUT the CUDA path.
# The oracle's own functions run in complex64 (fp32 psi, mu, eps and link variables; fp64 scalars K, J_av as
# in the library).  C1 relaxes into the single-sweep regime (criterion (34) met after one sweep, rule S8); there
# the band around the checkerboard mode is amplified by 1.186 per step (pin above), fp32 rounding noise grows to
# the tolerance level |r| = 1e-3, and criterion (34) itself then asks for a second sweep on a few steps.  The
# fp32-vs-fp64 difference after 100 steps is therefore set by the tolerance, not by fp32 rounding: about 1e-5
# in relative L2, on either side of BASELINE.json's 1e-5 depending on the seed.  At eps_tol = 1e-10 (no
# single-sweep steps) the same fp32 run stays below 2e-6.
# ------------------------------------------------------------------------------------------------
def _c1_run(dtype, seed, eps_tol, counts=None, nsteps=100):
    import tdgl_inputs as I
    cfg = I.CONFIGS["C1"]
    f32 = lambda v: float(np.float32(v))
    p = O.Params(cfg.nx, cfg.ny, cfg.nz, hx=f32(cfg.h), hy=f32(cfg.h), hz=f32(cfg.h), dt=f32(cfg.dt), bc=tuple(cfg.bc),
                 eps_tol=f32(eps_tol), max_sweeps=200)
    bx, bz = cfg.requested_field()
    Bx, Bz, _, nzq = O.snap_field(p, f32(bx), f32(bz))
    assert nzq == 4
    psi0 = I.initial_psi(cfg, seed=seed)                                   # fp32 values on both sides
    real = np.float32 if dtype == np.complex64 else np.float64
    st = O.State(psi=psi0.astype(dtype), mu=np.zeros(p.shape, real))
    O.run(p, st, np.ones(p.shape, real), Bx, Bz, 0.0, nsteps, sweep_counts=counts)
    assert st.psi.dtype == dtype and st.mu.dtype == real
    return p, st


def _rel_l2(a, b):
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


def test_R3_single_precision_deviation_on_C1_without_cuda():
    rels = []
    for seed in (0, 1, 3):
        p, s64 = _c1_run(np.complex128, seed, 1e-6)
        _, s32 = _c1_run(np.complex64, seed, 1e-6)
        # (i) the single-sweep regime: from about step 33 on the fp64 run accepts every step after ONE sweep
        first1 = s64.sweep_log.index(1)
        assert 25 <= first1 <= 45 and all(c == 1 for c in s64.sweep_log[first1:])
        # (ii) the fp32 run agrees on every decision before that, and later takes a second sweep on a few steps
        assert s32.sweep_log[:first1] == s64.sweep_log[:first1]
        extra = [n for n, (a, b) in enumerate(zip(s32.sweep_log, s64.sweep_log)) if a != b]
        assert 1 <= len(extra) <= 8 and all(s32.sweep_log[n] == 2 and n > first1 + 20 for n in extra)
        # each such decision is forced by criterion (34): the fp32 residual of the first sweep is above eps_tol
        for n in extra:
            assert s32.resid_trace[n][0] >= p.eps_tol > s32.resid_trace[n][1]
        # (iii) against the fp64 oracle replaying the fp32 run's counts (S9)
        _, rep = _c1_run(np.complex128, seed, 1e-6, counts=s32.sweep_log)
        rel = _rel_l2(s32.psi, rep.psi)
        assert np.max(np.abs(s32.psi - rep.psi)) <= 1e-4                   # BASELINE.json's max-norm gate holds
        assert 5e-6 < rel < 2e-5
        rels.append(rel)
    assert max(rels) > 1e-5                                                # ... the rel-L2 gate of 1e-5 does not, for some seeds
    # (iv) the same fp32 arithmetic away from the single-sweep regime
    _, t64 = _c1_run(np.complex128, 0, 1e-10)
    _, t32 = _c1_run(np.complex64, 0, 1e-10)
    assert min(t64.sweep_log) >= 3
    assert _rel_l2(t32.psi, t64.psi) < 2e-6 and np.max(np.abs(t32.psi - t64.psi)) < 1e-5


# ------------------------------------------------------------------------------------------------
# The paper's own mu solver (Eq. 40; readings S5, S20): pseudo-time relaxation + Crank-Nicolson + Jacobi
# ------------------------------------------------------------------------------------------------
def _assemble_N(p, h_tau):
    """Dense N from the printed entries: N_mm = 1 + h_tau sum c, N_{m,m+-alpha} = -h_tau c_alpha/2;
    periodic wrap, and on an open face the single neighbour's entry doubles (mirror ghost, S6/S21)."""
    n = p.n_sites
    N = np.zeros((n, n))
    idx = lambda i, j, k: i + p.nx * (j + p.ny * k)
    dims = (p.nx, p.ny, p.nz)
    cs = (p.cx, p.cy, p.cz)
    for k in range(p.nz):
        for j in range(p.ny):
            for i in range(p.nx):
                m = idx(i, j, k)
                N[m, m] += 1.0 + h_tau * sum(cs)
                pos = [i, j, k]
                for a in range(3):
                    for sgn in (+1, -1):
                        q = list(pos)
                        q[a] += sgn
                        if q[a] < 0 or q[a] >= dims[a]:
                            if p.bc[a] == O_:
                                q[a] = pos[a] - sgn            # mirror ghost
                            else:
                                q[a] %= dims[a]
                        N[m, idx(*q)] += -0.5 * h_tau * cs[a]
    return N


@pytest.mark.parametrize("bc", [(P_, P_, P_), (P_, P_, O_), (O_, O_, O_), (O_, P_, O_)])
def test_Eq40_one_pseudo_time_step_is_the_dense_solve_of_N_mu_equals_c(bc):
    p = O.Params(6, 5, 4, hx=0.5, hy=0.4, hz=0.6, g=1.2, bc=bc)
    rng = np.random.default_rng(3)
    w = O.site_weights(p)
    rho = rng.standard_normal(p.shape)
    rho -= np.sum(w * rho) / np.sum(w)
    mu0 = 0.3 * rng.standard_normal(p.shape)
    h_tau = 0.7
    N = _assemble_N(p, h_tau)
    # c from the printed formula with the stable sign (S5): mu^- + h_tau [ (Delta_h mu^-)/2 - rho ]
    c = mu0 + h_tau * (0.5 * O.laplacian_real(p, mu0) - rho)
    want = np.linalg.solve(N, c.ravel()).reshape(p.shape)
    got, log = O.solve_poisson_pseudotime(p, rho, mu0, h_tau=h_tau, eps_in=1e-30, max_inner=5000, max_outer=1)
    assert len(log) == 1 and np.max(np.abs(got - want)) < 1e-12
    # N = I - (h_tau/2) Delta_h, strictly diagonally dominant: every row sums to 1
    assert np.allclose(N.sum(axis=1), 1.0) and np.all(np.diag(N) > np.sum(np.abs(N), axis=1) - np.diag(N))
    assert np.max(np.abs((N @ mu0.ravel()).reshape(p.shape) - (mu0 - 0.5 * h_tau * O.laplacian_real(p, mu0)))) < 1e-12
    # the replay of prescribed inner counts runs exactly those
    got2, log2 = O.solve_poisson_pseudotime(p, rho, mu0, h_tau=h_tau, inner_counts=[3, 2])
    assert [l[0] for l in log2] == [3, 2]


@pytest.mark.parametrize("bc", [(P_, P_, P_), (P_, P_, O_), (O_, O_, O_)])
def test_Eq40_fixed_point_is_the_direct_solve(bc):
    p = O.Params(8, 8, 8, bc=bc)
    rng = np.random.default_rng(5)
    w = O.site_weights(p)
    rho = rng.standard_normal(p.shape)
    rho -= np.sum(w * rho) / np.sum(w)
    ref = O.solve_poisson(p, rho)
    mu, log = O.solve_poisson_pseudotime(p, rho, np.zeros(p.shape), h_tau=1.0, eps_mu=1e-26, eps_in=1e-28, max_outer=2000,
                                         max_inner=5000)
    assert len(log) < 2000
    assert np.max(np.abs(mu - ref)) < 1e-10
    assert abs(np.sum(w * mu)) < 1e-10                       # the weighted mean of the start value is conserved (S7)
    # the paper's tolerance (eps_mu = 1e-6) stops early: |Delta_h mu - rho| ~ 1e-3, still the same field to ~1e-3
    mu6, log6 = O.solve_poisson_pseudotime(p, rho, np.zeros(p.shape))
    assert len(log6) < len(log) and np.max(np.abs(O.laplacian_real(p, mu6) - rho)) < 5e-2
    assert max(l[0] for l in log6) <= 12                     # h_tau = 0.1: N is as dominant as M, a handful of sweeps


def test_S5_the_printed_sign_has_no_fixed_point():
    """As printed c_m = mu^- + h_tau [ -(Delta_h mu^-)/2 + rho ] with N = I - (h_tau/2) Delta_h: at the
    solution of Delta_h mu = rho the printed equation N mu = c is violated by exactly h_tau rho (it holds only for
    rho = 0), whereas the stable-sign c of reading S5 satisfies it."""
    p = O.Params(8, 8, 8)
    rng = np.random.default_rng(7)
    rho = rng.standard_normal(p.shape)
    rho -= rho.mean()
    mu = O.solve_poisson(p, rho)
    h_tau = 0.9
    Nmu = mu - 0.5 * h_tau * O.laplacian_real(p, mu)
    c_printed = mu + h_tau * (-0.5 * O.laplacian_real(p, mu) + rho)
    c_stable = mu + h_tau * (0.5 * O.laplacian_real(p, mu) - rho)
    assert np.max(np.abs(Nmu - c_stable)) < 1e-12
    assert np.max(np.abs((Nmu - c_printed) + h_tau * rho)) < 1e-12 and np.max(np.abs(Nmu - c_printed)) > 0.1


# ------------------------------------------------------------------------------------------------
# S25: insulating inclusions = cut links (P:511 (ii): "no-current (open) boundary conditions across internal grid edges")
# ------------------------------------------------------------------------------------------------
def _mask_with_holes(p, seed):
    """A cuboid hole, an L-shaped hole (re-entrant corners) and a few single removed sites; never the whole of a row."""
    rng = np.random.default_rng(seed)
    m = np.ones(p.shape, bool)
    m[2:5, 1:4, 3:6] = False
    m[5:7, 4:7, 0:2] = False
    m[6:7, 6:8, 0:4] = False
    for _ in range(6):
        m[tuple(rng.integers(0, n) for n in p.shape)] = False
    return m


def _site_terms(p, i, j, k, K, Bx, Bz):
    """The six neighbour terms of site (i, j, k) of the paper's operator, as (neighbour index, factor, c_alpha): the value
    (S+-_alpha psi)_m = factor * psi[neighbour].  Written out from P:272-276 (Eq. 29a), P:449-455 (jump), P:471-505 (open
    faces: S- := S+ at the first site, S+ := S- at the last) site by site -- independently of the oracle's array code."""
    Ly = p.length("y")
    ybar = j * p.hy - Ly / 2
    Ux = np.exp(1j * p.hx * (K + Bz * ybar))
    Uz = np.exp(-1j * p.hz * Bx * ybar)
    Pik = np.exp(1j * (i * p.hx * Ly * Bz - k * p.hz * Ly * Bx))
    out = []
    n = (p.nx, p.ny, p.nz)
    pos = (i, j, k)
    for a, (U, c) in enumerate(((Ux, p.cx), (1.0, p.cy), (Uz, p.cz))):
        fw = list(pos); fw[a] += 1
        bw = list(pos); bw[a] -= 1
        tf, tb = (tuple(fw), U), (tuple(bw), np.conj(U))
        if p.bc[a] == P_:
            if fw[a] == n[a]:
                fw[a] = 0
                tf = (tuple(fw), U * (np.conj(Pik) if a == 1 else 1.0))
            if bw[a] < 0:
                bw[a] = n[a] - 1
                tb = (tuple(bw), np.conj(U) * (Pik if a == 1 else 1.0))
        else:
            if bw[a] < 0:
                tb = tf                                        # S- := S+
            if fw[a] == n[a]:
                tf = tb                                        # S+ := S-
        out += [(tf[0], tf[1], c), (tb[0], tb[1], c)]
    return out


def dense_M_cut(p, psi_prev, mu, eps, K, Bx, Bz, mask):
    """Dense M of the implicit step with insulating inclusions: every term whose neighbour is a removed site is
    dropped from the row AND from the diagonal's sum over links; rows of removed sites are the identity."""
    N = p.n_sites
    M = np.zeros((N, N), dtype=np.complex128)
    idx = lambda i, j, k: i + p.nx * (j + p.ny * k)
    ht = p.ht
    for k in range(p.nz):
        for j in range(p.ny):
            for i in range(p.nx):
                m = idx(i, j, k)
                if not mask[k, j, i]:
                    M[m, m] = 1.0
                    continue
                diag = abs(psi_prev[k, j, i]) ** 2 + 1j * p.u * mu[k, j, i] - eps[k, j, i]
                for (ii, jj, kk), fac, c in _site_terms(p, i, j, k, K, Bx, Bz):
                    if mask[kk, jj, ii]:
                        M[m, idx(ii, jj, kk)] += -(ht / 2) * c * fac
                        diag += c
                M[m, m] = 1 + (ht / 2) * diag
    return M


@pytest.mark.parametrize("bc", [(P_, P_, P_), (P_, P_, O_), (O_, O_, O_), (O_, P_, P_)])
def test_S25_implicit_step_with_cut_links_dense_solve(bc):
    mask = _mask_with_holes(O.Params(8, 8, 8), 3)
    p = O.Params(8, 8, 8, hx=0.5, hy=0.55, hz=0.45, g=1.1, u=1.7, bc=bc, eps_tol=1e-28, max_sweeps=5000, solve_mu=False,
                 sc_mask=mask)
    Bx, Bz, _, _ = O.snap_field(p, 0.12, 0.35)
    K = 0.21 if bc[0] == P_ else 0.0
    rng = np.random.default_rng(4)
    psi0 = (1.0 + 0.4 * rand_psi(p, 7)) * mask
    mu0 = rng.uniform(-0.2, 0.2, p.shape) * mask
    eps = np.where(rng.uniform(size=p.shape) < 0.3, -1.0, 1.0)
    # without holes the site-by-site assembly is the printed matrix (the function of the P9 pin)
    pfull = O.Params(8, 8, 8, hx=0.5, hy=0.55, hz=0.45, g=1.1, u=1.7, bc=bc)
    full = np.ones(p.shape, bool)
    assert np.max(np.abs(dense_M_cut(pfull, psi0, mu0, eps, K, Bx, Bz, full) - dense_M(pfull, psi0, mu0, eps, K, Bx, Bz))) < 1e-14
    M = dense_M_cut(p, psi0, mu0, eps, K, Bx, Bz, mask)
    b_dense = 2 * psi0.ravel() - M @ psi0.ravel()
    links = O.paper_links(p, K, Bx, Bz)
    b, d = O.build_system(p, psi0, mu0, eps, links)
    sc = mask.ravel()
    assert np.max(np.abs(b.ravel() - b_dense)[sc]) < 1e-13 and np.max(np.abs(b.ravel()[~sc])) == 0.0
    assert np.max(np.abs(d.ravel() - np.diag(M))[sc]) < 1e-15
    off = np.sum(np.abs(M), axis=1) - np.abs(np.diag(M))
    assert np.all(np.abs(np.diag(M)) > off)                              # still strictly diagonally dominant
    x_dense = np.linalg.solve(M, b_dense)
    st = O.State(psi=psi0.copy(), mu=mu0.copy(), K=K)
    O.step(p, st, eps, Bx, Bz, 0.0)
    assert np.max(np.abs(st.psi.ravel() - x_dense)) < 1e-12
    assert np.all(st.psi[~mask] == 0.0)                                  # removed sites stay empty


@pytest.mark.parametrize("bc", ALL_BC)
def test_S25_cut_links_conserve_current_and_the_operator_is_hermitian(bc):
    """With cut links the covariant Laplacian is Hermitian in the weighted inner product (the mirror rule applied at
    the re-entrant corners of a voxelised hole would not be), so the weighted sum of rho = div j_s vanishes exactly:
    the Neumann problem for mu stays solvable.  And div(j_s + j_n) = rho - Delta_h mu on the links that exist (P7)."""
    mask = _mask_with_holes(O.Params(8, 8, 8), 5)
    p = O.Params(8, 8, 8, hx=0.5, hy=0.4, hz=0.6, g=1.2, bc=bc, sc_mask=mask)
    Bx, Bz, _, _ = O.snap_field(p, 0.1, 0.3)
    links = O.paper_links(p, 0.2 if bc[0] == P_ else 0.0, Bx, Bz)
    w = O.site_weights(p)
    f, g_ = rand_psi(p, 1) * mask, rand_psi(p, 2) * mask
    lhs = np.sum(w * np.conj(f) * O.covariant_laplacian(p, g_, links))
    rhs = np.sum(w * np.conj(O.covariant_laplacian(p, f, links)) * g_)
    assert abs(lhs - rhs) < 1e-11
    rho = O.supercurrent_divergence(p, f, links)
    assert abs(np.sum(w * rho)) < 1e-12 and np.all(rho[~mask] == 0.0)
    # discrete divergence of the link currents = rho - Delta_h mu, site by site (open faces: weight 1/2 doubles the link)
    mu = np.random.default_rng(3).standard_normal(p.shape) * mask
    js = O.link_supercurrents(p, f, links)
    div = np.zeros(p.shape)
    for a, axis, h, c in ((0, 2, p.hx, p.cx), (1, 1, p.hy, p.cy), (2, 0, p.hz, p.cz)):
        exist = (mask & np.roll(mask, -1, axis)).astype(float)
        if p.bc[a] == O_:
            sl = [slice(None)] * 3
            sl[axis] = -1
            exist[tuple(sl)] = 0.0
        gg = p.g ** 2 if a == 2 else 1.0
        jn = -(np.roll(mu, -1, axis) - mu) / (h * gg) * exist
        flux = (js[a] + jn) / h                                          # through the forward link
        wa = np.ones(p.shape)
        if p.bc[a] == O_:
            sl = [slice(None)] * 3
            sl[axis] = 0
            wa[tuple(sl)] = 0.5
            sl[axis] = -1
            wa[tuple(sl)] = 0.5
        div += (flux - np.roll(flux, 1, axis)) / wa
    assert np.max(np.abs(div - (rho - O.laplacian_real(p, mu)))[mask]) < 1e-11


def test_S25_pseudo_time_solver_with_holes_and_gauge_invariance():
    mask = _mask_with_holes(O.Params(8, 8, 8), 7)
    p = O.Params(8, 8, 8, bc=(P_, P_, O_), sc_mask=mask, mu_solver="pseudotime", h_tau=1.0, eps_mu=1e-26, eps_mu_in=1e-28,
                 mu_max_outer=4000, mu_max_inner=4000, eps_tol=1e-26, max_sweeps=4000)
    Bx, Bz, _, _ = O.snap_field(p, 0.0, 0.3)
    psi0 = nonzero_psi(p, 4) * mask
    eps = np.ones(p.shape)
    # the direct solver refuses; the iteration reaches Delta_h mu = rho on every superconducting site
    with pytest.raises(ValueError):
        O.solve_poisson(p, np.zeros(p.shape))
    st = O.State(psi=psi0.copy(), mu=np.zeros(p.shape), K=0.1)
    O.step(p, st, eps, Bx, Bz, 0.02)
    links = O.paper_links(p, st.K, Bx, Bz)
    res = O.laplacian_real(p, st.mu) - O.supercurrent_divergence(p, st.psi, links)
    assert np.max(np.abs(res[mask])) < 1e-10 and np.all(st.mu[~mask] == 0.0) and np.all(st.psi[~mask] == 0.0)
    assert abs(np.sum(O.site_weights(p) * st.mu)) < 1e-10
    # gauge invariance (P8) with holes: psi -> psi e^{i chi}, th(m) -> th(m) + chi(m) - chi(m + alpha)
    chi = np.random.default_rng(9).uniform(-3, 3, p.shape)

    def gauged(K):
        thx, thy, thz = O.paper_links(p, K, Bx, Bz)
        return (thx + chi - np.roll(chi, -1, 2), thy + chi - np.roll(chi, -1, 1), thz + chi - np.roll(chi, -1, 0))
    st2 = O.State(psi=psi0 * np.exp(1j * chi), mu=np.zeros(p.shape), K=0.1)
    O.step(p, st2, eps, Bx, Bz, 0.02, links_fn=gauged)
    assert np.max(np.abs(np.abs(st2.psi) - np.abs(st.psi))) < 1e-11
    assert np.max(np.abs(st2.mu - st.mu)) < 1e-9 and abs(st2.K - st.K) < 1e-12
    F1 = O.free_energy(p, st.psi, eps, links)
    F2 = O.free_energy(p, st2.psi, eps, gauged(st2.K))
    assert abs(F1 - F2) < 1e-10 * abs(F1)
