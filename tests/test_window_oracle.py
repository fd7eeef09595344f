"""CPU check of the windowed oracle used by the full-size sampled parity test: on a grid small enough for
a whole oracle step, the window result equals the full result at every site the window declares valid."""
import numpy as np
import pytest

import tdgl_inputs as I
from oracle import tdgl_oracle as O
from gpu_common import f32, oracle_params, oracle_window_solve, window_indices


@pytest.mark.parametrize("bc,origin", [((0, 0, 1), (-7, 30, -3)), ((0, 0, 1), (20, -5, 14)), ((0, 0, 0), (35, 35, 10)),
                                       ((1, 1, 1), (-2, 28, 9)), ((0, 1, 1), (10, -4, 0))])
def test_window_equals_full_oracle(bc, origin):
    cfg = I.Config("w", 44, 40, 22, bc, Bz=0.25, Bx=0.07, Jx=0.02, temperature=1e-3, incl_fraction=0.15,
                   incl_rmin=1.5, incl_rmax=2.5, seed=5)
    p = oracle_params(cfg)
    eps = O.epsilon_from_spheres(p, I.sphere_list(cfg), cfg.eps_in, cfg.eps_out)
    Bx, Bz, _, _ = O.snap_field(p, f32(cfg.Bx), f32(cfg.Bz))
    psi0 = I.initial_psi(cfg).astype(np.complex128)
    rng = np.random.default_rng(3)
    mu0 = 0.05 * rng.standard_normal(p.shape)
    K, step, sweeps = 0.31, 4, 6
    links = O.paper_links(p, K, Bx, Bz)
    zeta = O.langevin_noise(p, step)
    b, d = O.build_system(p, psi0, mu0, eps, links, zeta)
    x = psi0
    for _ in range(sweeps):
        x, _ = O.jacobi_sweep(p, x, b, d, links)
    n = (p.nx, p.ny, p.nz)
    ii, jj, kk = (window_indices(origin[a], 26, n[a], bc[a] == 0) for a in range(3))
    sel = np.ix_(kk, jj, ii)
    xw, valid = oracle_window_solve(p, psi0[sel], eps[sel], Bx, Bz, K, step, sweeps, ii, jj, kk, mu=mu0[sel])
    assert valid.sum() > 100
    assert np.max(np.abs(xw[valid] - x[sel][valid])) < 1e-13
    # and the mask is not overly generous: one site inside the artificial margin does differ somewhere
    if (~valid).any():
        assert np.max(np.abs(xw[~valid] - x[sel][~valid])) > 1e-9


def test_noise_and_links_at_match_full_arrays():
    cfg = I.Config("w", 12, 10, 6, (0, 0, 0), Bz=0.3, Bx=0.1, temperature=1e-3, seed=11)
    p = oracle_params(cfg)
    full = O.langevin_noise(p, 7)
    m = np.array([[0, 5], [59, 719]], dtype=np.uint64)
    assert np.array_equal(O.langevin_noise_at(p, 7, m), full.ravel()[m.astype(np.int64)])
    thx, thy, thz = O.paper_links(p, 0.2, 0.1, 0.3)
    ii, jj, kk = np.array([11, 0, 3]), np.array([9, 0]), np.array([5, 2])
    wx, wy, wz = O.paper_links_at(p, 0.2, 0.1, 0.3, ii, jj, kk)
    sel = np.ix_(kk, jj, ii)
    assert np.array_equal(wx, thx[sel]) and np.array_equal(wy, thy[sel]) and np.array_equal(wz, thz[sel])
