"""`-m gpu`: parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (CUDA graph
per step, WHILE node around the sweep, noise, inclusions, current), where a whole oracle step is out of reach.

(1) Sampled pointwise parity: one time step from the seeded initial state (mu = 0, K = 0).  The psi solve is
    local -- Jacobi information travels one site per sweep -- so the fp64 oracle recomputes psi^+ on windows of the
    grid from the window's own seeded inputs (tests/gpu_common.oracle_window_solve, validated against whole-grid
    oracle steps on the CPU in tests/test_window_oracle.py).  Windows sit at the quasi-periodic wraps, on both
    open z faces, across tile (128 x 8) and z-chunk boundaries and at random places.
(2) Properties that hold at any size, on the outputs of that step and of 20 further steps: Eq. (35) and the K
    update evaluated by the oracle's own functions on the returned psi, Delta_h mu = rho on windows, the
    weighted zero mode, and flux quantisation (exactly n_z vortices per slice).
(3) Sampled pointwise parity of a step with LIVE mu and K: step 22 is recomputed by the oracle on the same windows
    from the GPU's own (psi, mu, K) after 21 steps, so that the i u mu psi part of b, d and a non-zero K in U_x are
    compared at full size too.
(4) mu itself (not a local residual, which cannot see a low-mode error): at 256 x 256 x 128, the largest size whose
    whole-grid fp64 solve fits comfortably in host memory, mu of a driven noisy state against oracle.solve_poisson.
C5 is tested in both readings of S14: C5a = the literal "open on all faces" (J = 0), C5b = x periodic (J = 0.01).
"""
import numpy as np
import pytest

import tdgl_inputs as I
from oracle import tdgl_oracle as O
from gpu_common import f32, oracle_params, oracle_window_solve, window_indices

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def bench_solver(cfg):
    """Exactly bench.make_solver (graph mode, eps_tol 1e-6, max_sweeps 100, noise, pinning, field, current)."""
    import bench
    return bench.make_solver(cfg)


def windows_for(cfg, rng, size=(64, 56, 48), nrandom=3):
    if cfg.nz == 1:                                    # film: larger windows in the plane
        size = (160, 160, 1)
    n = (cfg.nx, cfg.ny, cfg.nz)
    per = [b == 0 for b in cfg.bc]
    origins = [(-20, -18, 40),                         # x wrap and y wrap (jump rows j = 0, ny - 1) / the open corner edge
               (n[0] // 2 - 10, -22, n[2] - size[2]),  # y wrap (or open y face) at the top z face
               (118, 3, 0 if not per[2] else -9),      # tile edge in x (i = 128), bottom z face / z wrap
               (n[0] - 30, n[1] // 2 - 3, 20),         # x wrap (or open x face), 8-row tile edges, z-chunk edge (k = 32)
               ]
    if not any(per) and cfg.nz > 1:                    # all open: the two opposite corners and the remaining faces
        origins += [(0, 0, 0), (n[0] - size[0], n[1] - size[1], n[2] - size[2]), (0, n[1] // 2, n[2] // 2),
                    (n[0] // 2, n[1] - size[1], n[2] // 3)]
    if cfg.nz == 1:                                    # film: strip seams (i = 1024 k), row-chunk edges, both wraps
        origins = [(-70, -80, 0), (1024 - 60, n[1] // 2 - 80, 0), (n[0] - 90, 64 - 80, 0), (3 * 1024 - 100, n[1] - 85, 0)]
    for _ in range(nrandom):
        origins.append(tuple(int(rng.integers(0, n[a] - size[a] + 1)) for a in range(3)))
    out = []
    for o in origins:
        idx = [window_indices(o[a], size[a], n[a], per[a]) for a in range(3)]
        out.append(tuple(idx))
    return out


@pytest.mark.parametrize("name,shape", [("C4", (512, 512, 256)), ("C5a", (1024, 1024, 512)), ("C5b", (1024, 1024, 512)),
                                        ("F2D", (8192, 8192, 1))])
def test_full_size_sampled_parity_and_properties(name, shape):
    cfg = I.CONFIGS[name]
    assert (cfg.nx, cfg.ny, cfg.nz) == shape
    p = oracle_params(cfg)
    rng = np.random.default_rng(2024)
    bx_req, bz_req = cfg.requested_field()
    Bx, Bz, _, nzq = O.snap_field(p, f32(bx_req), f32(bz_req))
    psi0 = I.initial_psi(cfg)                                           # seeded, complex64, (nz, ny, nx)
    eps = O.epsilon_from_spheres(p, I.sphere_list(cfg), cfg.eps_in, cfg.eps_out).astype(np.float32)

    s = bench_solver(cfg)
    s.set_state(torch.from_numpy(psi0), None, 0.0)
    # the inclusion mask of the full grid is bit-identical to the oracle's
    assert np.array_equal(s.get_eps().cpu().numpy(), eps)
    s.step(1)
    psi1_t, mu1_t = s.get_psi_mu()
    psi1, mu1 = psi1_t.cpu().numpy(), mu1_t.cpu().numpy()
    counts, resid = s.sweep_log(1)
    sweeps = int(counts[0])
    ob = s.observables()
    assert 3 <= sweeps <= 30 and ob.status == 0

    # (1) sampled pointwise parity of psi^+
    worst, nchecked = 0.0, 0
    for ii, jj, kk in windows_for(cfg, rng):
        sel = np.ix_(kk, jj, ii)
        xw, valid = oracle_window_solve(p, psi0[sel], eps[sel].astype(np.float64), Bx, Bz, 0.0, 0, sweeps, ii, jj, kk)
        assert valid.sum() > 1000
        err = np.abs(psi1[sel][valid] - xw[valid])
        worst = max(worst, float(err.max()))
        nchecked += int(valid.sum())
    assert nchecked > 50000
    print(f"full-size {name}: {sweeps} sweeps, {nchecked} sampled sites, max|dpsi| = {worst:.2e}")
    assert worst < 5e-6, worst                                          # one step, fp32 vs fp64

    # (2a) Eq. (35), E_x and K from the returned psi by the oracle's own functions
    def check_scalars(psi, K_old, ob):
        if p.bc[0] == O.OPEN:                                           # no current, no K with open x (oracle step 5)
            assert ob.Jav == 0.0 and ob.Ex == 0.0 and ob.K == 0.0
            return
        links_x = O.paper_links_at(p, K_old, Bx, Bz, np.arange(p.nx), np.arange(p.ny), np.arange(1))[0][0]
        jav = 0.0
        for k in range(p.nz):                                           # plane by plane: fp64 temporaries stay small
            f = psi[k].astype(np.complex128)[None]
            pk = O.Params(p.nx, p.ny, 1, hx=p.hx, hy=p.hy, hz=p.hz, dt=p.dt, bc=(p.bc[0], p.bc[1], 0))
            jav += O.average_supercurrent(pk, f, (links_x[None], None, None)) * (p.nx * p.ny)
        jav /= p.n_sites
        assert abs(ob.Jav - jav) < 2e-7, (ob.Jav, jav)
        ex = f32(cfg.Jx) - jav
        assert abs(ob.Ex - ex) < 2e-7
        assert abs(ob.K - O.rewind(p, K_old + p.dt * ex)) < 1e-6

    check_scalars(psi1, 0.0, ob)

    # (2b) Poisson: Delta_h mu = rho(psi^+, K^+) on windows, weighted zero mode, (2c) flux quantisation
    def check_mu(psi, mu, K):
        w1 = []                                                         # S7: w = 1/2 on the open faces of every axis
        for a, n in ((0, p.nx), (1, p.ny), (2, p.nz)):
            w = np.ones(n)
            if p.bc[a] == O.OPEN:
                w[0] = w[-1] = 0.5
            w1.append(w)
        wsum = float(np.einsum("kji,k,j,i->", mu.astype(np.float64), w1[2], w1[1], w1[0]))
        mscale = max(float(np.max(np.abs(mu))), 1e-6)
        assert abs(wsum) / (p.n_sites * mscale) < 1e-5
        for ii, jj, kk in windows_for(cfg, rng, nrandom=1):
            sel = np.ix_(kk, jj, ii)
            pw = O.Params(len(ii), len(jj), len(kk), hx=p.hx, hy=p.hy, hz=p.hz, dt=p.dt,
                          bc=tuple(O.OPEN if (p.bc[a] == O.OPEN and (idx[0] == 0 or idx[-1] == n - 1)) else O.PERIODIC
                                   for a, idx, n in ((0, ii, p.nx), (1, jj, p.ny), (2, kk, p.nz))))
            links = O.paper_links_at(p, K, Bx, Bz, ii, jj, kk)
            rho = O.supercurrent_divergence(pw, psi[sel].astype(np.complex128), links)
            lap = O.laplacian_real(pw, mu[sel].astype(np.float64))
            inner = np.zeros(pw.shape, bool)
            if p.nz == 1:
                inner[:, 1:-1, 1:-1] = True
            else:
                inner[1:-1, 1:-1, 1:-1] = True
            if p.bc[2] == O.OPEN and kk[0] == 0:
                inner[0, 1:-1, 1:-1] = True
            if p.bc[2] == O.OPEN and kk[-1] == p.nz - 1:
                inner[-1, 1:-1, 1:-1] = True
            # fp32 mu: the 7-point operator amplifies the error of mu (fp32 transforms: ~1e-6 relative) by 2 sum c = 24
            tol = 5e-5 * (24.0 * mscale + float(np.max(np.abs(rho))))
            assert np.max(np.abs(lap - rho)[inner]) < tol

    check_mu(psi1, mu1, ob.K)
    if nzq is not None:                                                 # x, y periodic: flux quantisation
        assert ob.vortices_per_slice == float(nzq) and (name != "C4" or nzq == 3129)

    s.step(20)
    ob_a = s.observables()
    psi_a, mu_a = s.get_psi_mu()
    psi_a, mu_a = psi_a.cpu().numpy(), mu_a.cpu().numpy()
    s.step(1)
    ob_b = s.observables()
    psi_b, mu_b = s.get_psi_mu()
    psi_b, mu_b = psi_b.cpu().numpy(), mu_b.cpu().numpy()
    check_scalars(psi_b, ob_a.K, ob_b)
    check_mu(psi_b, mu_b, ob_b.K)

    # (3) step 22 with live mu and K: the oracle recomputes it on the windows from the GPU's state after 21 steps
    assert ob_a.steps == 21 and (p.bc[0] == O.OPEN or cfg.Jx == 0.0 or abs(ob_a.K) > 1e-4)
    assert float(np.max(np.abs(mu_a))) > 1e-6
    sweeps_b = int(s.sweep_log(1)[0][0])
    worst_b, nchecked = 0.0, 0
    for ii, jj, kk in windows_for(cfg, rng, nrandom=2):
        sel = np.ix_(kk, jj, ii)
        xw, valid = oracle_window_solve(p, psi_a[sel], eps[sel].astype(np.float64), Bx, Bz, ob_a.K, int(ob_a.steps), sweeps_b,
                                        ii, jj, kk, mu=mu_a[sel])
        worst_b = max(worst_b, float(np.abs(psi_b[sel][valid] - xw[valid]).max()))
        nchecked += int(valid.sum())
    print(f"full-size {name}: step 22 with live mu (max {np.max(np.abs(mu_a)):.2e}) and K = {ob_a.K:.4f}: {sweeps_b} sweeps, "
          f"{nchecked} sampled sites, max|dpsi| = {worst_b:.2e}")
    assert nchecked > 50000 and worst_b < 5e-6, worst_b
    assert (nzq is None or ob_b.vortices_per_slice == float(nzq)) and ob_b.status == 0 and ob_b.steps == 22
    assert 0.0 < ob_b.mean_abs2 < 1.1
    s.close()


@pytest.mark.parametrize("name", ["C3", "C5a", "C5b"])
def test_mu_itself_at_256x256x128(name):
    """(4): mu of a driven, noisy state after 25 steps against the fp64 definition on the WHOLE grid (low modes
    included), at C3's size -- for C3 itself and for the boundary types of C5a / C5b.  Two comparisons: the solver
    on the rho the GPU produced, and the whole path against the oracle's own rho of the GPU's psi."""
    cfg = I.CONFIGS[name].scaled(256, 256, 128)
    p = oracle_params(cfg)
    bx_req, bz_req = cfg.requested_field()
    Bx, Bz, _, _ = O.snap_field(p, f32(bx_req), f32(bz_req))
    s = bench_solver(cfg)
    s.set_state(torch.from_numpy(I.initial_psi(cfg)), None, 0.0)
    s.step(25)
    ob = s.observables()
    psi, mu = s.get_psi_mu()
    rho = s.debug_rho().cpu().numpy()
    psi, mu = psi.cpu().numpy(), mu.cpu().numpy().astype(np.float64)
    ref_same_rho = O.solve_poisson(p, rho.astype(np.float64))
    scale = max(1.0, float(np.max(np.abs(ref_same_rho))))
    e1 = float(np.max(np.abs(mu - ref_same_rho)))
    links = O.paper_links(p, ob.K, Bx, Bz)
    ref = O.solve_poisson(p, O.supercurrent_divergence(p, psi.astype(np.complex128), links))
    e2 = float(np.max(np.abs(mu - ref)))
    print(f"{cfg.name}: max|mu| = {np.max(np.abs(ref)):.3e}, solver error {e1:.2e}, whole path {e2:.2e}, gain {s.mu_gain():.2f}")
    assert e1 < 2e-5 * scale and e2 < 2e-5 * scale
    # the coarse-grained field (8^3 block means: the low modes) agrees as well
    blk = lambda a: a.reshape(16, 8, 32, 8, 32, 8).mean(axis=(1, 3, 5))
    assert np.max(np.abs(blk(mu) - blk(ref))) < 5e-6 * scale
    w = O.site_weights(p)
    assert abs(np.sum(w * mu)) / np.sum(w) < 1e-5 * scale
    s.close()
