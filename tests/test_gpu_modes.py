"""`-m gpu`: the two further modes of the library against the fp64 oracle, through the C ABI.

TDGL_FLAG_MU_ITERATIVE -- the paper's own mu solver (Eq. 40: pseudo-time relaxation, Crank-Nicolson, Jacobi;
readings S5, S20).  It is an iteration stopped by tolerances, so parity follows reading S9: the GPU takes its own
decisions, logs the Jacobi sweep count of every outer iteration, and oracle.solve_poisson_pseudotime replays them.
TDGL_FLAG_FP64 -- the double-precision build (the paper's DP mode): every kernel of the step in fp64,
mu by the pseudo-time iteration in double; parity at the fp64 rounding level.
"""
import math

import numpy as np
import pytest

import tdgl_inputs as I
from oracle import tdgl_oracle as O
from gpu_common import f32, make_solver, oracle_params, rel_l2, setup_pair

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

P_, O_ = I.PERIODIC, I.OPEN
ALL_BC = [(a, b, c) for a in (P_, O_) for b in (P_, O_) for c in (P_, O_)]


def cfg_of(nx, ny, nz, bc, **kw):
    return I.Config(f"m{nx}x{ny}x{nz}", nx, ny, nz, tuple(bc), **kw)


# ---------------------------------------------------------------------------------------------------
# the pseudo-time mu iteration in fp32
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc", ALL_BC)
@pytest.mark.parametrize("shape", [(36, 14, 10), (130, 9, 1)])
def test_mu_iterative_solve_replayed_by_the_oracle(bc, shape):
    nx, ny, nz = shape
    if nz == 1:
        bc = (bc[0], bc[1], P_)
    cfg = cfg_of(nx, ny, nz, bc)
    p = oracle_params(cfg, mu_iterative=True)
    s = make_solver(cfg, mu_iterative=True)
    rng = np.random.default_rng(4)
    w = O.site_weights(p)
    rho = rng.standard_normal(p.shape)
    rho -= np.sum(w * rho) / np.sum(w)
    rho32 = rho.astype(np.float32)
    mu = s.debug_poisson(torch.from_numpy(rho32)).cpu().numpy().astype(np.float64)
    outer, inner = s.mu_log(1)
    assert outer[0] == len(inner[0]) >= 1 and max(inner[0]) <= 30
    ref, log = O.solve_poisson_pseudotime(p, rho32.astype(np.float64), np.zeros(p.shape), p.h_tau, p.eps_mu, p.eps_mu_in,
                                          inner_counts=inner[0])
    scale = max(1.0, float(np.max(np.abs(ref))))
    assert np.max(np.abs(mu - ref)) < 5e-6 * scale
    # the GPU's stopping decision is a valid outcome of criterion P:421 (S9).  From this cold start (white rho, |mu| of
    # order 10) max|d_tau mu|^2 falls by only ~1 % per outer iteration near the threshold, while the fp32 rounding of mu
    # (1e-6) is 1 % of the change per iteration (1e-4): the crossing moves by up to ~10 % of the count.  The GPU's stop
    # index must lie within 15 % of the fp64 oracle's own (or both hit the cap, S20: max_outer = 1000).
    free, flog = O.solve_poisson_pseudotime(p, rho32.astype(np.float64), np.zeros(p.shape), p.h_tau, p.eps_mu, p.eps_mu_in,
                                            max_outer=p.mu_max_outer)
    assert abs(len(flog) - len(log)) <= max(2, 0.15 * len(flog))
    assert len(log) == p.mu_max_outer or log[-1][1] < 2.0 * p.eps_mu
    s.close()


def test_mu_iterative_fixed_point_is_the_direct_solve():
    """Driven to fp32's floor (eps_mu = 1e-11, i.e. |d_tau mu| < 3e-6) the iteration reaches Delta_h mu = rho."""
    cfg = cfg_of(32, 16, 8, (P_, P_, O_))
    p = oracle_params(cfg)
    s = make_solver(cfg, mu_iterative=True)
    s.set_mu_solver(h_tau=1.0, eps_mu=1e-11, eps_in=1e-12, max_outer=5000, max_inner=400)
    rng = np.random.default_rng(5)
    w = O.site_weights(p)
    rho = rng.standard_normal(p.shape)
    rho -= np.sum(w * rho) / np.sum(w)
    rho32 = rho.astype(np.float32)
    mu = s.debug_poisson(torch.from_numpy(rho32)).cpu().numpy().astype(np.float64)
    ref = O.solve_poisson(p, rho32.astype(np.float64))
    assert np.max(np.abs(mu - ref)) < 2e-4 * np.max(np.abs(ref))
    s.close()


@pytest.mark.parametrize("name,shape", [("C2", (32, 32, 32)), ("C4", (48, 40, 24))])
def test_mu_iterative_run(name, shape):
    """30 steps with field, inclusions and current, the GPU taking every decision (psi sweeps, mu outer and inner
    counts); the oracle replays them all.  BASELINE.json's pointwise numbers."""
    cfg = I.CONFIGS[name].scaled(*shape)
    nsteps = 30
    p, st, eps, (Bx, Bz), s = setup_pair(cfg, temperature=0.0, mu_iterative=True)
    s.step(nsteps)
    psi, mu = s.get_psi_mu()
    counts, _ = s.sweep_log(nsteps)
    outer, inner = s.mu_log(nsteps)
    O.run(p, st, eps, Bx, Bz, f32(cfg.Jx), nsteps, sweep_counts=counts, mu_schedule=inner)
    assert np.max(np.abs(psi.cpu().numpy() - st.psi)) <= 1e-4
    assert rel_l2(psi.cpu().numpy(), st.psi) <= 1e-5
    assert np.max(np.abs(mu.cpu().numpy() - st.mu)) <= 1e-4 * max(1.0, np.max(np.abs(st.mu)))
    ob = s.observables()
    assert abs(ob.K - st.K) < 1e-6
    # N is as diagonally dominant as M: a few Jacobi sweeps per outer iteration; warm-started from the previous step the
    # number of outer iterations falls as the state settles (in this 30-step transient from a random state it is still
    # tens per step: a diffusive relaxation with h_tau = 0.1 is a slow Poisson solver, which is why the direct solver
    # is the default)
    assert max(max(i) for i in inner) <= 12 and np.mean(outer[-5:]) < np.mean(outer[:5])
    print(f"{cfg.name}: mu iteration, outer/step {np.mean(outer):.2f}, inner/outer {np.mean([np.mean(i) for i in inner]):.2f}")
    s.close()


# ---------------------------------------------------------------------------------------------------
# the double-precision build
# ---------------------------------------------------------------------------------------------------
def fp64_pair(cfg, psi0, mu0, K0, fixed_sweeps=0, yz=None, eps_tol=1e-6, with_pinning=True):
    """Oracle and fp64 Solver with identical inputs (xz gauge via setup_pair; yz gauge by hand)."""
    if yz is None:
        return setup_pair(cfg, psi0=psi0, mu0=mu0, K0=K0, fixed_sweeps=fixed_sweeps, fp64=True, eps_tol=eps_tol,
                          with_pinning=with_pinning) + (None,)
    from paper_1409_8340_b200 import Solver
    By_req, Bz_req = yz
    p = oracle_params(cfg, fp64=True, eps_tol=eps_tol)
    s = Solver(cfg.nx, cfg.ny, cfg.nz, bc=cfg.bc, h=cfg.h, dt=cfg.dt, eps_tol=eps_tol, fixed_sweeps=fixed_sweeps,
               temperature=cfg.temperature, seed=cfg.seed, gauge_yz=True, fp64=True)
    spheres = I.sphere_list(cfg)
    eps = O.epsilon_from_spheres(p, spheres, cfg.eps_in, cfg.eps_out)
    s.set_pinning(spheres, cfg.eps_in, cfg.eps_out)
    By, Bz, _, _ = O.snap_field_yz(p, f32(By_req), f32(Bz_req))
    s.set_field_current(By=By_req, Bz=Bz_req, Jx=cfg.Jx)
    st = O.State(psi=psi0.astype(np.complex128), mu=mu0.astype(np.float64), K=float(K0))
    s.set_state(torch.from_numpy(psi0), torch.from_numpy(mu0), float(K0))
    return p, st, eps, (By, Bz), s, (lambda K: O.paper_links_yz(p, K, By, Bz))


@pytest.mark.parametrize("bc", ALL_BC)
@pytest.mark.parametrize("gauge", ["xz", "yz"])
def test_fp64_two_steps_fixed_sweeps(bc, gauge):
    cfg = cfg_of(36, 14, 10, bc, Bx=0.05 if gauge == "xz" else 0.0, Bz=0.3, Jx=0.02 if bc[0] == P_ else 0.0,
                 temperature=1e-3, incl_fraction=0.15, incl_rmin=1.0, incl_rmax=2.0, seed=2)
    psi0, mu0 = I.random_state(cfg, seed=21, amp=0.8)
    K0 = 0.11 if bc[0] == P_ else 0.0
    p, st, eps, (B1, Bz), s, links_fn = fp64_pair(cfg, psi0, mu0, K0, fixed_sweeps=5, yz=(0.07, 0.3) if gauge == "yz" else None)
    s.step(2)
    psi, mu = s.get_psi_mu()
    assert psi.dtype == torch.complex128 and mu.dtype == torch.float64
    outer, inner = s.mu_log(2)
    for n in range(2):
        O.step(p, st, eps, B1 if gauge == "xz" else 0.0, Bz, f32(cfg.Jx), fixed_sweeps=5, links_fn=links_fn, mu_inner_counts=inner[n])
    ob = s.observables()
    assert ob.steps == 2 and ob.sweeps_last == 5 and ob.sweeps_total == 10
    assert np.max(np.abs(psi.cpu().numpy() - st.psi)) < 1e-12
    assert np.max(np.abs(mu.cpu().numpy() - st.mu)) < 1e-12 * max(1.0, np.max(np.abs(st.mu)))
    assert abs(ob.K - st.K) < 1e-13 and abs(ob.Ex - st.Ex) < 1e-13 and abs(ob.Jav - st.Jav) < 1e-13
    assert abs(ob.max_resid2 - st.max_resid2) <= 1e-6 * st.max_resid2          # reduced in fp64, reported as fp32
    # the oracle's own decisions on the mu iteration are the GPU's (fp64 on both sides)
    free = O.State(psi=psi0.astype(np.complex128), mu=mu0.astype(np.float64), K=K0)
    O.step(p, free, eps, B1 if gauge == "xz" else 0.0, Bz, f32(cfg.Jx), fixed_sweeps=5, links_fn=links_fn)
    assert [l[0] for l in free.mu_log[0]] == inner[0]
    s.close()


@pytest.mark.parametrize("bc", [(P_, P_, P_), (O_, P_, P_), (P_, O_, P_), (O_, O_, P_)])
def test_fp64_film(bc):
    cfg = cfg_of(132, 21, 1, bc, Bz=0.3, Jx=0.02 if bc[0] == P_ else 0.0, temperature=1e-3, incl_fraction=0.15,
                 incl_rmin=1.0, incl_rmax=2.0, seed=3)
    psi0, mu0 = I.random_state(cfg, seed=7, amp=0.8)
    K0 = 0.2 if bc[0] == P_ else 0.0
    p, st, eps, (Bx, Bz), s, _ = fp64_pair(cfg, psi0, mu0, K0, fixed_sweeps=4)
    s.step(2)
    psi, mu = s.get_psi_mu()
    outer, inner = s.mu_log(2)
    for n in range(2):
        O.step(p, st, eps, Bx, Bz, f32(cfg.Jx), fixed_sweeps=4, mu_inner_counts=inner[n])
    assert np.max(np.abs(psi.cpu().numpy() - st.psi)) < 1e-12
    assert np.max(np.abs(mu.cpu().numpy() - st.mu)) < 1e-12 * max(1.0, np.max(np.abs(st.mu)))
    assert abs(s.observables().K - st.K) < 1e-13
    s.close()


def test_fp64_C1_100_steps():
    """BASELINE.json configs[0] in the double-precision build, both sides taking their own decisions: the sweep counts
    agree on every step and psi agrees to 1e-10 -- the fp32 deviation of reading R3 is a property of single precision."""
    cfg = I.CONFIGS["C1"]
    p, st, eps, (Bx, Bz), s = setup_pair(cfg, fp64=True)
    s.step(100)
    psi, mu = s.get_psi_mu()
    counts, resid = s.sweep_log(100)
    outer, inner = s.mu_log(100)
    O.run(p, st, eps, Bx, Bz, 0.0, 100)
    assert list(counts) == st.sweep_log
    assert [[l[0] for l in step] for step in st.mu_log] == inner
    psi = psi.cpu().numpy()
    print(f"fp64 C1: max|dpsi| = {np.max(np.abs(psi - st.psi)):.2e}, rel-L2 = {rel_l2(psi, st.psi):.2e}")
    assert np.max(np.abs(psi - st.psi)) <= 1e-10 and rel_l2(psi, st.psi) <= 1e-11
    assert np.max(np.abs(mu.cpu().numpy() - st.mu)) <= 1e-11
    ob = s.observables()
    assert ob.vortices_per_slice == 4.0 and ob.steps == 100
    s.close()


def test_fp64_noise_initial_state_and_observables():
    cfg = cfg_of(32, 24, 10, (P_, P_, O_), Bx=0.04, nz_flux=3, temperature=2e-3, incl_fraction=0.1, incl_rmin=1.0,
                 incl_rmax=2.0, seed=77)
    p = oracle_params(cfg, fp64=True)
    s = make_solver(cfg, fp64=True)
    # initial condition (S13) and Langevin term (S11) in double
    psi, mu = s.get_psi_mu()
    assert np.max(np.abs(psi.cpu().numpy() - O.initial_state(p, f32(cfg.init_amp)).psi)) < 1e-15
    assert float(mu.abs().max()) == 0.0
    z = s.debug_noise(9).cpu().numpy()
    assert np.max(np.abs(z - O.langevin_noise(p, 9))) < 1e-16
    s.close()
    rng = np.random.default_rng(8)
    shape = (cfg.nz, cfg.ny, cfg.nx)
    psi0 = ((1.0 + 0.4 * rng.uniform(-1, 1, shape)) * np.exp(1j * rng.uniform(-math.pi, math.pi, shape))).astype(np.complex64)
    p, st, eps, (Bx, Bz), s = setup_pair(cfg, psi0=psi0, K0=0.2, fp64=True)
    ob = s.observables()
    links = O.paper_links(p, st.K, Bx, Bz)
    F = O.free_energy(p, st.psi, eps, links)
    assert abs(ob.free_energy - F) < 1e-12 * abs(F)
    assert abs(ob.mean_abs2 - O.mean_abs2(st.psi)) < 1e-14
    assert ob.vortices_per_slice == O.vortices_per_slice(p, st.psi, links, Bz) == 3.0
    rho = s.debug_rho().cpu().numpy()
    assert np.max(np.abs(rho - O.supercurrent_divergence(p, st.psi, links))) < 1e-12
    s.close()


def test_mode_flags_are_validated():
    from paper_1409_8340_b200 import Solver
    from paper_1409_8340_b200.binding import TdglError
    with pytest.raises(TdglError):
        Solver(16, 8, 4, mu_iterative=True, mu_refine=True)       # refinement belongs to the direct solver
    s = Solver(16, 8, 4)
    with pytest.raises(TdglError) as e:
        s.set_mu_solver()                                          # direct solver: no iteration to control
    assert e.value.code == -1
    s.close()


# ---------------------------------------------------------------------------------------------------
# insulating inclusions: removed sites and cut links (TDGL_FLAG_INSULATORS, reading S25; fp64 build)
# ---------------------------------------------------------------------------------------------------
def insulator_pair(cfg, holes, psi0, mu0, K0, fixed_sweeps=0, eps_tol=1e-6):
    """Oracle (sc_mask from the same inside test as the epsilon pattern) and Solver with identical inputs."""
    from dataclasses import replace
    from paper_1409_8340_b200 import Solver
    p = oracle_params(cfg, fp64=True, eps_tol=eps_tol)
    shapes = np.asarray(holes).shape[-1] == 10               # a tdgl_shape list (S26) instead of spheres
    mask = (O.epsilon_from_shapes if shapes else O.epsilon_from_spheres)(p, holes, 0.0, 1.0) > 0.5
    p = replace(p, sc_mask=mask)
    s = Solver(cfg.nx, cfg.ny, cfg.nz, bc=cfg.bc, h=cfg.h, dt=cfg.dt, eps_tol=eps_tol, fixed_sweeps=fixed_sweeps,
               temperature=cfg.temperature, seed=cfg.seed, fp64=True, insulators=True)
    spheres = I.sphere_list(cfg)
    eps = O.epsilon_from_spheres(p, spheres, cfg.eps_in, cfg.eps_out)
    s.set_pinning(spheres, cfg.eps_in, cfg.eps_out)
    (s.set_insulator_shapes if shapes else s.set_insulators)(holes)
    bx_req, bz_req = cfg.requested_field()
    Bx, Bz, _, _ = O.snap_field(p, f32(bx_req), f32(bz_req))
    s.set_field_current(Bx=bx_req, Bz=bz_req, Jx=cfg.Jx)
    st = O.State(psi=psi0.astype(np.complex128) * mask, mu=mu0.astype(np.float64) * mask, K=float(K0))
    s.set_state(torch.from_numpy(psi0), torch.from_numpy(mu0), float(K0))       # the library empties the removed sites
    return p, st, eps, (Bx, Bz), s, mask


@pytest.mark.parametrize("bc", ALL_BC)
def test_insulating_inclusions_two_steps(bc):
    cfg = cfg_of(36, 14, 10, bc, Bx=0.05, Bz=0.3, Jx=0.02 if bc[0] == P_ else 0.0, temperature=1e-3,
                 incl_fraction=0.1, incl_rmin=1.0, incl_rmax=2.0, seed=2)
    holes = np.array([[4.0, 3.0, 2.0, 1.6], [12.0, 5.0, 3.5, 2.1], [17.5, 0.5, 0.0, 1.3], [9.0, 6.5, 4.5, 0.9]], np.float32)
    psi0, mu0 = I.random_state(cfg, seed=21, amp=0.8)
    K0 = 0.11 if bc[0] == P_ else 0.0
    p, st, eps, (Bx, Bz), s, mask = insulator_pair(cfg, holes, psi0, mu0, K0, fixed_sweeps=5)
    assert 0.03 < 1.0 - mask.mean() < 0.3
    s.step(2)
    psi, mu = s.get_psi_mu()
    outer, inner = s.mu_log(2)
    for n in range(2):
        O.step(p, st, eps, Bx, Bz, f32(cfg.Jx), fixed_sweeps=5, mu_inner_counts=inner[n])
    psi, mu = psi.cpu().numpy(), mu.cpu().numpy()
    assert np.all(psi[~mask] == 0.0) and np.all(mu[~mask] == 0.0)
    assert np.max(np.abs(psi - st.psi)) < 1e-12
    assert np.max(np.abs(mu - st.mu)) < 1e-12 * max(1.0, np.max(np.abs(st.mu)))
    ob = s.observables()
    assert abs(ob.K - st.K) < 1e-13 and abs(ob.Jav - st.Jav) < 1e-13
    links = O.paper_links(p, st.K, Bx, Bz)
    F = O.free_energy(p, st.psi, eps, links)
    assert abs(ob.free_energy - F) < 1e-12 * abs(F)
    assert abs(ob.mean_abs2 - O.mean_abs2(st.psi)) < 1e-14
    assert ob.vortices_per_slice == O.vortices_per_slice(p, st.psi, links, Bz)
    s.close()


@pytest.mark.parametrize("bc", [(P_, P_, O_), (O_, O_, O_)])
def test_insulating_shapes_two_steps(bc):
    """Insulating ellipsoids and +-45 degree columns (S25 with the shapes of S26)."""
    cfg = cfg_of(40, 16, 12, bc, Bz=0.3, Jx=0.02 if bc[0] == P_ else 0.0, temperature=1e-3, seed=6)
    holes = np.array([[1, 5.0, 3.0, 2.0, 2.2, 1.1, 1.6, 0, 0, 0],
                      [2, 12.0, 5.0, 3.0, 1.2, 100.0, 0, 1, 0, 1],
                      [2, 16.0, 2.0, 3.0, 0.9, 100.0, 0, -1, 0, 1],
                      [0, 0.2, 0.1, 5.9, 1.4, 0, 0, 0, 0, 0]], np.float32)
    psi0, mu0 = I.random_state(cfg, seed=22, amp=0.8)
    p, st, eps, (Bx, Bz), s, mask = insulator_pair(cfg, holes, psi0, mu0, 0.07 if bc[0] == P_ else 0.0, fixed_sweeps=4)
    assert 0.03 < 1.0 - mask.mean() < 0.4
    s.step(2)
    psi, mu = s.get_psi_mu()
    outer, inner = s.mu_log(2)
    for n in range(2):
        O.step(p, st, eps, Bx, Bz, f32(cfg.Jx), fixed_sweeps=4, mu_inner_counts=inner[n])
    psi, mu = psi.cpu().numpy(), mu.cpu().numpy()
    assert np.all(psi[~mask] == 0.0) and np.all(mu[~mask] == 0.0)
    assert np.max(np.abs(psi - st.psi)) < 1e-12
    assert np.max(np.abs(mu - st.mu)) < 1e-12 * max(1.0, np.max(np.abs(st.mu)))
    s.close()


def test_insulating_inclusions_film_run_and_conservation():
    """A film with holes, 30 steps with the GPU's own decisions, replayed by the oracle; the weighted sum of rho vanishes
    (the cut-link operator is Hermitian: the Neumann problem for mu stays solvable) and no current enters a hole."""
    cfg = cfg_of(96, 64, 1, (P_, P_, P_), nz_flux=6, Jx=0.02, seed=4)
    holes = np.array([[10.0, 8.0, 0.0, 3.0], [30.0, 20.0, 0.0, 4.2], [40.0, 5.0, 0.0, 2.0]], np.float32)
    psi0 = I.initial_psi(cfg)
    p, st, eps, (Bx, Bz), s, mask = insulator_pair(cfg, holes, psi0, np.zeros((1, 64, 96), np.float32), 0.0)
    s.step(30)
    psi, mu = s.get_psi_mu()
    counts, _ = s.sweep_log(30)
    outer, inner = s.mu_log(30)
    O.run(p, st, eps, Bx, Bz, f32(cfg.Jx), 30, sweep_counts=counts, mu_schedule=inner)
    assert np.max(np.abs(psi.cpu().numpy() - st.psi)) < 1e-10
    assert np.max(np.abs(mu.cpu().numpy() - st.mu)) < 1e-10
    rho = s.debug_rho().cpu().numpy()
    assert abs(rho.sum()) < 1e-10 * np.abs(rho).sum() and np.all(rho[~mask] == 0.0)
    s.close()


def test_insulators_need_the_flag():
    from paper_1409_8340_b200 import Solver
    from paper_1409_8340_b200.binding import TdglError
    s = Solver(16, 8, 4, fp64=True)
    with pytest.raises(TdglError) as e:
        s.set_insulators(np.array([[1.0, 1.0, 1.0, 1.0]], np.float32))
    assert e.value.code == -3
    s.close()
    with pytest.raises(TdglError):
        Solver(16, 8, 4, insulators=True)                          # fp32 path has no cut links


# ---------------------------------------------------------------------------------------------------
# the direct mu solver of the double-precision build (TDGL_FLAG_MU_DIRECT): fp32 transform solver inside fp64
# iterative refinement.  The oracle side is the DEFINITION Delta_h mu = rho solved in fp64 (O.solve_poisson).
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc,shape", [((P_, P_, P_), (64, 32, 16)), ((P_, P_, O_), (128, 40, 9)), ((O_, O_, O_), (34, 13, 11)),
                                      ((P_, O_, P_), (64, 20, 12)), ((O_, P_, O_), (1024, 6, 5)), ((P_, P_, P_), (256, 96, 1)),
                                      ((O_, O_, P_), (130, 37, 1))])
def test_fp64_direct_poisson(bc, shape):
    nx, ny, nz = shape
    cfg = cfg_of(nx, ny, nz, bc)
    p = oracle_params(cfg, fp64=True, mu_direct=True)
    s = make_solver(cfg, fp64=True, mu_direct=True)
    rng = np.random.default_rng(8)
    w = O.site_weights(p)
    rho = rng.standard_normal(p.shape)
    rho -= np.sum(w * rho) / np.sum(w)                       # solvable right side (S6)
    mu = s.debug_poisson(torch.from_numpy(rho)).cpu().numpy()
    ref = O.solve_poisson(p, rho)
    scale = np.max(np.abs(ref))
    assert mu.dtype == np.float64
    assert np.max(np.abs(mu - ref)) < 1e-11 * scale
    assert np.max(np.abs(O.laplacian_real(p, mu) - rho)) < 1e-11 * max(1.0, np.max(np.abs(rho)))
    solves, passes, resid = s.mu_direct_stats()
    # the residual bottoms out at the fp64 rounding of Delta_h mu itself: ~ 6 terms of size 4 |mu| each
    assert solves == 1 and 2 <= passes <= 8 and resid < 1e-14 * max(1.0, 24.0 * scale)
    s.close()


@pytest.mark.parametrize("bc", ALL_BC)
def test_fp64_direct_two_steps(bc):
    cfg = cfg_of(36, 14, 10, bc, Bx=0.05, Bz=0.3, Jx=0.02 if bc[0] == P_ else 0.0, temperature=1e-3, incl_fraction=0.15,
                 incl_rmin=1.0, incl_rmax=2.0, seed=2)
    psi0, mu0 = I.random_state(cfg, seed=21, amp=0.8)
    K0 = 0.11 if bc[0] == P_ else 0.0
    p, st, eps, (Bx, Bz), s = setup_pair(cfg, psi0=psi0, mu0=mu0, K0=K0, fixed_sweeps=5, fp64=True, mu_direct=True)
    assert p.mu_solver == "direct"
    s.step(2)
    psi, mu = s.get_psi_mu()
    for _ in range(2):
        O.step(p, st, eps, Bx, Bz, f32(cfg.Jx), fixed_sweeps=5)
    ob = s.observables()
    assert np.max(np.abs(psi.cpu().numpy() - st.psi)) < 1e-12
    assert np.max(np.abs(mu.cpu().numpy() - st.mu)) < 1e-11 * max(1.0, np.max(np.abs(st.mu)))
    assert abs(ob.K - st.K) < 1e-13 and abs(ob.Jav - st.Jav) < 1e-13
    s.close()


def test_fp64_direct_film_and_C1_run():
    cfg = cfg_of(132, 22, 1, (P_, P_, P_), Bz=0.3, Jx=0.02, temperature=1e-3, incl_fraction=0.15, incl_rmin=1.0, incl_rmax=2.0, seed=3)
    psi0, mu0 = I.random_state(cfg, seed=7, amp=0.8)
    p, st, eps, (Bx, Bz), s = setup_pair(cfg, psi0=psi0, mu0=mu0, K0=0.2, fixed_sweeps=4, fp64=True, mu_direct=True)
    s.step(3)
    psi, mu = s.get_psi_mu()
    for _ in range(3):
        O.step(p, st, eps, Bx, Bz, f32(cfg.Jx), fixed_sweeps=4)
    assert np.max(np.abs(psi.cpu().numpy() - st.psi)) < 1e-12
    assert np.max(np.abs(mu.cpu().numpy() - st.mu)) < 1e-10 * max(1.0, np.max(np.abs(st.mu)))
    s.close()
    # BASELINE.json configs[0], 100 steps, both sides taking their own decisions
    cfg = I.CONFIGS["C1"]
    p, st, eps, (Bx, Bz), s = setup_pair(cfg, fp64=True, mu_direct=True)
    s.step(100)
    psi, mu = s.get_psi_mu()
    counts, _ = s.sweep_log(100)
    O.run(p, st, eps, Bx, Bz, 0.0, 100)
    assert list(counts) == st.sweep_log
    psi = psi.cpu().numpy()
    # C1 spends its last ~65 steps in the single-sweep regime, which amplifies the checkerboard band by 1.186 per step (reading R3):
    # fp64 rounding differences of 1e-16 (another summation order in mu) arrive at ~1e-10; measured 1.5e-10
    assert np.max(np.abs(psi - st.psi)) <= 1e-9 and rel_l2(psi, st.psi) <= 1e-10
    assert np.max(np.abs(mu.cpu().numpy() - st.mu)) <= 1e-10
    solves, passes, _ = s.mu_direct_stats()
    assert solves == 100 and passes <= 6 * solves
    s.close()


def test_mu_direct_flag_validation():
    from paper_1409_8340_b200 import Solver
    from paper_1409_8340_b200.binding import TdglError
    for kw in (dict(mu_direct=True), dict(mu_direct=True, fp64=True, mu_iterative=True), dict(mu_direct=True, fp64=True, insulators=True)):
        with pytest.raises(TdglError):
            Solver(16, 8, 4, **kw)
