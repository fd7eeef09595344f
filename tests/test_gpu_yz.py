"""`-m gpu`: the yz Landau gauge (TDGL_FLAG_GAUGE_YZ: Eq. 24b/29b, quasi-periodic jump in x; P:205, 278-283,
457-465) of the CUDA path against the fp64 oracle (oracle.paper_links_yz), through the C ABI."""
import math

import numpy as np
import pytest

import tdgl_inputs as I
from oracle import tdgl_oracle as O
from gpu_common import f32, oracle_params, rel_l2

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

P_, O_ = I.PERIODIC, I.OPEN
ALL_BC = [(a, b, c) for a in (P_, O_) for b in (P_, O_) for c in (P_, O_)]


def setup_yz(cfg, By, Bz, psi0, mu0=None, K0=0.0, host_loop=False, fixed_sweeps=0, eps_tol=1e-6, temperature=None):
    """Oracle params/state/links_fn and the CUDA solver in the yz gauge, identical inputs."""
    from paper_1409_8340_b200 import Solver
    T = cfg.temperature if temperature is None else temperature
    p = oracle_params(cfg, eps_tol=eps_tol, temperature=T)
    s = Solver(cfg.nx, cfg.ny, cfg.nz, bc=cfg.bc, h=cfg.h, dt=cfg.dt, eps_tol=eps_tol, max_sweeps=100,
               fixed_sweeps=fixed_sweeps, temperature=T, seed=cfg.seed, init_amp=cfg.init_amp, solve_mu=True,
               host_loop=host_loop, gauge_yz=True)
    spheres = I.sphere_list(cfg)
    eps = O.epsilon_from_spheres(p, spheres, cfg.eps_in, cfg.eps_out)
    s.set_pinning(spheres, cfg.eps_in, cfg.eps_out)
    By_e, Bz_e, _, _ = O.snap_field_yz(p, f32(By), f32(Bz))
    s.set_field_current(By=By, Bz=Bz, Jx=cfg.Jx)
    mu_np = np.zeros(p.shape, np.float32) if mu0 is None else mu0
    st = O.State(psi=psi0.astype(np.complex128), mu=mu_np.astype(np.float64), K=float(K0))
    s.set_state(torch.from_numpy(psi0), torch.from_numpy(mu_np), float(K0))

    def links_fn(K):
        return O.paper_links_yz(p, K, By_e, Bz_e)
    return p, st, eps, (By_e, Bz_e), links_fn, s


@pytest.mark.parametrize("bc", ALL_BC)
@pytest.mark.parametrize("host_loop", [False, True])
def test_yz_one_step_fixed_sweeps(bc, host_loop):
    cfg = I.Config("yz", 36, 14, 10, tuple(bc), Jx=0.02 if bc[0] == P_ else 0.0, temperature=1e-3, incl_fraction=0.15,
                   incl_rmin=1.0, incl_rmax=2.0, seed=2)
    psi0, mu0 = I.random_state(cfg, seed=21, amp=0.8)
    K0 = 0.11 if bc[0] == P_ else 0.0
    p, st, eps, (By, Bz), links_fn, s = setup_yz(cfg, 0.07, 0.3, psi0, mu0, K0, host_loop=host_loop, fixed_sweeps=5)
    s.step(2)
    psi, mu = s.get_psi_mu()
    psi, mu = psi.cpu().numpy(), mu.cpu().numpy()
    for _ in range(2):
        O.step(p, st, eps, 0.0, Bz, f32(cfg.Jx), fixed_sweeps=5, links_fn=links_fn)
    ob = s.observables()
    assert ob.steps == 2 and ob.sweeps_total == 10
    assert np.max(np.abs(psi - st.psi)) < 5e-6
    assert np.max(np.abs(mu - st.mu)) < 2e-5 * max(1.0, np.max(np.abs(st.mu)))
    assert abs(ob.K - st.K) < 1e-7 and abs(ob.Ex - st.Ex) < 1e-7 and abs(ob.Jav - st.Jav) < 1e-7
    assert abs(ob.max_resid2 - st.max_resid2) <= 2e-3 * st.max_resid2 + 1e-12
    assert abs(ob.Bx_eff - By) < 1e-7 and abs(ob.Bz_eff - Bz) < 1e-7          # Bx_eff reports B_y in this gauge
    s.close()


@pytest.mark.parametrize("bc", [(P_, P_, P_), (O_, O_, O_), (P_, O_, P_)])
def test_yz_mu_refinement(bc):
    """The fp64 residual of the mu refinement step (refine.cu) in the yz gauge: per-column U_y(i), U_z(i), jump in x.
    A long thin mesh and a rough state, refinement forced on: mu meets the 2e-5 gate after one step."""
    from paper_1409_8340_b200 import Solver
    cfg = I.Config("yzr", 900, 6, 5, tuple(bc), Jx=0.02 if bc[0] == P_ else 0.0, seed=4)
    psi0, mu0 = I.random_state(cfg, seed=6, amp=0.8)
    K0 = 0.2 if bc[0] == P_ else 0.0
    p = oracle_params(cfg)
    By, Bz, _, _ = O.snap_field_yz(p, f32(0.05), f32(0.3))
    st = O.State(psi=psi0.astype(np.complex128), mu=mu0.astype(np.float64), K=K0)
    s = Solver(cfg.nx, cfg.ny, cfg.nz, bc=cfg.bc, h=cfg.h, dt=cfg.dt, fixed_sweeps=1, gauge_yz=True, mu_refine=True)
    s.set_field_current(By=0.05, Bz=0.3, Jx=cfg.Jx)
    s.set_state(torch.from_numpy(psi0), torch.from_numpy(mu0), K0)
    s.step(1)
    O.step(p, st, np.ones(p.shape), 0.0, Bz, f32(cfg.Jx), fixed_sweeps=1, links_fn=lambda K: O.paper_links_yz(p, K, By, Bz))
    psi, mu = s.get_psi_mu()
    assert np.max(np.abs(psi.cpu().numpy() - st.psi)) < 5e-6
    assert np.max(np.abs(mu.cpu().numpy() - st.mu)) < 2e-5 * max(1.0, np.max(np.abs(st.mu)))
    s.close()


@pytest.mark.parametrize("shape", [(132, 37, 9), (260, 20, 12)])
def test_yz_ragged_tiles_and_seams(shape):
    """Several tiles in x (the jump acts on the first and the last one only), ragged tiles in x and y."""
    nx, ny, nz = shape
    cfg = I.Config("yz", nx, ny, nz, (P_, P_, P_), Jx=0.01, seed=3)
    psi0, mu0 = I.random_state(cfg, seed=5, amp=0.9)
    p, st, eps, (By, Bz), links_fn, s = setup_yz(cfg, 0.1, 0.25, psi0, mu0, 0.3, fixed_sweeps=4)
    s.step(1)
    psi, mu = s.get_psi_mu()
    O.step(p, st, eps, 0.0, Bz, f32(cfg.Jx), fixed_sweeps=4, links_fn=links_fn)
    assert np.max(np.abs(psi.cpu().numpy() - st.psi)) < 5e-6
    assert np.max(np.abs(mu.cpu().numpy() - st.mu)) < 2e-5 * max(1.0, np.max(np.abs(st.mu)))
    s.close()


@pytest.mark.parametrize("bc", [(P_, P_, P_), (P_, P_, O_), (O_, O_, O_)])
def test_yz_observables(bc):
    cfg = I.Config("yz", 32, 24, 10, tuple(bc), incl_fraction=0.1, incl_rmin=1.0, incl_rmax=2.0)
    rng = np.random.default_rng(8)
    shape = (cfg.nz, cfg.ny, cfg.nx)
    psi0 = ((1.0 + 0.4 * rng.uniform(-1, 1, shape)) * np.exp(1j * rng.uniform(-math.pi, math.pi, shape))).astype(np.complex64)
    Lx, Ly, _ = cfg.lengths()
    Bz_req = 2 * math.pi * 3 / (Lx * Ly)
    p, st, eps, (By, Bz), links_fn, s = setup_yz(cfg, 0.05, Bz_req, psi0, K0=0.2 if bc[0] == P_ else 0.0)
    ob = s.observables()
    links = links_fn(st.K)
    F = O.free_energy(p, st.psi, eps, links)
    assert abs(ob.free_energy - F) < 2e-6 * abs(F) + 1e-6 * p.n_sites
    assert abs(ob.vortices_per_slice - O.vortices_per_slice(p, st.psi, links, Bz)) < 1e-9
    if bc[0] == P_ and bc[1] == P_:
        assert ob.vortices_per_slice == 3.0                              # flux quantisation in this gauge
    s.close()


def test_yz_run_pointwise_40_steps():
    """Tilted field in the yz plane, current, inclusions, the GPU taking its own convergence decisions."""
    from test_gpu_runs import check_decisions
    cfg = I.Config("yz", 64, 48, 24, (P_, P_, O_), Jx=0.02, incl_fraction=0.1, incl_rmin=1.5, incl_rmax=2.5, seed=4)
    psi0 = I.initial_psi(cfg)
    p, st, eps, (By, Bz), links_fn, s = setup_yz(cfg, 0.1, 0.2, psi0)
    s.step(40)
    psi, mu = s.get_psi_mu()
    counts, _ = s.sweep_log(40)
    O.run(p, st, eps, 0.0, Bz, f32(cfg.Jx), 40, sweep_counts=counts, links_fn=links_fn)
    check_decisions(p, st, counts)
    psi, mu = psi.cpu().numpy(), mu.cpu().numpy()
    assert np.max(np.abs(psi - st.psi)) <= 1e-4 and rel_l2(psi, st.psi) <= 1e-5
    assert np.max(np.abs(mu - st.mu)) <= 1e-4 * max(1.0, np.max(np.abs(st.mu)))
    s.close()


def test_gauges_are_equivalent_on_the_gpu():
    """B || z, x and y open: the xz-gauge run from psi0 and the yz-gauge run from psi0 e^{i chi}, chi = B_z xbar ybar,
    stay related by the same phase (both are the CUDA path; the oracle pins the same identity in fp64)."""
    from paper_1409_8340_b200 import Solver
    cfg = I.Config("g", 40, 36, 12, (O_, O_, P_))
    Bz = 0.3
    p = oracle_params(cfg)
    xbar = (np.arange(cfg.nx) * p.hx - p.length("x") / 2)[None, None, :]
    ybar = (np.arange(cfg.ny) * p.hy - p.length("y") / 2)[None, :, None]
    chi = np.broadcast_to(f32(Bz) * xbar * ybar, p.shape)
    psi0 = I.initial_psi(cfg)
    out = []
    for yz in (False, True):
        s = Solver(cfg.nx, cfg.ny, cfg.nz, bc=cfg.bc, eps_tol=1e-10, max_sweeps=200, gauge_yz=yz)
        s.set_pinning(np.zeros((0, 4), np.float32), -1.0, 1.0)
        s.set_field_current(Bz=Bz)
        start = (psi0 * np.exp(1j * chi)).astype(np.complex64) if yz else psi0
        s.set_state(torch.from_numpy(start), None, 0.0)
        s.step(20)
        psi, mu = s.get_psi_mu()
        out.append((psi.cpu().numpy().astype(np.complex128), mu.cpu().numpy()))
        s.close()
    assert np.max(np.abs(out[1][0] - out[0][0] * np.exp(1j * chi))) < 2e-5
    assert np.max(np.abs(out[1][1] - out[0][1])) < 2e-5


def test_yz_error_codes():
    from paper_1409_8340_b200 import Solver
    from paper_1409_8340_b200.binding import TdglError
    s = Solver(32, 32, 8, gauge_yz=True)
    with pytest.raises(TdglError) as e:
        s.set_field_current(Bx=0.1, Bz=0.1)                              # B_x needs the xz gauge
    assert e.value.code == -3
    s.close()
    s = Solver(32, 32, 8)
    with pytest.raises(TdglError) as e:
        s.set_field_current(By=0.1, Bz=0.1)                              # B_y needs the yz gauge
    assert e.value.code == -3
    s.close()
    with pytest.raises(TdglError) as e:
        Solver(32, 32, 1, gauge_yz=True)                                 # films use the xz gauge
    assert e.value.code == -1
