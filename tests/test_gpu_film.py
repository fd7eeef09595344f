"""`-m gpu`: film mode (N_z = 1, the paper's 2D workloads P:527, 579-583; reading S22) of the CUDA path against the
fp64 oracle, through the C ABI: the y-marching kernels of march_film.cu (init + sweep, sweep, rho, fused J_av),
the film view of the Poisson solver, noise, observables, multi-step runs."""
import math

import numpy as np
import pytest

import tdgl_inputs as I
from oracle import tdgl_oracle as O
from gpu_common import f32, rel_l2, setup_pair

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

P_, O_ = I.PERIODIC, I.OPEN
BC2 = [(a, b, P_) for a in (P_, O_) for b in (P_, O_)]


def film(nx, ny, bc, **kw):
    return I.Config(f"film{nx}x{ny}", nx, ny, 1, tuple(bc), **kw)


@pytest.mark.parametrize("bc", BC2)
@pytest.mark.parametrize("shape,host_loop", [((36, 14), False), ((36, 14), True), ((1100, 21), False), ((2050, 9), False)])
def test_film_one_step_fixed_sweeps(bc, shape, host_loop):
    """Two steps of five sweeps: ragged strips (1100 = 1024 + 76, 2050 = 2 x 1024 + 2), short chunks, every
    boundary combination, noise, inclusions, current."""
    nx, ny = shape
    cfg = film(nx, ny, bc, Bz=0.3, Jx=0.02 if bc[0] == P_ else 0.0, temperature=1e-3, incl_fraction=0.15,
               incl_rmin=1.0, incl_rmax=2.0, seed=2)
    psi0, mu0 = I.random_state(cfg, seed=21, amp=0.8)
    K0 = 0.11 if bc[0] == P_ else 0.0
    p, st, eps, (Bx, Bz), s = setup_pair(cfg, psi0=psi0, mu0=mu0, K0=K0, host_loop=host_loop, fixed_sweeps=5)
    s.step(2)
    psi, mu = s.get_psi_mu()
    psi, mu = psi.cpu().numpy(), mu.cpu().numpy()
    for _ in range(2):
        O.step(p, st, eps, Bx, Bz, f32(cfg.Jx), fixed_sweeps=5)
    ob = s.observables()
    assert ob.steps == 2 and ob.sweeps_last == 5 and ob.sweeps_total == 10
    assert np.max(np.abs(psi - st.psi)) < 5e-6
    assert np.max(np.abs(mu - st.mu)) < 2e-5 * max(1.0, np.max(np.abs(st.mu)))
    assert abs(ob.K - st.K) < 1e-7 and abs(ob.Ex - st.Ex) < 1e-7 and abs(ob.Jav - st.Jav) < 1e-7
    assert abs(ob.max_resid2 - st.max_resid2) <= 2e-3 * st.max_resid2 + 1e-12
    s.close()


@pytest.mark.parametrize("bc", BC2)
@pytest.mark.parametrize("shape", [(64, 64), (128, 40), (34, 22), (512, 256), (2048, 24), (24, 2048), (4096, 12),
                                   (16, 4096), (8192, 8), (8, 8192)])
def test_film_poisson(bc, shape):
    nx, ny = shape
    cfg = film(nx, ny, bc)
    p, st, eps, B, s = setup_pair(cfg, with_pinning=False)
    rng = np.random.default_rng(5)
    rho = rng.uniform(-1, 1, p.shape)
    w = O.site_weights(p)
    rho -= np.sum(w * rho) / np.sum(w)
    rho32 = rho.astype(np.float32)
    mu = s.debug_poisson(torch.from_numpy(rho32)).cpu().numpy()
    ref = O.solve_poisson(p, rho32.astype(np.float64))
    assert np.max(np.abs(mu - ref)) < 2e-5 * np.max(np.abs(ref))
    s.close()


def test_film_noise_amplitude_and_stream():
    """The Langevin term of a film uses zeta_max of d = 2 (no h_z) and the same Philox stream as the oracle."""
    cfg = film(64, 32, (P_, P_, P_), temperature=2e-3, seed=77)
    p, st, eps, B, s = setup_pair(cfg, with_pinning=False)
    z = s.debug_noise(9).cpu().numpy()
    ref = O.langevin_noise(p, 9)
    # uniform words are exact in fp32; the product with zeta_max (d = 2: no h_z) is rounded once on each side
    zm = np.float32(O.zeta_max(p))
    assert abs(float(zm) - math.sqrt(3 * f32(2e-3) / (2 * f32(0.1) * 0.25))) < 1e-6
    assert np.array_equal(z.real, (ref.real / O.zeta_max(p)).astype(np.float32) * zm)
    assert np.array_equal(z.imag, (ref.imag / O.zeta_max(p)).astype(np.float32) * zm)
    s.close()


@pytest.mark.parametrize("bc", BC2)
def test_film_observables(bc):
    cfg = film(48, 40, bc, nz_flux=3 if bc[0] == P_ and bc[1] == P_ else None, Bz=0.2, incl_fraction=0.1,
               incl_rmin=1.0, incl_rmax=2.0)
    rng = np.random.default_rng(8)
    shape = (1, cfg.ny, cfg.nx)
    psi0 = ((1.0 + 0.4 * rng.uniform(-1, 1, shape)) * np.exp(1j * rng.uniform(-math.pi, math.pi, shape))).astype(np.complex64)
    p, st, eps, (Bx, Bz), s = setup_pair(cfg, psi0=psi0, K0=0.2 if bc[0] == P_ else 0.0)
    ob = s.observables()
    links = O.paper_links(p, st.K, Bx, Bz)
    F = O.free_energy(p, st.psi, eps, links)
    assert abs(ob.free_energy - F) < 2e-6 * abs(F) + 1e-6 * p.n_sites
    assert abs(ob.mean_abs2 - O.mean_abs2(st.psi)) < 1e-6
    assert abs(ob.vortices_per_slice - O.vortices_per_slice(p, st.psi, links, Bz)) < 1e-9
    if bc[0] == P_ and bc[1] == P_:
        assert ob.vortices_per_slice == 3.0
    s.close()


def test_film_rejects_an_in_plane_field():
    from paper_1409_8340_b200.binding import TdglError
    cfg = film(32, 32, (P_, P_, P_))
    p, st, eps, B, s = setup_pair(cfg, with_pinning=False)
    with pytest.raises(TdglError) as e:
        s.set_field_current(Bx=0.1, Bz=0.1, Jx=0.0)
    assert e.value.code == -3
    s.close()


@pytest.mark.parametrize("bc,nsteps", [((P_, P_, P_), 100), ((P_, O_, P_), 40), ((O_, O_, P_), 40)])
def test_film_run_pointwise(bc, nsteps):
    """A driven film (field, current, inclusions) without noise: the stated 1e-4 / 1e-5 gate after nsteps steps,
    the GPU taking its own convergence decisions (S9)."""
    from test_gpu_runs import check_decisions, run_pair
    cfg = film(96, 64, bc, nz_flux=6 if bc[0] == P_ and bc[1] == P_ else None, Bz=0.25,
               Jx=0.02 if bc[0] == P_ else 0.0, incl_fraction=0.1, incl_rmin=1.5, incl_rmax=2.5, seed=4)
    p, st, eps, B, s, psi, mu, counts, resid, ob = run_pair(cfg, nsteps)
    check_decisions(p, st, counts)
    assert np.max(np.abs(psi - st.psi)) <= 1e-4
    assert rel_l2(psi, st.psi) <= 1e-5
    assert np.max(np.abs(mu - st.mu)) <= 1e-4 * max(1.0, np.max(np.abs(st.mu)))
    assert abs(ob.K - st.K) < 1e-6
    s.close()


def test_film_run_with_noise_statistics():
    from test_gpu_runs import check_decisions, run_pair
    cfg = film(128, 128, (P_, P_, P_), nz_flux=10, Jx=0.02, temperature=1e-3, seed=6)
    p, st, eps, (Bx, Bz), s, psi, mu, counts, resid, ob = run_pair(cfg, 60)
    check_decisions(p, st, counts)
    links = O.paper_links(p, st.K, Bx, Bz)
    assert abs(ob.mean_abs2 - O.mean_abs2(st.psi)) <= 1e-3
    assert abs(ob.vortices_per_slice - O.vortices_per_slice(p, st.psi, links, Bz)) <= 1e-3
    assert np.max(np.abs(psi - st.psi)) <= 1e-4
    s.close()
