"""`-m gpu`: kernel-level parity of the CUDA path (through the C ABI) against the fp64 oracle.

Tolerances: integer / mask / Philox work is bit-exact; single fp32
operators are compared with the oracle evaluated on the same fp32 inputs, with a bound of a few fp32
ulps of the largest intermediate.
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
    return I.Config(f"t{nx}x{ny}x{nz}", nx, ny, nz, tuple(bc), **kw)


# ---------------------------------------------------------------------------------------------------
# a2: Philox stream, bit-exact
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed,step", [(0, 0), (12345, 7), ((1 << 40) + 99, 123456)])
def test_noise_bit_exact(seed, step):
    cfg = cfg_of(34, 10, 6, (P_, P_, P_), temperature=1e-3, seed=seed)
    p = oracle_params(cfg)
    s = make_solver(cfg)
    z = s.debug_noise(step).cpu().numpy()
    ref = O.langevin_noise(p, step)
    # uniform words are exact in fp32; the product with zeta_max is rounded once on each side
    zm = np.float32(O.zeta_max(p))
    ref32 = (np.float32(1) * (ref.real / O.zeta_max(p)).astype(np.float32) * zm) + 1j * (
        (ref.imag / O.zeta_max(p)).astype(np.float32) * zm)
    assert np.array_equal(z.real, ref32.real.astype(np.float32))
    assert np.array_equal(z.imag, ref32.imag.astype(np.float32))
    s.close()


@pytest.mark.parametrize("shape,bc", [((34, 10, 6), (P_, P_, P_)), ((130, 12, 9), (P_, O_, O_)), ((256, 32, 8), (P_, P_, O_)),
                                      ((66, 20, 1), (P_, P_, P_)), ((2050, 9, 1), (O_, P_, P_))])
@pytest.mark.parametrize("seed,nsteps", [(0, 1), ((1 << 40) + 99, 3)])
def test_fused_noise_draw_is_the_oracles(shape, bc, seed, nsteps):
    """The draw INSIDE the init kernels (k_march_tma<INIT>, k_march_film<INIT>; test_noise_bit_exact above exercises the copy
    in k_noise).  From psi = 0 with eps = 0, mu = 0, B = 0 and one sweep per step, Eq. (31) leaves b = h_t zeta and the
    sweep returns psi+ = h_t zeta / d with a constant real d: the new state IS the noise field, site by site.  A wrong
    word, counter, pair assignment or step index anywhere shows as an O(0.1) difference; agreement is asked to 1e-7
    (a few fp32 roundings of |psi+| ~ 0.02).  Several steps: the step index enters the counter (after step one psi is no longer zero, so this
    part is ordinary parity with the noise as the only source)."""
    nx, ny, nz = shape
    cfg = cfg_of(nx, ny, nz, bc, temperature=1e-3, seed=seed)
    psi0 = np.zeros((nz, ny, nx), np.complex64)
    p, st, eps, (Bx, Bz), s = setup_pair(cfg, psi0=psi0, with_pinning=False, solve_mu=False, fixed_sweeps=1)
    s.set_pinning(np.zeros((0, 4), np.float32), 0.0, 0.0)
    eps = np.zeros_like(eps)
    for n in range(nsteps):
        s.step(1)
        O.step(p, st, eps, Bx, Bz, 0.0, fixed_sweeps=1)
        psi = s.get_psi_mu()[0].cpu().numpy()
        if n == 0:
            zeta = O.langevin_noise(p, 0)
            ratio = st.psi / zeta                                     # h_t / d: one real constant over the whole mesh
            assert np.max(np.abs(ratio - ratio.flat[0])) < 1e-12 and abs(ratio.flat[0].imag) < 1e-15
        assert np.max(np.abs(psi - st.psi)) < 1e-7, (n, np.max(np.abs(psi - st.psi)))
    s.close()


def test_initial_state_matches_oracle_box_muller():
    cfg = cfg_of(32, 12, 6, (P_, P_, P_), seed=3)
    p = oracle_params(cfg)
    s = make_solver(cfg)
    psi, mu = s.get_psi_mu()
    ref = O.initial_state(p, f32(cfg.init_amp)).psi
    assert np.max(np.abs(psi.cpu().numpy() - ref)) < 2e-7
    assert float(mu.abs().max()) == 0.0
    s.close()


# ---------------------------------------------------------------------------------------------------
# a0: inclusion mask, bit-identical
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc", [(P_, P_, P_), (P_, P_, O_), (O_, O_, O_), (P_, O_, O_)])
def test_epsilon_mask_identical(bc):
    cfg = cfg_of(40, 28, 18, bc, incl_fraction=0.2, incl_rmin=1.0, incl_rmax=3.0, seed=5)
    p = oracle_params(cfg)
    s = make_solver(cfg)
    sph = I.sphere_list(cfg)
    assert len(sph) > 5
    s.set_pinning(sph, -1.0, 1.0)
    eps = s.get_eps().cpu().numpy()
    ref = O.epsilon_from_spheres(p, sph, -1.0, 1.0)
    assert np.array_equal(eps, ref.astype(np.float32))
    assert 0.05 < (eps < 0).mean() < 0.5
    s.set_pinning(np.zeros((0, 4), np.float32), -1.0, 0.5)          # empty list
    assert np.all(s.get_eps().cpu().numpy() == np.float32(0.5))
    s.close()


def test_epsilon_mask_sphere_larger_than_box():
    cfg = cfg_of(16, 16, 16, (P_, P_, O_))
    p = oracle_params(cfg)
    s = make_solver(cfg)
    sph = np.array([[3.0, 4.0, 2.0, 30.0], [1.0, 1.0, 1.0, 0.2]], np.float32)
    s.set_pinning(sph, -1.0, 1.0)
    assert np.array_equal(s.get_eps().cpu().numpy(), O.epsilon_from_spheres(p, sph, -1.0, 1.0).astype(np.float32))
    s.close()


@pytest.mark.parametrize("bc", [(P_, P_, P_), (P_, P_, O_), (O_, O_, O_), (O_, P_, O_)])
def test_shape_mask_identical(bc):
    """Further generator shapes (S26; Fig. 2d/e): ellipsoids, +-45 degree columns, a few spheres and
    arbitrarily oriented capped cylinders -- the mask must be the oracle's bit for bit."""
    cfg = cfg_of(44, 30, 20, bc, incl_rmin=0.8, incl_rmax=1.7, seed=8)
    p = oracle_params(cfg)
    s = make_solver(cfg)
    sh = I.shape_list(cfg, 9, 5)
    rng = np.random.default_rng(3)
    extra = np.zeros((6, 10), np.float32)
    extra[:3, 0] = 2                                                 # capped cylinders with any axis
    extra[:, 1:4] = rng.uniform(0, 10, (6, 3))
    extra[:, 4:7] = rng.uniform(0.6, 2.5, (6, 3))
    extra[:, 7:10] = rng.normal(size=(6, 3))
    extra[5, 1:5] = (0.1, 0.2, 0.1, 3.0)                             # a sphere through the corner (kind 0)
    sh = np.concatenate([sh, extra])
    s.set_pinning_shapes(sh, -1.0, 1.0)
    eps = s.get_eps().cpu().numpy()
    ref = O.epsilon_from_shapes(p, sh, -1.0, 1.0)
    assert np.array_equal(eps, ref.astype(np.float32))
    assert 0.05 < (eps < 0).mean() < 0.7
    for kind in (0, 1, 2):
        one = sh[sh[:, 0] == kind]
        s.set_pinning_shapes(one, -0.5, 1.0)
        assert np.array_equal(s.get_eps().cpu().numpy(), O.epsilon_from_shapes(p, one, -0.5, 1.0).astype(np.float32))
    s.set_pinning_shapes(np.zeros((0, 10), np.float32), -1.0, 0.5)  # empty list
    assert np.all(s.get_eps().cpu().numpy() == np.float32(0.5))
    from paper_1409_8340_b200.binding import TdglError
    bad = sh[:2].copy()
    bad[1, 0] = 3                                                    # unknown kind
    with pytest.raises(TdglError):
        s.set_pinning_shapes(bad)
    bad = sh[-8:-7].copy()
    bad[0, 7:10] = 0                                                 # a column without an axis
    assert bad[0, 0] == 2
    with pytest.raises(TdglError):
        s.set_pinning_shapes(bad)
    s.close()


def test_columnar_defects_run():
    """Fig. 2(e): +-45 degree columnar defects in a vertical field, 40 noisy driven steps against the oracle."""
    cfg = cfg_of(64, 32, 24, (P_, P_, O_), Bz=0.3, Jx=0.02, temperature=1e-3, incl_rmin=1.0, incl_rmax=1.5, seed=12)
    p = oracle_params(cfg)
    s = make_solver(cfg)
    sh = I.shape_list(cfg, 3, 6)
    eps = O.epsilon_from_shapes(p, sh, -1.0, 1.0)
    s.set_pinning_shapes(sh, -1.0, 1.0)
    bx_req, bz_req = cfg.requested_field()
    Bx, Bz, _, _ = O.snap_field(p, f32(bx_req), f32(bz_req))
    s.set_field_current(Bx=bx_req, Bz=bz_req, Jx=cfg.Jx)
    psi0 = I.initial_psi(cfg)
    st = O.State(psi=psi0.astype(np.complex128), mu=np.zeros(p.shape))
    s.set_state(torch.from_numpy(psi0), torch.zeros(p.shape, dtype=torch.float32), 0.0)
    s.step(40)
    counts, _ = s.sweep_log(40)
    O.run(p, st, eps, Bx, Bz, f32(cfg.Jx), 40, sweep_counts=counts)
    psi, mu = s.get_psi_mu()
    assert np.max(np.abs(psi.cpu().numpy() - st.psi)) <= 1e-4
    assert rel_l2(psi.cpu().numpy(), st.psi) <= 1e-5
    assert np.max(np.abs(mu.cpu().numpy() - st.mu)) <= 1e-4 * max(1.0, np.max(np.abs(st.mu)))
    s.close()


# ---------------------------------------------------------------------------------------------------
# a6: rho = div j_s
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc", ALL_BC)
@pytest.mark.parametrize("shape", [(34, 13, 11), (132, 37, 9)])
def test_rho_kernel(bc, shape):
    nx, ny, nz = shape
    cfg = cfg_of(nx, ny, nz, bc, Bx=0.07, Bz=0.21)
    psi0, mu0 = I.random_state(cfg, seed=11)
    K0 = 0.37 if bc[0] == P_ else 0.0
    p, st, eps, (Bx, Bz), s = setup_pair(cfg, psi0=psi0, mu0=mu0, K0=K0)
    rho = s.debug_rho().cpu().numpy()
    ref = O.supercurrent_divergence(p, st.psi, O.paper_links(p, K0, Bx, Bz))
    scale = np.max(np.abs(ref))
    assert np.max(np.abs(rho - ref)) < 2e-6 * max(scale, 1.0) * 24
    assert rel_l2(rho, ref) < 2e-6
    s.close()


# ---------------------------------------------------------------------------------------------------
# a7: Poisson solve
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc", ALL_BC)
@pytest.mark.parametrize("shape", [(32, 16, 8), (30, 12, 10), (64, 64, 32)])
def test_poisson_solve(bc, shape):
    nx, ny, nz = shape
    cfg = cfg_of(nx, ny, nz, bc)
    p = oracle_params(cfg)
    s = make_solver(cfg)
    rng = np.random.default_rng(4)
    w = O.site_weights(p)
    rho = rng.standard_normal(p.shape)
    rho -= np.sum(w * rho) / np.sum(w)                       # solvable right side (S6)
    rho32 = rho.astype(np.float32)
    mu = s.debug_poisson(torch.from_numpy(rho32)).cpu().numpy().astype(np.float64)
    ref = O.solve_poisson(p, rho32.astype(np.float64))
    scale = np.max(np.abs(ref))
    assert np.max(np.abs(mu - ref)) < 2e-5 * scale
    assert abs(np.sum(w * mu)) / np.sum(w) < 1e-5 * scale           # S7: weighted zero mode removed
    # and it solves the equation: Delta_h mu = rho up to fp32 rounding of mu times |Delta_h|
    res = O.laplacian_real(p, mu) - rho32
    assert np.max(np.abs(res)) < 24 * 4e-6 * scale + 1e-4
    s.close()


@pytest.mark.parametrize("bc,shape", [((P_, P_, O_), (512, 256, 6)), ((P_, P_, P_), (256, 128, 64)),
                                      ((P_, P_, O_), (128, 1024, 3)), ((P_, P_, P_), (1024, 64, 128)),
                                      ((P_, O_, P_), (64, 20, 256)), ((O_, P_, P_), (30, 512, 64)),
                                      ((O_, O_, O_), (1024, 40, 6)), ((P_, O_, O_), (64, 1000, 5)),
                                      ((O_, O_, P_), (514, 300, 8)), ((O_, P_, O_), (1366, 64, 3)),
                                      # prime-factor DCT-I (dct_pfa.cu): n = 1024, 256, 64 along x (rows) and y (columns),
                                      # odd row counts, ragged column groups, film
                                      ((O_, O_, P_), (64, 1024, 4)), ((O_, O_, O_), (256, 256, 8)), ((O_, P_, P_), (1024, 5, 3)),
                                      ((P_, O_, O_), (36, 1024, 3)), ((O_, O_, P_), (1024, 64, 1)), ((P_, O_, P_), (70, 256, 5)),
                                      ((O_, O_, O_), (1024, 1024, 4))])
def test_poisson_solve_fast_transform_sizes(bc, shape):
    """The register-blocked Hartley kernels (n = 64..1024), x pass, strided pass and the fused
    transform-divide-transform of a periodic z axis; Bluestein and prime-factor DCT-I on open axes."""
    nx, ny, nz = shape
    cfg = cfg_of(nx, ny, nz, bc)
    p = oracle_params(cfg)
    s = make_solver(cfg)
    rng = np.random.default_rng(6)
    w = O.site_weights(p)
    rho = rng.standard_normal(p.shape)
    rho -= np.sum(w * rho) / np.sum(w)
    rho32 = rho.astype(np.float32)
    mu = s.debug_poisson(torch.from_numpy(rho32)).cpu().numpy().astype(np.float64)
    ref = O.solve_poisson(p, rho32.astype(np.float64))
    scale = np.max(np.abs(ref))
    assert np.max(np.abs(mu - ref)) < 2e-5 * scale
    assert rel_l2(mu, ref) < 5e-6
    s.close()


def test_poisson_anisotropic_mesh():
    cfg = cfg_of(32, 16, 12, (P_, P_, O_))
    hxyz = (0.5, 0.4, 0.7)
    p = oracle_params(cfg, hxyz=hxyz, g=1.3)
    s = make_solver(cfg, hxyz=hxyz, g=1.3)
    rng = np.random.default_rng(5)
    w = O.site_weights(p)
    rho = rng.standard_normal(p.shape)
    rho -= np.sum(w * rho) / np.sum(w)
    rho32 = rho.astype(np.float32)
    mu = s.debug_poisson(torch.from_numpy(rho32)).cpu().numpy()
    ref = O.solve_poisson(p, rho32.astype(np.float64))
    assert np.max(np.abs(mu - ref)) < 2e-5 * np.max(np.abs(ref))
    s.close()


# ---------------------------------------------------------------------------------------------------
# a7: iterative refinement of the mu solve on meshes with a large white-noise gain (refine.cu)
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("shape,bc", [((1026, 9, 17), (O_, O_, O_)), ((1026, 3, 1), (O_, O_, P_)), ((1300, 9, 1), (O_, P_, P_)),
                                      ((700, 6, 5), (P_, P_, P_)), ((600, 8, 9), (P_, O_, O_))])
def test_mu_refinement_restores_the_gate_for_rough_states(shape, bc):
    """rho = div j_s of a ROUGH state (|psi| ~ 0.8, random phase per site: max|rho| ~ 15) on meshes with one long
    axis.  Without refinement the fp32 roundings of rho and of the transform passes, amplified by the low modes,
    miss the 2e-5 gate; one refinement step with the fp64 residual (rho re-evaluated from psi in fp64) meets it."""
    nx, ny, nz = shape
    cfg = cfg_of(nx, ny, nz, bc, Bz=0.3, Bx=0.0 if nz == 1 else 0.04, Jx=0.02 if bc[0] == P_ else 0.0, seed=1)
    psi0, mu0 = I.random_state(cfg, seed=2, amp=0.8)
    K0 = 0.1 if bc[0] == P_ else 0.0
    err = {}
    for refine in (False, True):
        p, st, eps, (Bx, Bz), s = setup_pair(cfg, psi0=psi0, mu0=mu0, K0=K0, fixed_sweeps=1, with_pinning=False,
                                             mu_refine=refine)
        assert s.mu_refine_enabled() == refine
        # (a) the solver alone, on the fp32 rho the kernel produced: mu vs the fp64 solve of that same rho
        rho = s.debug_rho()
        mu_s = s.debug_poisson(rho).cpu().numpy()
        ref_s = O.solve_poisson(p, rho.cpu().numpy().astype(np.float64))
        err[refine, "solver"] = float(np.max(np.abs(mu_s - ref_s))) / max(1.0, float(np.max(np.abs(ref_s))))
        # (b) the whole path of a time step (rho from psi, K update in between): one step of one sweep on both sides
        s.step(1)
        O.step(p, st, eps, Bx, Bz, f32(cfg.Jx), fixed_sweeps=1)
        psi, mu = s.get_psi_mu()
        assert np.max(np.abs(psi.cpu().numpy() - st.psi)) < 5e-6
        err[refine, "step"] = float(np.max(np.abs(mu.cpu().numpy() - st.mu))) / max(1.0, float(np.max(np.abs(st.mu))))
        s.close()
    print(shape, bc, {k: f"{v:.1e}" for k, v in err.items()})
    assert err[True, "solver"] < 2e-6 and err[True, "step"] < 2e-5
    assert err[False, "solver"] > 3 * err[True, "solver"]        # the refinement is what does it


def test_mu_gain_and_the_automatic_refinement_rule():
    """tdgl_mu_gain is the white-noise gain of Delta_h^{-1} (exact sum by numpy on small meshes); refinement is
    automatic above TDGL_MU_REFINE_GAIN = 200 and off for the 3D BASELINE grids."""
    from paper_1409_8340_b200 import Solver, TdglParams
    from paper_1409_8340_b200.binding import lib
    import ctypes as C

    def gain_c(nx, ny, nz, bc, h=(0.5, 0.5, 0.5), g=1.0):
        p = TdglParams()
        p.struct_size = C.sizeof(TdglParams)
        p.nx, p.ny, p.nz = nx, ny, nz
        p.hx, p.hy, p.hz = h
        p.dt, p.u, p.g, p.eps_tol, p.max_sweeps = 0.1, 1.0, g, 1e-6, 10
        p.bc[0], p.bc[1], p.bc[2] = bc
        p.flags = 1
        return lib().tdgl_mu_gain(C.byref(p))

    for (nx, ny, nz), bc, h, g in [((34, 13, 11), (P_, O_, O_), (0.5, 0.4, 0.7), 1.3), ((200, 6, 1), (O_, P_, P_), (0.5, 0.5, 0.5), 1.0),
                                   ((64, 64, 32), (P_, P_, O_), (0.5, 0.5, 0.5), 1.0)]:
        p = O.Params(nx, ny, nz, hx=h[0], hy=h[1], hz=h[2], g=g, bc=(bc[0], bc[1], P_ if nz == 1 else bc[2]))
        lam = O.laplacian_eigenvalues(p).ravel()
        lam = lam[np.abs(lam) > 1e-12]
        exact = math.sqrt(np.sum(1.0 / lam ** 2) / p.n_sites)
        assert abs(gain_c(nx, ny, nz, bc, h, g) - exact) < 1e-2 * exact
    assert gain_c(512, 512, 256, (P_, P_, O_)) < 1.0 and gain_c(1024, 1024, 512, (O_, O_, O_)) < 3.0
    assert gain_c(1026, 3, 1, (O_, O_, P_)) > 400.0
    s = Solver(1026, 4, 1, bc=(O_, P_, P_))
    assert s.mu_refine_enabled() and s.mu_gain() > 200.0
    s.close()
    s = Solver(64, 64, 32, bc=(P_, P_, O_))
    assert not s.mu_refine_enabled()
    s.close()


# ---------------------------------------------------------------------------------------------------
# a3 + a4 + a5 + a6 + a7: one full step with a prescribed number of sweeps, every boundary combination
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc", ALL_BC)
@pytest.mark.parametrize("host_loop", [False, True])
def test_one_step_fixed_sweeps(bc, host_loop):
    cfg = cfg_of(36, 14, 10, bc, Bx=0.05, Bz=0.3, Jx=0.02 if bc[0] == P_ else 0.0, temperature=1e-3,
                 incl_fraction=0.15, incl_rmin=1.0, incl_rmax=2.0, seed=2)
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
    # the residual the kernel reduced is the oracle's
    assert abs(ob.max_resid2 - st.max_resid2) <= 2e-3 * st.max_resid2 + 1e-12
    s.close()


def test_convergence_test_and_cap():
    """Eq. (34): stop at the first sweep whose input residual is below eps_tol; S10: cap + warning."""
    cfg = cfg_of(32, 16, 8, (P_, P_, P_), Bz=0.2)
    psi0, _ = I.random_state(cfg, seed=3, amp=0.7)
    p, st, eps, (Bx, Bz), s = setup_pair(cfg, psi0=psi0)
    s.step(1)
    O.step(p, st, eps, Bx, Bz, 0.0)
    ob = s.observables()
    assert ob.sweeps_last == st.sweeps_last and ob.status == 0
    tr = st.resid_trace[0]
    assert tr[-1] < p.eps_tol <= tr[-2]
    s.set_solver(1e-30, 3, 0)
    s.step(1)
    from paper_1409_8340_b200 import lib, TdglObs
    import ctypes
    o = TdglObs()
    rc = lib().tdgl_observables(s.h, ctypes.byref(o))
    assert rc == 1 and o.status == 1 and o.sweeps_last == 3           # TDGL_WMAXSWEEPS
    s.close()


def test_graph_and_host_loop_are_bit_identical():
    cfg = cfg_of(64, 32, 16, (P_, P_, O_), Bz=0.2, Jx=0.02, temperature=1e-3, incl_fraction=0.1, incl_rmin=1.5,
                 incl_rmax=1.5)
    out = []
    for host_loop in (False, True):
        p, st, eps, B, s = setup_pair(cfg, host_loop=host_loop)
        s.step(12)
        psi, mu = s.get_psi_mu()
        c, r = s.sweep_log(12)
        out.append((psi.cpu().numpy(), mu.cpu().numpy(), c, r, s.launch_count()))
        s.close()
    assert np.array_equal(out[0][0], out[1][0]) and np.array_equal(out[0][1], out[1][1])
    assert np.array_equal(out[0][2], out[1][2]) and np.array_equal(out[0][3], out[1][3])
    assert out[0][4] > 12 * 8


# ---------------------------------------------------------------------------------------------------
# a8: observables
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc", [(P_, P_, P_), (P_, P_, O_), (O_, O_, O_), (P_, O_, P_)])
def test_observables(bc):
    cfg = cfg_of(32, 24, 10, bc, Bx=0.04, nz_flux=3 if bc[0] == P_ and bc[1] == P_ else None, Bz=0.2,
                 incl_fraction=0.1, incl_rmin=1.0, incl_rmax=2.0)
    rng = np.random.default_rng(8)
    shape = (cfg.nz, cfg.ny, cfg.nx)
    psi0 = ((1.0 + 0.4 * rng.uniform(-1, 1, shape)) * np.exp(1j * rng.uniform(-math.pi, math.pi, shape))).astype(np.complex64)
    p, st, eps, (Bx, Bz), s = setup_pair(cfg, psi0=psi0, K0=0.2 if bc[0] == P_ else 0.0)
    ob = s.observables()
    links = O.paper_links(p, st.K, Bx, Bz)
    F = O.free_energy(p, st.psi, eps, links)
    assert abs(ob.free_energy - F) < 2e-6 * abs(F) + 1e-6 * p.n_sites
    assert abs(ob.mean_abs2 - O.mean_abs2(st.psi)) < 1e-6
    assert abs(ob.vortices_per_slice - O.vortices_per_slice(p, st.psi, links, Bz)) < 1e-9
    if bc[0] == P_ and bc[1] == P_:
        assert ob.vortices_per_slice == 3.0                              # flux quantisation
    assert abs(ob.Bz_eff - Bz) < 1e-7 and abs(ob.Bx_eff - Bx) < 1e-7
    s.close()


# ---------------------------------------------------------------------------------------------------
# boundary: error behaviour
# ---------------------------------------------------------------------------------------------------
def test_error_codes():
    import ctypes as C
    from paper_1409_8340_b200 import TdglParams, lib, tdgl_workspace_bytes
    from paper_1409_8340_b200.binding import TdglError
    p = TdglParams()
    p.nx, p.ny, p.nz = 31, 8, 8                                          # odd nx
    p.hx = p.hy = p.hz = 0.5
    p.dt, p.u, p.g, p.eps_tol, p.max_sweeps = 0.1, 1.0, 1.0, 1e-6, 10
    assert tdgl_workspace_bytes(p) == 0
    h = C.c_void_p()
    assert lib().tdgl_create(C.byref(p), C.byref(h)) == -1               # TDGL_EINVAL
    p.nx = 32
    need = tdgl_workspace_bytes(p)
    assert need > 32 * 8 * 8 * 44
    buf = torch.empty(need // 2, dtype=torch.uint8, device="cuda")
    p.workspace_dev, p.workspace_bytes = (buf.data_ptr() + 255) // 256 * 256, need // 2 - 256
    assert lib().tdgl_create(C.byref(p), C.byref(h)) == -2               # TDGL_ENOMEM
    s = make_solver(cfg_of(32, 8, 8, (O_, P_, P_)))
    with pytest.raises(TdglError) as e:
        s.set_field_current(Bz=0.1, Jx=0.01)                             # open x + current
    assert e.value.code == -3
    with pytest.raises(TdglError) as e:
        s.set_field_current(By=0.1)
    assert e.value.code == -3
    s.close()


# ---------------------------------------------------------------------------------------------------
# degenerate sizes: the smallest meshes the ABI accepts (2 x 2 x 2, films 2 x 2), one-site-wide tiles, a single
# ragged pair past a tile / strip edge, a z extent of two planes
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("shape", [(2, 2, 2), (4, 3, 2), (2, 5, 3), (130, 9, 17), (256, 8, 33), (6, 2, 1), (2, 2, 1),
                                   (1026, 3, 1)])
@pytest.mark.parametrize("bc", [(P_, P_, P_), (O_, O_, O_), (P_, O_, P_)])
def test_degenerate_sizes(shape, bc):
    nx, ny, nz = shape
    if nz == 1:
        bc = (bc[0], bc[1], P_)
    cfg = cfg_of(nx, ny, nz, bc, Bz=0.3, Jx=0.02 if bc[0] == P_ else 0.0, temperature=1e-3, seed=1)
    psi0, mu0 = I.random_state(cfg, seed=2, amp=0.8)
    p, st, eps, (Bx, Bz), s = setup_pair(cfg, psi0=psi0, mu0=mu0, K0=0.1 if bc[0] == P_ else 0.0, fixed_sweeps=4,
                                         with_pinning=False)
    s.step(2)
    psi, mu = s.get_psi_mu()
    for _ in range(2):
        O.step(p, st, eps, Bx, Bz, f32(cfg.Jx), fixed_sweeps=4)
    assert np.max(np.abs(psi.cpu().numpy() - st.psi)) < 5e-6
    assert np.max(np.abs(mu.cpu().numpy() - st.mu)) < 2e-5 * max(1.0, np.max(np.abs(st.mu)))
    assert abs(s.observables().K - st.K) < 1e-7
    s.close()


# ---------------------------------------------------------------------------------------------------
# parameters away from the defaults: anisotropic mesh, anisotropy g, relaxation constant u (S1)
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc,nz", [((P_, P_, O_), 12), ((O_, P_, P_), 9), ((P_, O_, P_), 1)])
def test_anisotropic_mesh_g_and_u(bc, nz):
    cfg = cfg_of(40, 18, nz, bc, Bz=0.25, Bx=0.05 if nz > 1 else 0.0, Jx=0.02 if bc[0] == P_ else 0.0, temperature=1e-3,
                 incl_fraction=0.1, incl_rmin=1.0, incl_rmax=2.0, seed=9)
    psi0, mu0 = I.random_state(cfg, seed=4, amp=0.8)
    kw = dict(hxyz=(0.5, 0.4, 0.6), g=1.3, u=1.7)
    p, st, eps, (Bx, Bz), s = setup_pair(cfg, psi0=psi0, mu0=mu0, K0=0.1 if bc[0] == P_ else 0.0, fixed_sweeps=5, **kw)
    s.step(2)
    psi, mu = s.get_psi_mu()
    for _ in range(2):
        O.step(p, st, eps, Bx, Bz, f32(cfg.Jx), fixed_sweeps=5)
    ob = s.observables()
    assert np.max(np.abs(psi.cpu().numpy() - st.psi)) < 5e-6
    assert np.max(np.abs(mu.cpu().numpy() - st.mu)) < 2e-5 * max(1.0, np.max(np.abs(st.mu)))
    assert abs(ob.K - st.K) < 1e-7 and abs(ob.Ex - st.Ex) < 1e-7
    links = O.paper_links(p, st.K, Bx, Bz)
    F = O.free_energy(p, st.psi, eps, links)
    assert abs(ob.free_energy - F) < 2e-6 * abs(F) + 1e-6 * p.n_sites
    s.close()


@pytest.mark.parametrize("nz", [8, 1])
def test_free_energy_descends_on_the_gpu(nz):
    """P12 on the CUDA path: without drive, noise and potential the discrete free energy never increases
    (relaxation dynamics of Eq. 16; soft property of the CN + linearised scheme at h_t = 0.1)."""
    cfg = cfg_of(48, 48, nz, (P_, P_, P_), nz_flux=4, incl_fraction=0.1, incl_rmin=1.5, incl_rmax=2.5, seed=12)
    p, st, eps, B, s = setup_pair(cfg, solve_mu=False)
    last = s.observables().free_energy
    for _ in range(30):
        s.step(2)
        F = s.observables().free_energy
        assert F <= last + 1e-6 * abs(last)
        last = F
    s.close()
