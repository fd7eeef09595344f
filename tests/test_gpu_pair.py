"""`-m gpu`: the fused two-sweep kernel (march_pair.cu; temporal blocking of Eq. 33).

Two gates.  (1) Against the fp64 oracle, with the tolerances of the plain path.  (2) Against the
plain sweep kernel: x^{l+1}, x^{l+2}, both residuals and the J_av partial sums use the same arithmetic in the same
order, and criterion (34) is kept exact by discarding a pair whose first sweep already met it, so psi, mu, K, the sweep
counts and the residual log must be BIT-identical whether pairs are never used (mode 0), used when predicted (mode 1) or
forced (mode 2, which exercises the discard-and-redo path; mode 3 also forces the separate J_av pass k_jav_tiles).
"""
import numpy as np
import pytest

import tdgl_inputs as I
from oracle import tdgl_oracle as O
from gpu_common import f32, rel_l2, setup_pair

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

P_, O_ = I.PERIODIC, I.OPEN
ALL_BC = [(a, b, c) for a in (P_, O_) for b in (P_, O_) for c in (P_, O_)]


def cfg_of(nx, ny, nz, bc, **kw):
    return I.Config(f"t{nx}x{ny}x{nz}", nx, ny, nz, tuple(bc), **kw)


def state_of(s):
    psi, mu = s.get_psi_mu()
    ob = s.observables()
    return psi.cpu().numpy().copy(), mu.cpu().numpy().copy(), ob


def test_eligibility():
    from paper_1409_8340_b200 import Solver
    for shape, yz, want in [((128, 32, 8), False, True), ((256, 48, 5), False, True), ((128, 32, 3), False, False),
                            ((128, 16, 8), False, False), ((128, 40, 8), False, False), ((64, 32, 8), False, False),
                            ((192, 32, 8), False, False), ((128, 32, 8), True, False), ((128, 32, 1), False, False)]:
        s = Solver(*shape, gauge_yz=yz) if yz else Solver(*shape)
        assert s.pair_stats()[0] == want, shape
        s.close()


@pytest.mark.parametrize("bc", ALL_BC)
@pytest.mark.parametrize("nsweeps", [5, 6])
def test_fixed_sweeps_pairs_vs_plain_and_oracle(bc, nsweeps):
    """Prescribed counts: 5 = init + two pairs, 6 = init + two pairs + one plain sweep.  Two z chunks (planes 0-5 and
    6-11), tiles on both y seams, jump phases P_{i,k} with B_x != 0, noise, inclusions, current."""
    cfg = cfg_of(128, 32, 12, bc, Bx=0.05, Bz=0.3, Jx=0.02 if bc[0] == P_ else 0.0, temperature=1e-3,
                 incl_fraction=0.15, incl_rmin=1.0, incl_rmax=2.0, seed=2)
    psi0, mu0 = I.random_state(cfg, seed=21, amp=0.8)
    K0 = 0.11 if bc[0] == P_ else 0.0
    res = []
    for mode in (0, 1):
        p, st, eps, (Bx, Bz), s = setup_pair(cfg, psi0=psi0, mu0=mu0, K0=K0, fixed_sweeps=nsweeps)
        assert s.pair_stats()[0]
        s.set_pair_mode(mode)
        s.step(2)
        res.append(state_of(s))
        _, pairs, redone = s.pair_stats()
        assert pairs == (0 if mode == 0 else 4) and redone == 0
        s.close()
    (psi_a, mu_a, ob_a), (psi_b, mu_b, ob_b) = res
    assert np.array_equal(psi_a.view(np.float32), psi_b.view(np.float32))
    assert np.array_equal(mu_a, mu_b)
    assert ob_a.K == ob_b.K and ob_a.Jav == ob_b.Jav and ob_a.max_resid2 == ob_b.max_resid2
    assert ob_b.sweeps_last == nsweeps and ob_b.sweeps_total == 2 * nsweeps
    for _ in range(2):
        O.step(p, st, eps, Bx, Bz, f32(cfg.Jx), fixed_sweeps=nsweeps)
    assert np.max(np.abs(psi_b - st.psi)) < 5e-6
    assert np.max(np.abs(mu_b - st.mu)) < 2e-5 * max(1.0, np.max(np.abs(st.mu)))
    assert abs(ob_b.K - st.K) < 1e-7 and abs(ob_b.Jav - st.Jav) < 1e-7
    assert abs(ob_b.max_resid2 - st.max_resid2) <= 2e-3 * st.max_resid2 + 1e-12


@pytest.mark.parametrize("bc,shape", [((P_, P_, O_), (256, 48, 20)), ((P_, P_, P_), (128, 64, 9)), ((O_, O_, O_), (256, 32, 7)),
                                      ((P_, O_, O_), (128, 48, 16))])
@pytest.mark.parametrize("host_loop", [False, True])
def test_tolerance_runs_are_bit_identical_in_all_pair_modes(bc, shape, host_loop):
    """Criterion (34) with the GPU's own decisions over 25 driven noisy steps: never / predicted / forced pairs give the
    same sweep counts, the same residual log and the same bits; forced pairs must hit the discard-and-redo path."""
    nx, ny, nz = shape
    cfg = cfg_of(nx, ny, nz, bc, Bx=0.04 if bc[1] == P_ and bc[2] == P_ else 0.03, Bz=0.3, Jx=0.02 if bc[0] == P_ else 0.0,
                 temperature=1e-3, incl_fraction=0.15, incl_rmin=1.0, incl_rmax=2.0, seed=5)
    nsteps = 25
    out = []
    for mode in (0, 1, 2, 3):                                         # 3: forced pairs that never sum J_av (k_jav_tiles does)
        p, st, eps, (Bx, Bz), s = setup_pair(cfg, host_loop=host_loop)
        s.set_pair_mode(mode)
        s.step(nsteps)
        psi, mu, ob = state_of(s)
        counts, resid = s.sweep_log(nsteps)
        out.append((psi, mu, ob, list(counts), list(resid), s.pair_stats()))
        s.close()
    ref = out[0]
    assert ref[5][1] == 0
    assert out[1][5][1] > 0                                           # the prediction did launch pairs
    assert out[2][5][1] >= out[1][5][1] and out[2][5][2] > 0          # forced: some pairs discarded and redone
    assert out[3][5][1:] == out[2][5][1:]
    for o in out[1:]:
        assert o[3] == ref[3] and o[4] == ref[4]
        assert np.array_equal(o[0].view(np.float32), ref[0].view(np.float32)) and np.array_equal(o[1], ref[1])
        assert o[2].K == ref[2].K and o[2].Jav == ref[2].Jav and o[2].Ex_mean == ref[2].Ex_mean
    assert min(ref[3]) >= 2 and max(ref[3]) >= 4
    # the predicted mode wastes little: at most one discarded pair per ten steps
    assert out[1][5][2] <= nsteps // 10 + 1, out[1][5]
    # and the run is the oracle's (replaying the GPU's counts; every decision valid on the oracle's own residuals)
    if not host_loop:
        O.run(p, st, eps, Bx, Bz, f32(cfg.Jx), nsteps, sweep_counts=ref[3])
        assert np.max(np.abs(out[1][0] - st.psi)) <= 1e-4
        assert rel_l2(out[1][0], st.psi) <= 1e-5
        assert np.max(np.abs(out[1][1] - st.mu)) <= 1e-4 * max(1.0, np.max(np.abs(st.mu)))


def test_schedule_and_cap_with_pairs():
    """Prescribed per-step schedules (2, 3, 4, 7 sweeps) never overshoot; the cap max_sweeps is honoured."""
    cfg = cfg_of(128, 32, 8, (P_, P_, O_), Bz=0.3, Jx=0.02, temperature=1e-3, seed=9)
    sched = [2, 3, 4, 7, 1, 5]
    res = []
    for mode in (0, 1):
        p, st, eps, (Bx, Bz), s = setup_pair(cfg)
        s.set_pair_mode(mode)
        s.set_sweep_schedule(sched)
        s.step(len(sched))
        counts, _ = s.sweep_log(len(sched))
        assert list(counts) == sched
        res.append(state_of(s))
        if mode == 1:
            assert s.pair_stats()[1] == 0 + 1 + 1 + 3 + 0 + 2
        s.set_solver(1e-30, 6, 0)                                      # tolerance never met: the cap ends the step
        s.set_pair_mode(2 if mode else 0)
        s.step(1)
        ob = s.observables()
        assert ob.sweeps_last == 6 and ob.status == 1
        res.append(state_of(s))
        s.close()
    assert np.array_equal(res[0][0].view(np.float32), res[2][0].view(np.float32))
    assert np.array_equal(res[1][0].view(np.float32), res[3][0].view(np.float32))


@pytest.mark.parametrize("shape", [(128, 32, 4), (128, 32, 33), (384, 32, 5), (128, 96, 17)])
@pytest.mark.parametrize("bc", [(P_, P_, P_), (O_, P_, O_), (P_, O_, P_)])
def test_smallest_and_ragged_meshes_forced_pairs(shape, bc):
    """The smallest eligible mesh (nz = 4, ny = 32), one-plane and ragged last z chunks (nz = 33, 17, 5), three tiles in x:
    forced pairs (incl. the discard-and-redo path and k_jav_tiles) against plain sweeps, bit for bit, 12 noisy steps."""
    nx, ny, nz = shape
    cfg = cfg_of(nx, ny, nz, bc, Bx=0.03, Bz=0.3, Jx=0.02 if bc[0] == P_ else 0.0, temperature=1e-3, incl_fraction=0.1,
                 incl_rmin=1.0, incl_rmax=2.0, seed=11)
    out = []
    for mode in (0, 3):
        p, st, eps, (Bx, Bz), s = setup_pair(cfg)
        s.set_pair_mode(mode)
        s.step(12)
        psi, mu, ob = state_of(s)
        out.append((psi, mu, ob, list(s.sweep_log(12)[0]), s.pair_stats()))
        s.close()
    a, b = out
    assert b[4][1] > 0 and a[3] == b[3]
    assert np.array_equal(a[0].view(np.float32), b[0].view(np.float32)) and np.array_equal(a[1], b[1])
    assert a[2].K == b[2].K and a[2].Jav == b[2].Jav
    O.run(p, st, eps, Bx, Bz, f32(cfg.Jx), 12, sweep_counts=a[3])
    assert np.max(np.abs(b[0] - st.psi)) <= 1e-4 and rel_l2(b[0], st.psi) <= 1e-5
