"""`-m gpu`: host-side bookkeeping of libtdgl that the parity tests do not reach -- the launch counter in graph mode
(bench.py's `gpu_launches`), the warning latched when the pseudo-time mu iteration stops at a cap, per-device set-up
when one process drives two GPUs."""
import numpy as np
import pytest

import tdgl_inputs as I
from gpu_common import make_solver, setup_pair

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

P_, O_ = I.PERIODIC, I.OPEN


@pytest.mark.parametrize("shape,pair_mode", [((64, 48, 1), 0), ((128, 32, 8), 0), ((128, 32, 8), 2), ((34, 10, 6), 0)])
def test_graph_mode_launch_count_equals_the_host_loop_count(shape, pair_mode):
    """With a prescribed sweep count the host loop launches exactly the kernels the graph's WHILE node runs (no speculative
    launch once its predictor has seen one step), so the two counters must advance alike: the film sweep kernel, the plain
    3D sweep and the fused pair kernel all count themselves on the device (Ctl::body_launches)."""
    nx, ny, nz = shape
    cfg = I.Config("lc", nx, ny, nz, (P_, P_, P_ if nz == 1 else O_), Bz=0.3, Jx=0.02)
    deltas, states = [], []
    for host_loop in (False, True):
        _, _, _, _, s = setup_pair(cfg, host_loop=host_loop, fixed_sweeps=5, with_pinning=False)
        s.set_pair_mode(pair_mode)
        s.step(2)
        c0 = s.launch_count()
        s.step(6)
        deltas.append(s.launch_count() - c0)
        psi, mu = s.get_psi_mu()
        states.append((psi.cpu().numpy(), mu.cpu().numpy()))
        eligible, pairs, _ = s.pair_stats()
        assert (pairs > 0) == (pair_mode == 2 and eligible)
        s.close()
    assert deltas[0] == deltas[1] and deltas[0] >= 6 * (4 + 4), deltas      # 4 loop-body sweeps after the fused init + first sweep
    assert np.array_equal(states[0][0], states[1][0]) and np.array_equal(states[0][1], states[1][1])


def test_mu_iteration_stopped_by_a_cap_latches_a_warning():
    from paper_1409_8340_b200.binding import TDGL_WMUCAP, TDGL_WMAXSWEEPS, lib, TdglObs
    import ctypes as C
    cfg = I.Config("cap", 36, 14, 10, (P_, P_, O_), Bz=0.3, Jx=0.05)
    s = make_solver(cfg, mu_iterative=True)
    s.set_field_current(Bz=0.3, Jx=0.05)
    s.step(2)
    assert s.observables().status == 0                       # defaults: the iteration converges well inside its caps
    s.set_mu_solver(max_outer=1, max_inner=2)
    s.step(1)
    o = TdglObs()
    rc = lib().tdgl_observables(s.h, C.byref(o))
    assert rc == TDGL_WMUCAP and o.status == TDGL_WMUCAP
    s.set_mu_solver()                                        # latched: it stays after the caps are lifted again
    s.set_solver(1e-6, 2)                                    # ... and a Jacobi cap adds its own bit
    s.step(1)
    rc = lib().tdgl_observables(s.h, C.byref(o))
    assert o.status == (TDGL_WMUCAP | TDGL_WMAXSWEEPS) and rc == TDGL_WMAXSWEEPS
    s.close()


def test_open_axis_transform_tables_reach_every_device():
    """The prime-factor DCT-I keeps its twiddles in __constant__ memory, which exists once PER DEVICE: a second GPU driven
    by the same process must get its own copy (it used to be uploaded once per process).  Needs two GPUs."""
    if torch.cuda.device_count() < 2:
        pytest.skip("one GPU on this box: the per-device upload cannot be exercised")
    from oracle import tdgl_oracle as O
    from gpu_common import oracle_params
    cfg = I.Config("twodev", 64, 64, 8, (O_, O_, P_))
    p = oracle_params(cfg)
    rng = np.random.default_rng(2)
    w = O.site_weights(p)
    rho = rng.standard_normal(p.shape)
    rho -= np.sum(w * rho) / np.sum(w)
    ref = O.solve_poisson(p, rho.astype(np.float32).astype(np.float64))
    for dev in (0, 1):
        with torch.cuda.device(dev):
            s = make_solver(cfg)
            mu = s.debug_poisson(torch.from_numpy(rho.astype(np.float32))).cpu().numpy()
            assert np.max(np.abs(mu - ref)) < 1e-4 * max(1.0, np.max(np.abs(ref))), dev
            s.close()
