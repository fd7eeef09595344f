"""`-m gpu`: multi-step parity of the CUDA path against the fp64 oracle on the BASELINE.json configs.

Stated-up-front numbers (BASELINE.json north_star): without noise max|psi_gpu - psi_oracle| <= 1e-4 and
relative L2 <= 1e-5 after 100 steps in fp32; with noise (same Philox stream) vortex count and <|psi|^2>
within 1e-3.  mu: max|d mu| <= 1e-4 max(1, max|mu|).  Reading S9 (several results are correct
at the threshold): the GPU takes its own convergence decisions; the oracle re-runs with the GPU's
per-step sweep counts and must find each decision valid (its own residual trace crosses eps_tol at
that sweep, within the relative ambiguity band AMBIG), and parity is taken against that run.
"""
import numpy as np
import pytest

import tdgl_inputs as I
from oracle import tdgl_oracle as O
from gpu_common import f32, rel_l2, setup_pair

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

AMBIG = 2e-3     # relative half-width of the band around eps_tol inside which either decision is valid


def run_pair(cfg, nsteps, with_pinning=True, **kw):
    p, st, eps, (Bx, Bz), s = setup_pair(cfg, with_pinning=with_pinning, **kw)
    s.step(nsteps)
    psi, mu = s.get_psi_mu()
    counts, resid = s.sweep_log(nsteps)
    ob = s.observables()
    O.run(p, st, eps, Bx, Bz, f32(cfg.Jx), nsteps, sweep_counts=counts)
    return p, st, eps, (Bx, Bz), s, psi.cpu().numpy(), mu.cpu().numpy(), counts, resid, ob


def check_decisions(p, st, counts, fixed=False):
    """Every GPU decision is a valid outcome of Eq. (34) on the oracle's own residual trace."""
    n_amb = 0
    for step, (c, tr) in enumerate(zip(counts, st.resid_trace)):
        assert len(tr) == c
        if c < p.max_sweeps:
            assert tr[-1] < p.eps_tol * (1 + AMBIG), (step, c, tr)
        for l in range(c - 1):
            assert tr[l] >= p.eps_tol * (1 - AMBIG), (step, c, l, tr)
        if abs(tr[-1] / p.eps_tol - 1) < AMBIG or (c > 1 and abs(tr[-2] / p.eps_tol - 1) < AMBIG):
            n_amb += 1
    return n_amb


def test_C1_100_steps_pointwise():
    cfg = I.CONFIGS["C1"]
    p, st, eps, B, s, psi, mu, counts, resid, ob = run_pair(cfg, 100)
    check_decisions(p, st, counts)
    assert np.max(np.abs(psi - st.psi)) <= 1e-4
    assert rel_l2(psi, st.psi) <= 1e-5
    assert np.max(np.abs(mu - st.mu)) <= 1e-4 * max(1.0, np.max(np.abs(st.mu)))
    assert ob.vortices_per_slice == 4.0 and ob.steps == 100
    assert ob.sweeps_total == int(np.sum(counts))
    s.close()


def test_C1_tight_tolerance_gate():
    """S9 (iv): at eps_tol = 1e-10 the sweep count is immaterial; fp32 vs fp64 after 100 steps."""
    cfg = I.CONFIGS["C1"]
    p, st, eps, (Bx, Bz), s = setup_pair(cfg, eps_tol=1e-10, max_sweeps=200)
    s.step(100)
    psi, mu = s.get_psi_mu()
    O.run(p, st, eps, Bx, Bz, 0.0, 100)
    assert np.max(np.abs(psi.cpu().numpy() - st.psi)) <= 2e-5
    assert rel_l2(psi.cpu().numpy(), st.psi) <= 5e-6
    s.close()


def test_C2_no_noise_100_steps_pointwise():
    """C2 (64^3, inclusions, current) with the Langevin term off: pointwise gate."""
    cfg = I.CONFIGS["C2"]
    p, st, eps, B, s, psi, mu, counts, resid, ob = run_pair(cfg, 100, temperature=0.0)
    check_decisions(p, st, counts)
    assert np.max(np.abs(psi - st.psi)) <= 1e-4
    assert rel_l2(psi, st.psi) <= 1e-5
    assert np.max(np.abs(mu - st.mu)) <= 1e-4 * max(1.0, np.max(np.abs(st.mu)))
    assert abs(ob.K - st.K) < 1e-6 and abs(ob.Ex - st.Ex) < 1e-6
    s.close()


def test_C2_with_noise_statistics():
    """C2 with T = 1e-3: same Philox stream on both sides; vortex count and <|psi|^2> within 1e-3, and in
    fact pointwise agreement far below the noise amplitude."""
    cfg = I.CONFIGS["C2"]
    nsteps = 60
    p, st, eps, (Bx, Bz), s, psi, mu, counts, resid, ob = run_pair(cfg, nsteps)
    check_decisions(p, st, counts)
    links = O.paper_links(p, st.K, Bx, Bz)
    assert abs(ob.mean_abs2 - O.mean_abs2(st.psi)) <= 1e-3
    assert abs(ob.vortices_per_slice - O.vortices_per_slice(p, st.psi, links, Bz)) <= 1e-3
    assert np.max(np.abs(psi - st.psi)) <= 1e-4
    assert 5.0 <= np.mean(counts[20:]) <= 9.0          # paper: 6-7 sweeps in a dynamic steady state
    s.close()


@pytest.mark.parametrize("name,shape,nsteps", [("C3", (64, 64, 32), 30), ("C4", (64, 64, 32), 30),
                                                ("C5a", (48, 40, 24), 20), ("C5b", (48, 40, 24), 20)])
def test_replicas_of_large_configs(name, shape, nsteps):
    """C3..C5 physics (boundary types, tilted field, inclusions, current) on grids the oracle finishes in
    seconds, noise off for the pointwise gate and on for the statistics."""
    cfg = I.CONFIGS[name].scaled(*shape)
    p, st, eps, B, s, psi, mu, counts, resid, ob = run_pair(cfg, nsteps, temperature=0.0)
    check_decisions(p, st, counts)
    assert np.max(np.abs(psi - st.psi)) <= 1e-4
    assert rel_l2(psi, st.psi) <= 1e-5
    assert np.max(np.abs(mu - st.mu)) <= 1e-4 * max(1.0, np.max(np.abs(st.mu)))
    s.close()
    p, st, eps, (Bx, Bz), s, psi, mu, counts, resid, ob = run_pair(cfg, nsteps)
    check_decisions(p, st, counts)
    assert abs(ob.mean_abs2 - O.mean_abs2(st.psi)) <= 1e-3
    assert np.max(np.abs(psi - st.psi)) <= 1e-4
    s.close()


def test_smoke_entry():
    import __graft_entry__
    __graft_entry__.smoke()
