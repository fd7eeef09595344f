"""Helpers shared by the `-m gpu` parity tests: build the oracle's Params and the CUDA Solver from the
same seeded configuration (tdgl_inputs.py) and drive both."""
from __future__ import annotations

import numpy as np

import tdgl_inputs as I
from oracle import tdgl_oracle as O


def f32(x: float) -> float:
    """The fp32 value the C ABI receives, widened: the oracle is fed the very same number."""
    return float(np.float32(x))


def oracle_params(cfg: I.Config, eps_tol=1e-6, max_sweeps=100, solve_mu=True, temperature=None, hxyz=None, g=1.0, u=1.0,
                  mu_iterative=False, fp64=False, mu_direct=False):
    hx, hy, hz = hxyz if hxyz is not None else (cfg.h, cfg.h, cfg.h)
    return O.Params(cfg.nx, cfg.ny, cfg.nz, hx=f32(hx), hy=f32(hy), hz=f32(hz), dt=f32(cfg.dt), u=f32(u), g=f32(g),
                    bc=tuple(cfg.bc), eps_tol=f32(eps_tol), max_sweeps=max_sweeps,
                    temperature=f32(cfg.temperature if temperature is None else temperature), seed=cfg.seed,
                    solve_mu=solve_mu, mu_solver="pseudotime" if ((mu_iterative or fp64) and not mu_direct) else "direct",
                    h_tau=f32(0.1), eps_mu=f32(1e-6), eps_mu_in=f32(1e-6))


def make_solver(cfg: I.Config, eps_tol=1e-6, max_sweeps=100, solve_mu=True, temperature=None, host_loop=False,
                fixed_sweeps=0, hxyz=None, g=1.0, u=1.0, mu_refine=None, mu_iterative=False, fp64=False, mu_direct=False):
    from paper_1409_8340_b200 import Solver
    return Solver(cfg.nx, cfg.ny, cfg.nz, bc=cfg.bc, h=cfg.h, dt=cfg.dt, g=g, u=u, eps_tol=eps_tol, max_sweeps=max_sweeps,
                  fixed_sweeps=fixed_sweeps, temperature=cfg.temperature if temperature is None else temperature,
                  seed=cfg.seed, init_amp=cfg.init_amp, solve_mu=solve_mu, host_loop=host_loop, hxyz=hxyz, mu_refine=mu_refine, mu_iterative=mu_iterative, fp64=fp64,
                  mu_direct=mu_direct)


def setup_pair(cfg: I.Config, psi0=None, mu0=None, K0=0.0, with_pinning=True, **kw):
    """Returns (oracle params, oracle state, eps, (Bx, Bz) effective, solver) with identical inputs."""
    import torch
    p = oracle_params(cfg, **{k: v for k, v in kw.items() if k not in ("host_loop", "fixed_sweeps", "mu_refine")})
    s = make_solver(cfg, **kw)
    spheres = I.sphere_list(cfg) if with_pinning else np.zeros((0, 4), np.float32)
    eps = O.epsilon_from_spheres(p, spheres, cfg.eps_in, cfg.eps_out)
    s.set_pinning(spheres, cfg.eps_in, cfg.eps_out)
    bx_req, bz_req = cfg.requested_field()
    Bx, Bz, _, _ = O.snap_field(p, f32(bx_req), f32(bz_req))
    s.set_field_current(Bx=bx_req, Bz=bz_req, Jx=cfg.Jx)
    if psi0 is None:
        psi0 = I.initial_psi(cfg)
    mu_np = np.zeros(p.shape, np.float32) if mu0 is None else mu0
    st = O.State(psi=psi0.astype(np.complex128), mu=mu_np.astype(np.float64), K=float(K0))
    s.set_state(torch.from_numpy(psi0), torch.from_numpy(mu_np), float(K0))
    return p, st, eps, (Bx, Bz), s


def rel_l2(a, b):
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


# ---- sampled parity at sizes where a whole oracle step is out of reach ---------------------------------
def window_indices(origin, size, n, periodic):
    """Global indices of a window along one axis: origin may be negative / run past n on a periodic axis
    (indices wrap); on an open axis the window is clipped to [0, n)."""
    q = np.arange(origin, origin + size)
    if periodic:
        return np.mod(q, n)
    return q[(q >= 0) & (q < n)]


def oracle_window_solve(p, psi0, eps, Bx, Bz, K, step, sweeps, ii, jj, kk, mu=None):
    """The oracle's psi solve (build_system + `sweeps` Jacobi sweeps, Eq. 31/33) on the window ii x jj x kk of a
    large grid, from the window's own inputs only.  Jacobi information travels one site per sweep, so
    the result is the full-grid result at every site farther than `sweeps` sites from an ARTIFICIAL
    window edge; real open faces inside the window keep the oracle's open boundary rule.  `psi0`, `eps`
    (and `mu`) are window arrays of shape (len(kk), len(jj), len(ii)).  Returns (x, valid mask)."""
    n = (p.nx, p.ny, p.nz)
    idx = (ii, jj, kk)
    bcw, lo_real, hi_real = [], [], []
    for a in range(3):
        op = p.bc[a] == O.OPEN
        whole = (not op) and len(idx[a]) == n[a]             # the window spans a periodic axis: its wrap is the real one
        lo_real.append(whole or (op and idx[a][0] == 0))
        hi_real.append(whole or (op and idx[a][-1] == n[a] - 1))
        bcw.append(O.OPEN if (op and (lo_real[a] or hi_real[a])) else O.PERIODIC)
    pw = O.Params(len(ii), len(jj), len(kk), hx=p.hx, hy=p.hy, hz=p.hz, dt=p.dt, u=p.u, g=p.g, bc=tuple(bcw),
                  eps_tol=p.eps_tol, max_sweeps=p.max_sweeps, temperature=p.temperature, seed=p.seed,
                  solve_mu=p.solve_mu)
    links = O.paper_links_at(p, K, Bx, Bz, ii, jj, kk)
    zeta = None
    if p.temperature > 0.0:
        m = (kk[:, None, None].astype(np.uint64) * np.uint64(p.ny) + jj[None, :, None].astype(np.uint64)) \
            * np.uint64(p.nx) + ii[None, None, :].astype(np.uint64)
        zeta = O.langevin_noise_at(p, step, m)
    psi0 = psi0.astype(np.complex128)
    b, d = O.build_system(pw, psi0, np.zeros(pw.shape) if mu is None else mu.astype(np.float64), eps, links, zeta)
    x = psi0
    for _ in range(sweeps):
        x, _r = O.jacobi_sweep(pw, x, b, d, links)
    valid = np.ones(pw.shape, bool)
    for a, axis in ((0, 2), (1, 1), (2, 0)):
        m1 = np.ones(len(idx[a]), bool)
        if not lo_real[a]:
            m1[:sweeps + 1] = False
        if not hi_real[a]:
            m1[len(idx[a]) - sweeps - 1:] = False
        sh = [1, 1, 1]
        sh[axis] = len(idx[a])
        valid &= m1.reshape(sh)
    return x, valid
