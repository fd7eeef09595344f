#!/usr/bin/env python
"""I-V characteristic of a pinned vortex lattice (the protocol of BASELINE.json's third configuration; PAPER.md:129,
183: the voltage follows from E_x = d_t K): for every applied current J_x the solver runs `--steps` time steps and
the electric field is averaged over the second half of the leg.

    python -m paper_1409_8340_b200.examples.iv_curve --grid 128 128 64 --steps 400

Uses only the six calls of include/tdgl.h through the ctypes binding; needs a CUDA device (there is no CPU path).
"""
from __future__ import annotations

import argparse
import math
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--grid", type=int, nargs=3, default=[128, 128, 64], metavar=("NX", "NY", "NZ"))
    ap.add_argument("--field", type=float, default=0.2, help="|B| in H_c2")
    ap.add_argument("--tilt", type=float, default=30.0, help="tilt of B from z towards x, degrees")
    ap.add_argument("--currents", type=float, nargs="+", default=[0.005 * (i + 1) for i in range(10)])
    ap.add_argument("--steps", type=int, default=400, help="time steps per current")
    ap.add_argument("--temperature", type=float, default=1e-3)
    ap.add_argument("--fraction", type=float, default=0.15, help="volume fraction of spherical inclusions")
    ap.add_argument("--seed", type=int, default=0)
    args = ap.parse_args(argv)

    import tdgl_inputs as I
    from paper_1409_8340_b200 import Solver

    nx, ny, nz = args.grid
    cfg = I.Config("iv", nx, ny, nz, (I.PERIODIC, I.PERIODIC, I.OPEN if nz > 1 else I.PERIODIC),
                   Bx=args.field * math.sin(math.radians(args.tilt)) if nz > 1 else 0.0,
                   Bz=args.field * math.cos(math.radians(args.tilt)), temperature=args.temperature,
                   incl_fraction=args.fraction, incl_rmin=1.5, incl_rmax=3.0, seed=args.seed)
    s = Solver(nx, ny, nz, bc=cfg.bc, h=cfg.h, dt=cfg.dt, temperature=cfg.temperature, seed=cfg.seed)
    s.set_pinning(I.sphere_list(cfg), cfg.eps_in, cfg.eps_out)
    lx = cfg.lengths()[0]
    print(f"# grid {nx}x{ny}x{nz}, B = ({cfg.Bx:.4f}, 0, {cfg.Bz:.4f}), T = {cfg.temperature}, {args.steps} steps per point")
    print("#      J_x      <E_x>          V   sweeps/step   <|psi|^2>   vortices/slice")
    half = args.steps // 2
    for J in args.currents:
        s.set_field_current(Bx=cfg.Bx, Bz=cfg.Bz, Jx=J)       # restarts the running mean of E_x
        s.step(args.steps - half)                             # transient of this leg
        sw0 = s.observables().sweeps_total
        s.set_field_current(Bx=cfg.Bx, Bz=cfg.Bz, Jx=J)       # same drive: only restarts the mean
        s.step(half)
        ob = s.observables()
        print(f"{J:10.4f} {ob.Ex_mean:12.5e} {ob.Ex_mean * lx:10.4e} {(ob.sweeps_total - sw0) / max(half, 1):10.2f} "
              f"{ob.mean_abs2:11.4f} {ob.vortices_per_slice:12.1f}")
    s.close()


if __name__ == "__main__":
    main()
