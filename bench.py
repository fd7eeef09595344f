#!/usr/bin/env python
"""bench.py -- TDGL hot-path throughput on B200 (BASELINE.json metric) with roofline, e2e and CPU baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C4] [--impl ours|reference]

A bench "step" is one TDGL time step (tdgl_step(h, 1)): fused init + first Jacobi sweep, the further
sweeps to criterion (34), J_av/K, rho, Poisson solve.  Prints ONE JSON line (rank 0).
  value      site-iterations/s = sites x Jacobi sweeps executed / device time of the K timed steps, state
             resident in HBM (CUDA events on the launching stream, max over ranks)
  e2e        the same metric with, every step, the state uploaded from pinned host memory
             (tdgl_set_state), one tdgl_step, and psi, mu and the observables read back to the host
  roofline   the sweep kernel with the largest share of the timed step (on C4 the fused two-sweep kernel k_march_pair,
             else the plain sweep): 32 B/site/sweep algorithmic bytes / mean launch duration (CUDA events around every
             launch of a host-loop run of the same workload) vs the measured HBM peak; `frac_of_min_traffic` for the
             pair kernel; both kernels also under roofline_sweep / roofline_pair; step_traffic = the whole step
  c5a        (C4 run only) a short resident leg on 1024x1024x512, open on all faces: steps/s at the largest grid
  cpu_baseline  the fp64 oracle (oracle/, numpy) timed on this box's host cores on a bounded sample
N > 1 (torchrun): independent replicas, one per GPU ("replicas only"); no collective on the
data path.  `--impl reference` times the oracle alone (rank 0).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

import numpy as np  # noqa: E402

import tdgl_inputs as I  # noqa: E402

METRIC = "TDGL site-iterations/s (whole time step) at 512x512x256 fp32"
UNIT = "site-iterations/s"
SWEEP_BYTES_PER_SITE = 32.0      # x^l 8 + b 8 + d 8 read, x^{l+1} 8 written


def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


def ncu_traffic(name="sweep_traffic.txt"):
    """Per-launch DRAM bytes of a sweep kernel from the committed ncu capture (profiles/sweep_traffic.txt, pair_traffic.txt)."""
    try:
        d = {}
        with open(os.path.join(ROOT, "profiles", name)) as f:
            for line in f:
                if line.startswith("#") or not line.strip():
                    continue
                k, v = line.split()
                d[k] = int(v)
        return d
    except Exception:
        return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)."""

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def reduce_over_ranks(vals, dist=None, device=None):
    """[time, count, count, ...] of this rank -> (max over ranks of vals[0], sums over ranks of the rest).
    Replicas only: this all-reduce of a few scalars AFTER the timed region is the only
    communication of the N > 1 bench; nothing on the data path is exchanged."""
    import torch
    t = torch.tensor([float(v) for v in vals], dtype=torch.float64, device=device)
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return [float(x) for x in t]
    tmax = t.clone(); dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
    tsum = t.clone(); dist.all_reduce(tsum, op=dist.ReduceOp.SUM)
    return [float(tmax[0])] + [float(x) for x in tsum[1:]]


def throughput(n_sites, sweeps_all, steps_per_rank, world, ms):
    """(site-iterations/s, steps/s) of the whole job: units all ranks processed / max-over-ranks time."""
    return n_sites * sweeps_all / (ms * 1e-3), world * steps_per_rank / (ms * 1e-3)


def replica_seed(cfg: I.Config, rank: int) -> int:
    """Replicas are independent problems: rank r draws its initial state and noise from Philox key seed + r."""
    return cfg.seed + rank


def config_dict(cfg: I.Config, world: int = 1):
    """The `config` object of the JSON line; the same keys for our arm and for `--impl reference`."""
    N = cfg.n_sites
    return {"workload": cfg.name, "grid": [cfg.nx, cfg.ny, cfg.nz], "bc": list(cfg.bc), "h": cfg.h, "dt": cfg.dt,
            "Bz": cfg.Bz, "Bx": cfg.Bx, "Jx": cfg.Jx, "T": cfg.temperature, "inclusion_fraction": cfg.incl_fraction,
            "eps_tol": 1e-6, "parallelism": "replicas only" if world > 1 else "1 GPU",
            "l2": "working set %.2f GB >> 126 MB L2, no flush needed" % (44.0 * N / 1e9),
            "loop": "CUDA graph per step, WHILE node around the sweep, no host sync"}


def make_solver(cfg: I.Config, host_loop=False, seed_offset=0, fp64=False, mu_iterative=False, mu_direct=False):
    from paper_1409_8340_b200 import Solver
    s = Solver(cfg.nx, cfg.ny, cfg.nz, bc=cfg.bc, h=cfg.h, dt=cfg.dt, eps_tol=1e-6, max_sweeps=100,
               temperature=cfg.temperature, seed=replica_seed(cfg, seed_offset), init_amp=cfg.init_amp, solve_mu=True,
               host_loop=host_loop, fp64=fp64, mu_iterative=mu_iterative, mu_direct=mu_direct)
    s.set_pinning(I.sphere_list(cfg), cfg.eps_in, cfg.eps_out)
    bx, bz = cfg.requested_field()
    s.set_field_current(Bx=bx, Bz=bz, Jx=cfg.Jx)
    return s


def _slab(cfg: I.Config):
    """The bounded sample: the same physics (boundary types, field, inclusions, current, noise) on a z-slab of
    the grid with the full x, y extent and 16 planes."""
    nz = min(cfg.nz, 16)
    return cfg.scaled(cfg.nx, cfg.ny, nz, f"{cfg.name} slab {cfg.nx}x{cfg.ny}x{nz}")


def _oracle_worker(args):
    """One host core: the fp64 oracle as it stands (numpy, one thread) stepping its own replica of the slab
    (Philox key and initial state offset by the worker index) until the time budget is spent."""
    name, widx, budget_s = args
    for v in ("OMP_NUM_THREADS", "OPENBLAS_NUM_THREADS", "MKL_NUM_THREADS"):
        os.environ[v] = "1"
    from dataclasses import replace
    from oracle import tdgl_oracle as O
    from gpu_common import f32, oracle_params
    sub = replace(_slab(I.CONFIGS[name]), seed=I.CONFIGS[name].seed + widx)
    p = oracle_params(sub)
    eps = O.epsilon_from_spheres(p, I.sphere_list(sub), sub.eps_in, sub.eps_out)
    bx, bz = sub.requested_field()
    Bx, Bz, _, _ = O.snap_field(p, f32(bx), f32(bz))
    st = O.State(psi=I.initial_psi(sub).astype(np.complex128), mu=np.zeros(p.shape))
    O.step(p, st, eps, Bx, Bz, f32(sub.Jx))                     # untimed: page-in, FFT plans
    t0 = time.perf_counter()
    sw0 = st.sweeps_total
    steps = 0
    while steps < 2 or (time.perf_counter() - t0 < budget_s and steps < 1000):
        O.step(p, st, eps, Bx, Bz, f32(sub.Jx))
        steps += 1
    return p.n_sites, steps, st.sweeps_total - sw0, time.perf_counter() - t0


def host_cores() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def oracle_sample(cfg: I.Config, budget_s: float = 20.0, cores: int = 0):
    """The fp64 oracle timed on ALL host cores of this box: one process per core (the oracle is single-threaded
    numpy), each stepping an independent replica of the slab sample for `budget_s` seconds.
    value = site-iterations of all workers / the slowest worker's time."""
    import multiprocessing as mp
    cores = cores or host_cores()
    sub = _slab(cfg)
    slab_gb = 16.0 * sub.n_sites * 40 / 1e9                    # ~40 fp64-complex temporaries per oracle step
    try:
        avail = os.sysconf("SC_AVPHYS_PAGES") * os.sysconf("SC_PAGE_SIZE") / 1e9
        cores = max(1, min(cores, int(0.6 * avail / slab_gb)))
    except (ValueError, OSError):
        pass
    t0 = time.perf_counter()
    if cores == 1:
        res = [_oracle_worker((cfg.name, 0, budget_s))]
    else:
        with mp.get_context("spawn").Pool(cores) as pool:
            res = pool.map(_oracle_worker, [(cfg.name, w, budget_s) for w in range(cores)])
    wall = time.perf_counter() - t0
    n_sites = res[0][0]
    steps_per_worker = max(r[1] for r in res)
    steps = sum(r[1] for r in res)
    sweeps = sum(r[2] for r in res)
    dt = max(r[3] for r in res)
    return {"value": n_sites * sweeps / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{sub.name} (C-order numpy fp64 oracle as it stands), {cores} independent replicas on {cores} "
                      f"host cores, {steps} steps and {sweeps} sweeps in {dt:.1f} s",
            "steps_per_s_on_sample": steps / dt, "ms_per_step_sample": 1e3 * dt * cores / steps,
            "steps_per_worker": steps_per_worker, "ms_per_worker_step": 1e3 * dt / steps_per_worker,
            "host_cores_available": host_cores(), "wall_s": wall}


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    # one pool of workers for the whole run: an untimed first step per worker (warm-up: page-in, FFT plans), then
    # oracle steps until the budget is spent (>= 2 per worker); sized so that the run ends within a few minutes
    t_all = time.perf_counter()
    res = oracle_sample(cfg, budget_s=min(60.0, max(10.0, 2.0 * args.steps)))
    v = res["value"]
    # `steps` / `ms_per_step` describe what was EXECUTED: every host core advanced its own replica of the slab sample by
    # `steps` oracle steps (the slowest worker's count) in parallel, `ms_per_step` wall milliseconds each, after one
    # untimed step; ms_per_step x steps is the timed wall time.  The K of the command line (`steps_requested`) only sizes
    # the time budget: K = 200 oracle steps of this slab would take half an hour.
    out = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": res["steps_per_worker"],
           "steps_requested": args.steps, "warmup": 1, "warmup_requested": args.warmup,
           "ms_per_step": res["ms_per_worker_step"], "ms_per_slab_step_per_core": res["ms_per_step_sample"], "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": dict(config_dict(cfg), parallelism="%d host cores" % res["cores"], l2="n/a (host)",
                          loop="oracle.step on a bounded slab sample per bench step; " + res["sample"]),
           "cpu_baseline": {"value": v, "unit": UNIT, "cores": res["cores"], "kind": "oracle", "sample": res["sample"]},
           "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0, "wall_s": time.perf_counter() - t_all}
    print(json.dumps(out), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=100)
    ap.add_argument("--config", default="C4")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-c5a", action="store_true", help="skip the short 1024x1024x512 leg that follows the C4 run")
    ap.add_argument("--pair-mode", type=int, default=1, help="tdgl_set_pair_mode: 1 automatic (default), 2 whenever the cap allows")
    ap.add_argument("--no-pairs", action="store_true", help="plain Jacobi sweeps only (tdgl_set_pair_mode 0): A/B against the fused two-sweep kernel")
    ap.add_argument("--fp64", action="store_true", help="the double-precision build (TDGL_FLAG_FP64; the paper's DP mode)")
    ap.add_argument("--mu-direct", action="store_true", help="with --fp64: direct mu solver (fp32 transforms inside fp64 iterative refinement, TDGL_FLAG_MU_DIRECT)")
    ap.add_argument("--mu-iterative", action="store_true", help="the paper's own pseudo-time mu solver (TDGL_FLAG_MU_ITERATIVE)")
    ap.add_argument("--h-tau", type=float, default=0.1, help="virtual time step of the pseudo-time mu solver (S20)")
    args = ap.parse_args()
    cfg = I.CONFIGS[args.config]
    if args.impl == "reference":
        run_reference(args, cfg)
        return

    import torch
    import torch.distributed as dist
    from paper_1409_8340_b200 import build as B
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if rank == 0:
        B.build()
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local_rank}"))
        dist.barrier()
    torch.cuda.set_device(local_rank)
    dev = torch.device(f"cuda:{local_rank}")
    W = max(args.warmup, 3)
    K = args.steps

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    # ---- resident run (graph mode) --------------------------------------------------------------
    mode = dict(fp64=args.fp64, mu_iterative=args.mu_iterative, mu_direct=args.mu_direct)
    iter_mu = (args.fp64 or args.mu_iterative) and not args.mu_direct
    bytes_per_site = SWEEP_BYTES_PER_SITE * (2.0 if args.fp64 else 1.0)
    s = make_solver(cfg, seed_offset=rank, **mode)
    if iter_mu:
        s.set_mu_solver(h_tau=args.h_tau)
    if args.no_pairs or args.pair_mode != 1:
        s.set_pair_mode(0 if args.no_pairs else args.pair_mode)
    s.step(W)
    barrier()
    ob0 = s.observables()
    l0 = s.launch_count()
    pair0 = s.pair_stats()
    sampler = ClockSampler(local_rank)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    s.step(K)
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop()
    ob1 = s.observables()
    mu_stats = None
    if args.mu_direct:
        sv, ps, rl = s.mu_direct_stats()
        mu_stats = {"refinement_passes_per_solve": ps / max(sv, 1), "last_max_residual": rl}
    elif iter_mu:
        outer, inner = s.mu_log(min(K, 1000))
        mu_stats = {"outer_per_step": float(np.mean(outer)), "inner_per_outer": float(np.mean([np.mean(i) for i in inner if i]))}
    launches = s.launch_count() - l0 - 2           # minus the two observables kernels
    pair1 = s.pair_stats()
    pairs = {"eligible": pair1[0], "mode": "off (--no-pairs)" if args.no_pairs else "automatic",
             "pairs_per_step": (pair1[1] - pair0[1]) / K, "discarded_per_step": (pair1[2] - pair0[2]) / K,
             "note": "a pair = two Jacobi sweeps in one pass over HBM (march_pair.cu); bit-identical to plain sweeps; a pair "
                     "whose first sweep already met criterion (34) is discarded and redone as one plain sweep"}
    sweeps = ob1.sweeps_total - ob0.sweeps_total
    ms, sweeps_all, launches_all = reduce_over_ranks([ms, sweeps, launches], dist if world > 1 else None, dev)
    launches_all = int(launches_all)
    N = cfg.n_sites
    value, steps_per_s = throughput(N, sweeps_all, K, world, ms)

    # ---- roofline of the sweep kernel: CUDA events around every sweep launch (host-loop run) ----
    roof = None
    roof_pair = None
    e2e = None
    if rank == 0 or world > 1:
        psi, mu = s.get_psi_mu()
        K0 = s.observables().K
        sh = make_solver(cfg, host_loop=True, seed_offset=rank, **mode)
        if iter_mu:
            sh.set_mu_solver(h_tau=args.h_tau)
        sh.set_state(psi, mu, K0)
        sh.set_pair_mode(0)                          # every sweep a plain sweep: the kernel this figure is about
        sh.step(3)
        sh.sweep_timing(1)
        sh.step(max(3, min(K, 40)))
        t_ms, n_l = sh.sweep_timing(0)
        peak, how = measured_peak()
        roof_pair = None
        if pair1[0] and not args.no_pairs:
            # the fused two-sweep kernel, timed the same way (pairs chosen by the library as in the resident run)
            sh.set_pair_mode(1)
            sh.step(3)
            sh.sweep_timing(2)
            sh.step(max(3, min(K, 40)))
            tp_ms, np_l = sh.sweep_timing(0)
            if np_l > 0:
                avg_p = tp_ms / np_l
                roof_pair = {"bound": "hbm", "kernel": "k_march_pair (two Jacobi sweeps in one pass, both residuals)",
                             "avg_launch_ms": avg_p, "launches_timed": int(np_l),
                             "algorithmic_bytes_per_launch": 2.0 * bytes_per_site * N,
                             "achieved": 2.0 * bytes_per_site * N / (avg_p * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                             "frac": 2.0 * bytes_per_site * N / (avg_p * 1e-3) / 1e9 / peak,
                             "min_traffic_bytes_per_launch": bytes_per_site * N,
                             "traffic": (ncu_traffic("pair_traffic.txt") or {}).get("dram_bytes_per_launch")
                             if (ncu_traffic("pair_traffic.txt") or {}).get("sites") == N else None,
                             "traffic_source": "profiles/pair_traffic.txt (one committed ncu --set full capture; not measured in this run)",
                             "frac_of_min_traffic": bytes_per_site * N / (avg_p * 1e-3) / 1e9 / peak,
                             "note": "`achieved` uses SURVEY 8(d)'s definition, 32 B/site/sweep x 2 sweeps per launch: a value "
                                     "above the peak is the point of temporal blocking (x^{l+1} never goes to HBM, b and d are "
                                     "read once for both sweeps: 32 B/site of DRAM traffic per PAIR, measured 2.16 GB per launch "
                                     "on C4, profiles/r02_pair_ncu_full.md); `frac_of_min_traffic` is that traffic over the peak"}
        if n_l > 0:
            avg_ms = t_ms / n_l
            ach = bytes_per_site * N / (avg_ms * 1e-3) / 1e9
            tr = ncu_traffic()
            kname = "k_march64<SWEEP>" if args.fp64 else ("k_march_film<SWEEP>" if cfg.nz == 1 else "k_march_tma<SWEEP>")
            roof = {"bound": "hbm", "kernel": kname + " (Jacobi sweep + max-residual)", "achieved": ach,
                    "peak": peak, "unit": "GB/s", "frac": ach / peak, "peak_source": how,
                    "avg_launch_ms": avg_ms, "launches_timed": int(n_l),
                    "algorithmic_bytes_per_launch": bytes_per_site * N,
                    "timed_in": "host-loop mode (TDGL_FLAG_HOST_LOOP): CUDA events around each single sweep launch after a "
                                "stream sync; `value` is timed in graph mode, where launches overlap their predecessors' tails",
                    "traffic": (tr or {}).get("dram_bytes_per_launch") if ((tr or {}).get("sites") == N and not args.fp64) else None,
                    "traffic_source": "profiles/sweep_traffic.txt (dram__bytes_read.sum + dram__bytes_write.sum of one committed "
                                      "ncu --set full capture of this kernel on this grid; not measured in this run)"}
        sh.close()
        del sh

        # ---- e2e: host buffers, per step H2D state -> step -> D2H state + observables ------------
        # Every step uploads its input state from pinned host memory, steps, and brings the new state and the
        # observables back to the host.  The copies run on their own streams (PCIe is full duplex): the upload of step
        # n + 1 and the download of step n - 1 overlap the kernels of step n, double-buffered on the device; the
        # observables read of every step synchronises with that step's kernels.
        if not args.no_e2e:
            Ke = max(1, min(K, 30))
            hp = torch.view_as_real(psi).cpu().pin_memory()
            hm = mu.cpu().pin_memory()
            dp = [torch.empty_like(torch.view_as_real(psi)) for _ in range(2)]
            dm = [torch.empty_like(mu) for _ in range(2)]
            op = [torch.empty_like(hp).pin_memory() for _ in range(2)]
            om = [torch.empty_like(hm).pin_memory() for _ in range(2)]
            h2d = hp.numel() * hp.element_size() + hm.numel() * hm.element_size()
            d2h = h2d + 136
            main = torch.cuda.current_stream()
            s_in, s_out = torch.cuda.Stream(), torch.cuda.Stream()
            ev_in = [torch.cuda.Event() for _ in range(2)]          # upload into slot done
            ev_used = [torch.cuda.Event() for _ in range(2)]        # the library has consumed the slot (set_state)
            ev_res = [torch.cuda.Event() for _ in range(2)]         # result of the step in its device buffers
            ev_out = [torch.cuda.Event() for _ in range(2)]         # download of the slot done
            keep = [None, None]

            def upload(slot):
                s_in.wait_event(ev_used[slot])
                with torch.cuda.stream(s_in):
                    dp[slot].copy_(hp, non_blocking=True)
                    dm[slot].copy_(hm, non_blocking=True)
                    ev_in[slot].record(s_in)

            for e in ev_used + ev_out:
                e.record(main)
            torch.cuda.synchronize()
            obx = s.observables()
            upload(0)
            nit = 2 + Ke
            for it in range(nit):
                slot = it & 1
                if it == 2:
                    torch.cuda.synchronize()
                    barrier()
                    sw_a = s.observables().sweeps_total
                    t0 = time.perf_counter()
                if it + 1 < nit:
                    upload(slot ^ 1)                      # next step's input: in flight during this step
                main.wait_event(ev_in[slot])
                s.set_state(torch.view_as_complex(dp[slot]), dm[slot], obx.K)
                ev_used[slot].record(main)
                s.step(1)
                main.wait_event(ev_out[slot])             # the download of two steps ago has left these buffers
                a, b2 = s.get_psi_mu()
                ev_res[slot].record(main)
                keep[slot] = (a, b2)
                s_out.wait_event(ev_res[slot])
                with torch.cuda.stream(s_out):
                    op[slot].copy_(torch.view_as_real(a), non_blocking=True)
                    om[slot].copy_(b2, non_blocking=True)
                    ev_out[slot].record(s_out)
                obx = s.observables()                     # syncs the library's stream: this step is done
            torch.cuda.synchronize()                      # ... and the last downloads
            te = time.perf_counter() - t0
            sw_e = obx.sweeps_total - sw_a
            te, sw_e = reduce_over_ranks([te, sw_e], dist if world > 1 else None, dev)
            e2e = {"value": N * sw_e / te, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                   "steps": Ke, "ms_per_step": 1e3 * te / Ke, "steps_per_s": world * Ke / te,
                   "how": "per step: state uploaded from pinned host memory, tdgl_set_state + tdgl_step + tdgl_get_psi_mu + "
                          "tdgl_observables, state downloaded to pinned host memory; uploads / downloads on their own streams "
                          "(double-buffered: the copies of neighbouring steps overlap this step's kernels)"}
    # ---- which kernel dominates the timed step: that one is `roofline` (the other stays under its own key) ------------
    step_ms = ms / K
    pps = (pair1[1] - pair0[1]) / K
    sweeps_ps = sweeps / K
    plain_ps = max(0.0, sweeps_ps - 1.0 - 2.0 * pps)          # sweep 1 is fused into the init kernel
    roofline, step_traffic = roof, None
    if roof is not None:
        roof["launches_per_step"] = plain_ps
        roof["share_of_step"] = plain_ps * roof["avg_launch_ms"] / step_ms
    if roof_pair is not None:
        roof_pair["peak_source"] = how
        roof_pair["launches_per_step"] = pps
        roof_pair["share_of_step"] = pps * roof_pair["avg_launch_ms"] / step_ms
        if roof is None or roof_pair["share_of_step"] > roof["share_of_step"]:
            roofline = roof_pair
    if roofline is not None:
        roofline = dict(roofline, dominant="largest share of the timed step among the kernels timed here; the other sweep "
                                          "kernel is under roofline_sweep / roofline_pair")
    if roof is not None and cfg.nz > 1 and not args.fp64 and not iter_mu:
        # minimum DRAM bytes of the step AS EXECUTED: init + first sweep 40 B/site, every fused pair 32, every
        # plain sweep 32, rho + J_av 12, the direct mu solve 56 (five passes over 4-8 B), over the time of the whole step
        per_site = 40.0 + 32.0 * pps + 32.0 * plain_ps + 12.0 + 56.0
        step_traffic = {"min_bytes_per_site": per_site, "achieved": per_site * N / (step_ms * 1e-3) / 1e9, "peak": peak,
                        "unit": "GB/s", "frac": per_site * N / (step_ms * 1e-3) / 1e9 / peak,
                        "note": "whole time step in graph mode: minimum real traffic of the kernels executed / ms_per_step / peak"}
    s.close()
    del s
    torch.cuda.empty_cache()

    # ---- steps/s at the largest BASELINE grid (C5a: 1024 x 1024 x 512, open on all faces), a short resident leg -----------
    c5a = None
    if args.config == "C4" and world == 1 and not args.no_c5a and not (args.fp64 or args.mu_iterative):
        c5 = I.CONFIGS["C5a"]
        if torch.cuda.mem_get_info()[0] > 60 * c5.n_sites:
            s5 = make_solver(c5)
            W5, K5 = 20, 30
            s5.step(W5)
            torch.cuda.synchronize()
            o0 = s5.observables()
            l5 = s5.launch_count()
            f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            f0.record()
            s5.step(K5)
            f1.record()
            torch.cuda.synchronize()
            ms5 = f0.elapsed_time(f1)
            l5 = s5.launch_count() - l5
            o1 = s5.observables()
            v5, sps5 = throughput(c5.n_sites, o1.sweeps_total - o0.sweeps_total, K5, 1, ms5)
            c5a = {"workload": "C5a", "grid": [c5.nx, c5.ny, c5.nz], "bc": list(c5.bc), "steps": K5, "warmup": W5,
                   "ms_per_step": ms5 / K5, "steps_per_s": sps5, "value": v5, "unit": UNIT,
                   "sweeps_per_step": (o1.sweeps_total - o0.sweeps_total) / K5, "gpu_launches": int(l5),
                   "state": {"mean_abs2": o1.mean_abs2, "status": o1.status},
                   "note": "north_star: steps/s up to 1024x1024x512; the literal all-open configs[4] with Jx = 0 (reading S14); the "
                           "run starts from the random initial state (protocol length is 500 steps: BASELINE.md section 4)"}
            s5.close()
            del s5

    if rank != 0:
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        cpu = oracle_sample(cfg)
    out = {
        "metric": METRIC if args.config == "C4" else METRIC.replace("512x512x256", "%dx%dx%d" % (cfg.nx, cfg.ny, cfg.nz)),
        "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64" if args.fp64 else "f32",
        "data": "synthetic", "steps_per_s": steps_per_s, "sweeps_per_step": sweeps_all / (K * world),
        "config": dict(config_dict(cfg, world), **({"mu_solver": "pseudo-time iteration (Eq. 40), host-driven loop"} if iter_mu else
                                                   ({"mu_solver": "direct: fp32 transform solver inside fp64 iterative refinement"} if args.mu_direct else {}))),
        "mu_iteration": mu_stats,
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches_all, "roofline": roofline, "roofline_sweep": roof,
        "roofline_pair": roof_pair, "step_traffic": step_traffic, "c5a": c5a,
        "pairs": pairs, "cpu_baseline": cpu,
        "state": {"mean_abs2": ob1.mean_abs2, "Ex": ob1.Ex, "K": ob1.K, "vortices_per_slice": ob1.vortices_per_slice,
                  "status": ob1.status},
    }
    print(json.dumps(out), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
