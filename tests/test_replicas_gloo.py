"""N > 1 is "replicas only": the only communication of bench.py is the reduction of a few
scalars after the timed region.  World-size-2 gloo test of exactly that code, on the CPU."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    # rank r: time 10 + r ms, 70 + r sweeps, 300 + r launches over K = 10 steps
    ms, sweeps, launches = bench.reduce_over_ranks([10.0 + rank, 70 + rank, 300 + rank], dist, torch.device("cpu"))
    value, sps = bench.throughput(1000, sweeps, 10, world, ms)
    if rank == 0:
        torch.save({"ms": ms, "sweeps": sweeps, "launches": launches, "value": value, "sps": sps}, out)
    dist.barrier()
    dist.destroy_process_group()


def test_rank_reduction_world_size_2(tmp_path):
    world, out = 2, str(tmp_path / "r.pt")
    mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
    r = torch.load(out)
    assert r["ms"] == 11.0                       # max over ranks
    assert r["sweeps"] == 141.0 and r["launches"] == 601.0      # sums over ranks
    assert r["value"] == pytest.approx(1000 * 141 / 11e-3)      # whole-job units / max time
    assert r["sps"] == pytest.approx(2 * 10 / 11e-3)


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_over_ranks([3.0, 5, 7]) == [3.0, 5.0, 7.0]
    v, s = bench.throughput(10, 5.0, 2, 1, 1.0)
    assert v == pytest.approx(10 * 5 / 1e-3) and s == pytest.approx(2 / 1e-3)


def _seed_worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    import tdgl_inputs as I
    from oracle import tdgl_oracle as O
    cfg = I.CONFIGS["C2"].scaled(8, 8, 4)
    seed = bench.replica_seed(cfg, rank)
    # what the replica's seed feeds: the Philox key of its initial state and Langevin stream
    psi0 = O.initial_state(O.Params(8, 8, 4, seed=seed), cfg.init_amp).psi
    t = torch.zeros(world, 1 + psi0.size, dtype=torch.float64)
    t[rank, 0] = seed
    t[rank, 1:] = torch.from_numpy(psi0.real.ravel().copy())
    dist.all_reduce(t)
    if rank == 0:
        torch.save(t, out)
    dist.barrier()
    dist.destroy_process_group()


def test_replicas_draw_from_different_philox_keys(tmp_path):
    """Replicas are independent problems: each rank's seed is distinct and gives a different initial field."""
    world, out = 2, str(tmp_path / "s.pt")
    mp.spawn(_seed_worker, args=(world, _free_port(), out), nprocs=world, join=True)
    t = torch.load(out)
    assert t[0, 0] != t[1, 0]
    assert float((t[0, 1:] - t[1, 1:]).abs().max()) > 1e-3


@pytest.mark.gpu
def test_solver_binds_to_the_current_device_not_to_cuda0():
    """One process per GPU: bench.py calls torch.cuda.set_device(LOCAL_RANK); the Solver allocates its workspace on
    the CURRENT device and enqueues on that device's current stream."""
    from paper_1409_8340_b200 import Solver
    cur = torch.cuda.current_device()
    s = Solver(16, 8, 4)
    assert s.device.index == cur and s.workspace.device.index == cur
    assert s.stream.cuda_stream == torch.cuda.current_stream(s.device).cuda_stream
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        s2 = Solver(16, 8, 4)
        assert s2.stream.cuda_stream == side.cuda_stream
        s2.step(2)
        assert s2.observables().steps == 2
        s2.close()
    s.close()
