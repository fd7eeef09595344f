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


def test_replica_seeds_differ_per_rank():
    """Replicas are independent problems: bench.make_solver offsets the Philox seed by the rank."""
    import inspect
    sys.path.insert(0, ROOT)
    import bench
    src = inspect.getsource(bench.main)
    assert "seed_offset=rank" in src


def test_solver_binds_to_the_current_device_not_to_cuda0():
    """One process per GPU: bench.py calls torch.cuda.set_device(LOCAL_RANK) and the Solver must allocate there."""
    import inspect
    from paper_1409_8340_b200.binding import Solver
    sig = inspect.signature(Solver.__init__)
    assert sig.parameters["device"].default is None
    src = inspect.getsource(Solver.__init__)
    assert "current_device()" in src
    sys.path.insert(0, ROOT)
    import bench
    assert "torch.cuda.set_device(local_rank)" in inspect.getsource(bench.main)
