"""The N > 1 path of bench.py on CPU: DESIGN.md section 7 ("replicas only") -- every rank steps its own
replica and the only cross-rank traffic is the contract's reduction (time = MAX over ranks, units =
SUM over ranks).  world_size 2, gloo, rendezvous on 127.0.0.1."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank: int, world: int, port: int, out):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    # rank r "measured" (r + 1) ms for 10 (r + 1) units
    t, u = bench.rank_reduce(float(rank + 1), 10.0 * (rank + 1), torch.device("cpu"))
    out.put((rank, t, u))
    dist.barrier()
    dist.destroy_process_group()


def test_rank_reduce_world2_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert got == [(0, 2.0, 30.0), (1, 2.0, 30.0)]


def test_rank_reduce_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.rank_reduce(3.5, 7.0, torch.device("cpu")) == (3.5, 7.0)


def test_reference_arm_runs_on_rank0_only(monkeypatch):
    """bench.py --impl reference under torchrun: ranks other than 0 return without work."""
    sys.path.insert(0, ROOT)
    import bench
    monkeypatch.setenv("RANK", "1")

    def boom(*a, **k):
        raise AssertionError("rank 1 must not build a workload")
    monkeypatch.setattr(bench, "make_workload", boom)

    class A:
        workload = "c0"; steps = 1; warmup = 0; gpus = 2
    bench.run_reference(A())


def test_bench_refuses_to_time_fewer_gpus_than_asked(capsys):
    """`python bench.py --gpus N` outside torchrun starts the N replica ranks itself; with fewer than N devices
    visible (none here) it must refuse with a clear message instead of timing one GPU and calling it N."""
    import argparse
    import bench
    rc = bench._respawn_under_torchrun(argparse.Namespace(gpus=8))
    assert rc == 2
    assert "refusing" in capsys.readouterr().err
