"""Host logic of bench.py's N > 1 path (N independent replicas, no data-path
collective): the timing is the maximum over ranks, the value the aggregate of all replicas.
Runs a world_size-2 gloo group on CPU."""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    import torch.distributed as dist
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 * (rank + 1), dist, "cpu")
    dist.barrier()
    out.put((rank, ms, bench.aggregate_value(world, 1000, 3, 5, ms)))
    dist.destroy_process_group()


def test_replicas_time_is_max_over_ranks_and_value_is_aggregate():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, value in got:
        assert ms == 20.0                                  # the slower replica's time, on every rank
        assert value == pytest.approx(2 * 1000 * 3 * 5 / 20e-3)


def test_single_process_needs_no_group():
    import bench
    assert bench.max_over_ranks(3.5, None, "cpu") == 3.5
    assert bench.aggregate_value(1, 10, 3, 2, 1.0) == pytest.approx(60000.0)


def test_reference_arm_runs_on_rank0_only(monkeypatch, capsys):
    """Ranks other than 0 exit without work in --impl reference."""
    import argparse
    import bench
    monkeypatch.setenv("RANK", "1")
    rc = bench.run_reference(argparse.Namespace(config=4, steps=1, warmup=0, gpus=2, n=None))
    assert rc == 0 and capsys.readouterr().out == ""
