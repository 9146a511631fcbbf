"""N > 1 path of bench.py on CPU: two gloo ranks, replicas only.

The data path has no collective; what the ranks share is the timing protocol: barrier, MAX over ranks of the
per-step time, job throughput = pairs of all ranks / that time.  This runs bench.aggregate_over_ranks under a real
torch.distributed process group (backend gloo, world_size 2, 127.0.0.1)."""
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
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)

    def all_reduce_max(x):
        t = torch.tensor([x], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t[0])

    dist.barrier()
    local_ms = 100.0 + 25.0 * rank                      # rank 1 is the slow replica
    step_ms, value = bench.aggregate_over_ranks(local_ms, 8256, world, all_reduce_max)
    out[rank] = (step_ms, value)
    dist.barrier()
    dist.destroy_process_group()


def test_two_replicas_max_over_ranks():
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
    assert set(out.keys()) == {0, 1}
    for rank in range(world):
        step_ms, value = out[rank]
        assert step_ms == pytest.approx(125.0)          # the slowest replica sets the job's time
        assert value == pytest.approx(2 * 8256 / 0.125)


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate_over_ranks(50.0, 36, 1) == (50.0, pytest.approx(36 / 0.05))


def test_rank_plumbing_and_step_counts(monkeypatch):
    """bench.py's launch plumbing without a GPU: under torchrun the ranks come from the environment; a plain
    `python bench.py --gpus N` (WORLD_SIZE unset) must spawn its N ranks itself; the driver's --steps / --warmup are
    honoured up to the per-configuration caps and never fall below three warm-up steps."""
    sys.path.insert(0, ROOT)
    import bench
    for k in ("WORLD_SIZE", "RANK", "LOCAL_RANK"):
        monkeypatch.delenv(k, raising=False)
    assert bench.rank_env(1) == (0, 0, 1, False)
    assert bench.rank_env(8) == (0, 0, 1, True)                  # nobody launched the ranks: bench spawns them
    monkeypatch.setenv("WORLD_SIZE", "4")
    monkeypatch.setenv("RANK", "3")
    monkeypatch.setenv("LOCAL_RANK", "3")
    assert bench.rank_env(4) == (3, 3, 4, False)
    assert bench.effective_counts("C5", None, 3) == (2, 3)
    assert bench.effective_counts("C5", 20, 5) == (2, 3)         # capped: a C5 apply takes the better part of a minute
    assert bench.effective_counts("C3", 20, 1) == (20, 3)        # at least three warm-up steps
    assert bench.effective_counts("C3", 1000, 50) == (50, 5)
    assert bench.effective_counts("C4", None, 3, quick=True) == (1, 1)


def test_reference_arm_exits_quietly_on_other_ranks(monkeypatch, capsys):
    """--impl reference under torchrun: rank 0 alone runs the oracle; the other ranks return without work or output."""
    sys.path.insert(0, ROOT)
    import argparse

    import bench
    args = argparse.Namespace(config="C1", steps=1, warmup=1, gpus=2)
    bench.run_reference(args, rank=1, world=2)
    assert capsys.readouterr().out == ""
