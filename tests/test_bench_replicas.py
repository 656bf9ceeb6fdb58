"""The N > 1 path of bench.py on CPU: two gloo ranks (replicas only, no
collective on the data path; the only exchange is the max-over-ranks of the timed region)."""
import os
import sys

import pytest

torch = pytest.importorskip("torch")
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _rank(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    ms = [1500.0, 1725.5][rank]                         # rank 1 is the slower replica
    agreed = bench.max_over_ranks(ms, world)
    value = bench.replicas_value(8388608.0, 3, agreed * 1e-3, world)
    dist.barrier()
    out[rank] = (agreed, value)
    dist.destroy_process_group()


def test_two_replicas_report_whole_job_throughput_over_the_slowest_rank():
    world, port = 2, 29517 + os.getpid() % 200
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_rank, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0] == res[1]                             # every rank agrees on the figure
    agreed, value = res[0]
    assert agreed == 1725.5
    assert abs(value - 2 * 8388608.0 * 3 / 1.7255) < 1e-6 * value


def test_single_rank_is_the_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(12.5, 1) == 12.5
    assert bench.replicas_value(100.0, 2, 4.0, 1) == 50.0


def test_reference_arm_is_rank_zero_only(monkeypatch, capsys):
    sys.path.insert(0, ROOT)
    import bench
    from workloads import get_config

    class A:
        steps, warmup, gpus = 1, 0, 2
    bench.run_reference(A, get_config(1), rank=1)       # other ranks: no work, no output
    assert capsys.readouterr().out == ""
