"""The N>1 path of bench.py is "replicas only": no data-path collective, only the
max-over-ranks of the timings and the whole-job aggregate.  Covered here with world_size 2 over gloo."""
import os
import socket
import sys

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
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    assert bench.rank_env() == (world, rank, rank)
    mine = 10.0 + 5.0 * rank                       # rank 1 is the slow replica
    ms = bench.max_over_ranks(mine, world, torch.device("cpu"))
    out[rank] = (ms, bench.aggregate_value(world, 2.0736, ms))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_world2_gloo():
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    for r in range(world):
        ms, val = res[r]
        assert ms == 15.0                          # every rank sees the slowest rank's time
        assert abs(val - 2 * 2.0736 / 15e-3) < 1e-9


def test_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, 1, torch.device("cpu")) == 3.5
    assert bench.aggregate_value(1, 2.0, 1000.0) == 2.0


def test_reference_arm_runs_on_rank0_only(monkeypatch):
    sys.path.insert(0, ROOT)
    import bench
    monkeypatch.setenv("RANK", "1")
    monkeypatch.setenv("WORLD_SIZE", "2")

    class A:
        config, view, steps, warmup, gpus = 1, 0, 1, 0, 2
    assert bench.run_reference(A) is None          # other ranks exit without work
