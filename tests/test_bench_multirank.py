"""Host logic of bench.py's N > 1 path on CPU: two gloo ranks, max-over-ranks timing and the replicas-only
aggregate (the path does not shard inside the library; --gpus N runs N independent replicas)."""
import os
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from paper_2504_16446_b200 import synth
    ms = [100.0, 140.0][rank]                      # rank 1 is the slow one
    dist.barrier()
    agreed = bench.max_over_ranks(ms, world, torch.device("cpu"))
    cfg = synth.get_config("C1")
    out[rank] = (agreed, bench.aggregate_throughput(cfg, world, agreed))
    dist.destroy_process_group()


def test_two_rank_max_and_aggregate():
    world, port = 2, 29500 + os.getpid() % 2000
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    from paper_2504_16446_b200 import synth
    cfg = synth.get_config("C1")
    for rank in range(world):
        agreed, value = res[rank]
        assert agreed == 140.0                                     # every rank reports the slowest rank's time
        assert value == pytest.approx(2 * cfg.vcp / 0.140 / 1e9)   # whole-job aggregate of two replicas


def test_single_rank_is_identity():
    import bench
    assert bench.max_over_ranks(12.5, 1, torch.device("cpu")) == 12.5
