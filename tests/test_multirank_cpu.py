"""N > 1 plumbing of bench.py on CPU: two gloo ranks (the path does not shard without an
exchange step, so --gpus N runs N independent replicas; the only collective is the max-over-ranks of the times)."""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r "measured" (10 + r) ms in total, (1 + r) ms hot, (2 + 3 r) s end to end
    ms_total, ms_hot, t_e2e = bench.allreduce_max([10.0 + rank, 1.0 + rank, 2.0 + 3 * rank], torch.device("cpu"), world)
    val = bench.aggregate_throughput(world, 1000, 5, ms_total)
    out.put((rank, ms_total, ms_hot, t_e2e, val))
    dist.barrier()
    dist.destroy_process_group()


def test_two_replicas_max_time_and_aggregate():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms_total, ms_hot, t_e2e, val in res:
        assert (ms_total, ms_hot, t_e2e) == (11.0, 2.0, 5.0)          # max over ranks, on every rank
        assert val == pytest.approx(2 * 1000 * 5 / 11.0e-3)           # whole-job aggregate of the two replicas


def test_single_rank_is_identity():
    import torch
    sys.path.insert(0, ROOT)
    import bench
    assert bench.allreduce_max([3.0, 4.0], torch.device("cpu"), 1) == [3.0, 4.0]
    assert bench.aggregate_throughput(1, 10, 2, 1000.0) == 20.0
