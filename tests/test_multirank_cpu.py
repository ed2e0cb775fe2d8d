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


# ---- partitioned convolution (include/demag.h "Several GPUs"): host-side arithmetic and handle exchange ----------
def _shard_worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from paper_2308_08447_b200 import binding as B
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # every rank computes ITS ranges through the C ABI (no GPU needed) and "exports" 128 recognisable bytes
    rows = B.demag_shard_range(256, world, rank, 16)
    pairs = B.demag_shard_range(129, world, rank, 1)
    handles = B.gather_handles(bytes([rank]) * B.IPC_BYTES)
    out.put((rank, rows, pairs, handles))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_partition_and_handle_gather():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + os.getpid() % 2000
    procs = [ctx.Process(target=_shard_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, rows0, pairs0, h0), (r1, rows1, pairs1, h1) = res
    assert rows0 == (0, 128) and rows1 == (128, 128)                  # M / H rows (split along y here)
    assert pairs0 == (0, 64) and pairs1 == (64, 65)                   # frequency pairs: the last rank takes the remainder
    assert h0 == h1 == bytes([0]) * 128 + bytes([1]) * 128            # rank-major, the same on every rank


@pytest.mark.parametrize("n,align", [(129, 1), (256, 16), (4096, 4), (33, 1), (48, 16), (513, 1)])
@pytest.mark.parametrize("world", [1, 2, 3, 4, 5, 8, 16])
def test_shard_range_tiles_the_axis(n, world, align):
    sys.path.insert(0, ROOT)
    from paper_2308_08447_b200 import binding as B
    per = n // world // align * align
    if per == 0:
        with pytest.raises(B.DemagError) as e:
            B.demag_shard_range(n, world, 0, align)
        assert e.value.status == 2
        return
    pos = 0
    for r in range(world):
        b, c = B.demag_shard_range(n, world, r, align)
        assert b == pos and c >= per and b % align == 0
        assert c == per or r == world - 1                              # only the last rank differs
        pos += c
    assert pos == n
    for bad in [(n, world, world, align), (n, world, -1, align), (0, world, 0, align), (n, 0, 0, align), (n, world, 0, 0)]:
        with pytest.raises(B.DemagError) as e:
            B.demag_shard_range(*bad)
        assert e.value.status == 1


def test_exchange_volume_model():
    """Per-rank traffic of the two spectrum exchanges: every rank sends the pairs it does not own of its rows and the
    rows it does not own of its pairs, 2 x 3 (hq ny nz / G) (G-1)/G complex numbers -- with hq ~ nx/2 pairs of two
    frequencies that is 12 n_c (G-1)/G^2 reals, against the 18 n_c (G-1)/G^2 of the paper's x split."""
    sys.path.insert(0, ROOT)
    from paper_2308_08447_b200 import binding as B
    nx, ny, nz = 256, 256, 64
    hq = nx // 2 + 1
    for G in (2, 4, 8):
        sent = 0
        for r in range(G):
            _, nyr = B.demag_shard_range(ny, G, r, 16)
            _, nqr = B.demag_shard_range(hq, G, r, 1)
            sent += 3 * nz * nyr * (hq - nqr) * 4        # phase 0: 4 reals per pair quad, to the other ranks
            sent += 3 * nz * nqr * (ny - nyr) * 4        # phase 1
        model = 12 * nx * ny * nz * (G - 1) / G**2 * G   # all ranks
        assert abs(sent / model - 1) < 0.02              # hq = nx/2 + 1: the extra pair
