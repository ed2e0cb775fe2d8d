"""The partitioned (several-GPU) convolution of include/demag.h "Several GPUs" (Fig. 1, Appendix A).

Only one GPU is available to the tests, and kernels of different ranks must never wait on one another on one device,
so the G ranks are G sharded plans in ONE process on ONE device, wired to each other's buffers with
demag_shard_set_peers and driven phase by phase (all ranks' phase 0, then all ranks' phase 1, ...): stream order
replaces the inter-rank barrier.  Every kernel, every peer address and the partition arithmetic are exactly those of a
G-process run; what differs is only how the pointers were obtained (IPC, covered by the two-process test below) and
the barrier (an NCCL all-reduce in binding.ShardedPlan.apply).

Bars: against the fp64 oracle as everywhere (2e-5 / 1e-11 of Ms), and BIT-EXACT against the one-GPU plan -- the
partitioned run executes the same butterflies on the same values in the same order, only the addresses differ.
"""
import os
import subprocess
import sys

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL32 = 2e-5
TOL64 = 1e-11
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


@pytest.fixture(scope="module")
def B():
    from paper_2308_08447_b200 import binding
    binding.lib()
    return binding


class Ranks:
    """G sharded plans on one device, wired together."""

    def __init__(self, B, n, h, prec, G, T=None, slab=0):
        self.B, self.G, self.n = B, G, n
        self.plans = [B.ShardedPlan(n, h, prec, rank=r, world=G, connect=False) for r in range(G)]
        bufs = [B.demag_shard_buffers(p.handle) for p in self.plans]
        for p in self.plans:
            B.demag_shard_set_peers(p.handle, [b[0] for b in bufs], [b[2] for b in bufs])
            p.set_kernel(T)
            if slab:
                B.demag_set_slab(p.handle, slab)

    def split(self, torch, M, dt):
        out = []
        for p in self.plans:
            y0, nyl = p.info["y0"], p.info["ny_loc"]
            out.append(torch.from_numpy(np.ascontiguousarray(M[:, :, y0:y0 + nyl, :])).to("cuda", dt))
        return out

    def apply(self, torch, Ml):
        Hl = [torch.full_like(m, float("nan")) for m in Ml]
        for ph in range(3):
            for p, m, h in zip(self.plans, Ml, Hl):
                self.B.demag_apply_sharded(p.handle, ph, m if ph == 0 else None, h if ph == 2 else None)
        torch.cuda.synchronize()
        return Hl

    def join(self, Hl):
        return np.concatenate([h.cpu().numpy().astype(np.float64) for h in Hl], axis=2)

    def close(self):
        for p in self.plans:
            p.close()


def _single(torch, B, n, h, T, M, prec):
    dt = torch.float32 if prec == 0 else torch.float64
    with B.Plan(n, h, 0, prec) as p:
        assert p.path() == 1
        p.set_kernel(T)
        Md = torch.from_numpy(np.ascontiguousarray(M)).to("cuda", dt)
        Hd = torch.empty_like(Md)
        p.apply(Md, Hd)
        torch.cuda.synchronize()
        return Hd.cpu().numpy().astype(np.float64)


CASES = [((64, 64, 8), 2), ((64, 64, 8), 4), ((256, 128, 4), 3), ((32, 32, 2), 2), ((1024, 64, 2), 4),
         ((128, 256, 16), 8), ((16, 512, 2), 8), ((64, 256, 4), 16), ((64, 32, 64), 1), ((2048, 16, 2), 2)]


@pytest.mark.parametrize("n,G", CASES)
@pytest.mark.parametrize("prec", [0, 1])
def test_sharded_matches_oracle_and_single_gpu_bitwise(torch, B, oracle, n, G, prec, monkeypatch):
    from paper_2308_08447_b200 import workloads as W
    if prec == 1:
        monkeypatch.setenv("DEMAG_PATH", "fast")
    h, Ms = (2e-9, 3e-9, 1.5e-9), 8e5
    dt = torch.float32 if prec == 0 else torch.float64
    M = W.random_unit_vectors(n, Ms, 900 + sum(n) + G)
    T = oracle.tensor_table(n, h)
    ref = oracle.fft_conv(T, M.astype(np.float64))
    cells = W.sample_cells(n, 32, 3)
    Hs = oracle.direct_sum_sampled(T, M.astype(np.float64), cells)           # Eq. (1) itself at sampled cells
    assert np.abs(ref.reshape(3, -1)[:, cells].T - Hs).max() / Ms < 1e-12
    R = Ranks(B, n, h, prec, G, T)
    try:
        infos = [p.info for p in R.plans]
        assert sum(i["ny_loc"] for i in infos) == n[1] and sum(i["nq_loc"] for i in infos) == n[0] // 2 + 1
        H = R.join(R.apply(torch, R.split(torch, M, dt)))
        H2 = R.join(R.apply(torch, R.split(torch, M, dt)))                   # buffers are reusable back to back
    finally:
        R.close()
    assert H.shape == (3, n[2], n[1], n[0])
    err = np.abs(H - ref).max() / Ms
    assert err <= (TOL32 if prec == 0 else TOL64), err
    assert np.array_equal(H, H2)
    assert np.array_equal(H, _single(torch, B, n, h, T, M, prec))


def test_sharded_with_slabs_and_builtin_tensor(torch, B, oracle):
    """Several slabs per rank (the q loop of phase 1) and the built-in Newell builder on every rank."""
    from paper_2308_08447_b200 import workloads as W
    n, h, Ms, G = (64, 64, 8), (2e-9, 2e-9, 2e-9), 8e5, 2
    M = W.random_unit_vectors(n, Ms, 77)
    ref = oracle.fft_conv(oracle.tensor_table(n, h), M.astype(np.float64))
    R = Ranks(B, n, h, 0, G, None, slab=5)
    try:
        H = R.join(R.apply(torch, R.split(torch, M, torch.float32)))
    finally:
        R.close()
    assert np.abs(H - ref).max() / Ms <= TOL32


def test_sharded_energy_partial_sums(torch, B, oracle):
    from paper_2308_08447_b200 import workloads as W
    n, h, Ms, G = (64, 64, 8), (2e-9, 3e-9, 1e-9), 8e5, 4
    M = W.random_unit_vectors(n, Ms, 5)
    T = oracle.tensor_table(n, h)
    R = Ranks(B, n, h, 0, G, T)
    try:
        Ml = R.split(torch, M, torch.float32)
        Hl = R.apply(torch, Ml)
        E = torch.zeros(G, dtype=torch.float64, device="cuda")
        for r, p in enumerate(R.plans):
            B.demag_energy(p.handle, Ml[r], Hl[r], E[r:r + 1])
        torch.cuda.synchronize()
        H = R.join(Hl)
    finally:
        R.close()
    mu0 = 4e-7 * np.pi
    Eref = -0.5 * mu0 * np.prod(h) * np.sum(M.astype(np.float64) * H)
    assert abs(float(E.sum().cpu()) - Eref) <= 1e-12 * abs(Eref)


def test_full_size_c3_eight_ranks_sampled(torch, B, oracle):
    """BASELINE.json config C3 (256 x 256 x 64, fp32) split over 8 ranks: Eq. (1) at sampled cells + bitwise equality
    with the one-GPU plan."""
    from paper_2308_08447_b200 import workloads as W
    n, h, Ms, G = (256, 256, 64), (3e-9, 3e-9, 3e-9), 8.6e5, 8
    M = W.random_unit_vectors(n, Ms, 1003)
    T = oracle.tensor_table(n, h)
    R = Ranks(B, n, h, 0, G, T)
    try:
        H = R.join(R.apply(torch, R.split(torch, M, torch.float32)))
    finally:
        R.close()
    with B.Plan(n, h, 0, 0) as p:
        p.set_kernel(T)
        Md = torch.from_numpy(M).to("cuda", torch.float32)
        Hd = torch.empty_like(Md)
        p.apply(Md, Hd)
        torch.cuda.synchronize()
        assert np.array_equal(H, Hd.cpu().numpy().astype(np.float64))
    cells = W.sample_cells(n, 24, 11)
    Hs = oracle.direct_sum_sampled(T, M.astype(np.float64), cells)
    assert np.abs(H.reshape(3, -1)[:, cells].T - Hs).max() / Ms <= TOL32


def test_sharded_error_paths(torch, B):
    h = (2e-9, 2e-9, 2e-9)
    for args in [((48, 64, 8), 2), ((64, 64, 1), 2)]:                        # not a power of two; one cell thick
        with pytest.raises(B.DemagError) as e:
            B.demag_plan_create_sharded(*args[0], *h, 0, 0, 0, args[1])
        assert e.value.status == 2
    with pytest.raises(B.DemagError) as e:                                   # 16 rows cannot feed 2 ranks (tiles of 16 rows)
        B.demag_plan_create_sharded(64, 16, 8, *h, 0, 0, 0, 2)
    assert e.value.status == 2
    with pytest.raises(B.DemagError) as e:                                   # periodic axis
        B.demag_plan_create_sharded(64, 64, 8, *h, 1, 0, 0, 2)
    assert e.value.status == 2
    for rank, world in [(2, 2), (-1, 2), (0, 0), (0, 17)]:
        with pytest.raises(B.DemagError) as e:
            B.demag_plan_create_sharded(64, 64, 8, *h, 0, 0, rank, world)
        assert e.value.status == 1
    p = B.demag_plan_create_sharded(64, 64, 8, *h, 0, 0, 1, 2)
    try:
        M = torch.zeros((3, 8, 32, 64), device="cuda")
        H = torch.zeros_like(M)
        with pytest.raises(B.DemagError) as e:                               # a rank of 2 is not a whole convolution
            B.demag_apply(p, M, H)
        assert e.value.status == 1
        with pytest.raises(B.DemagError) as e:                               # peers not installed
            B.demag_apply_sharded(p, 0, M, None)
        assert e.value.status == 1
        a, _, b, _ = B.demag_shard_buffers(p)
        with pytest.raises(B.DemagError) as e:                               # entry `rank` must be the plan's own buffer
            B.demag_shard_set_peers(p, [a, a], [b, b + 16])
        assert e.value.status == 1
        B.demag_shard_set_peers(p, [a, a], [b, b])
        with pytest.raises(B.DemagError) as e:                               # no kernel yet
            B.demag_apply_sharded(p, 0, M, None)
        assert e.value.status == 5
        B.demag_set_kernel(p, None)
        with pytest.raises(B.DemagError) as e:
            B.demag_apply_sharded(p, 3, M, H)
        assert e.value.status == 1
        with pytest.raises(B.DemagError) as e:
            B.demag_apply_sharded(p, 0, None, None)
        assert e.value.status == 1
    finally:
        B.demag_plan_destroy(p)
    q = B.demag_plan_create(64, 64, 8, *h, 0, 0)
    try:
        with pytest.raises(B.DemagError) as e:                               # an ordinary plan has no shard
            B.demag_shard_info(q)
        assert e.value.status == 1
    finally:
        B.demag_plan_destroy(q)


_IPC_WORKER = r"""
import os, sys
import numpy as np, torch, torch.distributed as dist
sys.path.insert(0, sys.argv[1])
from paper_2308_08447_b200 import binding as B, workloads as W
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)
torch.cuda.set_device(0)
n, h, Ms = (64, 64, 8), (2e-9, 3e-9, 1.5e-9), 8e5
M = W.random_unit_vectors(n, Ms, 4242)
p = B.ShardedPlan(n, h, 0, rank=rank, world=world, connect=False)
B.demag_shard_ipc_connect(p.handle, B.gather_handles(B.demag_shard_ipc_export(p.handle)))
p.set_kernel(None)
y0, nyl = p.info["y0"], p.info["ny_loc"]
Ml = torch.from_numpy(np.ascontiguousarray(M[:, :, y0:y0 + nyl, :])).cuda()
Hl = torch.empty_like(Ml)
for ph in range(3):                    # host barrier between the phases: no kernel ever waits for another process
    B.demag_apply_sharded(p.handle, ph, Ml, Hl)
    torch.cuda.synchronize()
    dist.barrier()
out = [None] * world
dist.all_gather_object(out, Hl.cpu().numpy())
if rank == 0:
    H = np.concatenate(out, axis=2)
    with B.Plan(n, h, 0, 0) as q:
        q.set_kernel(None)
        Md = torch.from_numpy(M).cuda(); Hd = torch.empty_like(Md)
        q.apply(Md, Hd); torch.cuda.synchronize()
        assert np.array_equal(H, Hd.cpu().numpy()), np.abs(H - Hd.cpu().numpy()).max()
    print("IPC_OK")
dist.barrier()
p.close()
dist.destroy_process_group()
"""


def test_two_processes_exchange_ipc_handles(torch, B, tmp_path):
    """demag_shard_ipc_export / _connect between two PROCESSES (both on device 0), phases separated by host
    barriers (gloo), result bit-equal to the one-GPU plan."""
    script = tmp_path / "ipc_worker.py"
    script.write_text(_IPC_WORKER)
    port = 29500 + os.getpid() % 2000
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script), ROOT], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    outs = []
    for pr in procs:
        try:
            o, _ = pr.communicate(timeout=300)
        except subprocess.TimeoutExpired:
            pr.kill()
            o, _ = pr.communicate()
        outs.append(o)
    assert all(pr.returncode == 0 for pr in procs), "\n".join(outs)
    assert "IPC_OK" in outs[0]
