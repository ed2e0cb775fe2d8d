"""demag_apply_atomistic_static (include/demag.h): the atomistic front end for callers that cannot call cudaMalloc -- its two
macrocell arrays live in one fixed file-scope device array inside the library.  Checked against the existing path
(demag_atomistic_reserve + demag_apply_atomistic) and the oracle on two calls in a row (second call: another plan, another
mesh size, so stale contents of the shared array would show), in fp32 and fp64; oversized meshes are rejected.

This file is collected last on purpose (the suite runs with pytest -x).  It passes alone in a fresh process and after
the other tests."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL32, TOL64 = 2e-5, 1e-11


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


def _case(torch, B, oracle, L, c, prec, seed):
    """One lattice through the existing path, the no-allocation path and the oracle.  Returns nothing; asserts."""
    from paper_2308_08447_b200 import workloads as W
    a, mu_s = 0.3e-9, 2.0
    n = tuple(l // k for l, k in zip(L, c))
    h = tuple(k * a for k in c)
    dt = torch.float32 if prec == 0 else torch.float64
    tol = TOL32 if prec == 0 else TOL64
    S = W.random_spins_numpy(L, seed)
    Ms = oracle.MU_B * mu_s / a ** 3
    T = oracle.tensor_table(n, h)
    Mref = oracle.macrocell_average(S.astype(np.float64), c, mu_s, a)
    want = oracle.macrocell_scatter(oracle.direct_sum(T, Mref), c)
    with B.Plan(n, h, 0, prec) as p:
        p.set_kernel(T)
        Sd = torch.from_numpy(S).to("cuda", dt)
        H_old = torch.full_like(Sd, float("nan"))
        H_new = torch.full_like(Sd, float("nan"))
        p.reserve_atomistic()
        w0 = p.workspace_bytes()
        p.apply_atomistic(Sd, H_old, c, mu_s, a)                      # existing path (plan-owned macrocell arrays)
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]                          # device-wide free memory: any cudaMalloc would lower it
        p.apply_atomistic_static(Sd, H_new, c, mu_s, a)               # no-allocation path (library's static array)
        torch.cuda.synchronize()
        assert p.workspace_bytes() == w0 and torch.cuda.mem_get_info()[0] == free0
        assert not torch.isnan(H_new).any()
        got_old = H_old.cpu().numpy().astype(np.float64); got_new = H_new.cpu().numpy().astype(np.float64)
        assert np.abs(got_new - got_old).max() / Ms <= tol            # the tolerance of the other tests ...
        assert np.array_equal(got_new, got_old)                       # ... and in fact the same kernels on the same values
        assert np.abs(got_new - want).max() / Ms <= tol               # and the oracle (Eq. (9) -> Eq. (1) -> scatter)
        assert torch.equal(Sd.cpu(), torch.from_numpy(S).to(dt))      # input untouched
        # accumulate mode through the same entry point
        H_acc = H_new.clone()
        p.apply_atomistic_static(Sd, H_acc, c, mu_s, a, accumulate=True)
        torch.cuda.synchronize()
        assert np.allclose(H_acc.cpu().numpy(), 2 * got_new, rtol=1e-6 if prec == 0 else 1e-14, atol=0)


def test_static_scratch_entry_point_matches_existing_path_on_two_calls_in_a_row(torch, B, oracle):
    # call 1: 8x8x4 macrocells of 4x2x2 spins (fp32, the float4 kernels); call 2: a smaller, differently shaped mesh in fp32
    # (generic kernels) -- it reuses the front of the array the first call filled; then the same two in fp64
    _case(torch, B, oracle, (32, 16, 8), (4, 2, 2), 0, 31)
    _case(torch, B, oracle, (12, 10, 6), (2, 2, 3), 0, 32)
    _case(torch, B, oracle, (32, 16, 8), (4, 2, 2), 1, 33)
    _case(torch, B, oracle, (12, 10, 6), (2, 2, 3), 1, 34)


def test_static_scratch_limit_and_errors(torch, B):
    assert B.demag_static_scratch_bytes() == 16 << 20
    a = 0.3e-9
    n = (128, 128, 64)                                               # 1,048,576 cells > 699,050: does not fit the 16 MiB array
    with B.Plan(n, (a, a, a), 0, 0) as p:
        p.set_kernel(None)
        S = torch.zeros((3, n[2], n[1], n[0]), dtype=torch.float32, device="cuda"); H = torch.empty_like(S)
        with pytest.raises(B.DemagError) as e:
            p.apply_atomistic_static(S, H, (1, 1, 1), 2.0, a)
        assert e.value.status == 2 and "static array holds" in str(e.value)
        p.reserve_atomistic(); p.apply_atomistic(S, H, (1, 1, 1), 2.0, a)        # the allocating path still serves it
        torch.cuda.synchronize()
    with B.Plan((8, 8, 4), (a, a, a), 0, 0) as p:
        S = torch.zeros((3, 4, 8, 8), dtype=torch.float32, device="cuda"); H = torch.empty_like(S)
        with pytest.raises(B.DemagError) as e:
            p.apply_atomistic_static(S, H, (1, 1, 1), 2.0, a)
        assert e.value.status == 5                                   # no kernel yet
        p.set_kernel(None)
        with pytest.raises(B.DemagError) as e:
            p.apply_atomistic_static(S, H, (2, 2, 2), 2.0, a)
        assert e.value.status == 1                                   # h != c * a
        with pytest.raises(B.DemagError) as e:
            p.apply_atomistic_static(S, S, (1, 1, 1), 2.0, a)
        assert e.value.status == 1                                   # aliasing
