"""Parity of the compile-time specialised kernel family (kernels_v2.cuh, demag_path() == 1) against the fp64
oracle, one case per instantiated transform length of every stage, plus agreement with the size-generic family.

Tolerances as everywhere (BASELINE.json north_star): 2e-5 (fp32) / 1e-11 (fp64) of Ms, the oracle's tensor
pushed through demag_set_kernel.
"""
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL32 = 2e-5
TOL64 = 1e-11


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


def _run(torch, B, n, h, T, M, prec, expect_path=None, slab=0):
    dt = torch.float32 if prec == 0 else torch.float64
    with B.Plan(n, h, 0, prec) as p:
        if expect_path is not None:
            assert p.path() == expect_path, f"plan for {n} took kernel family {p.path()}"
        p.set_kernel(T)
        if slab:
            p.set_slab(slab)
        Md = torch.from_numpy(np.ascontiguousarray(M)).to("cuda", dt)
        Hd = torch.full_like(Md, float("nan"))
        p.apply(Md, Hd)
        torch.cuda.synchronize()
        assert not torch.isnan(Hd).any()
        return Hd.cpu().numpy().astype(np.float64)


def _reference(oracle, n, h, M):
    """Full field: Eq. (1) by direct summation when small, else the NumPy-FFT cross-check O-C, itself checked
    against Eq. (1) at sampled cells."""
    from paper_2308_08447_b200 import workloads as W
    T = oracle.tensor_table(n, h)
    M64 = M.astype(np.float64)
    if np.prod(n) <= 4096:
        return T, oracle.direct_sum(T, M64)
    ref = oracle.fft_conv(T, M64)
    cells = W.sample_cells(n, 48, 7)
    Hs = oracle.direct_sum_sampled(T, M64, cells)
    assert np.abs(ref.reshape(3, -1)[:, cells].T - Hs).max() / 8e5 < 1e-12
    return T, ref


# one shape per x length (Lc = nx = 16 .. 4096), per y length (Ny = 32 .. 8192), per z length (Nz = 4 .. 2048);
# the other two axes small but spanning several tiles / a ragged last tile where the stage allows it
X_SHAPES = [(16, 16, 2), (32, 16, 4), (64, 32, 2), (128, 16, 2), (256, 48 // 3 * 2, 2), (512, 16, 2), (1024, 16, 2),
            (2048, 16, 2), (4096, 16, 2)]
Y_SHAPES = [(16, 16, 4), (16, 32, 2), (32, 64, 2), (16, 128, 2), (16, 256, 4), (16, 512, 2), (16, 1024, 2),
            (16, 2048, 2), (16, 4096, 2)]
Z_SHAPES = [(16, 16, 2), (16, 16, 4), (16, 16, 8), (16, 16, 16), (16, 32, 32), (16, 16, 64), (16, 16, 128),
            (16, 16, 256), (16, 16, 512), (16, 16, 1024)]
FILM_SHAPES = [(16, 16, 1), (64, 128, 1), (256, 32, 1)]          # nz = 1: no z transform, multiply only (row a3')
SHAPES = sorted(set(X_SHAPES + Y_SHAPES + Z_SHAPES + FILM_SHAPES + [(64, 64, 8), (32, 48 // 3 * 2, 16), (256, 64, 16)]))


@pytest.mark.parametrize("n", SHAPES)
@pytest.mark.parametrize("prec", [0, 1])
def test_fast_family_against_oracle(torch, B, oracle, n, prec, monkeypatch):
    from paper_2308_08447_b200 import workloads as W
    if prec == 1:
        monkeypatch.setenv("DEMAG_PATH", "fast")      # fp64 plans take the generic family unless asked
    if prec == 1 and 2 * n[1] > 4096:
        pytest.skip("fp64 fast path stops at Ny = 4096 (shared memory)")
    h = (2e-9, 3e-9, 1.5e-9)
    Ms = 8e5
    M = W.random_unit_vectors(n, Ms, 300 + sum(n))
    T, ref = _reference(oracle, n, h, M)
    H = _run(torch, B, n, h, T, M, prec, expect_path=1)
    err = np.abs(H - ref).max() / Ms
    assert err <= (TOL32 if prec == 0 else TOL64), err


@pytest.mark.parametrize("n", [(64, 32, 4), (128, 64, 16), (32, 16, 64)])
def test_fast_and_generic_families_agree(torch, B, oracle, n, monkeypatch):
    from paper_2308_08447_b200 import workloads as W
    h = (2e-9, 2e-9, 2e-9)
    Ms = 8e5
    M = W.random_unit_vectors(n, Ms, 11)
    T = oracle.tensor_table(n, h)
    monkeypatch.setenv("DEMAG_PATH", "fast")
    Hf = _run(torch, B, n, h, T, M, 1, expect_path=1)
    monkeypatch.setenv("DEMAG_PATH", "generic")
    Hg = _run(torch, B, n, h, T, M, 1, expect_path=0)
    monkeypatch.delenv("DEMAG_PATH")
    assert np.abs(Hf - Hg).max() / Ms <= 1e-12


@pytest.mark.parametrize("n", [(16, 32, 128), (32, 16, 256), (64, 64, 128)])
def test_long_z_columns_both_z_kernels(torch, B, oracle, n, monkeypatch):
    """Nz = 256 / 512 (fp32): the even / odd two-pass z kernel (k_z_eo_v, default) and the three-pass kernel it replaces
    (DEMAG_NO_ZEO) against the oracle, and against each other at rounding level."""
    from paper_2308_08447_b200 import workloads as W
    h, Ms = (2e-9, 3e-9, 1e-9), 8e5
    M = W.random_unit_vectors(n, Ms, 23)
    T = oracle.tensor_table(n, h)
    ref = oracle.fft_conv(T, M.astype(np.float64))
    cells = W.sample_cells(n, 24, 5)
    Hs = oracle.direct_sum_sampled(T, M.astype(np.float64), cells)
    assert np.abs(ref.reshape(3, -1)[:, cells].T - Hs).max() / Ms < 1e-12       # the cross-check is Eq. (1) where sampled
    He = _run(torch, B, n, h, T, M, 0, expect_path=1)
    monkeypatch.setenv("DEMAG_NO_ZEO", "1")
    H3 = _run(torch, B, n, h, T, M, 0, expect_path=1)
    monkeypatch.delenv("DEMAG_NO_ZEO")
    assert np.abs(He - ref).max() / Ms <= TOL32 and np.abs(H3 - ref).max() / Ms <= TOL32
    assert np.abs(He - H3).max() / Ms <= 2e-6
    assert not np.array_equal(He, H3)                                           # two different kernels did run


@pytest.mark.parametrize("slab", [1, 2, 5])
def test_fast_family_slab_size_does_not_change_result(torch, B, oracle, slab):
    from paper_2308_08447_b200 import workloads as W
    n, h = (32, 16, 8), (2e-9, 2e-9, 2e-9)
    M = W.random_unit_vectors(n, 8e5, 5)
    T = oracle.tensor_table(n, h)
    H0 = _run(torch, B, n, h, T, M, 0, expect_path=1)
    H1 = _run(torch, B, n, h, T, M, 0, expect_path=1, slab=slab)
    assert np.array_equal(H0, H1)


def test_fast_family_impulse_returns_tensor_column(torch, B, oracle, monkeypatch):
    """A single magnetised cell reads the stored kernel back through the whole pipeline: H_a(i) = -N_ab(i-j) M_b."""
    monkeypatch.setenv("DEMAG_PATH", "fast")
    n, h = (32, 16, 8), (2e-9, 3e-9, 1e-9)
    T = oracle.tensor_table(n, h)
    for (jx, jy, jz), comp in [((0, 0, 0), 0), ((31, 15, 7), 1), ((13, 6, 2), 2)]:
        M = np.zeros((3,) + n[::-1], dtype=np.float32)
        M[comp, jz, jy, jx] = 1.0
        ref = oracle.direct_sum(T, M.astype(np.float64))
        H = _run(torch, B, n, h, T, M, 1, expect_path=1)
        assert np.abs(H - ref).max() <= 1e-13


@pytest.mark.parametrize("n", [(64, 64, 8), (256, 32, 1), (2048, 16, 2), (16, 4096, 2), (256, 256, 64)])
@pytest.mark.parametrize("pdl", ["2", "1", "0"])
def test_back_to_back_applies_are_ordered(torch, B, n, pdl, monkeypatch):
    """The kernels of the fast family are launched with programmatic stream serialization (kernels_v2.cuh pdl_enter /
    pdl_leave): the next grid is let in when every block of the current one has started (mode 1, tiny meshes) or has
    stored its last result (mode 2); DEMAG_PDL forces a mode, or 0 = off, for any size (read at plan creation).  Eight applies queued
    back to back on one plan, alternating between two magnetisations, without a host synchronisation in between,
    must each equal bit for bit the field of the same magnetisation applied alone (workspaces are reused from apply
    to apply: any early start would show up as a mixed field)."""
    from paper_2308_08447_b200 import workloads as W
    monkeypatch.setenv("DEMAG_PDL", pdl)
    h, Ms = (2e-9, 2e-9, 1e-9), 8e5
    Ma = torch.from_numpy(W.random_unit_vectors(n, Ms, 31)).to("cuda", torch.float32)
    Mb = torch.from_numpy(W.random_unit_vectors(n, Ms, 32)).to("cuda", torch.float32)
    with B.Plan(n, h, 0, B.DEMAG_FP32) as p:
        p.set_kernel(None)
        assert p.path() == 1
        alone = []
        for Md in (Ma, Mb):
            Hd = torch.empty_like(Md)
            p.apply(Md, Hd); torch.cuda.synchronize()
            alone.append(Hd.clone())
        assert not torch.equal(alone[0], alone[1])
        outs = [torch.full_like(Ma, float("nan")) for _ in range(8)]
        for i, Hd in enumerate(outs):
            p.apply(Ma if i % 2 == 0 else Mb, Hd)
        acc = torch.zeros_like(Ma)
        p.apply_add(Ma, acc); p.apply_add(Mb, acc)
        torch.cuda.synchronize()
        for i, Hd in enumerate(outs):
            assert torch.equal(Hd, alone[i % 2]), f"apply {i} differs from the same apply run alone"
        assert (acc.double() - alone[0].double() - alone[1].double()).abs().max().item() / Ms <= 4e-7
