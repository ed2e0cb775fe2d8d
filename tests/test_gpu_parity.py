"""Parity of the CUDA path (through the C ABI) against the fp64 oracle -- needs a B200.

Tolerances (BASELINE.json north_star): max |H_gpu - H_ref| / Ms <= 2e-5 for fp32, <= 1e-11 for fp64,
with the oracle's N pushed through demag_set_kernel (R5 "convolution parity").
"""
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
    binding.lib()          # fail loudly if the CUDA library is missing
    return binding


def run_gpu(torch, B, n, h, T, M, prec, slab=0, builtin=False):
    dt = torch.float32 if prec == B.DEMAG_FP32 else torch.float64
    with B.Plan(n, h, 0, prec) as p:
        p.set_kernel(None if builtin else T)
        if slab:
            p.set_slab(slab)
        Md = torch.from_numpy(np.ascontiguousarray(M)).to("cuda", dt)
        Hd = torch.full_like(Md, float("nan"))
        p.apply(Md, Hd)
        torch.cuda.synchronize()
        assert torch.equal(Md.cpu(), torch.from_numpy(np.ascontiguousarray(M)).to(dt)), "M was modified"
        return Hd.cpu().numpy().astype(np.float64)


def rand_M(n, Ms, seed):
    from paper_2308_08447_b200 import workloads as W
    return W.random_unit_vectors(n, Ms, seed)


# --------------------------------------------------------------------------------- config 1
def test_config1_full_direct_sum_and_naive_dft(torch, B, oracle):
    from paper_2308_08447_b200 import workloads as W
    cfg = W.CONFIGS["C1"]
    M = W.make_magnetisation(cfg)
    T = oracle.tensor_table(cfg.n, cfg.h)
    HA = oracle.direct_sum(T, M.astype(np.float64))
    HB = oracle.naive_dft_conv(T, M.astype(np.float64))
    assert np.abs(HA - HB).max() / cfg.Ms < 1e-13
    H32 = run_gpu(torch, B, cfg.n, cfg.h, T, M, B.DEMAG_FP32)
    assert np.abs(H32 - HA).max() / cfg.Ms <= TOL32
    H64 = run_gpu(torch, B, cfg.n, cfg.h, T, M, B.DEMAG_FP64)
    assert np.abs(H64 - HA).max() / cfg.Ms <= TOL64
    assert np.abs(H64 - HB).max() / cfg.Ms <= TOL64


# --------------------------------------------------------------------------------- shape sweep
SHAPES = [(1, 1, 1), (2, 1, 1), (1, 2, 1), (1, 1, 2), (2, 2, 2), (4, 2, 8), (8, 8, 8), (16, 4, 2), (64, 1, 1),
          (1, 64, 1), (1, 1, 64), (1, 16, 4), (32, 16, 1), (4, 128, 8), (128, 4, 2), (2, 2, 128), (16, 32, 16),
          (512, 2, 1), (2, 512, 2), (64, 64, 4)]


@pytest.mark.parametrize("n", SHAPES)
@pytest.mark.parametrize("prec", [0, 1])
def test_shapes_against_oracle(torch, B, oracle, n, prec):
    """Every power-of-two length per axis incl. degenerate 1-cell axes, several tiles and ragged tile
    tails (line counts not divisible by the batch)."""
    h = (2e-9, 3e-9, 1e-9)
    Ms = 8e5
    M = rand_M(n, Ms, 100 + sum(n))
    T = oracle.tensor_table(n, h)
    ref = oracle.fft_conv(T, M.astype(np.float64))
    if np.prod(n) <= 4096:
        ref_ds = oracle.direct_sum(T, M.astype(np.float64))
        assert np.abs(ref - ref_ds).max() / Ms < 1e-12
        ref = ref_ds
    H = run_gpu(torch, B, n, h, T, M, prec)
    err = np.abs(H - ref).max() / Ms
    assert err <= (TOL32 if prec == 0 else TOL64), err


@pytest.mark.parametrize("n", [(16, 16, 2048), (4, 4, 4096), (4096, 4, 1), (2, 4096, 2), (8192, 32, 2), (8192, 4, 1)])
def test_maximum_axis_lengths(torch, B, oracle, n):
    """The longest transforms the library accepts (n_x = 8192 -> a 16384-point real transform; n_y, n_z = 4096 ->
    N_a = 8192) on every axis, incl. the z lengths beyond
    the fast family's range (size-generic kernels); full field against the NumPy-FFT cross-check O-C, which is itself
    checked against Eq. (1) at sampled cells."""
    from paper_2308_08447_b200 import workloads as W
    h, Ms = (2e-9, 3e-9, 1e-9), 8e5
    M = rand_M(n, Ms, 900 + sum(n))
    T = oracle.tensor_table(n, h)
    ref = oracle.fft_conv(T, M.astype(np.float64))
    cells = W.sample_cells(n, 32, 3)
    Hs = oracle.direct_sum_sampled(T, M.astype(np.float64), cells)
    assert np.abs(ref.reshape(3, -1)[:, cells].T - Hs).max() / Ms < 1e-12
    for prec in (0, 1):
        if prec == 1 and n[2] == 4096:           # an 8192-point fp64 z line does not fit in shared memory: refused
            with pytest.raises(B.DemagError) as e:
                B.demag_plan_create(*n, *h, 0, 1)
            assert e.value.status == 2
            continue
        H = run_gpu(torch, B, n, h, T, M, prec)
        assert np.abs(H - ref).max() / Ms <= (TOL32 if prec == 0 else TOL64)
    for bad in ((8193, 4, 1), (4, 4097, 1), (4, 4, 4097)):
        with pytest.raises(B.DemagError) as e:
            B.demag_plan_create(*bad, *h, 0, 0)
        assert e.value.status == 2


@pytest.mark.parametrize("slab", [1, 3, 7])
def test_slab_size_does_not_change_result(torch, B, oracle, slab):
    n, h = (32, 16, 8), (2e-9, 2e-9, 2e-9)
    M = rand_M(n, 8e5, 5)
    T = oracle.tensor_table(n, h)
    H0 = run_gpu(torch, B, n, h, T, M, 0)
    H1 = run_gpu(torch, B, n, h, T, M, 0, slab=slab)
    assert np.array_equal(H0, H1)


def test_impulse_returns_tensor_column(torch, B, oracle):
    """A single magnetised cell reads the kernel back through the whole pipeline: catches every
    padding / crop / packing / parity-sign bug."""
    n, h = (16, 8, 4), (1e-9, 1.5e-9, 0.5e-9)
    T = oracle.tensor_table(n, h)
    j = (5, 3, 1)
    for b in range(3):
        M = np.zeros((3, n[2], n[1], n[0]), dtype=np.float32)
        M[b, j[2], j[1], j[0]] = 1.0
        H = run_gpu(torch, B, n, h, T, M, B.DEMAG_FP64)
        for iz, iy, ix in [(0, 0, 0), (3, 7, 15), (1, 3, 5), (2, 0, 9), (0, 7, 0), (3, 2, 14)]:
            N6 = oracle.N_at(((ix - j[0]) * h[0], (iy - j[1]) * h[1], (iz - j[2]) * h[2]), h)
            want = -N6[oracle.COMP][:, b]
            assert np.abs(H[:, iz, iy, ix] - want).max() < 1e-12


def test_linearity(torch, B, oracle):
    n, h = (16, 16, 4), (2e-9, 2e-9, 2e-9)
    T = oracle.tensor_table(n, h)
    M1 = rand_M(n, 1.0, 1).astype(np.float64); M2 = rand_M(n, 1.0, 2).astype(np.float64)
    H1 = run_gpu(torch, B, n, h, T, M1, 1); H2 = run_gpu(torch, B, n, h, T, M2, 1)
    H3 = run_gpu(torch, B, n, h, T, 2.0 * M1 - 3.0 * M2, 1)
    assert np.abs(H3 - (2.0 * H1 - 3.0 * H2)).max() < 1e-12


# --------------------------------------------------------------------------------- general mesh sizes
GENERAL = [(12, 10, 3), (7, 1, 1), (1, 9, 5), (48, 48, 1), (33, 17, 9), (100, 36, 5), (65, 16, 2),
           (130, 70, 3), (18, 130, 6), (1030, 18, 2), (480, 30, 2)]     # even nx on the fast path: zeros / crop inside the x kernels


@pytest.mark.parametrize("n", GENERAL)
@pytest.mark.parametrize("prec", [0, 1])
def test_general_mesh_sizes(torch, B, oracle, n, prec):
    """DESIGN.md R10: sizes that are not powers of two (the paper's own meshes) are embedded in the
    next power-of-two mesh; the result is the same Eq. (1) sum (padding >= 2n - 1 is exact)."""
    h = (2e-9, 3e-9, 1e-9)
    Ms = 8e5
    M = rand_M(n, Ms, 500 + sum(n))
    T = oracle.tensor_table(n, h)
    ref = oracle.direct_sum(T, M.astype(np.float64)) if np.prod(n) <= 6000 else oracle.fft_conv(T, M.astype(np.float64))
    H = run_gpu(torch, B, n, h, T, M, prec)
    assert np.abs(H - ref).max() / Ms <= (TOL32 if prec == 0 else TOL64)
    Hb = run_gpu(torch, B, n, h, None, M, prec, builtin=True)      # built-in tensor on the embedding mesh
    assert np.abs(Hb - ref).max() / Ms <= (TOL32 if prec == 0 else 1e-9)


def test_general_mesh_builder_table_energy_atomistic(torch, B, oracle):
    n, h, Ms = (12, 10, 3), (2e-9, 3e-9, 1e-9), 8e5
    with B.Plan(n, h, 0, B.DEMAG_FP64) as p:
        assert np.abs(p.get_kernel_real() - oracle.tensor_table(n, h)).max() <= 1e-10
        M = rand_M(n, Ms, 9).astype(np.float64)
        T = oracle.tensor_table(n, h)
        p.set_kernel(T)
        Md = torch.from_numpy(M).cuda(); Hd = torch.empty_like(Md)
        E = torch.zeros(1, dtype=torch.float64, device="cuda")
        p.apply(Md, Hd); p.energy(Md, Hd, E); torch.cuda.synchronize()
        ref = oracle.direct_sum(T, M)
        Eref = oracle.energy(M, ref, h)
        assert abs(E.item() - Eref) <= 1e-10 * abs(Eref)
    # atomistic on a lattice whose macrocell mesh is 6 x 4 x 2
    from paper_2308_08447_b200 import workloads as W
    c, a, mu_s = (2, 2, 2), 0.3e-9, 2.0
    L = (12, 8, 4)
    S = W.random_spins_numpy(L, 77).astype(np.float64)
    nm, hm = (6, 4, 2), tuple(ci * a for ci in c)
    Tm = oracle.tensor_table(nm, hm)
    Mref = oracle.macrocell_average(S, c, mu_s, a)
    Href = oracle.macrocell_scatter(oracle.direct_sum(Tm, Mref), c)
    with B.Plan(nm, hm, 0, B.DEMAG_FP64) as p:
        p.set_kernel(Tm)
        Sd = torch.from_numpy(S).cuda(); Hs = torch.empty_like(Sd)
        p.reserve_atomistic()
        p.apply_atomistic(Sd, Hs, c, mu_s, a)
        torch.cuda.synchronize()
        assert np.abs(Hs.cpu().numpy() - Href).max() / np.abs(Mref).max() <= 1e-11


# --------------------------------------------------------------------------------- periodic axes (caller's kernel)
def _periodic_table(oracle, n, h, pbc, images=2):
    """Caller-side periodic kernel ("modified convolution kernel"; R11): the open-boundary tensor
    summed over `images` periodic images on each side along the periodic axes, at offsets 0 <= d_a < n_a."""
    nx, ny, nz = n
    T = np.zeros((6, nz, ny, nx))
    rng = [range(-images, images + 1) if p else range(1) for p in pbc]
    for dz in range(nz):
        for dy in range(ny):
            for dx in range(nx):
                acc = np.zeros(6)
                for mx in rng[0]:
                    for my in rng[1]:
                        for mz in rng[2]:
                            acc += oracle.N_at(((dx + mx * nx) * h[0], (dy + my * ny) * h[1], (dz + mz * nz) * h[2]), h)
                T[:, dz, dy, dx] = acc
    # a periodic kernel obeys K(n_a - d) = parity * K(d) on its periodic axes (include/demag.h); the truncated image sum
    # does so only up to its last images: symmetrise it
    for a, ax in ((0, 3), (1, 2), (2, 1)):
        if pbc[a]:
            idx = (-np.arange(n[a])) % n[a]
            par = oracle.PARITY[:, a].reshape(6, 1, 1, 1)
            T = 0.5 * (T + par * np.take(T, idx, axis=ax))
    return T


def _periodic_direct(oracle, T, M, pbc):
    """H_i = -sum_j K(i - j) M_j with the offset wrapped on periodic axes and reflected (parity of R1) on open ones."""
    PAR, COMP = oracle.PARITY, oracle.COMP
    _, nz, ny, nx = M.shape
    n = (nx, ny, nz)
    H = np.zeros_like(M)
    cells = [(x, y, z) for z in range(nz) for y in range(ny) for x in range(nx)]
    for (ix, iy, iz) in cells:
        for (jx, jy, jz) in cells:
            d = [ix - jx, iy - jy, iz - jz]
            sg = np.ones(6)
            for a in range(3):
                if pbc[a]:
                    d[a] %= n[a]
                elif d[a] < 0:
                    d[a] = -d[a]; sg = sg * PAR[:, a]
            k = T[:, d[2], d[1], d[0]] * sg
            for a in range(3):
                H[a, iz, iy, ix] -= sum(k[COMP[a, b]] * M[b, jz, jy, jx] for b in range(3))
    return H


@pytest.mark.parametrize("n,pbc", [((8, 4, 2), (True, False, False)), ((4, 8, 2), (False, True, False)),
                                   ((8, 8, 1), (True, True, False)), ((4, 2, 8), (False, False, True))])
def test_periodic_axes_with_callers_kernel(torch, B, oracle, n, pbc):
    """pbc_flags: a periodic axis is not padded and the caller's table is taken as the periodic kernel on
    it.  Reference = the wrapped direct sum written out here, cross-checked with the oracle's naive-DFT convolution on
    the unpadded axis."""
    h, Ms = (2e-9, 3e-9, 1e-9), 8e5
    T = _periodic_table(oracle, n, h, pbc)
    M = rand_M(n, Ms, 40 + sum(n)).astype(np.float64)
    ref = _periodic_direct(oracle, T, M, pbc)
    P = tuple(na if (p or na == 1) else 2 * na for na, p in zip(n, pbc))
    assert np.abs(oracle.naive_dft_conv(T, M, P) - ref).max() / Ms < 1e-12
    flags = sum(f for f, p in zip((B.DEMAG_PBC_X, B.DEMAG_PBC_Y, B.DEMAG_PBC_Z), pbc) if p)
    for prec, tol in ((0, TOL32), (1, TOL64)):
        dt = torch.float32 if prec == 0 else torch.float64
        with B.Plan(n, h, flags, prec) as p:
            p.set_kernel(T)
            Md = torch.from_numpy(M).to("cuda", dt); Hd = torch.empty_like(Md)
            p.apply(Md, Hd); torch.cuda.synchronize()
            Mq = Md.cpu().numpy().astype(np.float64)
            refq = ref if prec == 1 else _periodic_direct(oracle, T, Mq, pbc)
            assert np.abs(Hd.cpu().numpy().astype(np.float64) - refq).max() / Ms <= tol


@pytest.mark.parametrize("n,pbc,images", [((8, 4, 2), (True, False, False), 3), ((4, 8, 2), (True, True, False), 2),
                                          ((4, 4, 4), (False, False, True), 4), ((16, 16, 1), (True, True, False), 1),
                                          ((8, 8, 2), (True, True, True), 1), ((4, 4, 2), (True, False, False), 0)])
def test_builtin_periodic_tensor(torch, B, oracle, n, pbc, images):
    """NEXT row 1 (reading R11): the built-in builder's periodic tensor -- images summed on every periodic
    axis, symmetrised -- against oracle.periodic_tensor_table entry by entry (the GPU uses the multipole series beyond
    24 cells, the oracle quadrature: R4/R5 tolerance), then the field of that plan against the wrapped direct sum."""
    h, Ms = (2e-9, 3e-9, 1e-9), 8e5
    flags = sum(f for f, p in zip((B.DEMAG_PBC_X, B.DEMAG_PBC_Y, B.DEMAG_PBC_Z), pbc) if p)
    To = oracle.periodic_tensor_table(n, h, pbc, images)
    M = rand_M(n, Ms, 60 + sum(n)).astype(np.float64)
    ref = _periodic_direct(oracle, To, M, pbc)
    for prec, tol in ((1, 1e-9), (0, TOL32)):
        dt = torch.float32 if prec == 0 else torch.float64
        with B.Plan(n, h, flags, prec) as p:
            p.set_pbc_images(images)
            Tg = p.get_kernel_real()
            assert np.abs(Tg - To).max() <= 1e-10
            p.set_kernel(None)
            Md = torch.from_numpy(M).to("cuda", dt); Hd = torch.empty_like(Md)
            p.apply(Md, Hd); torch.cuda.synchronize()
            Mq = Md.cpu().numpy().astype(np.float64)
            refq = ref if prec == 1 else _periodic_direct(oracle, To, Mq, pbc)
            assert np.abs(Hd.cpu().numpy().astype(np.float64) - refq).max() / Ms <= tol


# --------------------------------------------------------------------------------- dipole-dipole (Eq. (8))
@pytest.mark.parametrize("L", [(16, 16, 4), (12, 10, 3), (32, 16, 8)])
@pytest.mark.parametrize("prec", [0, 1])
def test_dipole_dipole_field_through_set_kernel(torch, B, oracle, L, prec):
    """NEXT row 2: the atomistic dipole-dipole field of Eq. (8) "re-arranged into the form of
    Equation (1)": same engine, caller-supplied point-dipole tensor (N(0) = 0), one cell per spin.  Reference =
    Eq. (8) written out pair by pair on the small lattices, the direct sum of Eq. (1) with that tensor on the larger."""
    from paper_2308_08447_b200 import workloads as W
    a, mu_s = 0.3e-9, 2.0
    Ms = oracle.MU_B * mu_s / a ** 3
    S = W.random_spins_numpy(L, 21 + sum(L))
    M = (S.astype(np.float64) * Ms).astype(np.float32)
    T = oracle.dipole_table(L, a)
    if np.prod(L) <= 1100:
        ref = oracle.dipole_field_eq8(M.astype(np.float64) / Ms, mu_s, a)
    else:
        ref = oracle.direct_sum(T, M.astype(np.float64))
    H = run_gpu(torch, B, L, (a, a, a), T, M, prec)
    assert np.abs(H - ref).max() / Ms <= (TOL32 if prec == 0 else TOL64)


# --------------------------------------------------------------------------------- sub-step extrapolation
@pytest.mark.parametrize("n", [(12, 10, 3), (5, 3, 1), (64, 32, 8)])
@pytest.mark.parametrize("npts", [1, 2, 5, 6, 8])
@pytest.mark.parametrize("prec", [0, 1])
def test_extrapolate_against_oracle(torch, B, oracle, n, npts, prec):
    """demag_extrapolate == oracle.poly_extrapolate (the Lagrange polynomial through npts fields) entry by entry,
    overwrite and accumulate modes, vector body and scalar tail (3 n_c not a multiple of 4).  Tolerance from the
    arithmetic: npts FMAs and one rounding of each weight, (npts + 2) eps sum_k |L_k| max|H_k|."""
    rng = np.random.default_rng(70 + npts + sum(n))
    dt = torch.float32 if prec == 0 else torch.float64
    npd = np.float32 if prec == 0 else np.float64
    shape = (3, n[2], n[1], n[0])
    ts = np.sort(rng.uniform(0.0, 1.0, npts)) + np.arange(npts) * 0.05
    t = ts[-1] + 0.37 * (ts[-1] - ts[0] + 0.1)
    H = [(rng.normal(size=shape) * 8e5).astype(npd) for _ in range(npts)]
    ref = oracle.poly_extrapolate([h.astype(np.float64) for h in H], ts, t)
    Lk = [np.prod([(t - tj) / (tk - tj) for j, tj in enumerate(ts) if j != k]) for k, tk in enumerate(ts)]
    S = sum(abs(l) * np.abs(h).max() for l, h in zip(Lk, H))
    tol = (npts + 2) * np.finfo(npd).eps * S
    with B.Plan(n, (2e-9, 2e-9, 2e-9), 0, prec) as p:
        Hd = [torch.from_numpy(h).cuda() for h in H]
        out = torch.full(shape, float("nan"), dtype=dt, device="cuda")
        p.extrapolate(Hd, ts, t, out)
        torch.cuda.synchronize()
        assert np.abs(out.cpu().numpy().astype(np.float64) - ref).max() <= tol
        base = (rng.normal(size=shape) * 1e5).astype(npd)
        acc = torch.from_numpy(base).cuda()
        p.extrapolate(Hd, ts, t, acc, accumulate=True)
        torch.cuda.synchronize()
        assert np.abs(acc.cpu().numpy().astype(np.float64) - (ref + base.astype(np.float64))).max() <= tol + np.finfo(npd).eps * np.abs(ref).max()
        for h, h0 in zip(Hd, H):
            assert np.array_equal(h.cpu().numpy(), h0)                       # the history is read only


def test_extrapolated_field_follows_a_rotating_magnetisation(torch, B, oracle):
    """What the hook is for: fields computed at 5 past times, a quartic through them evaluated at a sub-step
    half a step ahead, against the convolution actually carried out at that time.  M rotates by 0.1 rad per step, so
    the quartic's error is O(0.1^5)."""
    n, h, Ms = (32, 16, 4), (2e-9, 2e-9, 2e-9), 8e5
    rng = np.random.default_rng(3)
    phi = rng.uniform(0, 2 * np.pi, size=(n[2], n[1], n[0]))
    Mt = lambda t: (Ms * np.stack([np.cos(phi + t), np.sin(phi + t), np.zeros_like(phi)])).astype(np.float32)
    ts = [0.1 * k for k in range(5)]
    with B.Plan(n, h, 0, 0) as p:
        p.set_kernel(oracle.tensor_table(n, h))
        Hs = []
        for t in ts + [0.45]:
            Md = torch.from_numpy(Mt(t)).cuda(); Hd = torch.empty_like(Md)
            p.apply(Md, Hd)
            Hs.append(Hd)
        out = torch.empty_like(Hs[0])
        p.extrapolate(Hs[:5], ts, 0.45, out)
        torch.cuda.synchronize()
        err = float((out - Hs[5]).abs().max()) / Ms
        assert err < 2e-5, err
        p.extrapolate(Hs[3:5], ts[3:5], 0.45, out)                          # a straight line through two fields is far worse
        torch.cuda.synchronize()
        assert float((out - Hs[5]).abs().max()) / Ms > 20 * err


def test_extrapolate_error_paths(torch, B):
    with B.Plan((8, 8, 2), (1e-9,) * 3) as p:
        H = [torch.zeros((3, 2, 8, 8), device="cuda") for _ in range(9)]
        out = torch.zeros_like(H[0])
        for hist, ts in [([], []), (H, list(range(9))), (H[:2], [0.5, 0.5]), (H[:2], [0.0, float("nan")]), ([out, H[0]], [0, 1])]:
            with pytest.raises(B.DemagError) as e:
                p.extrapolate(hist, ts, 2.0, out)
            assert e.value.status == 1
        with pytest.raises(B.DemagError) as e:
            B._check(B.lib().demag_extrapolate(p.handle, 1, None, None, 0.0, out.data_ptr(), 0, None))
        assert e.value.status == 1


# --------------------------------------------------------------------------------- accumulate into H_eff
@pytest.mark.parametrize("n", [(32, 16, 8), (64, 32, 1), (12, 10, 3), (1, 8, 4), (4, 4, 2)])
@pytest.mark.parametrize("prec", [0, 1])
def test_apply_add_accumulates_into_heff(torch, B, oracle, n, prec):
    """demag_apply_add: H_eff <- H_eff + H_d in the last kernel (both kernel families, film, embedded and 1-cell-wide
    meshes): equal to demag_apply's field added to the same start array, to rounding."""
    h, Ms = (2e-9, 3e-9, 1e-9), 8e5
    dt = torch.float32 if prec == 0 else torch.float64
    M = rand_M(n, Ms, 70 + sum(n))
    T = oracle.tensor_table(n, h)
    with B.Plan(n, h, 0, prec) as p:
        p.set_kernel(T)
        Md = torch.from_numpy(M).to("cuda", dt)
        Hd = torch.empty_like(Md)
        H0 = torch.randn_like(Md) * Ms
        Heff = H0.clone()
        p.apply(Md, Hd); p.apply_add(Md, Heff); torch.cuda.synchronize()
        want = (H0.double() + Hd.double()).cpu().numpy()
        got = Heff.double().cpu().numpy()
        assert np.abs(got - want).max() / Ms <= (4e-7 if prec == 0 else 1e-15)
        ref = oracle.direct_sum(T, M.astype(np.float64))
        assert np.abs(got - H0.double().cpu().numpy() - ref).max() / Ms <= (TOL32 if prec == 0 else TOL64)


# --------------------------------------------------------------------------------- tensor builder
@pytest.mark.parametrize("n,h", [((64, 32, 4), (2e-9, 2e-9, 1e-9)), ((128, 128, 1), (2e-9, 2e-9, 1e-9)),
                                 ((32, 32, 32), (3e-9, 3e-9, 3e-9)), ((256, 8, 2), (1e-9, 1.5e-9, 0.5e-9))])
def test_builtin_tensor_builder_vs_oracle(torch, B, oracle, n, h):
    """DESIGN.md R5 (ii): |dN| <= 1e-10 everywhere and <= 1e-6 |N| in the far field.  The builder uses
    a multipole series in the far field, the oracle Gauss-Legendre quadrature: independent routes."""
    with B.Plan(n, h, 0, B.DEMAG_FP64) as p:
        Tg = p.get_kernel_real()
    To = oracle.tensor_table(n, h)
    assert np.abs(Tg - To).max() <= 1e-10
    d = np.stack(np.meshgrid(np.arange(n[2]) * h[2], np.arange(n[1]) * h[1], np.arange(n[0]) * h[0], indexing="ij"))
    far = np.sqrt((d ** 2).sum(0)) > 30 * max(h)
    if far.any():
        rel = np.abs(Tg - To)[:, far] / np.maximum(np.abs(To[:, far]), 1e-300)
        big = np.abs(To[:, far]) > 1e-3 * np.abs(To[:, far]).max()
        assert rel[big].max() <= 1e-6


def test_builtin_kernel_end_to_end(torch, B, oracle):
    n, h, Ms = (32, 32, 2), (4e-9, 4e-9, 4e-9), 8e5
    M = rand_M(n, Ms, 1001)
    ref = oracle.direct_sum(oracle.tensor_table(n, h), M.astype(np.float64))
    H32 = run_gpu(torch, B, n, h, None, M, 0, builtin=True)
    assert np.abs(H32 - ref).max() / Ms <= TOL32
    H64 = run_gpu(torch, B, n, h, None, M, 1, builtin=True)
    assert np.abs(H64 - ref).max() / Ms <= 1e-9          # R5 (iii): reported, bounded by builder parity


# --------------------------------------------------------------------------------- energy
def test_energy(torch, B, oracle):
    n, h, Ms = (16, 8, 4), (2e-9, 3e-9, 1e-9), 8e5
    M = rand_M(n, Ms, 3)
    T = oracle.tensor_table(n, h)
    Href = oracle.direct_sum(T, M.astype(np.float64))
    for prec, dt, tol in ((0, torch.float32, 1e-5), (1, torch.float64, 1e-12)):
        with B.Plan(n, h, 0, prec) as p:
            p.set_kernel(T)
            Md = torch.from_numpy(M).to("cuda", dt); Hd = torch.empty_like(Md)
            E = torch.zeros(1, dtype=torch.float64, device="cuda")
            p.apply(Md, Hd); p.energy(Md, Hd, E)
            torch.cuda.synchronize()
            Eref = oracle.energy(M.astype(np.float64), Href, h)
            assert E.item() > 0
            assert abs(E.item() - Eref) <= tol * Eref


# --------------------------------------------------------------------------------- atomistic
def test_atomistic_small_lattice(torch, B, oracle):
    """64^3 spins -> 16^3 macrocells of 4x4x4 (Eq. (9)); scatter is bitwise the cell value."""
    from paper_2308_08447_b200 import workloads as W
    L, c, a, mu_s = (64, 64, 64), (4, 4, 4), 0.3e-9, 2.0
    n = (16, 16, 16); h = (1.2e-9,) * 3
    S = W.random_spins_numpy(L, 1005)
    Mref = oracle.macrocell_average(S.astype(np.float64), c, mu_s, a)
    Ms = oracle.MU_B * mu_s / a ** 3
    T = oracle.tensor_table(n, h)
    Href = oracle.fft_conv(T, Mref)
    with B.Plan(n, h, 0, B.DEMAG_FP32) as p:
        p.set_kernel(T)
        Sd = torch.from_numpy(S).cuda(); Hs = torch.full_like(Sd, float("nan"))
        p.reserve_atomistic()
        p.apply_atomistic(Sd, Hs, c, mu_s, a)
        torch.cuda.synchronize()
        Hs_h = Hs.cpu().numpy()
        want = oracle.macrocell_scatter(Href, c)
        assert np.abs(Hs_h - want).max() / Ms <= TOL32
        cells = Hs_h[:, ::4, ::4, ::4]
        assert np.array_equal(Hs_h, oracle.macrocell_scatter(cells, c))      # piecewise constant, bitwise
        Hs2 = Hs.clone()
        p.reserve_atomistic()
        p.apply_atomistic(Sd, Hs2, c, mu_s, a, accumulate=True)
        torch.cuda.synchronize()
        assert np.allclose(Hs2.cpu().numpy(), 2 * Hs_h, rtol=1e-6, atol=0)
    # non-cubic macrocell, fp64
    L2, c2 = (32, 16, 8), (2, 4, 1)
    n2 = (16, 4, 8); h2 = (2 * a, 4 * a, 1 * a)
    S2 = W.random_spins_numpy(L2, 7).astype(np.float64)
    M2 = oracle.macrocell_average(S2, c2, mu_s, a)
    T2 = oracle.tensor_table(n2, h2)
    want = oracle.macrocell_scatter(oracle.direct_sum(T2, M2), c2)
    with B.Plan(n2, h2, 0, B.DEMAG_FP64) as p:
        p.set_kernel(T2)
        Sd = torch.from_numpy(S2).cuda(); Hs = torch.empty_like(Sd)
        p.reserve_atomistic()
        p.apply_atomistic(Sd, Hs, c2, mu_s, a)
        torch.cuda.synchronize()
        assert np.abs(Hs.cpu().numpy() - want).max() / Ms <= TOL64


# --------------------------------------------------------------------------------- no write outside H, M untouched
GUARD = 1 << 16          # elements of sentinel on either side of every caller array


def _guarded(torch, shape, dt, fill=None):
    """A caller array cut out of the middle of a larger buffer whose margins hold a sentinel bit pattern."""
    nel = int(np.prod(shape))
    pad = (-nel) % 4                                     # keep the next view 16-byte aligned
    buf = torch.full((GUARD + nel + pad + GUARD,), -7.25e33, device="cuda", dtype=dt)
    view = buf[GUARD:GUARD + nel].view(*shape)
    if fill is not None:
        view.copy_(fill)
    return buf, view


def _margins_intact(torch, buf, nel):
    s = torch.tensor(-7.25e33, device="cuda", dtype=buf.dtype)
    return bool((buf[:GUARD] == s).all()) and bool((buf[GUARD + nel:] == s).all())


@pytest.mark.parametrize("n", [(64, 64, 8), (16, 32, 16), (32, 16, 1), (256, 32, 1), (4, 128, 8), (24, 10, 6), (1, 1, 64),
                               (130, 70, 3), (1030, 18, 2)])
@pytest.mark.parametrize("prec", [0, 1])
def test_apply_writes_exactly_H_and_leaves_M_untouched(torch, B, oracle, n, prec):
    """demag_apply / demag_apply_add / demag_energy on caller arrays surrounded by sentinel margins: every element of
    H is written, nothing outside H is, M keeps its bits (include/demag.h: "does not modify M, overwrites H") --
    both kernel families, one-cell-thick, embedded and one-cell-wide meshes."""
    h, Ms = (2e-9, 3e-9, 1e-9), 8e5
    dt = torch.float32 if prec == 0 else torch.float64
    M = torch.from_numpy(rand_M(n, Ms, 90 + sum(n))).to(dt)
    nel = 3 * int(np.prod(n))
    shape = (3, n[2], n[1], n[0])
    with B.Plan(n, h, 0, prec) as p:
        p.set_kernel(None)
        mb, Md = _guarded(torch, shape, dt, M.cuda())
        hb, Hd = _guarded(torch, shape, dt)
        ab, Ha = _guarded(torch, shape, dt, torch.zeros(shape, dtype=dt))
        E = torch.zeros(1, device="cuda", dtype=torch.float64)
        p.apply(Md, Hd); p.apply_add(Md, Ha); p.energy(Md, Hd, E)
        torch.cuda.synchronize()
        assert _margins_intact(torch, mb, nel) and _margins_intact(torch, hb, nel) and _margins_intact(torch, ab, nel)
        assert torch.equal(Md.cpu(), M), "M was modified"
        assert not bool((Hd == torch.tensor(-7.25e33, device="cuda", dtype=dt)).any()), "an element of H was not written"
        assert bool(torch.isfinite(Hd).all())
        assert (Ha.double() - Hd.double()).abs().max().item() / Ms <= (4e-7 if prec == 0 else 1e-15)
        assert E.item() >= 0.0


def test_atomistic_and_extrapolate_write_exactly_their_outputs(torch, B):
    """The spin-field scatter and the sub-step extrapolation on sentinel-guarded arrays."""
    from paper_2308_08447_b200 import workloads as W
    L, c, a, mu_s = (32, 16, 8), (4, 2, 2), 0.3e-9, 2.0
    n = (8, 8, 4); h = (4 * a, 2 * a, 2 * a)
    S = torch.from_numpy(W.random_spins_numpy(L, 11))
    shape = (3, L[2], L[1], L[0]); nel = 3 * int(np.prod(L))
    with B.Plan(n, h, 0, B.DEMAG_FP32) as p:
        p.set_kernel(None)
        sb, Sd = _guarded(torch, shape, torch.float32, S.cuda())
        ob, Hs = _guarded(torch, shape, torch.float32)
        p.reserve_atomistic()
        p.apply_atomistic(Sd, Hs, c, mu_s, a)
        torch.cuda.synchronize()
        assert _margins_intact(torch, sb, nel) and _margins_intact(torch, ob, nel)
        assert torch.equal(Sd.cpu(), S) and bool(torch.isfinite(Hs).all())
        mshape = (3, n[2], n[1], n[0]); mel = 3 * int(np.prod(n))
        hist = [torch.randn(mshape, device="cuda") for _ in range(3)]
        eb, He = _guarded(torch, mshape, torch.float32)
        p.extrapolate(hist, [0.0, 1.0, 2.0], 2.5, He)
        torch.cuda.synchronize()
        assert _margins_intact(torch, eb, mel) and bool(torch.isfinite(He).all())


# --------------------------------------------------------------------------------- ABI error paths
def test_error_paths(torch, B):
    with pytest.raises(B.DemagError) as e:
        B.demag_plan_create(0, 4, 4, 1e-9, 1e-9, 1e-9)
    assert e.value.status == 1
    with pytest.raises(B.DemagError) as e:
        B.demag_plan_create(12, 4, 4, 1e-9, 1e-9, 1e-9, B.DEMAG_PBC_X)
    assert e.value.status == 2                          # a periodic axis cannot be padded
    with pytest.raises(B.DemagError) as e:
        B.demag_plan_create(8193, 4, 4, 1e-9, 1e-9, 1e-9)
    assert e.value.status == 2
    with pytest.raises(B.DemagError) as e:
        B.demag_plan_create(4, 4, 4, -1e-9, 1e-9, 1e-9)
    assert e.value.status == 1
    with pytest.raises(B.DemagError) as e:
        B.demag_plan_create(4, 4, 4, 1e-9, 1e-9, 1e-9, 0, 7)
    assert e.value.status == 1
    with B.Plan((4, 4, 4), (1e-9,) * 3) as p:
        M = torch.zeros((3, 4, 4, 4), device="cuda"); H = torch.zeros_like(M)
        with pytest.raises(B.DemagError) as e:
            p.apply(M, H)
        assert e.value.status == 5                      # NO_KERNEL
        p.set_kernel(None)
        with pytest.raises(B.DemagError) as e:
            p.apply(M, M)
        assert e.value.status == 1                      # aliasing
        with pytest.raises(B.DemagError) as e:
            B._check(B.lib().demag_apply(p.handle, None, H.data_ptr(), None))
        assert e.value.status == 1
        with pytest.raises(B.DemagError) as e:
            B._check(B.lib().demag_apply(p.handle, M.data_ptr() + 4, H.data_ptr(), None))
        assert e.value.status == 1                      # misaligned
        assert p.workspace_bytes() > 0 and p.launches_per_apply() >= 5
        with pytest.raises(B.DemagError) as e:
            p.reserve_atomistic()
            p.apply_atomistic(M, H, (2, 2, 2), 2.0, 0.3e-9)
        assert e.value.status == 1                      # h != c*a
    with B.Plan((4, 4, 4), (1e-9,) * 3, B.DEMAG_PBC_X) as p:
        for bad in (-1, 1001):
            with pytest.raises(B.DemagError) as e:
                p.set_pbc_images(bad)
            assert e.value.status == 1                  # image count out of range


# --------------------------------------------------------------------------------- stream semantics of the hot path
def test_apply_is_capturable_in_a_cuda_graph(torch, B, oracle):
    """include/demag.h: demag_apply "never allocates, never synchronises, never touches the host" -- so a time
    integrator can capture it (and demag_apply_add / demag_extrapolate / demag_energy) into a CUDA graph.  The replayed
    graph must give the eager result bit for bit, for both kernel families and an embedded mesh."""
    for n in [(32, 32, 2), (64, 32, 8), (12, 10, 3), (64, 64, 1)]:
        h, Ms = (2e-9, 2e-9, 2e-9), 8e5
        M = rand_M(n, Ms, 17)
        with B.Plan(n, h, 0, 0) as p:
            p.set_kernel(None)
            Md = torch.from_numpy(M).cuda()
            H0, H1, Heff = torch.empty_like(Md), torch.empty_like(Md), torch.zeros_like(Md)
            E = torch.zeros(1, dtype=torch.float64, device="cuda")
            p.apply(Md, H0); torch.cuda.synchronize()
            g = torch.cuda.CUDAGraph()
            s = torch.cuda.Stream()
            with torch.cuda.stream(s):
                with torch.cuda.graph(g, stream=s):
                    p.apply(Md, H1)
                    p.apply_add(Md, Heff)
                    p.energy(Md, H1, E)
            Md.copy_(torch.from_numpy(rand_M(n, Ms, 18)).cuda())          # new input, same addresses
            p.apply(Md, H0); torch.cuda.synchronize()
            for rep in range(3):
                g.replay()
            torch.cuda.synchronize()
            assert torch.equal(H0, H1)
            assert torch.allclose(Heff, 3 * H0, rtol=1e-5, atol=1e-5 * Ms)
            assert abs(E.item() - oracle.energy(Md.cpu().numpy().astype(np.float64), H0.cpu().numpy().astype(np.float64), h)) <= 1e-6 * abs(E.item())


def test_apply_atomistic_never_allocates_and_its_first_call_is_capturable(torch, B, oracle):
    """include/demag.h: the macrocell arrays are allocated by demag_atomistic_reserve, never by demag_apply_atomistic:
    without them the call fails with INVALID_ARG; with them the workspace does not change any more and the very FIRST
    atomistic call of a plan can be captured in a CUDA graph (replay == Eq. (9) average -> Eq. (1) -> scatter)."""
    from paper_2308_08447_b200 import workloads as W
    L, c, a, mu_s = (32, 16, 8), (4, 2, 2), 0.3e-9, 2.0
    n = (8, 8, 4); h = (4 * a, 2 * a, 2 * a)
    S = W.random_spins_numpy(L, 21)
    Mref = oracle.macrocell_average(S.astype(np.float64), c, mu_s, a)
    T = oracle.tensor_table(n, h)
    want = oracle.macrocell_scatter(oracle.direct_sum(T, Mref), c)
    Ms = oracle.MU_B * mu_s / a ** 3
    with B.Plan(n, h, 0, B.DEMAG_FP32) as p:
        p.set_kernel(T)
        Sd = torch.from_numpy(S).cuda(); Hs = torch.full_like(Sd, float("nan"))
        w0 = p.workspace_bytes()
        with pytest.raises(B.DemagError) as e:
            p.apply_atomistic(Sd, Hs, c, mu_s, a)
        assert e.value.status == 1 and "demag_atomistic_reserve" in str(e.value)
        assert p.workspace_bytes() == w0
        p.reserve_atomistic()
        w1 = p.workspace_bytes()
        assert w1 == w0 + 2 * 3 * int(np.prod(n)) * 4
        p.reserve_atomistic()                                                # idempotent
        assert p.workspace_bytes() == w1
        g = torch.cuda.CUDAGraph()
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            with torch.cuda.graph(g, stream=st):
                p.apply_atomistic(Sd, Hs, c, mu_s, a)                        # first atomistic call of this plan
        g.replay(); torch.cuda.synchronize()
        assert p.workspace_bytes() == w1
        assert np.abs(Hs.cpu().numpy().astype(np.float64) - want).max() / Ms <= TOL32


def test_plan_is_bound_to_its_device_and_bad_tuning_values_are_ignored(torch, B, oracle, monkeypatch):
    """Tuning toggles with nonsense values must not break a plan (they are ignored), and the results stay the oracle's."""
    n, h, Ms = (32, 16, 16), (2e-9, 2e-9, 2e-9), 8e5
    M = rand_M(n, Ms, 5)
    T = oracle.tensor_table(n, h)
    ref = oracle.direct_sum(T, M.astype(np.float64))
    for k, v in (("DEMAG_TY", "0"), ("DEMAG_TY", "-3"), ("DEMAG_B2_KB", "0"), ("DEMAG_SLAB_MB", "-1"), ("DEMAG_PDL", "7"),
                 ("DEMAG_PF", "nan"), ("DEMAG_PF", "-2")):
        monkeypatch.setenv(k, v)
        for path in ("generic", "fast"):
            monkeypatch.setenv("DEMAG_PATH", path)
            H = run_gpu(torch, B, n, h, T, M, 0)
            assert np.abs(H - ref).max() / Ms <= TOL32, (k, v, path)
        monkeypatch.delenv(k)


def test_two_plans_on_two_streams_do_not_interfere(torch, B, oracle):
    n, h, Ms = (64, 64, 8), (2e-9, 2e-9, 2e-9), 8e5
    Ma, Mb = rand_M(n, Ms, 1), rand_M(n, Ms, 2)
    with B.Plan(n, h, 0, 0) as pa, B.Plan(n, h, 0, 0) as pb:
        pa.set_kernel(None); pb.set_kernel(None)
        A, Bm = torch.from_numpy(Ma).cuda(), torch.from_numpy(Mb).cuda()
        Ha0, Hb0 = torch.empty_like(A), torch.empty_like(A)
        pa.apply(A, Ha0); pb.apply(Bm, Hb0); torch.cuda.synchronize()
        sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
        Ha, Hb = torch.empty_like(A), torch.empty_like(A)
        for _ in range(20):
            pa.apply(A, Ha, stream=sa); pb.apply(Bm, Hb, stream=sb)
        torch.cuda.synchronize()
        assert torch.equal(Ha, Ha0) and torch.equal(Hb, Hb0)


def test_create_destroy_returns_all_device_memory(torch, B):
    torch.cuda.synchronize()
    with B.Plan((64, 64, 8), (2e-9,) * 3) as p:                          # first plan: one-time context / module allocations
        p.set_kernel(None)
    free0, _ = torch.cuda.mem_get_info()
    for i in range(20):
        with B.Plan((64, 64, 8), (2e-9,) * 3, 0, i % 2) as p:
            p.set_kernel(None)
            assert p.workspace_bytes() > 0
        sp = B.ShardedPlan((64, 64, 8), (2e-9,) * 3, 0, rank=i % 2, world=2, connect=False)
        sp.set_kernel(None); sp.close()
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free0 - free1 <= (8 << 20), (free0, free1)                    # nothing of 20 plans' ~10 MB each is left behind
