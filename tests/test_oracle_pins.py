"""Pins of the fp64 oracle against what the paper and the mathematics fix (CPU only).

The paper prints no worked example for this path (tests/golden/README.md), so every pin is a closed
form, an invariant, an independent evaluation of the DEFINITION, or brute force on tiny inputs.
Each test says which plausible mistake it would catch.
"""
import os

import numpy as np
import pytest

from paper_2308_08447_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")
CELLS = [(1.0, 1.0, 1.0), (2.0, 2.0, 1.0), (1.0, 1.5, 0.5), (3e-9, 2e-9, 5e-9)]


# ------------------------------------------------------------------------------------ tensor N
def test_golden_self_demag(oracle):
    """north_star: trace 1, cube 1/3; film / rod limits.  Catches a wrong prefactor or sign of N."""
    for line in open(os.path.join(GOLD, "self_demag.txt")):
        if line.startswith("#") or not line.strip():
            continue
        t = line.split()
        h = tuple(map(float, t[:3])); want = np.array(list(map(float, t[3:6]))); tol = float(t[6])
        got = oracle.newell_N((0, 0, 0), h)
        assert np.allclose(got[:3], want, atol=tol, rtol=0), (h, got)
        assert abs(got[:3].sum() - 1.0) < 1e-10   # 1000:1 aspect: closed-form cancellation
        assert np.abs(got[3:]).max() < 1e-15


@pytest.mark.parametrize("h", CELLS)
def test_self_term_trace_is_one(oracle, h):
    n = oracle.newell_N((0, 0, 0), h)
    assert abs(n[0] + n[1] + n[2] - 1.0) < 2e-12
    assert np.all(n[:3] > 0)


@pytest.mark.parametrize("h", CELLS)
def test_trace_vanishes_off_self(oracle, h):
    """Laplace: trace N(r) = 0 for r != 0.  Catches a dropped term in f."""
    rng = np.random.default_rng(3)
    for _ in range(40):
        d = rng.integers(-6, 7, size=3)
        if not d.any():
            continue
        n = oracle.N_at(d * np.array(h), h)
        assert abs(n[:3].sum()) < 2e-13 * max(1.0, 1.0), (d, n[:3].sum())


@pytest.mark.parametrize("h", CELLS)
def test_parity(oracle, h):
    """Diagonal even; xy odd in x,y; xz odd in x,z; yz odd in y,z; off-diagonals vanish on mirror planes."""
    r = np.array([3, 2, 1]) * np.array(h)
    n0 = oracle.N_at(r, h)
    for sx in (1, -1):
        for sy in (1, -1):
            for sz in (1, -1):
                n = oracle.N_at(r * np.array([sx, sy, sz]), h)
                want = n0 * np.array([1, 1, 1, sx * sy, sx * sz, sy * sz])
                assert np.allclose(n, want, rtol=0, atol=1e-14)
    z = lambda rr, cs: np.abs(oracle.N_at(rr, h)[list(cs)]).max() < 1e-15   # exact up to summation order
    assert z((0, r[1], r[2]), (3, 4)) and z((r[0], 0, r[2]), (3, 5)) and z((r[0], r[1], 0), (4, 5))


def test_component_permutation(oracle):
    """Swapping axes permutes components: catches a wrong argument order in Nyy/Nzz/Nxz/Nyz."""
    h = np.array([1.0, 1.5, 0.5]); r = np.array([2.0, -3.0, 1.0])
    n = oracle.newell_N(r, h)
    # swap x<->y: xx<->yy, xz<->yz
    m = oracle.newell_N(r[[1, 0, 2]], h[[1, 0, 2]])
    assert np.allclose(m, n[[1, 0, 2, 3, 5, 4]], rtol=1e-11, atol=1e-16)
    # swap x<->z: xx<->zz, xy<->yz
    m = oracle.newell_N(r[[2, 1, 0]], h[[2, 1, 0]])
    assert np.allclose(m, n[[2, 1, 0, 5, 4, 3]], rtol=1e-11, atol=1e-16)


def _dipole(r, V):
    r = np.asarray(r, float); R = np.linalg.norm(r)
    K = (np.eye(3) / R ** 3 - 3 * np.outer(r, r) / R ** 5) * V / (4 * np.pi)
    return np.array([K[0, 0], K[1, 1], K[2, 2], K[0, 1], K[0, 2], K[1, 2]])


def test_far_field_dipole_limit(oracle):
    """N(r) -> (V/4pi)(delta/r^3 - 3 r r/r^5).  Catches sign/scale errors of every component."""
    h = (3.0, 2.0, 1.0)
    r = (30.0, -20.0, 7.0)
    n = oracle.newell_N(r, h); d = _dipole(r, 6.0)
    assert np.allclose(n, d, rtol=0.02, atol=2e-8)
    r = (300.0, -200.0, 70.0)
    n = oracle.N_at(r, h); d = _dipole(r, 6.0)
    assert np.allclose(n, d, rtol=3e-4, atol=1e-12)


def _numpy_quadrature_N(r, h, m=24):
    """Independent evaluation of the DEFINITION: N = V int prod(tent) K(r+u) d3u with numpy leggauss
    (not the oracle's own node tables).  Valid when the two cells do not touch."""
    x, w = np.polynomial.legendre.leggauss(m)
    t = 0.5 * (x + 1.0); w = 0.5 * w
    nodes = []; wts = []
    for hc in h:
        nodes.append(np.concatenate([t * hc, -t * hc])); wts.append(np.concatenate([w * (1 - t), w * (1 - t)]))
    ux, uy, uz = np.meshgrid(*nodes, indexing="ij")
    Wt = wts[0][:, None, None] * wts[1][None, :, None] * wts[2][None, None, :]
    p = [r[0] + ux, r[1] + uy, r[2] + uz]
    R2 = p[0] ** 2 + p[1] ** 2 + p[2] ** 2; R = np.sqrt(R2)
    out = []
    for a, b in ((0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2)):
        K = ((a == b) / R ** 3 - 3 * p[a] * p[b] / R ** 5)
        out.append((Wt * K).sum())
    return np.array(out) * np.prod(h) / (4 * np.pi)


@pytest.mark.parametrize("h", CELLS[:3])
@pytest.mark.parametrize("d", [(2, 0, 0), (0, 2, 1), (1, 1, 2), (2, -1, 1), (3, 2, 0), (-2, 3, 4)])
def test_newell_equals_integral_definition(oracle, h, d):
    """Closed form vs the 6-fold integral (reduced to the tent-weighted 3-fold one), near field."""
    r = np.array(d) * np.array(h)
    want = _numpy_quadrature_N(r, h)
    got = oracle.newell_N(r, h)
    assert np.allclose(got, want, rtol=0, atol=2e-9), (got - want)


def test_oracle_quadrature_matches_numpy_quadrature(oracle):
    h = (2.0, 2.0, 1.0); r = (41.0, -13.0, 9.0)
    assert np.allclose(oracle.quad_N(r, h, 3), _numpy_quadrature_N(r, h, 12), rtol=0, atol=1e-14)
    assert np.allclose(oracle.quad_N(r, h, 6), _numpy_quadrature_N(r, h, 12), rtol=0, atol=1e-17)


def test_near_far_switch_band(oracle):
    """R4: Newell and quadrature agree to <= 5e-12 abs in the band around the switch radius (16 cells),
    and the m=2 / m=3 quadratures agree beyond 128 cells."""
    h = (2.0, 2.0, 1.0)
    rng = np.random.default_rng(11)
    for _ in range(200):
        u = rng.standard_normal(3); u /= np.linalg.norm(u)
        r = u * rng.uniform(12, 24) * 2.0
        r = np.round(r / np.array(h)) * np.array(h)
        a = oracle.newell_N(r, h); b = oracle.quad_N(r, h, 3); c = oracle.quad_N(r, h, 6)
        assert np.abs(a - c).max() < 5e-12 and np.abs(b - c).max() < 5e-12
    for _ in range(50):
        u = rng.standard_normal(3); u /= np.linalg.norm(u)
        r = u * rng.uniform(128, 400) * 2.0
        assert np.abs(oracle.quad_N(r, h, 2) - oracle.quad_N(r, h, 6)).max() < 1e-15


def test_refinement_identity_diagonal(oracle):
    """(1/n_c) sum_i sum_j N_aa(i-j; h) = N_aa(0; n*h): the body's own self term.  Ties the self term,
    the touching-neighbour terms and the parity folding together; catches any wrong near-field entry."""
    n = (4, 3, 2); h = (1.0, 1.5, 0.5)
    T = oracle.tensor_table(n, h)
    nc = np.prod(n)
    body = oracle.newell_N((0, 0, 0), tuple(np.array(n) * np.array(h)))
    for a in range(3):
        M = np.zeros((3, n[2], n[1], n[0])); M[a] = 1.0
        H = oracle.direct_sum(T, M)
        assert abs(-H[a].sum() / nc - body[a]) < 1e-14
    # survey-recorded digits for this body
    assert np.allclose(body[:3], [0.1793320815, 0.1585421340, 0.6621257845], atol=2e-10)


def test_block_refinement_off_diagonal(oracle):
    """N_ab(o*2h; cell 2h) = (1/8) sum over the 64 cell pairs of two 2x2x2 blocks of N_ab(.; cell h)."""
    h = np.array([1.0, 1.5, 0.5])
    for o in [(1, 1, 0), (1, 2, 1), (2, 0, 1), (0, 1, 1)]:
        big = oracle.newell_N(np.array(o) * 2 * h, tuple(2 * h))
        acc = np.zeros(6)
        for i in np.ndindex(2, 2, 2):
            for j in np.ndindex(2, 2, 2):
                d = 2 * np.array(o) + np.array(i) - np.array(j)
                acc += oracle.newell_N(d * h, tuple(h))
        assert np.allclose(acc / 8.0, big, rtol=0, atol=2e-14), (o, acc / 8 - big)


def test_far_field_refinement_detects_cancellation(oracle):
    """Uniform 256x256x1 body: the table with the far-field treatment satisfies the refinement
    identity to ~1e-12; a plain closed-form table would miss by ~1e-9 (catastrophic cancellation)."""
    n = (256, 256, 1); h = (2.0, 2.0, 1.0)
    T = oracle.tensor_table(n, h)
    body = oracle.newell_N((0, 0, 0), (512.0, 512.0, 1.0))
    # sum_i sum_j T(|i-j|) = sum_d mult(d) T(d), mult = prod (n_a - |d_a|), both signs of d
    wx = (n[0] - np.arange(n[0])) * np.where(np.arange(n[0]) == 0, 1, 2)
    wy = (n[1] - np.arange(n[1])) * np.where(np.arange(n[1]) == 0, 1, 2)
    for a in range(3):
        s = (T[a, 0] * wy[:, None] * wx[None, :]).sum() / (n[0] * n[1])
        assert abs(s - body[a]) < 2e-11, (a, s - body[a])


# ----------------------------------------------------------------------------- Eq. (1), O-A/O-B
def _tiny(oracle, n=(8, 6, 2), h=(1.0, 1.5, 0.5), seed=5):
    T = oracle.tensor_table(n, h)
    M = np.random.default_rng(seed).standard_normal((3, n[2], n[1], n[0]))
    return T, M


def test_direct_sum_vs_pure_python(oracle):
    """O-A against Eq. (1) typed as Python loops with SIGNED offsets through N_at (no table, no parity
    folding): catches an index or sign slip in the folded table lookup."""
    n = (3, 2, 2); h = (1.0, 1.5, 0.5)
    T, M = _tiny(oracle, n, h)
    H = oracle.direct_sum(T, M)
    comp = oracle.COMP
    for iz, iy, ix in np.ndindex(n[2], n[1], n[0]):
        acc = np.zeros(3)
        for jz, jy, jx in np.ndindex(n[2], n[1], n[0]):
            N6 = oracle.N_at(((ix - jx) * h[0], (iy - jy) * h[1], (iz - jz) * h[2]), h)
            N33 = N6[comp]
            acc -= N33 @ M[:, jz, jy, jx]
        assert np.allclose(H[:, iz, iy, ix], acc, rtol=0, atol=1e-14)


def test_impulse_response_is_minus_N(oracle):
    """A single magnetised cell at j returns the column -N(i-j) (Eq. (1) read backwards)."""
    n = (5, 4, 3); h = (1.0, 1.5, 0.5)
    T = oracle.tensor_table(n, h)
    j = (2, 1, 1)  # (jx, jy, jz)
    for b in range(3):
        M = np.zeros((3, n[2], n[1], n[0])); M[b, j[2], j[1], j[0]] = 1.0
        for H in (oracle.direct_sum(T, M), oracle.naive_dft_conv(T, M), oracle.fft_conv(T, M)):
            for iz, iy, ix in np.ndindex(n[2], n[1], n[0]):
                N6 = oracle.N_at(((ix - j[0]) * h[0], (iy - j[1]) * h[1], (iz - j[2]) * h[2]), h)
                want = -N6[oracle.COMP][:, b]
                assert np.allclose(H[:, iz, iy, ix], want, rtol=0, atol=1e-14)


def test_direct_sum_equals_naive_dft_convolution(oracle):
    """north_star: direct sum == FFT convolution on tiny grids (O-A vs O-B), for P = 2n and P = 2n-1."""
    T, M = _tiny(oracle)
    HA = oracle.direct_sum(T, M)
    HB = oracle.naive_dft_conv(T, M)
    assert np.abs(HA - HB).max() < 5e-15 * np.abs(M).max() * 10
    HB2 = oracle.naive_dft_conv(T, M, P=(15, 11, 3))
    assert np.abs(HA - HB2).max() < 5e-14
    HC = oracle.fft_conv(T, M)
    assert np.abs(HA - HC).max() < 5e-14


def test_thin_axis_is_not_padded(oracle):
    """R6: an axis with n_a = 1 is neither padded nor transformed (config 2)."""
    n = (8, 6, 1); T, M = _tiny(oracle, n, (2.0, 2.0, 1.0))
    assert oracle.padded_shape(n) == (16, 12, 1)
    assert np.abs(oracle.direct_sum(T, M) - oracle.naive_dft_conv(T, M)).max() < 1e-14
    assert np.abs(oracle.direct_sum(T, M) - oracle.fft_conv(T, M)).max() < 1e-14


def test_kernel_spectrum_is_real(oracle):
    """the transformed kernel can be stored as real arrays (two odd axes -> (-i)^2)."""
    T, _ = _tiny(oracle)
    assert oracle.kernel_spectrum_imag_ratio(T) < 1e-12


def test_sampled_equals_full(oracle):
    T, M = _tiny(oracle)
    H = oracle.direct_sum(T, M)
    cells = W.sample_cells((8, 6, 2), 40, 1)
    Hs = oracle.direct_sum_sampled(T, M, cells)
    assert np.array_equal(Hs, H.reshape(3, -1)[:, cells].T)


def test_linearity_and_translation(oracle):
    T, M = _tiny(oracle)
    M2 = np.random.default_rng(9).standard_normal(M.shape)
    H = oracle.direct_sum(T, 2.0 * M - 3.0 * M2)
    assert np.abs(H - (2.0 * oracle.direct_sum(T, M) - 3.0 * oracle.direct_sum(T, M2))).max() < 1e-13


def test_uniform_film_field(oracle):
    """north_star: uniformly z-magnetised large thin film gives H ~ -Mz z^.  Mean field equals
    -Nzz(0; body) Ms exactly (refinement identity through the convolution)."""
    n = (256, 256, 1); h = (2.0, 2.0, 1.0); Ms = 8e5
    T = oracle.tensor_table(n, h)
    M = np.zeros((3, 1, 256, 256)); M[2] = Ms
    H = oracle.fft_conv(T, M)
    body = oracle.newell_N((0, 0, 0), (512.0, 512.0, 1.0))
    assert abs(H[2].mean() / Ms + body[2]) < 1e-10
    assert abs(H[2, 0, 128, 128] / Ms + 1.0) < 5e-3           # centre: H ~ -Ms
    assert np.abs(H[:2, 0, 128, 128]).max() / Ms < 1e-9      # no in-plane field at the centre
    # sampled direct sum at the centre agrees with the FFT route
    c = np.array([128 * 256 + 128])
    assert np.abs(oracle.direct_sum_sampled(T, M, c)[0] - H[:, 0, 128, 128]).max() / Ms < 1e-11


def test_energy_nonnegative_and_prism_closed_form(oracle):
    """north_star: demag energy >= 0; uniformly magnetised prism: E = (mu0/2) Ms^2 V N_aa(0; body)."""
    n = (8, 6, 2); h = (1e-9, 1.5e-9, 0.5e-9)
    T = oracle.tensor_table(n, h)
    rng = np.random.default_rng(21)
    for _ in range(5):
        M = rng.standard_normal((3, n[2], n[1], n[0])) * 8e5
        assert oracle.energy(M, oracle.direct_sum(T, M), h) > 0
    body_h = tuple(np.array(n) * np.array(h)); Vb = np.prod(body_h)
    body = oracle.newell_N((0, 0, 0), body_h)
    for a in range(3):
        M = np.zeros((3, n[2], n[1], n[0])); M[a] = 8e5
        E = oracle.energy(M, oracle.direct_sum(T, M), h)
        assert abs(E - 0.5 * oracle.MU0 * 8e5 ** 2 * Vb * body[a]) < 1e-12 * E


# ----------------------------------------------------------------------------- atomistic, Eq. (9)
def test_macrocell_average_and_scatter(oracle):
    """Eq. (9): fully aligned spins give M = mu_B mu_s / a^3 whatever the macrocell; scatter copies."""
    a = 0.3e-9; mu_s = 2.0
    S = np.zeros((3, 8, 8, 8)); S[2] = 1.0
    M = oracle.macrocell_average(S, (4, 2, 2), mu_s, a)
    assert M.shape == (3, 4, 4, 2)
    assert np.allclose(M[2], oracle.MU_B * mu_s / a ** 3, rtol=1e-14) and np.all(M[:2] == 0)
    assert abs(oracle.MU_B * mu_s / a ** 3 - 6.870e5) < 5e1          # "Ms" of config 5
    S = W.random_spins_numpy((8, 4, 4), 3).astype(np.float64)
    M = oracle.macrocell_average(S, (4, 2, 2), mu_s, a)
    blk = S[:, 2:4, 0:2, 4:8].sum(axis=(1, 2, 3)) * oracle.MU_B * mu_s / (16 * a ** 3)
    assert np.allclose(M[:, 1, 0, 1], blk, rtol=1e-14)
    Hs = oracle.macrocell_scatter(M, (4, 2, 2))
    assert Hs.shape == S.shape and np.array_equal(Hs[:, 3, 1, 5], M[:, 1, 0, 1])
    assert np.allclose(oracle.macrocell_average(Hs, (4, 2, 2), 1.0, 1.0) * 16 / oracle.MU_B, M * 16, rtol=1e-13)


def test_dipole_tensor_rearranges_eq8_into_eq1(oracle):
    """"Equation (8) can be re-arranged into the form of Equation (1)".  The rearrangement
    (oracle.dipole_table + the direct sum of Eq. (1)) against Eq. (8) written out pair by pair; plus what the
    mathematics fixes for the tensor: zero trace (Laplace), zero self term, the parity of R1, and the far-field limit
    of the cell-averaged (Newell) tensor of a cube of edge a."""
    from paper_2308_08447_b200 import workloads as W
    L, a, mu_s = (6, 5, 3), 0.3e-9, 2.0
    S = W.random_spins_numpy(L, 5).astype(np.float64)
    T = oracle.dipole_table(L, a)
    M = S * (oracle.MU_B * mu_s / a ** 3)
    H1 = oracle.direct_sum(T, M)
    H8 = oracle.dipole_field_eq8(S, mu_s, a)
    assert np.abs(H1 - H8).max() <= 1e-12 * np.abs(H8).max()
    assert np.abs(T[0] + T[1] + T[2]).max() <= 1e-18 + 1e-15 * np.abs(T).max()
    assert np.all(T[:, 0, 0, 0] == 0)
    assert np.all(T[3, :, 0, :] == 0) and np.all(T[3, :, :, 0] == 0)          # xy vanishes on its mirror planes
    far = oracle.N_at((9 * a, 7 * a, 5 * a), (a, a, a))
    Tf = oracle.dipole_table((10, 8, 6), a)[:, 5, 7, 9]
    assert np.abs(far - Tf).max() <= 2e-3 * np.abs(Tf).max()                  # cube -> point dipole, O((a/r)^4)


def test_periodic_tensor_table_invariants_and_film_limit(oracle):
    """oracle.periodic_tensor_table (reading R11).  Pins: (i) trace identity Nxx + Nyy + Nzz = delta(d) survives the image
    sum (only the m = 0 image of d = 0 has r = 0); (ii) exact symmetry T(n - d) = parity T(d) on periodic axes, open axes
    untouched; (iii) the symmetrised sum equals the image sum over m = -I-1 .. I with weight 1/2 on the two end images
    for d > 0, the plain sum over |m| <= I for d = 0 (parity N(-x) = N(x)); (iv) physics: with x and y periodic, a uniformly z-magnetised mesh is a square plate of side
    L = (2 I + 1) n h seen from its centre, whose demagnetizing factor is 1 - Omega / 2 pi -> 1 - (2 sqrt2 / pi) t / L for
    a thin plate (solid angle of a square from a point t/2 above its centre): sum_d Tzz(d) tends to the infinite film's 1
    at exactly that rate."""
    h = (2e-9, 3e-9, 1e-9)
    n, pbc, I = (4, 3, 2), (True, False, True), 2
    T = oracle.periodic_tensor_table(n, h, pbc, I)
    tr = T[0] + T[1] + T[2]
    assert abs(tr[0, 0, 0] - 1) < 1e-12 and np.abs(tr.reshape(-1)[1:]).max() < 1e-12
    for a, ax in ((0, 3), (2, 1)):
        idx = (-np.arange(n[a])) % n[a]
        assert np.abs(T - oracle.PARITY[:, a].reshape(6, 1, 1, 1) * np.take(T, idx, axis=ax)).max() < 1e-15
    Topen = oracle.tensor_table((1, 3, 1), h)
    assert np.abs(oracle.periodic_tensor_table((1, 3, 1), h, (False, False, False), 5) - Topen).max() == 0
    W = np.zeros_like(T)
    wt = lambda m, d: 1.0 if d == 0 else 0.5 if m in (-I - 1, I) else 1.0
    for dz in range(n[2]):
        for dy in range(n[1]):
            for dx in range(n[0]):
                for mx in range(-I - (dx > 0), I + 1):
                    for mz in range(-I - (dz > 0), I + 1):
                        W[:, dz, dy, dx] += wt(mx, dx) * wt(mz, dz) * oracle.N_at(((dx + mx * n[0]) * h[0], dy * h[1], (dz + mz * n[2]) * h[2]), h)
    assert np.abs(W - T).max() < 1e-13
    # (iv) the film limit, cube cells of edge t, mesh 2 x 2 x 1
    t = 1e-9
    for I in (6, 12):
        Tf = oracle.periodic_tensor_table((2, 2, 1), (t, t, t), (True, True, False), I)
        L = (2 * I + 1) * 2 * t
        deficit = 1.0 - Tf[2].sum()
        assert 0 < deficit < 0.1
        assert abs(deficit / (2 * np.sqrt(2) / np.pi * t / L) - 1) < 0.05, (I, deficit, 2 * np.sqrt(2) / np.pi * t / L)


def test_poly_extrapolate_reproduces_polynomials(oracle):
    """oracle.poly_extrapolate (R19).  Pins: a field whose entries ARE polynomials in t of degree <= p is
    reproduced exactly at any time from p+1 samples (quartic for RK4: 5 samples; quintic for RKF56: 6), and not from
    p samples; at a sample time the sample itself comes back; the result equals NumPy's least-squares polynomial fit
    of the same degree (which interpolates when the system is square)."""
    rng = np.random.default_rng(7)
    for p in (4, 5):
        coef = rng.normal(size=(p + 1, 3, 2, 3, 4))
        f = lambda t: sum(coef[d] * t ** d for d in range(p + 1))
        ts = np.sort(rng.uniform(0.0, 1.0, p + 1))
        H = [f(t) for t in ts]
        for t in (1.3, 0.5 * (ts[0] + ts[1]), -0.2):
            assert np.abs(oracle.poly_extrapolate(H, ts, t) - f(t)).max() <= 1e-9 * np.abs(f(t)).max()
        assert np.abs(oracle.poly_extrapolate(H[1:], ts[1:], 1.3) - f(1.3)).max() > 1e-4      # one sample short: not exact
        assert np.abs(oracle.poly_extrapolate(H, ts, ts[2]) - H[2]).max() <= 1e-12 * np.abs(H[2]).max()
        flat = np.stack([h.reshape(-1) for h in H])
        fit = np.polynomial.polynomial.polyfit(ts, flat, p)
        ref = np.polynomial.polynomial.polyval(1.3, fit).reshape(H[0].shape)
        assert np.abs(oracle.poly_extrapolate(H, ts, 1.3) - ref).max() <= 1e-7 * np.abs(ref).max()
    one = oracle.poly_extrapolate([np.full((2, 2), 3.0)], [0.1], 9.0)                          # degree 0: constant
    assert np.array_equal(one, np.full((2, 2), 3.0))


# ------------------------------------------------------------------------------------ LLG (NEXT row 4)
def _macrospin(oracle, m0, H, alpha, dt, n, Ms=8e5):
    """One cell, no demagnetizing field: Eq. (5) in a static uniform field has a closed-form solution."""
    M0 = (Ms * np.asarray(m0, dtype=np.float64)).reshape(3, 1, 1, 1)
    Mf, avg, _ = oracle.llg_rk4_run(None, M0, Ms, H, alpha, dt, n, demag=lambda X: np.zeros_like(X))
    return Mf.ravel() / Ms, avg / Ms


def test_llg_macrospin_matches_the_closed_form(oracle):
    """Eq. (5) with H = H z^: m_z(t) = tanh(alpha g H t + atanh m_z(0)), azimuth phi(t) = phi(0) + g H t,
    g = gamma / (1 + alpha^2) (textbook solution of the LLG equation for a macrospin).  Catches a wrong sign of the
    precession or damping term, a missing 1/(1 + alpha^2), a wrong RK4 weight."""
    alpha, H = 0.1, 1.0e5
    g = oracle.GAMMA_LLG / (1.0 + alpha * alpha)
    th0, ph0 = 0.7, 0.3
    m0 = [np.sin(th0) * np.cos(ph0), np.sin(th0) * np.sin(ph0), np.cos(th0)]
    dt, n = 1.0e-13, 500
    m, avg = _macrospin(oracle, m0, (0.0, 0.0, H), alpha, dt, n)
    for i in (1, 100, n):
        t = i * dt
        mz = np.tanh(alpha * g * H * t + np.arctanh(np.cos(th0)))
        ph = ph0 + g * H * t
        want = np.array([np.sqrt(1 - mz * mz) * np.cos(ph), np.sqrt(1 - mz * mz) * np.sin(ph), mz])
        assert np.abs(avg[i] - want).max() < 1e-9, (i, avg[i], want)
    assert abs(np.linalg.norm(m) - 1.0) < 1e-12


def test_llg_rhs_is_orthogonal_to_m_and_vanishes_at_equilibrium(oracle):
    rng = np.random.default_rng(3)
    M = rng.standard_normal((3, 4, 5, 6)); H = 1e5 * rng.standard_normal((3, 4, 5, 6))
    Ms = 8e5
    M *= Ms / np.sqrt((M * M).sum(axis=0, keepdims=True))
    K = oracle.llg_rhs(M, H, Ms, 0.3)
    assert np.abs((K * M).sum(axis=0)).max() <= 1e-12 * np.abs(K).max() * Ms          # |M| is conserved by the flow
    assert np.abs(oracle.llg_rhs(M, 2.5 * M, Ms, 0.3)).max() <= 1e-9 * oracle.GAMMA_LLG * Ms * Ms * 1e-6   # M || H: no torque
    # alpha = 0: pure precession, dM/dt = -gamma M x H exactly
    assert np.allclose(oracle.llg_rhs(M, H, Ms, 0.0), -oracle.GAMMA_LLG * np.cross(M, H, axis=0), rtol=1e-14, atol=0)


def test_llg_rk4_is_fourth_order_and_conserves_energy_without_damping(oracle):
    alpha, H = 0.05, 2.0e5
    g = oracle.GAMMA_LLG / (1.0 + alpha * alpha)
    th0 = 1.1
    m0 = [np.sin(th0), 0.0, np.cos(th0)]
    T = 2.0e-11
    errs = []
    for n in (50, 100, 200):
        m, _ = _macrospin(oracle, m0, (0.0, 0.0, H), alpha, T / n, n)
        mz = np.tanh(alpha * g * H * T + np.arctanh(np.cos(th0)))
        ph = g * H * T
        want = np.array([np.sqrt(1 - mz * mz) * np.cos(ph), np.sqrt(1 - mz * mz) * np.sin(ph), mz])
        errs.append(np.abs(m - want).max())
    assert 12.0 < errs[0] / errs[1] < 20.0 and 12.0 < errs[1] / errs[2] < 20.0, errs      # error ~ dt^4
    m, avg = _macrospin(oracle, m0, (0.0, 0.0, H), 0.0, 1e-13, 300)
    assert np.abs(avg[:, 2] - np.cos(th0)).max() < 1e-10                                   # m . H conserved when alpha = 0


def test_llg_with_demag_dissipates_energy_and_extrapolation_tracks_the_full_run(oracle):
    """Small film with the demagnetizing field: (i) E_d + E_Zee never increases for alpha > 0 (the LLG flow is a
    gradient-like flow of the energy: dE/dt = -alpha mu0 g/Ms |M x H|^2 V <= 0); (ii) |M| stays Ms; (iii) the run that
    replaces the sub-step convolutions by the quartic through the five last full-step fields stays within
    1e-6 of the run that convolves at every stage, with 16 + (n - 4) convolutions instead of 4 n."""
    n, h, Ms = (16, 8, 2), (5e-9, 5e-9, 5e-9), 8e5
    Tn = oracle.tensor_table(n, h)
    M0 = W.random_unit_vectors(n, Ms, 5).astype(np.float64)
    M0[0] += 2.0 * Ms                                        # mostly along +x with a random tilt
    M0 *= Ms / np.sqrt((M0 * M0).sum(axis=0, keepdims=True))
    Hz = (-2.0e4, 1.0e3, 0.0)                                # the switching field of PAPER.md:47
    alpha, dt, steps = 0.1, 1.0e-13, 60
    V = float(np.prod(h))

    def energy_of(M):
        Hd = oracle.fft_conv(Tn, M)
        return oracle.energy(M, Hd, h) - oracle.MU0 * V * float((M * np.asarray(Hz).reshape(3, 1, 1, 1)).sum())
    Es, M = [energy_of(M0)], M0
    for _ in range(6):
        M, _, _ = oracle.llg_rk4_run(Tn, M, Ms, Hz, alpha, dt, 10)
        Es.append(energy_of(M))
        assert np.abs(np.sqrt((M * M).sum(axis=0)) / Ms - 1.0).max() < 1e-9
    assert all(b <= a + 1e-12 * abs(a) for a, b in zip(Es, Es[1:])), Es
    assert Es[-1] < Es[0]
    Mf, avg_full, nc_full = oracle.llg_rk4_run(Tn, M0, Ms, Hz, alpha, dt, steps)
    Mx, avg_ext, nc_ext = oracle.llg_rk4_run(Tn, M0, Ms, Hz, alpha, dt, steps, extrapolate=True)
    assert nc_full == 4 * steps and nc_ext == 16 + (steps - 4)
    assert np.allclose(M, Mf, rtol=0, atol=1e-9 * Ms)       # 6 x 10 steps == 60 steps (no hidden state)
    assert oracle.fig2_error(avg_ext, avg_full, Ms) < 1e-6
    assert np.abs(Mx - Mf).max() / Ms < 1e-5


def test_fig2_error_metric_by_hand(oracle):
    """eps = sum_i ||M(t_i) - M~(t_i)|| / (n Ms)."""
    ref = np.array([[1.0, 0.0, 0.0], [0.0, 2.0, 0.0], [0.0, 0.0, 3.0]])
    got = ref + np.array([[3.0, 4.0, 0.0], [0.0, 0.0, 0.0], [0.0, 0.0, -2.0]])
    assert abs(oracle.fig2_error(got, ref, 10.0) - (5.0 + 0.0 + 2.0) / (3 * 10.0)) < 1e-15
