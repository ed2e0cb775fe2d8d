"""fp64 CPU oracle for the demagnetizing-field convolution -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Python face of ``oracle/demag_oracle.c`` (ctypes) plus the few oracle pieces that are one-liners in
NumPy.  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this module; the CUDA path never does, and this module never
imports ``paper_2308_08447_b200``.

Citations are ``PAPER.md:<line>`` (arXiv 2308.08447) or a DESIGN.md reading (R<n>).

    tensor_table        N over non-negative offsets (R1, R4)          [C]
    direct_sum          O-A, Eq. (1) written out                   [C]
    direct_sum_sampled  O-S, Eq. (1) at chosen cells                                [C]
    naive_dft_conv      O-B, padded convolution via O(N^2) DFTs    [C]
    fft_conv            O-C, the same through numpy.fft (library cross-check)       [NumPy]
    energy              E = -(mu0/2) V_cell sum M.H (R12)                            [NumPy]
    macrocell_average   Eq. (9) (R13)                              [NumPy]
    macrocell_scatter   "applied equally to all spins" (R14)           [NumPy]
    dipole_table        point-dipole tensor that turns Eq. (8) into Eq. (1)   [NumPy]
    dipole_field_eq8    Eq. (8) written out, O(n^2)                [NumPy]
    poly_extrapolate    polynomial through previously computed fields, evaluated at a sub-step time (R19)  [NumPy]
    periodic_tensor_table  image-summed, symmetrised tensor on periodic axes (R11)   [NumPy loops over N_at]
    llg_rhs             Eq. (5) solved for dM/dt (R20)                          [NumPy]
    llg_rk4_run         classical RK4 on Eq. (5) with H_eff = H_d + H_Zee, H_d by fft_conv at every stage, or by the
                        quartic extrapolation of PAPER.md:96 at the sub-steps (R21, R22)       [NumPy]
    fig2_error          mean relative error of the average magnetisation        [NumPy]

All of them are pinned in tests/test_oracle_pins.py; none is "parity unpinned".
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "demag_oracle.c")
_LIB = os.path.join(_HERE, "libdemag_oracle.so")

MU0 = 4.0e-7 * np.pi           # vacuum permeability, T m / A
MU_B = 9.2740100783e-24        # Bohr magneton, J / T  (= A m^2)

_dp = ctypes.POINTER(ctypes.c_double)
_lib = None


def build(force: bool = False) -> str:
    """Compile the C oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        d, i = ctypes.c_double, ctypes.c_int
        lib.oracle_newell_N.argtypes = [d, d, d, d, d, d, _dp]
        lib.oracle_quad_N.argtypes = [d, d, d, d, d, d, i, _dp]
        lib.oracle_N_at.argtypes = [d, d, d, d, d, d, _dp]
        lib.oracle_tensor_table.argtypes = [i, i, i, d, d, d, _dp]
        lib.oracle_direct_sum.argtypes = [i, i, i, _dp, _dp, _dp]
        lib.oracle_direct_sum_sampled.argtypes = [i, i, i, _dp, _dp, i,
                                                  ctypes.POINTER(ctypes.c_longlong), _dp]
        lib.oracle_naive_dft_conv.argtypes = [i, i, i, i, i, i, _dp, _dp, _dp]
        lib.oracle_naive_dft_conv.restype = i
        lib.oracle_kernel_spectrum_imag_ratio.argtypes = [i, i, i, i, i, i, _dp]
        lib.oracle_kernel_spectrum_imag_ratio.restype = d
        lib.oracle_num_threads.restype = i
        _lib = lib
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(_dp)


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def _n6(fn, *args) -> np.ndarray:
    out = np.empty(6, dtype=np.float64)
    fn(*args, _p(out))
    return out


def newell_N(r, h) -> np.ndarray:
    """Closed-form N (xx,yy,zz,xy,xz,yz) at offset r [m] for cell h [m] (R1)."""
    return _n6(_load().oracle_newell_N, *map(float, r), *map(float, h))


def quad_N(r, h, m: int = 3) -> np.ndarray:
    """Integral definition of N by m-point Gauss-Legendre per half axis (R4)."""
    lib = _load()
    out = np.empty(6, dtype=np.float64)
    lib.oracle_quad_N(*map(float, r), *map(float, h), int(m), _p(out))
    return out


def N_at(r, h) -> np.ndarray:
    """N as the oracle uses it: Newell near, quadrature far (R4)."""
    return _n6(_load().oracle_N_at, *map(float, r), *map(float, h))


def tensor_table(n, h) -> np.ndarray:
    """T[6][nz][ny][nx] = N_c(d*h) over non-negative cell offsets d (scope row a0)."""
    nx, ny, nz = map(int, n)
    T = np.empty((6, nz, ny, nx), dtype=np.float64)
    _load().oracle_tensor_table(nx, ny, nz, *map(float, h), _p(T))
    return T


def _check(T, M):
    T = np.ascontiguousarray(T, dtype=np.float64)
    M = np.ascontiguousarray(M, dtype=np.float64)
    assert T.ndim == 4 and T.shape[0] == 6 and M.ndim == 4 and M.shape[0] == 3
    assert T.shape[1:] == M.shape[1:], (T.shape, M.shape)
    nz, ny, nx = M.shape[1:]
    return T, M, nx, ny, nz


def direct_sum(T, M) -> np.ndarray:
    """O-A: H_i = -sum_j N(i-j) M_j for every cell (Eq. (1))."""
    T, M, nx, ny, nz = _check(T, M)
    H = np.empty_like(M)
    _load().oracle_direct_sum(nx, ny, nz, _p(T), _p(M), _p(H))
    return H


def direct_sum_sampled(T, M, cells) -> np.ndarray:
    """O-S: Eq. (1) at flat cell indices ``cells`` ((iz*ny+iy)*nx+ix); returns [len(cells)][3]."""
    T, M, nx, ny, nz = _check(T, M)
    cells = np.ascontiguousarray(cells, dtype=np.int64)
    Hs = np.empty((len(cells), 3), dtype=np.float64)
    _load().oracle_direct_sum_sampled(nx, ny, nz, _p(T), _p(M), len(cells),
                                      cells.ctypes.data_as(ctypes.POINTER(ctypes.c_longlong)), _p(Hs))
    return Hs


def padded_shape(n, pbc=(False, False, False)):
    """P_a = 2 n_a for an open axis with n_a > 1, else n_a (R6)."""
    return tuple(int(na) if (na == 1 or p) else 2 * int(na) for na, p in zip(n, pbc))


def naive_dft_conv(T, M, P=None) -> np.ndarray:
    """O-B: zero-padded convolution through O(N^2) DFTs."""
    T, M, nx, ny, nz = _check(T, M)
    Px, Py, Pz = P if P is not None else padded_shape((nx, ny, nz))
    H = np.empty_like(M)
    rc = _load().oracle_naive_dft_conv(nx, ny, nz, Px, Py, Pz, _p(T), _p(M), _p(H))
    if rc != 0:
        raise ValueError(f"oracle_naive_dft_conv failed: {rc}")
    return H


def kernel_spectrum_imag_ratio(T, P=None) -> float:
    T = np.ascontiguousarray(T, dtype=np.float64)
    nz, ny, nx = T.shape[1:]
    Px, Py, Pz = P if P is not None else padded_shape((nx, ny, nz))
    return float(_load().oracle_kernel_spectrum_imag_ratio(nx, ny, nz, Px, Py, Pz, _p(T)))


# parity of component c along (x, y, z): diagonal even; xy odd in x,y; xz odd in x,z; yz odd in y,z
PARITY = np.array([[1, 1, 1], [1, 1, 1], [1, 1, 1], [-1, -1, 1], [-1, 1, -1], [1, -1, -1]])
# (row, col) -> component index of the symmetric 3x3 tensor
COMP = np.array([[0, 3, 4], [3, 1, 5], [4, 5, 2]])


def padded_kernel(T, P=None) -> np.ndarray:
    """K[6][Pz][Py][Px]: N(s(d)) with s_a = d_a (d_a<n_a), d_a-P_a (d_a>n_a), 0 at d_a=n_a (R6)."""
    T = np.asarray(T, dtype=np.float64)
    nz, ny, nx = T.shape[1:]
    Px, Py, Pz = P if P is not None else padded_shape((nx, ny, nz))
    K = np.zeros((6, Pz, Py, Px))
    for c in range(6):
        A = T[c]
        for axis, (na, Pa, par) in enumerate(zip((nz, ny, nx), (Pz, Py, Px), PARITY[c][::-1])):
            if Pa == na:
                continue
            shp = list(A.shape)
            shp[axis] = Pa
            B = np.zeros(shp)
            sl = [slice(None)] * 3
            sl[axis] = slice(0, na)
            B[tuple(sl)] = A
            src = [slice(None)] * 3
            src[axis] = slice(na - 1, 0, -1)         # offsets -(na-1) .. -1 -> slots Pa-na+1 .. Pa-1
            dst = [slice(None)] * 3
            dst[axis] = slice(Pa - na + 1, Pa)
            B[tuple(dst)] = par * A[tuple(src)]
            A = B
        K[c] = A
    return K


def fft_conv(T, M, P=None) -> np.ndarray:
    """O-C: the same padded convolution through numpy.fft (a library routine the path reduces to);
    a cross-check validated against O-A/O-B on small grids, not the authority."""
    T = np.asarray(T, dtype=np.float64)
    M = np.asarray(M, dtype=np.float64)
    nz, ny, nx = M.shape[1:]
    Px, Py, Pz = P if P is not None else padded_shape((nx, ny, nz))
    s = (Pz, Py, Px)
    try:                                   # same routine family (pocketfft), threaded
        import scipy.fft as _fft
        rfftn = lambda x: _fft.rfftn(x, s=s, axes=(0, 1, 2), workers=-1)
        irfftn = lambda x: _fft.irfftn(x, s=s, axes=(0, 1, 2), workers=-1)
    except ImportError:
        rfftn = lambda x: np.fft.rfftn(x, s=s, axes=(0, 1, 2))
        irfftn = lambda x: np.fft.irfftn(x, s=s, axes=(0, 1, 2))
    Mh = [rfftn(M[b]) for b in range(3)]
    H = np.empty_like(M)
    Kh = {}
    for a in range(3):
        acc = 0
        for b in range(3):
            c = int(COMP[a, b])
            if c not in Kh:
                Kh[c] = rfftn(_padded_one(T[c], c, (Px, Py, Pz)))
            acc = acc + Kh[c] * Mh[b]
        H[a] = -irfftn(acc)[:nz, :ny, :nx]
    return H


def _padded_one(Tc, c, P):
    """padded_kernel for a single component (avoids building all six at once)."""
    T6 = np.zeros((6,) + Tc.shape)
    T6[c] = Tc
    return padded_kernel(T6, P)[c]


def energy(M, H, h) -> float:
    """E = -(mu0/2) V_cell sum_i M_i . H_i  (R12; formula not printed in the paper)."""
    M = np.asarray(M, dtype=np.float64)
    H = np.asarray(H, dtype=np.float64)
    return float(-0.5 * MU0 * float(np.prod(h)) * np.sum(M * H))


def macrocell_average(S, c, mu_s, a) -> np.ndarray:
    """Eq. (9): M_cell = mu_B mu_s sum(S_hat) / (cx cy cz a^3)  [A/m]  (R13).
    S: unit spins [3][Lz][Ly][Lx]; c = (cx, cy, cz) spins per macrocell edge."""
    S = np.asarray(S, dtype=np.float64)
    cx, cy, cz = map(int, c)
    _, Lz, Ly, Lx = S.shape
    assert Lx % cx == 0 and Ly % cy == 0 and Lz % cz == 0
    R = S.reshape(3, Lz // cz, cz, Ly // cy, cy, Lx // cx, cx).sum(axis=(2, 4, 6))
    return R * (MU_B * mu_s / (cx * cy * cz * a ** 3))


def macrocell_scatter(H, c) -> np.ndarray:
    """the cell field is applied equally to all spins of the cell (R14)."""
    cx, cy, cz = map(int, c)
    return np.repeat(np.repeat(np.repeat(np.asarray(H), cz, axis=1), cy, axis=2), cx, axis=3)


def dipole_table(L, a) -> np.ndarray:
    """Point-dipole tensor on a simple cubic lattice of constant a over the non-negative offsets, [6][Lz][Ly][Lx]:
    the kernel that puts the dipole-dipole field of Eq. (8) ("can be re-arranged into the form of
    Equation (1)") into the form H = -sum_j N(i-j) M_j with M_j = mu_B mu_S S^_j / a^3:
        N_ab(r) = (a^3 / 4 pi) (delta_ab / r^3 - 3 r_a r_b / r^5),   N(0) = 0 (the sum of Eq. (8) runs over j != i)."""
    Lx, Ly, Lz = map(int, L)
    z, y, x = np.meshgrid(np.arange(Lz) * a, np.arange(Ly) * a, np.arange(Lx) * a, indexing="ij")
    r2 = x * x + y * y + z * z
    r2[0, 0, 0] = 1.0
    ir3 = r2 ** -1.5
    ir5 = r2 ** -2.5
    f = a ** 3 / (4.0 * np.pi)
    T = np.stack([f * (ir3 - 3 * x * x * ir5), f * (ir3 - 3 * y * y * ir5), f * (ir3 - 3 * z * z * ir5),
                  f * (-3 * x * y * ir5), f * (-3 * x * z * ir5), f * (-3 * y * z * ir5)])
    T[:, 0, 0, 0] = 0.0
    return T


def dipole_field_eq8(S, mu_s, a) -> np.ndarray:
    """Eq. (8) written out, O(n^2), small lattices only:
        H_i = (mu_B / 4 pi) sum_{j != i} [3 (S_j . r^_ij) r^_ij - S_j] / r_ij^3,   S_j = mu_S S^_j,
    r_ij the vector from spin i to spin j.  S: unit spins [3][Lz][Ly][Lx]; result in A/m, same layout."""
    S = np.asarray(S, dtype=np.float64)
    _, Lz, Ly, Lx = S.shape
    z, y, x = np.meshgrid(np.arange(Lz) * a, np.arange(Ly) * a, np.arange(Lx) * a, indexing="ij")
    pos = np.stack([x.ravel(), y.ravel(), z.ravel()], axis=1)
    Sv = S.reshape(3, -1).T * mu_s
    H = np.zeros_like(Sv)
    for i in range(pos.shape[0]):
        d = pos - pos[i]
        r = np.sqrt((d * d).sum(axis=1))
        r[i] = 1.0
        rh = d / r[:, None]
        t = (3.0 * (Sv * rh).sum(axis=1)[:, None] * rh - Sv) / (r ** 3)[:, None]
        t[i] = 0.0
        H[i] = MU_B / (4.0 * np.pi) * t.sum(axis=0)
    return H.T.reshape(3, Lz, Ly, Lx)


def periodic_tensor_table(n, h, pbc, images) -> np.ndarray:
    """Periodic tensor of reading R11 ("modified convolution kernel"; its reference [25] is absent), written as
    the definition: on every periodic axis a the open-boundary tensor is summed over `images` images on each side,

        S[d] = sum_{|m_a| <= images, a periodic} N((d + m o n) o h),        0 <= d_a < n_a,

    then made symmetric under d_a -> n_a - d_a with the component's parity on that axis (a periodic kernel is; the
    truncated sum only up to its last images):  T = sym_x sym_y sym_z S,  sym_a f(d_a) = (f(d_a) + parity_a f((n_a - d_a) mod n_a)) / 2.
    Small meshes only (one N_at call per offset and image)."""
    nx, ny, nz = map(int, n)
    rng = [range(-images, images + 1) if p else range(1) for p in pbc]
    T = np.zeros((6, nz, ny, nx))
    for dz in range(nz):
        for dy in range(ny):
            for dx in range(nx):
                acc = np.zeros(6)
                for mx in rng[0]:
                    for my in rng[1]:
                        for mz in rng[2]:
                            acc += N_at(((dx + mx * nx) * h[0], (dy + my * ny) * h[1], (dz + mz * nz) * h[2]), h)
                T[:, dz, dy, dx] = acc
    for a, ax in ((0, 3), (1, 2), (2, 1)):
        if pbc[a]:
            idx = (-np.arange((nx, ny, nz)[a])) % (nx, ny, nz)[a]
            T = 0.5 * (T + PARITY[:, a].reshape(6, 1, 1, 1) * np.take(T, idx, axis=ax))
    return T


def poly_extrapolate(H_hist, t_hist, t) -> np.ndarray:
    """Demagnetizing field at a sub-step time t from previously computed fields ("polynomial extrapolation
    of the demagnetizing field at sub-steps of the higher order evaluation method, using previously computed values ...
    the RK4 method requires a quartic polynomial, whilst the RKF56 method requires a quintic polynomial"; reading R19):
    the unique polynomial of degree p through the p+1 samples (t_k, H_k), every field entry on its own, in Lagrange form

        H(t) = sum_k L_k(t) H_k,      L_k(t) = prod_{j != k} (t - t_j) / (t_k - t_j).

    H_hist: sequence of p+1 equally shaped arrays; t_hist: p+1 distinct times."""
    ts = [float(v) for v in t_hist]
    out = np.zeros_like(np.asarray(H_hist[0], dtype=np.float64))
    for k, Hk in enumerate(H_hist):
        Lk = 1.0
        for j, tj in enumerate(ts):
            if j != k:
                Lk *= (float(t) - tj) / (ts[k] - tj)
        out += Lk * np.asarray(Hk, dtype=np.float64)
    return out


# ------------------------------------------------------------------------------------------------ LLG (NEXT row 4)
GAMMA_LLG = 2.212761569e5      # mu0 |gamma_e| in m / (A s): the gyromagnetic ratio of Eq. (5) when H is in A/m (R20)


def llg_rhs(M, H, Ms, alpha, gamma=GAMMA_LLG) -> np.ndarray:
    """Eq. (5):  dm/dt = -gamma m x H_eff + alpha m x dm/dt,  m = M / Ms, solved for the derivative
    (cross the equation with m, use |m| = 1):

        dM/dt = -gamma / (1 + alpha^2) * [ M x H + (alpha / Ms) M x (M x H) ].

    M, H: [3][...] in A/m; returns dM/dt in A/(m s).  (R20: the paper prints only the implicit form.)"""
    M = np.asarray(M, dtype=np.float64)
    H = np.asarray(H, dtype=np.float64)
    MxH = np.cross(M, H, axis=0)
    MxMxH = np.cross(M, MxH, axis=0)
    return (-gamma / (1.0 + alpha * alpha)) * (MxH + (alpha / Ms) * MxMxH)


def llg_rk4_run(T, M0, Ms, Hzee, alpha, dt, nsteps, gamma=GAMMA_LLG, extrapolate=False, demag=None):
    """Classical 4th-order Runge-Kutta on Eq. (5) ("typically evaluated using a higher order explicit
    evaluation method, e.g. RK4") with H_eff = H_d + H_Zee (the other interactions are out of scope),
    H_d = -N * M (Eq. (1)) through `demag` (default: fft_conv with the table T), H_Zee a uniform field (3-vector, A/m).

    Stages of one step from (t, M):  K1 = f(M),  K2 = f(M + dt/2 K1),  K3 = f(M + dt/2 K2),  K4 = f(M + dt K3),
    M(t + dt) = M + dt/6 (K1 + 2 K2 + 2 K3 + K4); no renormalisation of |M| (R21: none is stated).

    extrapolate = False: H_d is convolved at every stage (4 per step).
    extrapolate = True (R22): H_d is convolved only at the START of a step (stage 1, time t_n); the five
    most recent such fields are kept, and once five exist the fields of stages 2-4 (times t_n + dt/2, t_n + dt/2,
    t_n + dt) are the quartic polynomial through them (poly_extrapolate) evaluated at the stage time.

    Returns (M_final, Mavg [nsteps+1][3] mesh-averaged magnetisation at t_0..t_nsteps, n_convolutions)."""
    M = np.array(M0, dtype=np.float64)
    Hz = np.asarray(Hzee, dtype=np.float64).reshape(3, 1, 1, 1)
    conv = demag if demag is not None else (lambda X: fft_conv(T, X))
    nconv = 0
    hist, thist = [], []
    avg = [M.reshape(3, -1).mean(axis=1)]
    t = 0.0
    for _ in range(int(nsteps)):
        Hd1 = conv(M); nconv += 1
        hist.append(Hd1); thist.append(t)
        if len(hist) > 5:
            hist.pop(0); thist.pop(0)
        use = extrapolate and len(hist) == 5

        def field(X, ts):
            nonlocal nconv
            if use:
                return poly_extrapolate(hist, thist, ts)
            nconv += 1
            return conv(X)
        K1 = llg_rhs(M, Hd1 + Hz, Ms, alpha, gamma)
        X = M + 0.5 * dt * K1
        K2 = llg_rhs(X, field(X, t + 0.5 * dt) + Hz, Ms, alpha, gamma)
        X = M + 0.5 * dt * K2
        K3 = llg_rhs(X, field(X, t + 0.5 * dt) + Hz, Ms, alpha, gamma)
        X = M + dt * K3
        K4 = llg_rhs(X, field(X, t + dt) + Hz, Ms, alpha, gamma)
        M = M + (dt / 6.0) * (K1 + 2.0 * K2 + 2.0 * K3 + K4)
        t += dt
        avg.append(M.reshape(3, -1).mean(axis=1))
    return M, np.array(avg), nconv


def fig2_error(Mavg, Mavg_ref, Ms) -> float:
    """PAPER.md:47:  eps = sum_i || M(t_i) - M~(t_i) || / (n Ms)  over the n recorded points of the average
    magnetisation, M~ the reference dataset."""
    A = np.asarray(Mavg, dtype=np.float64); R = np.asarray(Mavg_ref, dtype=np.float64)
    assert A.shape == R.shape and A.shape[1] == 3
    return float(np.sqrt(((A - R) ** 2).sum(axis=1)).sum() / (A.shape[0] * Ms))
