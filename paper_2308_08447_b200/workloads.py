"""Seeded synthetic inputs for the five BASELINE.json configs.

This module holds NO arithmetic of the method (no tensor, no FFT, no convolution): it only makes
magnetisation / spin arrays and picks sample cells.  It is the one module that both the tests of the
CUDA path and the tests of the oracle use.  It imports neither
``oracle`` nor the CUDA binding.

The paper's own workloads are simulator states that cannot be regenerated here (thin-film S-state,
PAPER.md:47; FePt film); the shapes below stand in for them: a 1-cell-thick film
(Fig. 2/5 meshes), a 3D block, a macrocell mesh with N_S = 64 spins per cell (Fig. 6).

Arrays are planar ``[3][nz][ny][nx]`` (x fastest), float32 unless stated.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass(frozen=True)
class Config:
    name: str
    n: tuple          # (nx, ny, nz) demag mesh
    h: tuple          # cell size in metres
    Ms: float         # A/m (scale of the parity tolerance)
    seed: int
    kind: str         # "random" | "voronoi" | "vortex" | "atomistic"
    macro: tuple = (1, 1, 1)   # spins per macrocell edge (atomistic only)
    a: float = 0.0             # lattice constant (atomistic only)
    mu_s: float = 0.0          # moment in Bohr magnetons (atomistic only)


MU_B = 9.2740100783e-24

CONFIGS = {
    "C1": Config("C1 tiny 32x32x2", (32, 32, 2), (4e-9, 4e-9, 4e-9), 8e5, 1001, "random"),
    "C2": Config("C2 film 1024x1024x1", (1024, 1024, 1), (2e-9, 2e-9, 1e-9), 8e5, 1002, "voronoi"),
    "C3": Config("C3 3D 256x256x64", (256, 256, 64), (3e-9, 3e-9, 3e-9), 8.6e5, 1003, "vortex"),
    "C4": Config("C4 large film 4096x4096x8", (4096, 4096, 8), (2e-9, 2e-9, 2e-9), 1e6, 1004, "random"),
    "C5": Config("C5 atomistic 1024^3 spins -> 256^3 cells", (256, 256, 256),
                 (1.2e-9, 1.2e-9, 1.2e-9), MU_B * 2.0 / (0.3e-9) ** 3, 1005, "atomistic",
                 macro=(4, 4, 4), a=0.3e-9, mu_s=2.0),
}


def _rng(seed):
    return np.random.Generator(np.random.PCG64(seed))


def random_unit_vectors(n, Ms, seed) -> np.ndarray:
    """M = Ms * g/|g|, g ~ N(0, I3) per cell (configs 1 and 4); generated in z-slabs."""
    nx, ny, nz = n
    rng = _rng(seed)
    M = np.empty((3, nz, ny, nx), dtype=np.float32)
    for z in range(nz):
        g = rng.standard_normal((3, ny, nx))
        g /= np.sqrt((g * g).sum(axis=0, keepdims=True))
        M[:, z] = (Ms * g).astype(np.float32)
    return M


def voronoi_domains(n, Ms, seed, cells_per_grain=50) -> np.ndarray:
    """Random domains (config 2): Voronoi grains of ~cells_per_grain cells in the xy plane, each with a
    random unit direction; cell -> nearest seed (Euclidean, non-periodic), uniform along z."""
    from scipy.spatial import cKDTree
    nx, ny, nz = n
    rng = _rng(seed)
    ngr = max(1, int(round(nx * ny / cells_per_grain)))
    pts = rng.uniform(0.0, 1.0, size=(ngr, 2)) * np.array([nx, ny])
    d = rng.standard_normal((ngr, 3))
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    yy, xx = np.meshgrid(np.arange(ny) + 0.5, np.arange(nx) + 0.5, indexing="ij")
    _, idx = cKDTree(pts).query(np.stack([xx.ravel(), yy.ravel()], axis=1), workers=-1)
    m = d[idx].T.reshape(3, 1, ny, nx)
    return np.ascontiguousarray(np.broadcast_to(Ms * m, (3, nz, ny, nx))).astype(np.float32)


def vortex(n, Ms, seed, core_cells=10.0, tilt=0.05) -> np.ndarray:
    """Vortex (config 3): in-plane curl about the mesh centre, m_z = exp(-rho^2/r_c^2) core of radius
    ``core_cells``, uniform along z, then m <- normalise(m + tilt * xi), xi ~ N(0, I3)."""
    nx, ny, nz = n
    rng = _rng(seed)
    y, x = np.meshgrid(np.arange(ny) - (ny - 1) / 2.0, np.arange(nx) - (nx - 1) / 2.0, indexing="ij")
    rho = np.sqrt(x * x + y * y)
    mz = np.exp(-(rho / core_cells) ** 2)
    inp = np.sqrt(np.maximum(0.0, 1.0 - mz * mz)) / np.maximum(rho, 1e-30)
    m2d = np.stack([-y * inp, x * inp, mz])
    M = np.empty((3, nz, ny, nx), dtype=np.float32)
    for z in range(nz):
        m = m2d + tilt * rng.standard_normal((3, ny, nx))
        m /= np.sqrt((m * m).sum(axis=0, keepdims=True))
        M[:, z] = (Ms * m).astype(np.float32)
    return M


def random_spins_numpy(L, seed) -> np.ndarray:
    """Unit spins uniformly random on the sphere, float32 [3][Lz][Ly][Lx] (host; small lattices)."""
    return random_unit_vectors(L, 1.0, seed)


def random_spins_torch(L, seed, device="cuda", chunk_z=16):
    """Config 5 at full size: 1024^3 unit spins (12.9 GB) are made on the device with torch's seeded
    generator, z-slab by z-slab; nothing of the method is involved."""
    import torch
    Lx, Ly, Lz = L
    gen = torch.Generator(device=device)
    gen.manual_seed(int(seed))
    S = torch.empty((3, Lz, Ly, Lx), dtype=torch.float32, device=device)
    for z0 in range(0, Lz, chunk_z):
        z1 = min(Lz, z0 + chunk_z)
        g = torch.randn((3, z1 - z0, Ly, Lx), dtype=torch.float32, device=device, generator=gen)
        g /= torch.sqrt((g * g).sum(dim=0, keepdim=True))
        S[:, z0:z1] = g
        del g
    return S


def make_magnetisation(cfg: Config) -> np.ndarray:
    """Host magnetisation for the micromagnetic configs (C1..C4)."""
    if cfg.kind == "random":
        return random_unit_vectors(cfg.n, cfg.Ms, cfg.seed)
    if cfg.kind == "voronoi":
        return voronoi_domains(cfg.n, cfg.Ms, cfg.seed)
    if cfg.kind == "vortex":
        return vortex(cfg.n, cfg.Ms, cfg.seed)
    raise ValueError(f"{cfg.kind}: use random_spins_* for the atomistic config")


def sample_cells(n, K, seed) -> np.ndarray:
    """K flat cell indices ((iz*ny+iy)*nx+ix): the 8 corners, the 6 face centres, the 12 edge centres,
    the body centre, the rest uniform random without repetition (as far as K allows)."""
    nx, ny, nz = n
    lo_hi_mid = lambda m: sorted({0, m - 1, (m - 1) // 2})
    fixed = []
    for iz in lo_hi_mid(nz):
        for iy in lo_hi_mid(ny):
            for ix in lo_hi_mid(nx):
                fixed.append((iz * ny + iy) * nx + ix)
    fixed = list(dict.fromkeys(fixed))[:K]
    rng = _rng(seed + 7919)
    out = list(fixed)
    seen = set(out)
    nc = nx * ny * nz
    while len(out) < min(K, nc):
        i = int(rng.integers(0, nc))
        if i not in seen:
            seen.add(i)
            out.append(i)
    return np.array(out, dtype=np.int64)
