"""Seeded synthetic particle sets shaped like the paper's per-node workloads.

This module is the ONE piece shared by the CUDA path, the CPU oracle and the
tests: it only draws positions. It contains none of the method's arithmetic
(no cell index, no force law, no polynomial) and imports neither `oracle/`
nor the CUDA binding.

The five configurations are BASELINE.json `configs[0..4]`; how each clause
of those one-line descriptions is realised follows SURVEY.md Appendix C
(seeds, halo-count law, Plummer truncation, draw order).  The paper itself
fixes only the shape: 8192^3 particles on 16,384 nodes = 2^25 per node
(PAPER.md:113, 141), mean density one particle per PM cell (PAPER.md:141,
185), 20-46 % of particles in halos, smallest stored halo 40
particles, clusters of "more than 4 million particles"
(PAPER.md:81).  These inputs STAND IN for the paper's particle data, which
is not available.

All positions are float32, in PM grid units, inside [0, box) per axis, in
random memory order (worst case for the binning scatter); masses are 1.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

SEED_BASE = 141133960  # seed = 141133960 + config number (1-based)

N_MIN_HALO = 40          # PAPER.md:171 smallest stored halo
N_MAX_HALO = 4.0e6       # PAPER.md:81 "more than 4 million particles"
HALO_SLOPE = 0.9         # dN/dn ~ n^-1.9  (BASELINE.json configs[2..4])
PLUMMER_UMAX = (100.0 / 101.0) ** 1.5  # truncate the Plummer profile at 10 scale radii


@dataclass(frozen=True)
class Workload:
    """Geometry + solver parameters + generator recipe of one configuration."""
    name: str
    n: int
    box: tuple            # (Lx, Ly, Lz) in grid units
    ncell: tuple          # chaining-mesh cells per axis (cell edge 3.2)
    rcut: float
    eps: float
    seed: int
    background: str       # "uniform" | "lattice"
    frac_halo: float      # fraction of particles placed in Plummer spheres
    n_halo: int
    a_range: tuple        # Plummer scale radius range
    sigma: float = 0.0    # Gaussian displacement of the lattice background
    lattice: tuple = ()   # lattice sites per axis (background == "lattice")
    permute: bool = True
    steps: int = 1        # sub-cycle steps (config 4: 5 x (bin, force, kick))
    dt: float = 0.0
    note: str = ""
    extra: dict = field(default_factory=dict)


CONFIGS = {
    1: Workload("config1_uniform_32k", 32 ** 3, (32.0, 32.0, 32.0), (10, 10, 10), 3.0, 0.1,
                SEED_BASE + 1, "uniform32", 0.0, 0, (0.0, 0.0), permute=False,
                note="BASELINE.json configs[0]: 32^3 uniform fp32 in box 32"),
    2: Workload("config2_lattice_2m", 128 ** 3, (128.0, 128.0, 128.0), (40, 40, 40), 3.0, 0.1,
                SEED_BASE + 2, "lattice", 0.0, 0, (0.0, 0.0), sigma=0.5, lattice=(128, 128, 128),
                note="BASELINE.json configs[1]: 128^3 lattice + N(0,0.5^2)"),
    3: Workload("config3_clustered_16m", 256 ** 3, (256.0, 256.0, 256.0), (80, 80, 80), 3.0, 0.05,
                SEED_BASE + 3, "uniform", 0.5, 4000, (0.5, 4.0),
                note="BASELINE.json configs[2]: 50% uniform + 50% in 4000 Plummer halos"),
    4: Workload("config4_clustered_2p25", 2 ** 25, (256.0, 256.0, 512.0), (80, 80, 160), 3.0, 0.05,
                SEED_BASE + 4, "lattice", 0.6, 20000, (0.3, 3.0), sigma=0.7, lattice=(256, 256, 512),
                steps=5, dt=0.01,
                note="BASELINE.json configs[3]: the paper's per-node load, 40% lattice + 60% halos"),
    5: Workload("config5_clustered_512", 512 ** 3, (512.0, 512.0, 512.0), (160, 160, 160), 3.0, 0.02,
                SEED_BASE + 5, "uniform", 0.8, 100000, (0.2, 2.5),
                note="BASELINE.json configs[4]: 20% uniform + 80% in 100000 halos"),
}


def halo_counts(rng: np.random.Generator, n_halo: int, total: int) -> np.ndarray:
    """Per-halo particle counts from dN/dn ~ n^-1.9 on [40, 4e6], scaled to `total`.

    Inverse-CDF draw, scale to the halo-particle total, floor, and give the
    remainder to the largest fractional parts.
    """
    u = rng.random(n_halo)
    lo, hi = N_MIN_HALO ** (-HALO_SLOPE), N_MAX_HALO ** (-HALO_SLOPE)
    raw = (lo + u * (hi - lo)) ** (-1.0 / HALO_SLOPE)
    scaled = raw * (total / raw.sum())
    cnt = np.floor(scaled).astype(np.int64)
    rem = int(total - cnt.sum())
    if rem > 0:
        frac = scaled - cnt
        cnt[np.argsort(-frac, kind="stable")[:rem]] += 1
    assert cnt.sum() == total
    return cnt


def plummer_offsets(rng: np.random.Generator, a_per_particle: np.ndarray) -> np.ndarray:
    """Isotropic offsets with Plummer radial law r = a / sqrt(u^(-2/3) - 1), u in (0, u_max]."""
    m = a_per_particle.shape[0]
    u = (1.0 - rng.random(m)) * PLUMMER_UMAX          # (0, u_max]
    r = a_per_particle / np.sqrt(u ** (-2.0 / 3.0) - 1.0)
    del u
    cost = rng.uniform(-1.0, 1.0, m)
    phi = rng.uniform(0.0, 2.0 * np.pi, m)
    sint = np.sqrt(np.maximum(0.0, 1.0 - cost * cost))
    out = np.empty((m, 3), dtype=np.float64)
    out[:, 0] = r * sint * np.cos(phi)
    out[:, 1] = r * sint * np.sin(phi)
    out[:, 2] = r * cost
    return out


def _finish(rng, xyz64: np.ndarray, box, permute: bool) -> np.ndarray:
    """Permute memory order, wrap into the box in fp64, cast to fp32, map values that round to L to 0."""
    n = xyz64.shape[0]
    if permute:
        xyz64 = xyz64[rng.permutation(n)]
    out = np.empty((n, 4), dtype=np.float32)
    for ax in range(3):
        L = float(box[ax])
        w = np.mod(xyz64[:, ax], L)
        w32 = w.astype(np.float32)
        w32[w32 >= np.float32(L)] = np.float32(0.0)
        out[:, ax] = w32
    out[:, 3] = np.float32(1.0)
    return out


def make_clustered(n: int, box, seed: int, background: str, frac_halo: float, n_halo: int,
                   a_range, sigma: float = 0.0, lattice=(), permute: bool = True) -> np.ndarray:
    """General recipe: background (uniform or displaced lattice) + Plummer halos -> float32 [n,4]."""
    rng = np.random.Generator(np.random.PCG64(seed))
    box = tuple(float(b) for b in box)
    n_h = int(round(frac_halo * n)) if n_halo > 0 else 0
    n_bg = n - n_h
    parts = []
    if background == "uniform":
        if n_bg:
            parts.append(rng.random((n_bg, 3)) * np.asarray(box))
    elif background == "lattice":
        nx, ny, nz = lattice
        n_sites = nx * ny * nz
        if n_bg == n_sites:
            site = np.arange(n_sites, dtype=np.int64)
        else:
            site = rng.permutation(n_sites)[:n_bg]
        bg = np.empty((n_bg, 3), dtype=np.float64)
        bg[:, 0] = (site % nx) + 0.5
        bg[:, 1] = ((site // nx) % ny) + 0.5
        bg[:, 2] = (site // (nx * ny)) + 0.5
        del site
        sp = np.asarray(box) / np.asarray([nx, ny, nz], dtype=np.float64)
        bg *= sp
        bg += rng.normal(0.0, sigma, (n_bg, 3))
        parts.append(bg)
    else:
        raise ValueError(background)
    if n_h:
        cnt = halo_counts(rng, n_halo, n_h)
        centre = rng.random((n_halo, 3)) * np.asarray(box)
        a = rng.uniform(a_range[0], a_range[1], n_halo)
        off = plummer_offsets(rng, np.repeat(a, cnt))
        off += np.repeat(centre, cnt, axis=0)
        parts.append(off)
    xyz = parts[0] if len(parts) == 1 else np.concatenate(parts, axis=0)
    del parts
    return _finish(rng, xyz, box, permute)


def generate(cfg: int | Workload) -> np.ndarray:
    """float32 [N,4] (x, y, z, m=1) for BASELINE.json configs[cfg-1]."""
    w = CONFIGS[cfg] if isinstance(cfg, int) else cfg
    if w.background == "uniform32":
        # config 1 exactly as SURVEY.md Appendix C: fp32 draws scaled by 32 (exact, < 32), no permutation
        rng = np.random.Generator(np.random.PCG64(w.seed))
        out = np.empty((w.n, 4), dtype=np.float32)
        out[:, :3] = rng.random((w.n, 3), dtype=np.float32) * np.float32(w.box[0])
        out[:, 3] = np.float32(1.0)
        return out
    return make_clustered(w.n, w.box, w.seed, w.background, w.frac_halo, w.n_halo, w.a_range,
                          sigma=w.sigma, lattice=w.lattice, permute=w.permute)


def scaled_clustered(n: int, ncell, seed: int, frac_halo: float = 0.5, n_halo: int = 8,
                     a_range=(0.3, 2.0), cell: float = 3.2, background: str = "uniform",
                     sigma: float = 0.5) -> tuple:
    """Small test-sized particle set with the same recipe (box = ncell * cell). Returns (pos_mass, box)."""
    box = tuple(float(np.float32(c * cell)) for c in ncell)
    lattice = ()
    if background == "lattice":
        m = int(round(n ** (1.0 / 3.0)))
        lattice = (m, m, m)
        n = m ** 3 if frac_halo == 0.0 else n
    pos = make_clustered(n, box, seed, background, frac_halo, n_halo, a_range, sigma=sigma,
                         lattice=lattice, permute=True)
    return pos, box


def unit_lattice(m: int) -> np.ndarray:
    """Perfect cubic lattice, sites (i+1/2), spacing 1, in a box of m^3 (pin P3)."""
    g = np.arange(m, dtype=np.float32) + np.float32(0.5)
    z, y, x = np.meshgrid(g, g, g, indexing="ij")
    out = np.empty((m ** 3, 4), dtype=np.float32)
    out[:, 0], out[:, 1], out[:, 2], out[:, 3] = x.ravel(), y.ravel(), z.ravel(), 1.0
    return out
