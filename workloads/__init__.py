"""Seeded synthetic inputs for the five ENCORE configs (BASELINE.json `configs`).

This module only *draws points and weights*.  It holds none of the estimator's
arithmetic (no separations, bins, harmonics, couplings) and is imported by the
tests and by bench.py, which hand the same arrays to the CPU oracle and to the
CUDA library.  Neither `oracle/` nor `paper_2105_08722_b200/` imports it.

The paper's own workloads are uniform random points in a periodic box
(L=1500, N_r=10, r_max=200) and BOSS CMASS-like mocks with a
data-minus-random field on a cut-sky footprint.  The
Patchy mocks and survey randoms are not available here; the recipes below take
their shapes (densities 2-3e-4, r_max 160-200, N_r 8-10, lmax 3-10, a D-R field
whose weights sum to zero) and stand in for them.  Recipes: DESIGN.md §4.

Positions are returned SoA, shape (3, n) float64, C-contiguous; weights (n,).
"""
from __future__ import annotations

import dataclasses
import hashlib

import numpy as np


@dataclasses.dataclass(frozen=True)
class Config:
    """Estimator parameters + the recipe of one workload."""
    name: str
    order: int          # N of the NPCF (3, 4, 5)
    nbins: int          # N_r
    rmin: float
    rmax: float
    lmax: int
    box: float          # periodic cube side L; 0.0 = open (non-periodic) geometry
    n: int              # number of particles
    seed: int
    kind: str           # "uniform" | "lognormal" | "cutsky"
    weights: str        # "unit" | "uniform_0.8_1.2" | "data_minus_random"
    grid: int = 256     # lognormal mesh per side


# BASELINE.json configs[0..4]
CONFIGS = {
    "c1": Config("c1", 3, 5, 0.0, 200.0, 4, 1000.0, 2000, 1, "uniform", "unit"),
    "c2": Config("c2", 3, 10, 0.0, 200.0, 10, 1000.0, 200000, 2, "lognormal", "unit"),
    "c3": Config("c3", 4, 10, 20.0, 160.0, 5, 1000.0, 300000, 3, "lognormal", "uniform_0.8_1.2"),
    "c4": Config("c4", 4, 10, 20.0, 160.0, 5, 0.0, 1600000, 4, "cutsky", "data_minus_random"),
    "c5": Config("c5", 5, 8, 20.0, 160.0, 3, 1000.0, 300000, 5, "lognormal", "unit"),
}


# The input of the paper's Table 2: ~5e4 uniform points in a periodic box L = 1500, N_r = 10 bins up to
# r_max = 200.  Not a BASELINE.json config: bench.py's `next_rows.paper_table2_shapes` times it, tests/golden/ holds the
# oracle's 4PCF lmax = 10 run of it (the paper's largest 4PCF GPU shape: 381 multiplets x 120 bin triples).
TABLE2 = Config("table2", 4, 10, 0.0, 200.0, 5, 1500.0, 50625, 578, "uniform", "unit")
EXTRA = {"table2_4pcf_lmax10": dataclasses.replace(TABLE2, name="table2_4pcf_lmax10", lmax=10)}


def scaled(cfg: Config, box: float | None = None, n: int | None = None,
           grid: int | None = None, name: str | None = None) -> Config:
    """Same recipe at a reduced size (parity-test cases the oracle finishes in seconds).

    For periodic configs pass a smaller `box` (the mean density is kept unless `n` is
    given); for the cut-sky config pass `n` (the 1:3 data:random split is kept and the
    shell is shrunk so that the density is kept).
    """
    if cfg.box > 0.0:
        b = cfg.box if box is None else float(box)
        nn = n if n is not None else int(round(cfg.n * (b / cfg.box) ** 3))
        g = grid if grid is not None else max(16, int(round(cfg.grid * b / cfg.box)))
        return dataclasses.replace(cfg, box=b, n=nn, grid=g,
                                   name=name or f"{cfg.name}_L{b:g}_n{nn}")
    nn = cfg.n if n is None else int(n)
    return dataclasses.replace(cfg, n=nn, name=name or f"{cfg.name}_n{nn}")


# ----------------------------------------------------------------------------------
# generators
# ----------------------------------------------------------------------------------
def _lognormal_density(grid: int, rng: np.random.Generator) -> np.ndarray:
    """exp(g) with g a unit-variance Gaussian field, P(k) ∝ k^-1.5, on a grid^3 mesh."""
    white = rng.standard_normal((grid, grid, grid))
    fk = np.fft.rfftn(white)
    kx = np.fft.fftfreq(grid) * grid
    kz = np.fft.rfftfreq(grid) * grid
    k2 = kx[:, None, None] ** 2 + kx[None, :, None] ** 2 + kz[None, None, :] ** 2
    k2[0, 0, 0] = 1.0
    amp = k2 ** (-0.375)            # |k|^-0.75  ->  P(k) ∝ |k|^-1.5
    amp[0, 0, 0] = 0.0
    g = np.fft.irfftn(fk * amp, s=(grid, grid, grid), axes=(0, 1, 2))
    g -= g.mean()
    g /= g.std()
    return np.exp(g)


def lognormal_box(box: float, n: int, seed: int, grid: int = 256) -> np.ndarray:
    """n points Poisson-sampled (conditioned on the total) from a lognormal field in [0,L)^3."""
    rng = np.random.default_rng(seed)
    rho = _lognormal_density(grid, rng).ravel()
    p = rho / rho.sum()
    counts = rng.multinomial(n, p)
    cell = np.repeat(np.arange(grid ** 3, dtype=np.int64), counts)
    ix, rem = np.divmod(cell, grid * grid)
    iy, iz = np.divmod(rem, grid)
    u = rng.random((3, n))
    h = box / grid
    pos = np.empty((3, n), dtype=np.float64)
    pos[0] = (ix + u[0]) * h
    pos[1] = (iy + u[1]) * h
    pos[2] = (iz + u[2]) * h
    # guard the half-open interval against (idx + u) * h rounding up to L
    np.minimum(pos, np.nextafter(box, 0.0), out=pos)
    perm = rng.permutation(n)
    return np.ascontiguousarray(pos[:, perm])


def uniform_box(box: float, n: int, seed: int) -> np.ndarray:
    rng = np.random.default_rng(seed)
    pos = rng.random((3, n)) * box
    np.minimum(pos, np.nextafter(box, 0.0), out=pos)
    return np.ascontiguousarray(pos)


def _in_footprint(p: np.ndarray, r1: float, r2: float, half_deg: float) -> np.ndarray:
    r = np.sqrt((p ** 2).sum(axis=0))
    ra = np.degrees(np.arctan2(p[1], p[0]))
    dec = np.degrees(np.arcsin(np.clip(p[2] / np.maximum(r, 1e-300), -1.0, 1.0)))
    return (r >= r1) & (r < r2) & (np.abs(ra) <= half_deg) & (np.abs(dec) <= half_deg)


def cutsky(n_total: int, seed: int, grid: int = 256, r1: float = 1200.0, r2: float = 1800.0,
           half_deg: float = 30.0, field_box: float = 1000.0):
    """Data-minus-random field on a shell-patch footprint (open geometry).

    n_total/4 clustered 'data' points (w=+1) + 3 n_total/4 uniform 'randoms'
    (w = -N_D/N_R, so the weights sum to zero).  For reduced sizes the
    shell thickness is shrunk about its mid-radius so that the data density stays
    that of the full config (400000 points in the full footprint).
    """
    rng = np.random.default_rng(seed)
    n_data = n_total // 4
    n_rand = n_total - n_data
    full_data = 400000
    if n_data < full_data:
        # keep density: shrink the radial extent (volume ∝ r2^3 - r1^3 at fixed solid angle)
        vol_full = r2 ** 3 - r1 ** 3
        rm = 0.5 * (r1 + r2)
        target = vol_full * n_data / full_data
        lo, hi = 0.0, 0.5 * (r2 - r1)
        for _ in range(80):
            mid = 0.5 * (lo + hi)
            if (rm + mid) ** 3 - (rm - mid) ** 3 < target:
                lo = mid
            else:
                hi = mid
        r1, r2 = rm - hi, rm + hi
    # data: lognormal field tiled periodically, random tile choice, rejection to the footprint
    rho = _lognormal_density(grid, rng).ravel()
    p = rho / rho.sum()
    h = field_box / grid
    ntx = int(np.ceil(r2 / field_box))                                  # tiles: x in [0, ntx L)
    nty = int(np.ceil(r2 * np.sin(np.radians(half_deg)) / field_box))   #        y,z in [-nty L, nty L)
    data = np.empty((3, 0))
    omega = (2 * np.radians(half_deg)) * (2 * np.sin(np.radians(half_deg)))
    vol = omega * (r2 ** 3 - r1 ** 3) / 3.0
    tiles_vol = (ntx * field_box) * (2 * nty * field_box) ** 2
    while data.shape[1] < n_data:
        need = n_data - data.shape[1]
        m = int(1.3 * need * tiles_vol / vol) + 1000
        m = min(m, 8_000_000)
        cell = rng.choice(grid ** 3, size=m, p=p)
        ix, rem = np.divmod(cell, grid * grid)
        iy, iz = np.divmod(rem, grid)
        u = rng.random((3, m))
        q = np.empty((3, m))
        q[0] = (ix + u[0]) * h + field_box * rng.integers(0, ntx, m)
        q[1] = (iy + u[1]) * h + field_box * rng.integers(-nty, nty, m)
        q[2] = (iz + u[2]) * h + field_box * rng.integers(-nty, nty, m)
        q = q[:, _in_footprint(q, r1, r2, half_deg)]
        data = np.concatenate([data, q[:, :need]], axis=1)
    # randoms: uniform in volume over the same footprint
    ur = rng.random(n_rand)
    rr = (r1 ** 3 + ur * (r2 ** 3 - r1 ** 3)) ** (1.0 / 3.0)
    ra = np.radians(half_deg) * (2.0 * rng.random(n_rand) - 1.0)
    sd = np.sin(np.radians(half_deg)) * (2.0 * rng.random(n_rand) - 1.0)
    cd = np.sqrt(1.0 - sd * sd)
    rand = np.stack([rr * cd * np.cos(ra), rr * cd * np.sin(ra), rr * sd])
    pos = np.concatenate([data, rand], axis=1)
    w = np.concatenate([np.ones(n_data), np.full(n_rand, -float(n_data) / float(n_rand))])
    perm = rng.permutation(n_total)
    return np.ascontiguousarray(pos[:, perm]), np.ascontiguousarray(w[perm])


def make(cfg: Config | str):
    """Return (positions (3,n) float64, weights (n,) float64) for a config."""
    if isinstance(cfg, str):
        cfg = CONFIGS[cfg]
    if cfg.kind == "uniform":
        pos = uniform_box(cfg.box, cfg.n, cfg.seed)
    elif cfg.kind == "lognormal":
        pos = lognormal_box(cfg.box, cfg.n, cfg.seed, cfg.grid)
    elif cfg.kind == "cutsky":
        return cutsky(cfg.n, cfg.seed, cfg.grid)
    else:
        raise ValueError(cfg.kind)
    if cfg.weights == "unit":
        w = np.ones(cfg.n)
    elif cfg.weights == "uniform_0.8_1.2":
        w = np.random.default_rng(cfg.seed + 1000).uniform(0.8, 1.2, cfg.n)
    else:
        raise ValueError(cfg.weights)
    return pos, np.ascontiguousarray(w, dtype=np.float64)


def nearest_subset(pos: np.ndarray, centre, k: int) -> np.ndarray:
    """Indices of the k points nearest `centre` (ties by index) — c1's 40-point brute-force subset."""
    d2 = ((pos - np.asarray(centre, dtype=np.float64)[:, None]) ** 2).sum(axis=0)
    return np.argsort(d2, kind="stable")[:k]


def digest(pos: np.ndarray, w: np.ndarray) -> str:
    """sha256 of the input bytes: stored beside golden values so a stale fixture is detected."""
    hsh = hashlib.sha256()
    hsh.update(np.ascontiguousarray(pos, dtype=np.float64).tobytes())
    hsh.update(np.ascontiguousarray(w, dtype=np.float64).tobytes())
    return hsh.hexdigest()
