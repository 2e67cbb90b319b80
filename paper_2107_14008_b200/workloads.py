"""Seeded synthetic particle loads (input generators only).

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path, and therefore holds
none of the method's arithmetic: no force law, no truncation function, no tree, no lists.
It only draws positions and masses with numpy.

The recipes stand in for the particle distributions the paper measured on (its 2LPTic /
Zel'dovich initial conditions at z=99, and its evolved halo-rich z=0
states); none of those data are available here.  They are the five
configurations of BASELINE.json (``configs[0..4]`` == ``CONFIGS[1..5]``), see DESIGN.md §4.

Input flavours (reading A20):
  F  positions rounded once to the fp32 grid, then handed to every path (and the oracle) as
     that rounded value.  The paper's single-precision runs keep "all variable as SP"
     (PAPER.md:L206), so the particle data themselves live on the fp32 grid.
  D  unrounded fp64 positions (the paper's DP run).
"""
from __future__ import annotations

import dataclasses

import numpy as np


@dataclasses.dataclass(frozen=True)
class Config:
    """One BASELINE.json workload."""
    name: str
    n_side: int            # N = n_side**3 particles
    n_pm: int              # PM mesh cells per side; r_s = 1.2*boxsize/n_pm
    maxleaf: int
    kind: str              # "uniform" | "clustered" | "grid"
    seed: int
    clustered_fraction: float = 0.0
    n_spheres: int = 0
    grid_sigma: float = 0.0   # in units of the grid spacing
    boxsize: float = 1.0
    G: float = 1.0

    @property
    def n(self) -> int:
        return self.n_side ** 3


CONFIGS = {
    1: Config("c1_uniform_32", 32, 32, 32, "uniform", 1001),
    2: Config("c2_clustered_128", 128, 128, 32, "clustered", 1002, clustered_fraction=0.5, n_spheres=2000),
    3: Config("c3_grid_256", 256, 256, 32, "grid", 1003, grid_sigma=0.3),
    4: Config("c4_clustered_256", 256, 256, 32, "clustered", 1004, clustered_fraction=0.7, n_spheres=20000),
    5: Config("c5_clustered_512", 512, 512, 32, "clustered", 1005, clustered_fraction=0.7, n_spheres=20000),
}

PLUMMER_A_MAX = 0.002       # scale radius of the most massive sphere (BASELINE.json configs[1])
PLUMMER_TRUNC = 10.0        # radii beyond 10 a are re-drawn (the config is silent)
MASS_SLOPE = 1.9            # dn/dM ~ M^-1.9 over two decades


def _sphere_counts(rng: np.random.Generator, n_spheres: int, n_clustered: int):
    """Sphere masses from dn/dM ~ M^-1.9 on [1,100] and the particle count of each sphere."""
    u = rng.random(n_spheres)
    k = MASS_SLOPE - 1.0
    M = (1.0 + u * (100.0 ** (-k) - 1.0)) ** (-1.0 / k)
    share = M / M.sum() * n_clustered
    counts = np.floor(share).astype(np.int64)
    rem = int(n_clustered - counts.sum())
    order = np.argsort(-M, kind="stable")
    # hand the rounding remainder out one particle at a time, most massive first
    q, r = divmod(rem, n_spheres)
    counts += q
    counts[order[:r]] += 1
    return M, counts


def _plummer_offsets(rng: np.random.Generator, counts: np.ndarray, a: np.ndarray, dtype=np.float64):
    """Offsets from the sphere centre for every clustered particle (Plummer profile, cut at 10 a)."""
    total = int(counts.sum())
    a_of = np.repeat(a, counts)
    r = np.empty(total)
    todo = np.arange(total)
    while todo.size:
        u = rng.random(todo.size)
        u = np.clip(u, 1e-300, 1.0)
        rr = (u ** (-2.0 / 3.0) - 1.0) ** -0.5     # in units of a
        ok = rr <= PLUMMER_TRUNC
        r[todo[ok]] = rr[ok]
        todo = todo[~ok]
    r *= a_of
    cos_t = rng.uniform(-1.0, 1.0, total)
    sin_t = np.sqrt(1.0 - cos_t * cos_t)
    phi = rng.uniform(0.0, 2.0 * np.pi, total)
    off = np.empty((total, 3))
    off[:, 0] = r * sin_t * np.cos(phi)
    off[:, 1] = r * sin_t * np.sin(phi)
    off[:, 2] = r * cos_t
    return off


def positions(kind: str, n: int, seed: int, *, boxsize: float = 1.0, clustered_fraction: float = 0.0,
              n_spheres: int = 0, grid_sigma: float = 0.0, flavour: str = "F") -> np.ndarray:
    """n x 3 float64 positions in [0, boxsize).  flavour 'F' = values on the fp32 grid."""
    rng = np.random.default_rng(seed)
    if kind == "uniform":
        pos = rng.random((n, 3))
    elif kind == "grid":
        side = round(n ** (1.0 / 3.0))
        if side ** 3 != n:
            raise ValueError("grid load needs a cubic particle number")
        g = (np.arange(side) + 0.5) / side
        pos = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3)
        pos = pos + rng.normal(0.0, grid_sigma / side, size=pos.shape)
    elif kind == "clustered":
        n_cl = int(round(clustered_fraction * n))
        M, counts = _sphere_counts(rng, n_spheres, n_cl)
        a = PLUMMER_A_MAX * (M / M.max()) ** (1.0 / 3.0)
        centres = rng.random((n_spheres, 3))
        off = _plummer_offsets(rng, counts, a)
        cl = np.repeat(centres, counts, axis=0) + off
        un = rng.random((n - n_cl, 3))
        pos = np.concatenate([cl, un], axis=0)
        # caller order should not be sorted by sphere: shuffle once
        pos = pos[rng.permutation(n)]
    else:
        raise ValueError(f"unknown load kind {kind!r}")
    pos = np.mod(pos, 1.0)
    if flavour == "F":
        pos = pos.astype(np.float32)
        pos[pos >= 1.0] = 0.0          # rounding up to 1.0 wraps to 0
        pos = pos.astype(np.float64)
    elif flavour == "D":
        pos[pos >= 1.0] = 0.0
    else:
        raise ValueError("flavour must be 'F' or 'D'")
    return np.ascontiguousarray(pos * boxsize) if boxsize != 1.0 else np.ascontiguousarray(pos)


def make(cfg: Config | int, *, flavour: str = "F"):
    """(pos[n,3] float64, mass[n] float64) for a config (use ``scaled`` for test-sized copies)."""
    if isinstance(cfg, int):
        cfg = CONFIGS[cfg]
    pos = positions(cfg.kind, cfg.n, cfg.seed, boxsize=cfg.boxsize, clustered_fraction=cfg.clustered_fraction,
                    n_spheres=cfg.n_spheres, grid_sigma=cfg.grid_sigma, flavour=flavour)
    mass = np.full(cfg.n, 1.0 / cfg.n)
    return pos, mass


def scaled(cfg: Config | int, n_side: int) -> Config:
    """The same recipe at a smaller particle number (parity-test sizes); N_PM shrinks with it so
    the mean neighbour count inside r_cut stays the full config's."""
    if isinstance(cfg, int):
        cfg = CONFIGS[cfg]
    n_sph = max(1, int(round(cfg.n_spheres * n_side ** 3 / cfg.n))) if cfg.n_spheres else 0
    return dataclasses.replace(cfg, name=f"{cfg.name}@{n_side}", n_side=n_side, n_pm=n_side, n_spheres=n_sph)


def sample_targets(n: int, n_targets: int, seed: int) -> np.ndarray:
    """Plain uniform sample of target indices (sorted), for the sampled-target parity checks."""
    rng = np.random.default_rng(seed + 7_000_000)
    return np.sort(rng.choice(n, size=min(n, n_targets), replace=False)).astype(np.int64)
