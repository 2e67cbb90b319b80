"""Seeded input generators (paper_2107_14008_b200/workloads.py): shapes, determinism, flavours."""
import numpy as np
import pytest

from paper_2107_14008_b200 import workloads


@pytest.mark.parametrize("cfg_id", [1, 2, 3, 4])
def test_scaled_configs_are_seeded_and_in_box(cfg_id):
    cfg = workloads.scaled(cfg_id, 16)
    pos, mass = workloads.make(cfg)
    pos2, _ = workloads.make(cfg)
    assert pos.shape == (4096, 3) and pos.dtype == np.float64
    assert np.array_equal(pos, pos2)
    assert pos.min() >= 0.0 and pos.max() < 1.0
    assert mass.sum() == pytest.approx(1.0)
    # flavour F: every coordinate is exactly representable in fp32
    assert np.array_equal(pos.astype(np.float32).astype(np.float64), pos)
    posD, _ = workloads.make(cfg, flavour="D")
    assert not np.array_equal(posD.astype(np.float32).astype(np.float64), posD)
    assert np.abs(posD - pos).max() < 1e-7 or np.abs(np.abs(posD - pos).max() - 1.0) < 1e-7


def test_clustered_recipe_statistics():
    cfg = workloads.scaled(4, 32)              # 32768 particles, 39 spheres
    pos, _ = workloads.make(cfg, flavour="D")
    # 70 % of the particles sit in spheres of scale radius <= 0.002: the nearest-neighbour distance
    # distribution must be far more skewed than for a uniform load
    rng = np.random.default_rng(0)
    idx = rng.choice(cfg.n, 300, replace=False)
    d = pos[None, :, :] - pos[idx, None, :]
    d -= np.round(d)
    r = np.sqrt((d ** 2).sum(-1))
    r[r == 0] = 1.0
    nn = r.min(axis=1)
    uniform_nn = 0.554 * cfg.n ** (-1.0 / 3.0)
    assert np.median(nn) < 0.2 * uniform_nn
    assert (nn > 0.5 * uniform_nn).mean() > 0.1          # the 30 % uniform component is there


def test_grid_recipe_displacement():
    cfg = workloads.scaled(3, 16)
    pos, _ = workloads.make(cfg, flavour="D")
    g = (np.arange(16) + 0.5) / 16
    grid = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3)
    disp = pos - grid
    disp -= np.round(disp)
    assert disp.std() == pytest.approx(0.3 / 16, rel=0.03)


def test_sample_targets():
    t = workloads.sample_targets(1000, 100, 3)
    assert len(np.unique(t)) == 100 and t.min() >= 0 and t.max() < 1000
    assert np.array_equal(t, workloads.sample_targets(1000, 100, 3))
