"""Parity of the CUDA path (through the C ABI, include/photons.h) against the CPU oracle (oracle/),
element by element on the same seeded inputs.  GPU only: ``pytest -m gpu``.

Tolerances are north_star's (BASELINE.json), written out here:
    fp64                         max_i |a_gpu - a_ref| <= 1e-12 * rms|a_ref|
    fp32 / mixed, direct g       <= 1e-5 * rms|a_ref|
    interpolated g (table)       <= 1e-4 * rms|a_ref|
|.| is the Euclidean norm of the 3-vector, rms is taken over the compared targets.
The FMA-pipe polynomial g (PHOTONS_G_POLY) is not one of north_star's two variants; it is held to the
tighter of the two fp32 bounds (1e-5).

The fp32 bounds are met with the exact close-pair path on (close_pair_radius > 0, A12);
with it off the literal max-norm criterion is missed by a factor of about two on the closest pairs,
which test_fp32_without_close_pairs_documents_the_gap pins so that the statement in DESIGN.md stays true.
"""
import numpy as np
import pytest

from paper_2107_14008_b200 import workloads

pytestmark = pytest.mark.gpu

TOL_FP64 = 1e-12
TOL_FP32 = 1e-5
TOL_TABLE = 1e-4


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the CUDA path has no CPU fallback")
    from paper_2107_14008_b200 import binding
    binding.load()          # raises if libphotons.so is not built
    return binding


def _geom(cfg):
    r_s = 1.2 * cfg.boxsize / cfg.n_pm
    return r_s, 6.0 * r_s                       # r_cut = 6 r_s (north_star)


def _err(a, ref):
    rms = np.sqrt((ref ** 2).sum(axis=1).mean())
    return np.sqrt(((a - ref) ** 2).sum(axis=1)).max() / rms


def _close(cfg):
    # radius inside which fp32 pairs are redone in fp64: 0.02 r_cut (A12)
    return 0.02 * _geom(cfg)[1]


@pytest.fixture(scope="module")
def c1(oracle):
    """BASELINE config 1: N = 32^3 uniform, full O(N^2) oracle."""
    cfg = workloads.CONFIGS[1]
    pos, mass = workloads.make(cfg)
    r_s, r_cut = _geom(cfg)
    ref, cnt = oracle.p2p(pos, mass, boxsize=cfg.boxsize, r_s=r_s, r_cut=r_cut, G=cfg.G)
    return cfg, pos, mass, ref, cnt


def _run(B, cfg, pos, mass, **kw):
    kw.setdefault("maxleaf", cfg.maxleaf)
    out, st = B.short_range_acc(pos, mass, boxsize=cfg.boxsize, n_pm=cfg.n_pm, G=cfg.G, **kw)
    assert np.isfinite(out).all()
    return out, st


# ------------------------------------------------------------------------------------------ config 1

@pytest.mark.parametrize("maxleaf", [16, 32, 64, 128])
def test_c1_fp64_direct(B, c1, maxleaf):
    cfg, pos, mass, ref, _ = c1
    out, st = _run(B, cfg, pos, mass, precision="fp64", g_mode="direct", maxleaf=maxleaf)
    assert _err(out, ref) <= TOL_FP64
    assert st["n_leaves"] == cfg.n // maxleaf


@pytest.mark.parametrize("nodes,level,tol", [(4096, 4, TOL_FP64), (4096, 3, TOL_FP64), (512, 4, TOL_TABLE),
                                             (512, 2, TOL_TABLE), (256, 1, TOL_TABLE), (1024, 1, TOL_TABLE)])
def test_c1_fp64_table(B, c1, nodes, level, tol):
    # Eq. 2 in fp64: "T[4] for DP"; a 4096-node table at level >= 3 even meets the fp64 bound
    cfg, pos, mass, ref, _ = c1
    out, _ = _run(B, cfg, pos, mass, precision="fp64", g_mode="table", table_nodes=nodes, table_level=level)
    assert _err(out, ref) <= tol


@pytest.mark.parametrize("precision", ["fp32", "mixed"])
@pytest.mark.parametrize("maxleaf", [16, 32, 64, 128])
@pytest.mark.parametrize("g_mode", ["direct", "poly"])
def test_c1_fp32_direct_and_poly(B, c1, precision, maxleaf, g_mode):
    cfg, pos, mass, ref, _ = c1
    out, _ = _run(B, cfg, pos, mass, precision=precision, g_mode=g_mode, maxleaf=maxleaf,
                  close_pair_radius=_close(cfg))
    assert _err(out, ref) <= TOL_FP32


@pytest.mark.parametrize("precision", ["fp32", "mixed"])
@pytest.mark.parametrize("nodes,level", [(256, 1), (256, 2), (512, 2), (1024, 1), (1024, 2), (4096, 0), (4096, 1), (512, 3)])
def test_c1_fp32_table(B, c1, precision, nodes, level):
    cfg, pos, mass, ref, _ = c1
    out, _ = _run(B, cfg, pos, mass, precision=precision, g_mode="table", table_nodes=nodes, table_level=level,
                  close_pair_radius=_close(cfg))
    assert _err(out, ref) <= TOL_TABLE


def test_c1_table_level2_keeps_fp32_quality(B, c1):
    # "T[2] adequate for single precision" with 512 nodes
    cfg, pos, mass, ref, _ = c1
    out, _ = _run(B, cfg, pos, mass, precision="fp32", g_mode="table", table_nodes=512, table_level=2,
                  close_pair_radius=_close(cfg))
    assert _err(out, ref) <= TOL_FP32


def test_fp32_without_close_pairs_documents_the_gap(B, c1):
    # DESIGN.md A12: plain fp32 pair arithmetic misses the literal 1e-5*rms max-norm on the closest pairs
    # (one fp32 ulp of an acceleration ~100x the rms) but stays within a few 1e-5.
    cfg, pos, mass, ref, _ = c1
    out, _ = _run(B, cfg, pos, mass, precision="fp32", g_mode="direct", close_pair_radius=0.0)
    e = _err(out, ref)
    assert e <= 1e-4
    # relative to each target's own acceleration the error is at fp32 round-off level
    rms = np.sqrt((ref ** 2).sum(axis=1).mean())
    rel = np.sqrt(((out - ref) ** 2).sum(axis=1)) / np.maximum(np.sqrt((ref ** 2).sum(axis=1)), rms)
    assert rel.max() <= 5e-6


def test_c1_fp32_output_dtype_and_device_buffers(B, c1):
    import torch
    cfg, pos, mass, ref, _ = c1
    dpos = torch.from_numpy(pos).cuda()
    dmass = torch.from_numpy(mass).cuda()
    with B.Photons(n_pm=cfg.n_pm, precision="fp32", g_mode="poly", close_pair_radius=_close(cfg)) as ph:
        ph.set_particles(dpos, dmass)
        ph.build_leaves()
        out64 = torch.empty((cfg.n, 3), dtype=torch.float64, device="cuda")
        out32 = torch.empty((cfg.n, 3), dtype=torch.float32, device="cuda")
        ph.short_range_acc(out64)
        ph.short_range_acc(out32)
    torch.cuda.synchronize()
    assert _err(out64.cpu().numpy(), ref) <= TOL_FP32
    assert np.array_equal(out64.cpu().numpy().astype(np.float32), out32.cpu().numpy())
    # an fp32 *output* alone costs up to half an ulp of the largest acceleration
    assert _err(out32.cpu().numpy().astype(np.float64), ref) <= 2e-5


def test_c1_fp32_input_arrays(B, c1):
    # flavour F positions are exactly representable in fp32: float32 input must give the same bits
    cfg, pos, mass, ref, _ = c1
    a, _ = _run(B, cfg, pos, mass, precision="fp64", g_mode="direct")
    b, _ = _run(B, cfg, pos.astype(np.float32), None, precision="fp64", g_mode="direct")
    # mass = NULL means 1/n each, which is what the config uses
    assert np.array_equal(a, b)


def test_determinism_and_stream_invariance(B, c1):
    # each target's sum is owned by one CTA, no atomics (Alg. 1): bit-identical across runs and streams
    cfg, pos, mass, _, _ = c1
    for prec, g in (("fp64", "direct"), ("fp32", "poly"), ("mixed", "table")):
        a, _ = _run(B, cfg, pos, mass, precision=prec, g_mode=g, n_streams=1)
        b, _ = _run(B, cfg, pos, mass, precision=prec, g_mode=g, n_streams=1)
        c, _ = _run(B, cfg, pos, mass, precision=prec, g_mode=g, n_streams=4)
        assert np.array_equal(a, b)
        assert np.array_equal(a, c)


def test_launch_shape_invariance(B, c1):
    # the result may depend on chunking / warps per leaf only through rounding order
    cfg, pos, mass, ref, _ = c1
    for W in (1, 2, 4, 8):
        for chunk in (32, 64, 128, 256):
            out, _ = _run(B, cfg, pos, mass, precision="fp64", g_mode="direct", warps_per_leaf=W, chunk_max=chunk)
            assert _err(out, ref) <= TOL_FP64
    for W in (1, 8):
        out, _ = _run(B, cfg, pos, mass, precision="fp32", g_mode="poly", warps_per_leaf=W, chunk_max=64,
                      close_pair_radius=_close(cfg))
        assert _err(out, ref) <= TOL_FP32


@pytest.mark.parametrize("maxleaf,tpl", [(16, 1), (16, 2), (32, 1), (32, 2), (64, 2), (128, 4)])
def test_lane_mappings(B, c1, maxleaf, tpl):
    # every (MAXLEAF, targets per lane) shape of the fp32 kernel, with and without the exact close-pair path
    cfg, pos, mass, ref, _ = c1
    for prec, g, tol in (("fp32", "poly", TOL_FP32), ("mixed", "table", TOL_TABLE), ("fp32", "direct", TOL_FP32)):
        out, _ = _run(B, cfg, pos, mass, precision=prec, g_mode=g, maxleaf=maxleaf, targets_per_lane=tpl,
                      close_pair_radius=_close(cfg))
        assert _err(out, ref) <= tol
    out, _ = _run(B, cfg, pos, mass, precision="fp32", g_mode="poly", maxleaf=maxleaf, targets_per_lane=tpl)
    assert _err(out, ref) <= 1e-4
    with pytest.raises(B.PhotonsError):
        B.Photons(maxleaf=128, targets_per_lane=1)


def test_pairs_evaluated_and_list_cover(B, c1):
    """Host-visible feeder outputs: the permutation is a permutation, leaves are ORB-balanced, and the
    interaction list of every target leaf holds every leaf that has a particle pair inside r_cut (A11)."""
    cfg, pos, mass, _, cnt = c1
    r_s, r_cut = _geom(cfg)
    with B.Photons(n_pm=cfg.n_pm, precision="fp64", g_mode="direct") as ph:
        ph.set_particles(pos, mass)
        ph.build_leaves()
        st = ph.stats()
        perm, leaf_start = ph.leaf_order()
        ptr, first, nleaf, code = ph.interaction_list()
    n = cfg.n
    assert np.array_equal(np.sort(perm), np.arange(n))
    sizes = np.diff(leaf_start)
    assert sizes.min() == sizes.max() == 32 and st["n_leaves"] == 1024
    # evaluated pairs: all within-cut ordered pairs (incl. none of the self pairs) must be covered
    assert st["pairs_evaluated"] >= cnt["pairs_in_cut"]
    assert 4e3 < st["pairs_evaluated"] / n < 9e3            # SURVEY.md §8(c) "counts": 6.3e3 at MAXLEAF 32
    # expand the list to (target leaf, source leaf) pairs
    tl = np.repeat(np.arange(1024), np.diff(ptr))
    pairs = set()
    for t, f, k in zip(tl, first, nleaf):
        for j in range(f, f + k):
            pairs.add((int(t), int(j)))
    assert len(pairs) == st["n_leaf_pairs"] == int(nleaf.sum())
    assert all((i, i) in pairs for i in range(1024))
    # brute force on a sample of targets: every leaf within r_cut particle-to-particle must be listed
    leaf_of = np.empty(n, dtype=np.int64)
    leaf_of[perm] = np.repeat(np.arange(1024), 32)
    rng = np.random.default_rng(5)
    for i in rng.choice(n, 200, replace=False):
        d = pos - pos[i]
        d -= np.rint(d)
        near = np.nonzero((d * d).sum(axis=1) < r_cut * r_cut)[0]
        for j in np.unique(leaf_of[near]):
            assert (int(leaf_of[i]), int(j)) in pairs
    assert set(np.unique(code)) <= set(range(28))


# ------------------------------------------------------------------- ragged sizes and degenerate cases

@pytest.mark.parametrize("n", [1, 2, 3, 31, 33, 100, 1000, 5000, 20011])
@pytest.mark.parametrize("precision,g_mode,tol", [("fp64", "direct", TOL_FP64), ("fp32", "poly", TOL_FP32),
                                                   ("mixed", "table", TOL_TABLE)])
def test_ragged_and_tiny_n(B, oracle, n, precision, g_mode, tol):
    # N not a power of two: leaves of unequal size with padding slots; tiny N: leaves spanning the box
    # (per-pair minimum image, shift code 27)
    rng = np.random.default_rng(100 + n)
    pos = rng.random((n, 3)).astype(np.float32).astype(np.float64)
    mass = rng.uniform(0.5, 1.5, n) / n
    n_pm = 16
    r_s = 1.2 / n_pm
    ref, _ = oracle.p2p(pos, mass, boxsize=1.0, r_s=r_s, r_cut=6 * r_s)
    out, _ = B.short_range_acc(pos, mass, n_pm=n_pm, precision=precision, g_mode=g_mode,
                               close_pair_radius=0.02 * 6 * r_s)
    if n == 1:
        assert np.array_equal(out, np.zeros((1, 3)))
        return
    rms = np.sqrt((ref ** 2).sum(axis=1).mean())
    if rms == 0:
        assert np.abs(out).max() == 0
    else:
        assert _err(out, ref) <= tol


def test_two_body_closed_form_and_seam(B):
    # a_1 = +G m_2 g(d)/d^2 towards 2, also across the periodic seam (SURVEY.md §8(c) "two-body")
    import math
    n_pm = 32
    r_s = 1.2 / n_pm
    d = 0.03
    for x1 in (0.5, 0.99):
        pos = np.array([[x1, 0.25, 0.75], [(x1 + d) % 1.0, 0.25, 0.75]])
        mass = np.array([2.0, 3.0])
        out, _ = B.short_range_acc(pos, mass, n_pm=n_pm, precision="fp64", g_mode="direct", G=0.5)
        x = d / (2 * r_s)
        g = math.erfc(x) + 2 * x / math.sqrt(math.pi) * math.exp(-x * x)
        assert out[0, 0] == pytest.approx(0.5 * 3.0 * g / d ** 2, rel=1e-12)
        assert out[1, 0] == pytest.approx(-0.5 * 2.0 * g / d ** 2, rel=1e-12)
        assert np.abs(out[:, 1:]).max() == 0


def test_zero_beyond_cut_and_coincident(B):
    n_pm = 32
    r_cut = 6 * 1.2 / n_pm
    pos = np.array([[0.1, 0.1, 0.1], [0.1 + r_cut * 1.0001, 0.1, 0.1], [0.6, 0.6, 0.6], [0.6, 0.6, 0.6]])
    for prec, g in (("fp64", "direct"), ("fp32", "direct"), ("fp32", "poly"), ("fp32", "table"), ("mixed", "poly")):
        out, _ = B.short_range_acc(pos, None, n_pm=n_pm, precision=prec, g_mode=g)
        assert np.array_equal(out, np.zeros((4, 3)))       # beyond the cut: exactly 0; coincident: 0 (A7)


def test_perfect_lattice_has_zero_force(B):
    side = 16
    g = (np.arange(side) + 0.5) / side
    pos = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3)
    out, _ = B.short_range_acc(pos, None, n_pm=16, precision="fp64", g_mode="direct")
    scale = (1.0 / side ** 3) / (1.0 / side) ** 2           # G m / spacing^2
    assert np.abs(out).max() <= 1e-12 * scale


def test_isolated_boundaries(B, oracle):
    """periodic = 0: no images, no wrapping, negative coordinates; oracle with boxsize <= 0."""
    rng = np.random.default_rng(77)
    n = 20000
    n_pm = 32
    r_s = 1.2 / n_pm
    r_cut = 6 * r_s
    # a blob that straddles the origin and the faces of the nominal unit box
    pos = (rng.normal(0.0, 0.35, (n, 3)) + np.array([0.1, 0.9, -0.2])).astype(np.float32).astype(np.float64)
    mass = rng.uniform(0.5, 1.5, n) / n
    ref, _ = oracle.p2p(pos, mass, boxsize=0.0, r_s=r_s, r_cut=r_cut)
    per, _ = oracle.p2p(np.mod(pos, 1.0), mass, boxsize=1.0, r_s=r_s, r_cut=r_cut)
    assert _err(per, ref) > 1e-3                    # the periodic answer really is a different one
    for prec, g, tol, kw in (("fp64", "direct", TOL_FP64, {}), ("fp32", "poly", TOL_FP32, dict(close_pair_radius=0.02 * r_cut)),
                             ("mixed", "poly", TOL_FP32, dict(close_pair_radius=0.02 * r_cut)),
                             ("fp32", "table", TOL_TABLE, dict(close_pair_radius=0.02 * r_cut)),
                             ("fp32", "direct", TOL_FP32, dict(close_pair_radius=0.02 * r_cut, maxleaf=16))):
        out, _ = B.short_range_acc(pos, mass, n_pm=n_pm, periodic=0, precision=prec, g_mode=g, **kw)
        assert _err(out, ref) <= tol, (prec, g)
    # isolated mode has no r_cut < L/2 requirement
    out, _ = B.short_range_acc(pos[:50] * 0.01, mass[:50], boxsize=1.0, n_pm=8, periodic=0, precision="fp64", g_mode="direct")
    ref8, _ = oracle.p2p(pos[:50] * 0.01, mass[:50], boxsize=0.0, r_s=1.2 / 8, r_cut=6 * 1.2 / 8)
    assert _err(out, ref8) <= TOL_FP64


# ---------------------------------------------------------------------------- error behaviour (ABI)

def test_abi_errors(B):
    import ctypes
    with pytest.raises(B.PhotonsError) as e:
        B.Photons(n_pm=8)                      # r_cut = 0.9 >= boxsize/2
    assert e.value.code == B.EBOX
    for bad in (dict(maxleaf=48), dict(precision=7), dict(g_mode=9), dict(n_streams=0), dict(boxsize=-1.0),
                dict(precision="fp64", g_mode="poly"), dict(g_mode="table", table_nodes=5),
                dict(g_mode="poly", rcut_over_rs=7.0)):
        with pytest.raises(B.PhotonsError) as e:
            B.Photons(**bad)
        assert e.value.code == B.EINVAL
    with B.Photons(n_pm=32) as ph:
        with pytest.raises(B.PhotonsError) as e:
            ph.build_leaves()
        assert e.value.code == B.ESTATE
        out = np.empty((4, 3))
        ph.n = 4
        with pytest.raises(B.PhotonsError) as e:
            ph.short_range_acc(out)
        assert e.value.code == B.ESTATE
        pos = np.random.default_rng(0).random((4, 3))
        bad = pos.copy()
        bad[2, 1] = np.nan
        with pytest.raises(B.PhotonsError) as e:
            ph.set_particles(bad)
        assert e.value.code == B.ENONFINITE
        rc = ph._lib.photons_set_particles(ph._ctx, 0, pos.ctypes.data, None, B.DTYPE_F64, B.MEM_HOST, None)
        assert rc == B.EINVAL                   # empty input
        ph.set_particles(pos)
        ph.build_leaves()
        ph.short_range_acc(out)
        ph.set_particles(pos)                   # invalidates the leaves
        with pytest.raises(B.PhotonsError) as e:
            ph.short_range_acc(out)
        assert e.value.code == B.ESTATE
    B.load().photons_destroy(ctypes.c_void_p())  # NULL-safe


def test_positions_outside_the_box_are_wrapped(B, c1):
    cfg, pos, mass, ref, _ = c1
    shifted = pos + np.array([3.0, -2.0, 1.0])               # exact in fp64 for fp32-grid positions
    out, _ = _run(B, cfg, shifted, mass, precision="fp64", g_mode="direct")
    assert _err(out, ref) <= TOL_FP64


# ------------------------------------------------------------------ clustered and grid loads (sampled)

@pytest.mark.parametrize("cfg_id,n_side", [(2, 48), (3, 48), (4, 64)])
def test_scaled_configs_sampled_targets(B, oracle, cfg_id, n_side):
    """Configs 2-4 at test size (same recipe, N_PM scaled with N), oracle on sampled targets."""
    cfg = workloads.scaled(cfg_id, n_side)
    pos, mass = workloads.make(cfg)
    r_s, r_cut = _geom(cfg)
    tgt = workloads.sample_targets(cfg.n, 4000, cfg.seed)
    ref, _ = oracle.p2p_sampled(pos, mass, tgt, boxsize=cfg.boxsize, r_s=r_s, r_cut=r_cut)
    for prec, g, tol, kw in (("fp64", "direct", TOL_FP64, {}),
                             ("fp32", "direct", TOL_FP32, dict(close_pair_radius=0.02 * r_cut)),
                             ("fp32", "poly", TOL_FP32, dict(close_pair_radius=0.02 * r_cut)),
                             ("mixed", "poly", TOL_FP32, dict(close_pair_radius=0.02 * r_cut)),
                             ("fp32", "table", TOL_TABLE, dict(close_pair_radius=0.02 * r_cut, table_nodes=512, table_level=2))):
        out, _ = _run(B, cfg, pos, mass, precision=prec, g_mode=g, **kw)
        assert _err(out[tgt], ref) <= tol, (prec, g)


def test_mixed_precision_on_unrounded_positions(B, oracle):
    """Flavour D (genuine fp64 positions, A20): leaf-centre-relative fp32 is far closer to the oracle than
    absolute fp32; with the exact close-pair path (which reads the fp64 originals) it meets 1e-4."""
    cfg = workloads.scaled(4, 48)
    pos, mass = workloads.make(cfg, flavour="D")
    r_s, r_cut = _geom(cfg)
    tgt = workloads.sample_targets(cfg.n, 4000, cfg.seed)
    ref, _ = oracle.p2p_sampled(pos, mass, tgt, boxsize=cfg.boxsize, r_s=r_s, r_cut=r_cut)
    e = {}
    for prec in ("fp32", "mixed"):
        out, _ = _run(B, cfg, pos, mass, precision=prec, g_mode="poly", close_pair_radius=0.05 * r_cut)
        e[prec] = _err(out[tgt], ref)
    assert e["mixed"] < e["fp32"]
    assert e["mixed"] <= 1e-4
    out, _ = _run(B, cfg, pos, mass, precision="fp64", g_mode="direct")
    assert _err(out[tgt], ref) <= TOL_FP64


# ----------------------------------------------------------- full size, in bench.py's launch configuration

@pytest.mark.parametrize("cfg_id,n_targets", [(2, 2000), (3, 500)])
def test_full_size_configs_2_and_3_sampled(B, oracle, cfg_id, n_targets):
    """BASELINE configs 2 (128^3 clustered) and 3 (256^3 displaced grid) at full size in the headline launch
    configuration (fp32, poly g, bench.CLOSE_OVER_RCUT), sampled targets; config 3 also in fp64."""
    import bench
    import torch
    cfg = workloads.CONFIGS[cfg_id]
    pos, mass = workloads.make(cfg)
    r_s, r_cut = _geom(cfg)
    tgt = workloads.sample_targets(cfg.n, n_targets, cfg.seed)
    ref, cnt = oracle.p2p_sampled(pos, mass, tgt, boxsize=cfg.boxsize, r_s=r_s, r_cut=r_cut)
    if cfg_id == 3:   # homogeneous load: the closed-form neighbour count (4 pi / 3) 7.2^3 = 1563.5
        assert cnt["pairs_in_cut"] / len(tgt) == pytest.approx(1563.5, rel=0.02)
    dpos = torch.from_numpy(pos).cuda()
    out = torch.empty((cfg.n, 3), dtype=torch.float64, device="cuda")
    d_tgt = torch.from_numpy(tgt).cuda()
    runs = [(bench.headline_params(cfg), TOL_FP32), (bench.headline_params(cfg, precision="mixed"), TOL_FP32),
            (bench.headline_params(cfg, g_mode="table", table_nodes=512, table_level=2), TOL_TABLE)]
    if cfg_id == 3:
        runs.append((bench.headline_params(cfg, precision="fp64", g_mode="table", table_nodes=4096, table_level=3), TOL_FP64))
    for params, tol in runs:
        with B.Photons(**params) as ph:
            ph.set_particles(dpos, None)
            ph.build_leaves()
            st = ph.short_range_acc(out)
        assert _err(out[d_tgt].cpu().numpy(), ref) <= tol, params
        assert st["n_leaves"] == cfg.n // cfg.maxleaf


def test_full_size_config5_mixed_4_streams(B, oracle):
    """BASELINE config 5: N = 512^3 clustered, N_PM 512, MAXLEAF 32, mixed precision, leaf batches over 4 CUDA
    streams; oracle on sampled targets (128 here; bench-side studies use more)."""
    import bench
    import torch
    cfg = workloads.CONFIGS[5]
    pos, mass = workloads.make(cfg)
    r_s, r_cut = _geom(cfg)
    tgt = workloads.sample_targets(cfg.n, 128, cfg.seed)
    ref, _ = oracle.p2p_sampled(pos, mass, tgt, boxsize=cfg.boxsize, r_s=r_s, r_cut=r_cut)
    dpos = torch.from_numpy(pos.astype(np.float32)).cuda()       # flavour F: exact in fp32
    del pos
    out = torch.empty((cfg.n, 3), dtype=torch.float32, device="cuda")
    with B.Photons(**bench.headline_params(cfg, precision="mixed", n_streams=4)) as ph:
        ph.set_particles(dpos, None)
        ph.build_leaves()
        st = ph.short_range_acc(out)
    a = out[torch.from_numpy(tgt).cuda()].double().cpu().numpy()
    # an fp32 output array costs half an ulp of each acceleration on top of the arithmetic
    assert _err(a, ref) <= TOL_FP32
    assert st["n_leaves"] == cfg.n // 32 and bool(torch.isfinite(out).all())


def test_full_size_config4_sampled(B, oracle):
    """BASELINE config 4 (N = 256^3 clustered, MAXLEAF 32) exactly as bench.py times it (fp32, poly g,
    close pairs on, device-resident input), checked on sampled targets the oracle computes one by one."""
    import bench
    import torch
    cfg = workloads.CONFIGS[4]
    pos, mass = workloads.make(cfg)
    r_s, r_cut = _geom(cfg)
    tgt = workloads.sample_targets(cfg.n, 600, cfg.seed)
    ref, _ = oracle.p2p_sampled(pos, mass, tgt, boxsize=cfg.boxsize, r_s=r_s, r_cut=r_cut)
    params = bench.headline_params(cfg)
    dpos = torch.from_numpy(pos).cuda()
    out = torch.empty((cfg.n, 3), dtype=torch.float64, device="cuda")
    with B.Photons(**params) as ph:
        ph.set_particles(dpos, None)
        ph.build_leaves()
        st = ph.short_range_acc(out)
        a = out[torch.from_numpy(tgt).cuda()].cpu().numpy()
        assert _err(a, ref) <= TOL_FP32
        # properties that hold at any size: finite everywhere, Newton's third law to fp32 accuracy
        assert bool(torch.isfinite(out).all())
        tot = out.sum(dim=0).abs().max().item()
        scale = out.norm(dim=1).sum().item()
        assert tot / scale < 1e-6
        assert st["n_leaves"] == cfg.n // 32
        assert 4e3 < st["pairs_evaluated"] / cfg.n < 4e4
