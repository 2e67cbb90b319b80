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
@pytest.mark.parametrize("g_mode", ["direct", "fused", "poly"])
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
    for prec, g, tol in (("fp32", "poly", TOL_FP32), ("mixed", "table", TOL_TABLE), ("fp32", "direct", TOL_FP32),
                         ("mixed", "fused", TOL_FP32)):
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


@pytest.mark.parametrize("n,maxleaf", [(20011, 32), (5000, 16), (100003, 64)])
def test_pairs_evaluated_is_the_sum_over_the_list_with_ragged_leaves(B, n, maxleaf):
    """stats.pairs_evaluated (the numerator of the bench metric) against the list it describes, exactly: the sum over
    target leaves of (particles in the leaf) x (particles in its listed source leaves), with N chosen so that leaf
    counts differ (ORB halves odd nodes unevenly: DESIGN.md A13).  The list walk takes a leaf's count from the box
    record of its tree node."""
    rng = np.random.default_rng(91)
    pos = rng.random((n, 3)).astype(np.float32).astype(np.float64)
    with B.Photons(n_pm=32, maxleaf=maxleaf, precision="fp64", g_mode="direct") as ph:
        ph.set_particles(pos, np.full(n, 1.0 / n))
        ph.build_leaves()
        st = ph.stats()
        _, leaf_start = ph.leaf_order()
        ptr, first, nleaf, _ = ph.interaction_list()
    cnt = np.diff(leaf_start)
    assert cnt.min() < cnt.max() <= maxleaf            # ragged
    csum = np.concatenate([[0], np.cumsum(cnt)])
    src_per_entry = csum[first + nleaf] - csum[first]
    tl = np.repeat(np.arange(len(cnt)), np.diff(ptr))
    assert int((cnt[tl] * src_per_entry).sum()) == st["pairs_evaluated"]
    assert int(nleaf.sum()) == st["n_leaf_pairs"]


@pytest.mark.parametrize("n,maxleaf,clustered", [(32768, 32, False), (20011, 16, False), (5000, 64, False), (262144, 32, True),
                                                 (100003, 32, True), (262144, 16, True), (300007, 16, False)])
def test_orb_tree_is_a_median_split_along_the_widest_axis(B, n, maxleaf, clustered):
    """PAPER.md L35 / DESIGN.md A13, checked on the device-built tree itself: every node is cut along the widest axis of
    its particle bounding box (fp32 coordinates), the left child takes floor(size/2) particles and no particle of the
    left child lies beyond one of the right child (up to the 24-bit key quantum of the partition, ties either way).
    Covers both build phases: nodes above 4096 particles (global partition passes) and below (shared memory)."""
    rng = np.random.default_rng(77)
    if clustered:
        cen = rng.random((40, 3))
        pos = (cen[rng.integers(0, 40, n)] + 0.01 * rng.standard_normal((n, 3)) * rng.random((n, 1)) ** 3) % 1.0
        pos[: n // 5] = rng.random((n // 5, 3))
    else:
        pos = rng.random((n, 3))
    pos = pos.astype(np.float32).astype(np.float64)
    mass = np.full(n, 1.0 / n)
    with B.Photons(n_pm=32, maxleaf=maxleaf, precision="fp64", g_mode="direct") as ph:
        ph.set_particles(pos, mass)
        ph.build_leaves()
        perm, leaf_start = ph.leaf_order()
    assert np.array_equal(np.sort(perm), np.arange(n))
    n_leaves = len(leaf_start) - 1
    depth = int(np.log2(n_leaves))
    assert 1 << depth == n_leaves and np.diff(leaf_start).max() <= maxleaf
    x = pos[perm]
    for level in range(depth):
        step = n_leaves >> level
        bounds = leaf_start[::step]
        for k in range(1 << level):
            s0, s1 = int(bounds[k]), int(bounds[k + 1])
            mid = int(leaf_start[k * step + step // 2])
            assert mid - s0 == (s1 - s0) // 2
            node = x[s0:s1]
            ext = node.max(axis=0) - node.min(axis=0)
            axis = int(np.argmax(ext))              # ties -> lowest axis, as A13
            left, right = x[s0:mid, axis], x[mid:s1, axis]
            if len(left) and len(right):
                assert left.max() <= right.min() + ext[axis] * 2.0 ** -20, (level, k, axis)


def test_long_lists_take_the_second_walk_and_agree(B, c1):
    """Lists longer than the builder's stash (128 entries) are finished by a second walk that resumes where the first
    one ran out of stash.  With runs of a single leaf (chunk_max = maxleaf = 16) every list of config 1 is that long;
    the set of (target leaf, source leaf, image) triples must equal the one built with runs of 8 leaves."""
    cfg, pos, mass, _, _ = c1
    got = []
    for chunk_max in (16, 128):
        with B.Photons(n_pm=cfg.n_pm, maxleaf=16, chunk_max=chunk_max, precision="fp64", g_mode="direct") as ph:
            ph.set_particles(pos, mass)
            ph.build_leaves()
            st = ph.stats()
            ptr, first, nleaf, code = ph.interaction_list()
        tl = np.repeat(np.arange(len(ptr) - 1), np.diff(ptr))
        trip = np.concatenate([np.stack([np.full(k, t), np.arange(f, f + k), np.full(k, c)], axis=1)
                               for t, f, k, c in zip(tl, first, nleaf, code)])
        got.append((st, np.diff(ptr), trip[np.lexsort(trip.T[::-1])]))
    (st_a, len_a, trip_a), (st_b, len_b, trip_b) = got
    assert len_a.min() > 128 and len_b.max() <= 128          # the first build needed the second walk everywhere
    assert (nleaf_ok := st_a["n_leaf_pairs"]) == st_b["n_leaf_pairs"] == len(trip_a) == len(trip_b)
    assert np.array_equal(trip_a, trip_b)
    assert st_a["pairs_evaluated"] == st_b["pairs_evaluated"]


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
    for prec, g in (("fp64", "direct"), ("fp64", "table"), ("fp32", "direct"), ("fp32", "fused"), ("fp32", "poly"), ("fp32", "table"),
                    ("mixed", "poly")):
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


@pytest.mark.parametrize("n,maxleaf", [(40, 32), (33, 16), (1000, 32), (5000, 64), (20011, 16), (20011, 32), (20011, 128)])
@pytest.mark.parametrize("g_mode,tol", [("poly", TOL_FP32), ("fused", TOL_FP32), ("table", TOL_TABLE)])
def test_equal_mass_kernels(B, oracle, n, maxleaf, g_mode, tol):
    """photons_params.mass_path: with every mass equal (Alg. 2 L177 carries one GM) the fp32 kernels leave G m out of the
    pair core and apply it once per staged run.  Ragged N, so that padding slots (which these kernels cannot silence by a
    zero mass) are in every leaf; a G m that is not a power of two; against the oracle and against the per-pair path."""
    rng = np.random.default_rng(500 + n)
    pos = rng.random((n, 3)).astype(np.float32).astype(np.float64)
    m0, G = 7.5 / n, 43.0
    mass = np.full(n, m0)
    n_pm = 16
    r_s = 1.2 / n_pm
    ref, _ = oracle.p2p(pos, mass, boxsize=1.0, r_s=r_s, r_cut=6 * r_s, G=G)
    kw = dict(n_pm=n_pm, G=G, precision="fp32", g_mode=g_mode, maxleaf=maxleaf, close_pair_radius=0.02 * 6 * r_s)
    eq, st = B.short_range_acc(pos, mass, **kw)
    per, _ = B.short_range_acc(pos, mass, mass_path=1, **kw)
    none, _ = B.short_range_acc(pos * 1.0, None, **{**kw, "G": G * m0 * n})       # mass = NULL is 1/n each
    assert _err(eq, ref) <= tol and _err(per, ref) <= tol and _err(none, ref) <= tol
    assert _err(eq, per) <= 0.5 * TOL_FP32                             # two kernels, the same sum up to fp32 rounding
    assert n < 1000 or not np.array_equal(eq, per)
    # one particle of another mass: set_particles must notice and take the per-pair kernels
    mass2 = mass.copy()
    mass2[n // 2] *= 3.0
    ref2, _ = oracle.p2p(pos, mass2, boxsize=1.0, r_s=r_s, r_cut=6 * r_s, G=G)
    out2, _ = B.short_range_acc(pos, mass2, **kw)
    assert _err(out2, ref2) <= tol


@pytest.mark.parametrize("n,maxleaf", [(33, 16), (40, 32), (5000, 64), (20011, 32), (20011, 16)])
@pytest.mark.parametrize("g_mode,tol", [("poly", TOL_FP32), ("table", TOL_TABLE)])
def test_equal_mass_kernels_mixed(B, oracle, n, maxleaf, g_mode, tol):
    """The same for precision = mixed (offsets from the leaf origins): padding slots sit at PAD_FAR there too, and the
    tiny cases take the per-pair minimum image, which wraps offsets by whole box lengths and must leave them far."""
    rng = np.random.default_rng(700 + n)
    pos = rng.random((n, 3)).astype(np.float32).astype(np.float64)
    m0, G = 7.5 / n, 43.0
    mass = np.full(n, m0)
    n_pm = 16
    r_s = 1.2 / n_pm
    ref, _ = oracle.p2p(pos, mass, boxsize=1.0, r_s=r_s, r_cut=6 * r_s, G=G)
    kw = dict(n_pm=n_pm, G=G, precision="mixed", g_mode=g_mode, maxleaf=maxleaf, close_pair_radius=0.02 * 6 * r_s)
    eq, _ = B.short_range_acc(pos, mass, **kw)
    per, _ = B.short_range_acc(pos, mass, mass_path=1, **kw)
    assert _err(eq, ref) <= tol and _err(per, ref) <= tol
    assert _err(eq, per) <= 0.5 * TOL_FP32
    assert n < 1000 or not np.array_equal(eq, per)


def test_equal_mass_kernels_softened_isolated_and_negative(B, oracle):
    rng = np.random.default_rng(91)
    n, n_pm = 6001, 16
    r_s = 1.2 / n_pm
    r_cut = 6 * r_s
    pos = rng.random((n, 3)).astype(np.float32).astype(np.float64)
    mass = np.full(n, 1.0 / n)
    kw = dict(n_pm=n_pm, precision="fp32", g_mode="poly", close_pair_radius=0.02 * r_cut)
    ref, _ = oracle.p2p(pos, mass, boxsize=1.0, r_s=r_s, r_cut=r_cut, eps=0.01 * r_cut)
    out, _ = B.short_range_acc(pos, mass, softening=0.01 * r_cut, **kw)
    assert _err(out, ref) <= TOL_FP32
    # isolated boundaries: a blob that straddles the origin (as test_isolated_boundaries, with one mass)
    blob = (rng.normal(0.0, 0.35, (n, 3)) + np.array([0.1, 0.9, -0.2])).astype(np.float32).astype(np.float64)
    ref, _ = oracle.p2p(blob, mass, boxsize=0.0, r_s=1.2 / 32, r_cut=6 * 1.2 / 32)
    out, _ = B.short_range_acc(blob, mass, periodic=0, **{**kw, "n_pm": 32, "close_pair_radius": 0.02 * 6 * 1.2 / 32})
    assert _err(out, ref) <= TOL_FP32
    ref, _ = oracle.p2p(pos, -mass, boxsize=1.0, r_s=r_s, r_cut=r_cut)          # equal negative masses: the sign is kept
    out, _ = B.short_range_acc(pos, -mass, **kw)
    assert _err(out, ref) <= TOL_FP32


@pytest.mark.parametrize("maxleaf,tpl", [(16, 1), (16, 2), (32, 1), (32, 2), (64, 2), (128, 4)])
def test_c1_per_pair_mass_path(B, c1, maxleaf, tpl):
    # config 1 has equal masses, so every other config-1 test runs the equal-mass kernels: the per-pair ones here
    cfg, pos, mass, ref, _ = c1
    for g, tol in (("poly", TOL_FP32), ("fused", TOL_FP32), ("table", TOL_TABLE)):
        out, _ = _run(B, cfg, pos, mass, precision="fp32", g_mode=g, maxleaf=maxleaf, targets_per_lane=tpl, mass_path=1,
                      close_pair_radius=_close(cfg))
        assert _err(out, ref) <= tol


# ---------------------------------------------------------------------------- error behaviour (ABI)

def test_abi_errors(B):
    import ctypes
    with pytest.raises(B.PhotonsError) as e:
        B.Photons(n_pm=8)                      # r_cut = 0.9 >= boxsize/2
    assert e.value.code == B.EBOX
    for bad in (dict(maxleaf=48), dict(precision=7), dict(g_mode=9), dict(n_streams=0), dict(boxsize=-1.0),
                dict(precision="fp64", g_mode="poly"), dict(g_mode="table", table_nodes=5),
                dict(g_mode="poly", rcut_over_rs=7.0), dict(mass_path=2)):
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


# ------------------------------------------ units, mass ratios, softening, fp64 table layouts (test sizes)

def _two_population_masses(n, seed, ratio=1e3):
    rng = np.random.default_rng(seed)
    m = np.where(rng.random(n) < 0.05, ratio, 1.0)
    return m / m.sum()


@pytest.mark.parametrize("boxsize,G,unit_mass", [(1e-3, 43.0, False), (100.0, 43.0, False), (1.0, 43007.0, True),
                                                  (3.0e5, 6.674e-8, False)])
def test_units_box_G_and_mass_ratio(B, oracle, boxsize, G, unit_mass):
    """The fp32 / mixed kernels must not depend on the caller's units:
    box lengths that fp32 does not hold exactly (1e-3: the image shift is a two-float sum), Gadget-like G m >> 1
    (w = G m / r^3 overflowed fp32 at the self pair before the kernels normalised their units), a 10^3 mass ratio."""
    cfg = workloads.scaled(4, 40)
    pos1, _ = workloads.make(cfg)
    pos = (pos1 * boxsize).astype(np.float32).astype(np.float64)       # flavour F in the new units
    pos[pos >= np.float32(boxsize)] = 0.0
    n = cfg.n
    mass = np.ones(n) if unit_mass else _two_population_masses(n, 11) * 7.5
    r_s = 1.2 * boxsize / cfg.n_pm
    r_cut = 6 * r_s
    tgt = workloads.sample_targets(n, 4000, cfg.seed)
    ref, _ = oracle.p2p_sampled(pos, mass, tgt, boxsize=boxsize, r_s=r_s, r_cut=r_cut, G=G)
    assert np.isfinite(ref).all()
    for prec, g, tol, kw in (("fp64", "direct", TOL_FP64, {}),
                             ("fp64", "table", TOL_FP64, dict(table_nodes=4096, table_level=3)),
                             ("fp32", "direct", TOL_FP32, dict(close_pair_radius=0.02 * r_cut)),
                             ("fp32", "poly", TOL_FP32, dict(close_pair_radius=0.02 * r_cut)),
                             ("fp32", "fused", TOL_FP32, dict(close_pair_radius=0.02 * r_cut)),
                             ("fp32", "poly", TOL_FP32, dict(close_pair_radius=0.02 * r_cut, maxleaf=16)),
                             ("mixed", "poly", TOL_FP32, dict(close_pair_radius=0.02 * r_cut)),
                             ("mixed", "table", TOL_TABLE, dict(close_pair_radius=0.02 * r_cut)),
                             ("fp32", "table", TOL_TABLE, dict(close_pair_radius=0.02 * r_cut, table_nodes=512, table_level=2)),
                             ("fp32", "poly", 1e-4, {})):            # no exact close-pair path: still finite and close
        out, _ = B.short_range_acc(pos, mass, boxsize=boxsize, n_pm=cfg.n_pm, G=G, precision=prec, g_mode=g,
                                   **{"maxleaf": cfg.maxleaf, **kw})
        assert np.isfinite(out).all(), (prec, g, kw)
        assert _err(out[tgt], ref) <= tol, (prec, g, kw)


@pytest.mark.parametrize("eps_over_rcut", [1e-3, 3.56e-3, 0.02, 0.2])
def test_softened_parity(B, oracle, c1, eps_over_rcut):
    """Plummer-softened variant (A23) against the oracle's softened mode: config 1 (full
    O(N^2)) and config 4 at test size (sampled), every precision and g mode.  3.56e-3 r_cut is the paper's own ratio
    (100 kpc/h softening in a 1 Gpc/h box with N_PM = 256: r_cut = 6 * 1.2 * 1000/256 = 28.1 Mpc/h).
    eps = 0.2 r_cut is far outside that: on the uniform load the softened sum is cancellation-dominated
    (sum |a_ij| >> |a_i|), the fp32 pair arithmetic alone then sits at 1.1e-5 rms, and there is nothing left inside
    the softening core for the exact close-pair path to redo; the fp32 variants are held to 3e-5 there."""
    cfg, pos, mass, _, _ = c1
    f32 = 3.0 if eps_over_rcut > 0.1 else 1.0
    r_s, r_cut = _geom(cfg)
    eps = eps_over_rcut * r_cut
    ref, _ = oracle.p2p(pos, mass, boxsize=cfg.boxsize, r_s=r_s, r_cut=r_cut, G=cfg.G, eps=eps)
    runs = (("fp64", "direct", TOL_FP64, {}), ("fp64", "table", TOL_FP64, dict(table_nodes=4096, table_level=3)),
            ("fp64", "table", TOL_FP64, dict(table_nodes=4096, table_level=3, table_layout="coef")),
            ("fp32", "direct", f32 * TOL_FP32, dict(close_pair_radius=_close(cfg))),
            ("fp32", "poly", f32 * TOL_FP32, dict(close_pair_radius=_close(cfg))),
            ("fp32", "fused", f32 * TOL_FP32, dict(close_pair_radius=_close(cfg))),
            ("mixed", "poly", f32 * TOL_FP32, dict(close_pair_radius=_close(cfg))),
            ("fp32", "table", TOL_TABLE, dict(close_pair_radius=_close(cfg))),
            ("fp32", "poly", f32 * TOL_FP32, dict(close_pair_radius=_close(cfg), maxleaf=64)))
    for prec, g, tol, kw in runs:
        out, _ = _run(B, cfg, pos, mass, precision=prec, g_mode=g, softening=eps, **kw)
        assert _err(out, ref) <= tol, (prec, g, kw)
    cfg4 = workloads.scaled(4, 48)
    pos4, mass4 = workloads.make(cfg4)
    r_s4, r_cut4 = _geom(cfg4)
    tgt = workloads.sample_targets(cfg4.n, 3000, cfg4.seed)
    ref4, _ = oracle.p2p_sampled(pos4, mass4, tgt, boxsize=1.0, r_s=r_s4, r_cut=r_cut4, eps=eps_over_rcut * r_cut4)
    for prec, g, tol, kw in runs:
        kw = {k: (0.02 * r_cut4 if k == "close_pair_radius" else v) for k, v in kw.items()}
        out, _ = _run(B, cfg4, pos4, mass4, precision=prec, g_mode=g, softening=eps_over_rcut * r_cut4, **kw)
        assert _err(out[tgt], ref4) <= tol, (prec, g, kw)


@pytest.mark.parametrize("precision,g_mode", [("fp32", "direct"), ("fp32", "poly"), ("mixed", "poly")])
def test_per_pair_image_keeps_close_pairs_across_a_box_face(B, oracle, precision, g_mode):
    """Tiny N (16^3, r_cut = 0.45 L): every list entry takes the minimum image per pair.  With softening the exact path
    does not trigger, so the fp32 image arithmetic itself is on test: the shift must go to an operand it is exact for,
    or a close pair across a box face loses its separation to one ulp of the box length (1.2e-5 rms before the fix)."""
    cfg = workloads.scaled(1, 16)
    pos, mass = workloads.make(cfg)
    r_s, r_cut = _geom(cfg)
    eps = 0.01 * r_cut
    ref, _ = oracle.p2p(pos, mass, boxsize=cfg.boxsize, r_s=r_s, r_cut=r_cut, G=cfg.G, eps=eps)
    out, st = _run(B, cfg, pos, mass, precision=precision, g_mode=g_mode, softening=eps, close_pair_radius=0.0)
    assert _err(out, ref) <= 0.5 * TOL_FP32


def test_softening_changes_the_answer_and_zero_is_bitwise_off(B, c1):
    cfg, pos, mass, ref, _ = c1
    r_s, r_cut = _geom(cfg)
    for prec, g in (("fp64", "direct"), ("fp32", "poly")):
        a, _ = _run(B, cfg, pos, mass, precision=prec, g_mode=g)
        b, _ = _run(B, cfg, pos, mass, precision=prec, g_mode=g, softening=0.0)
        c, _ = _run(B, cfg, pos, mass, precision=prec, g_mode=g, softening=0.05 * r_cut)
        assert np.array_equal(a, b)
        assert _err(c, ref) > 1e-3
    with pytest.raises(B.PhotonsError):
        B.Photons(n_pm=cfg.n_pm, softening=-1.0)
    with pytest.raises(B.PhotonsError):
        B.Photons(n_pm=cfg.n_pm, softening=2 * r_cut)


@pytest.mark.parametrize("maxleaf", [16, 32, 64, 128])
@pytest.mark.parametrize("layout,nodes,level,tol", [("paper", 512, 4, 1e-10), ("coef", 512, 4, 1e-10), ("paper", 4096, 3, TOL_FP64),
                                                   ("coef", 4096, 3, TOL_FP64), ("coef", 4096, 4, TOL_FP64),
                                                   ("coef", 256, 2, TOL_TABLE), ("paper", 256, 1, TOL_TABLE), ("coef", 1024, 0, 1e-3),
                                                   ("quad", 512, 4, 1e-10), ("quad", 4096, 3, TOL_FP64), ("quad", 256, 2, TOL_TABLE),
                                                   ("quad", 256, 0, 1e-2)])
def test_c1_fp64_table_layouts(B, c1, maxleaf, layout, nodes, level, tol):
    # Eq. 2 in fp64, all three table layouts: the same Taylor series about the same node.  512 nodes / T[4]
    # ("T[4] for double") carries the table's own truncation error, ~5e-12 in T (SURVEY §8(c) "table")
    cfg, pos, mass, ref, _ = c1
    out, _ = _run(B, cfg, pos, mass, precision="fp64", g_mode="table", table_nodes=nodes, table_level=level,
                  table_layout=layout, maxleaf=maxleaf)
    assert _err(out, ref) <= tol
    with pytest.raises(B.PhotonsError):
        B.Photons(n_pm=cfg.n_pm, precision="fp32", g_mode="table", table_layout="coef")
    with pytest.raises(B.PhotonsError):
        B.Photons(n_pm=cfg.n_pm, precision="fp32", g_mode="table", table_level=4)


# ----------------------------------------------------------- full size, in bench.py's launch configuration
# The oracle's accelerations of 10^4 seeded targets per config (north_star: "oracle on 10^4 sampled targets") come
# from tests/golden/c{2,3,4,5}_acc_10k.npz, written by tests/golden/make_golden.py (oracle + workloads only).

T3 = 4.39849652838829e-4        # T(3): the jump of g at r_cut (A1, A9; pinned in test_oracle_pins.py)


def _golden(cfg_id, pos):
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", f"c{cfg_id}_acc_10k.npz")
    g = np.load(path)
    cfg = workloads.CONFIGS[cfg_id]
    tgt = g["targets"]
    assert len(tgt) == 10_000 and int(g["n"]) == cfg.n and int(g["seed"]) == cfg.seed
    assert np.array_equal(tgt, workloads.sample_targets(cfg.n, 10_000, cfg.seed))
    assert np.array_equal(g["pos_tgt"], pos[tgt])          # the generator still makes the golden's input
    return tgt, g["acc"], g


def _cut_flip_report(pos, tgt, a, ref, cfg, label, top=8):
    """A9: pairs within rounding of r_cut may fall on either side of the cut; each flip moves one target by the jump
    quantum q = T(3) G m / r_cut^2.  For the `top` largest errors, look for a source within 2e-7 r_cut of the cut whose
    flip explains the error vector, and report how many there are (not silently allowed: printed, and the literal
    criterion is asserted by the caller on ALL targets, flips included)."""
    r_s, r_cut = _geom(cfg)
    q = T3 * cfg.G * (1.0 / cfg.n) / r_cut ** 2
    err = a - ref
    mag = np.sqrt((err ** 2).sum(axis=1))
    rms = np.sqrt((ref ** 2).sum(axis=1).mean())
    near_q = int(((mag > 0.7 * q) & (mag < 1.3 * q)).sum())
    explained = 0
    for k in np.argsort(-mag)[:top]:
        if not 0.5 * q < mag[k] < 2.5 * q:
            continue
        d = pos - pos[tgt[k]]
        d -= cfg.boxsize * np.rint(d / cfg.boxsize)
        r = np.sqrt((d * d).sum(axis=1))
        cand = np.nonzero(np.abs(r - r_cut) < 2e-7 * r_cut)[0]
        for j in cand:
            jump = q * d[j] / r[j]
            if min(np.linalg.norm(err[k] - jump), np.linalg.norm(err[k] + jump)) < 0.3 * q:
                explained += 1
                break
    print(f"[A9] {label}: jump quantum q = {q / rms:.2e} rms; targets with |err| in [0.7, 1.3] q: {near_q} of {len(tgt)}; "
          f"of the {top} largest errors, explained by one flipped pair at the cut: {explained}; max err {mag.max() / rms:.2e} rms")
    return near_q, explained


@pytest.mark.parametrize("cfg_id", [2, 3])
def test_full_size_configs_2_and_3_golden_10k(B, cfg_id):
    """BASELINE configs 2 (128^3 clustered) and 3 (256^3 displaced grid) at full size in the headline launch
    configuration (fp32, poly g, bench.CLOSE_OVER_RCUT) and the other variants, on the golden's 10^4 targets."""
    import bench
    import torch
    cfg = workloads.CONFIGS[cfg_id]
    pos, mass = workloads.make(cfg)
    tgt, ref, g = _golden(cfg_id, pos)
    if cfg_id == 3:   # homogeneous load: the closed-form neighbour count (4 pi / 3) 7.2^3 = 1563.5
        assert int(g["pairs_in_cut"]) / len(tgt) == pytest.approx(1563.5, rel=0.01)
    dpos = torch.from_numpy(pos).cuda()
    out = torch.empty((cfg.n, 3), dtype=torch.float64, device="cuda")
    d_tgt = torch.from_numpy(tgt).cuda()
    runs = [(bench.headline_params(cfg), TOL_FP32), (bench.headline_params(cfg, precision="mixed"), TOL_FP32),
            (bench.headline_params(cfg, g_mode="direct"), TOL_FP32), (bench.headline_params(cfg, g_mode="fused"), TOL_FP32),
            (bench.headline_params(cfg, g_mode="table", table_nodes=512, table_level=2), TOL_TABLE)]
    if cfg_id == 3:
        runs.append((bench.headline_params(cfg, precision="fp64", g_mode="table", table_nodes=4096, table_level=3), TOL_FP64))
    else:
        runs.append((bench.headline_params(cfg, precision="fp64", g_mode="direct"), TOL_FP64))
    for params, tol in runs:
        with B.Photons(**params) as ph:
            ph.set_particles(dpos, None)
            ph.build_leaves()
            st = ph.short_range_acc(out)
        a = out[d_tgt].cpu().numpy()
        _cut_flip_report(pos, tgt, a, ref, cfg, f"config {cfg_id} {params['precision']}/{params['g_mode']}")
        assert _err(a, ref) <= tol, params
        assert st["n_leaves"] == cfg.n // cfg.maxleaf


def test_full_size_config5_mixed_4_streams_golden_10k(B):
    """BASELINE config 5: N = 512^3 clustered, N_PM 512, MAXLEAF 32, mixed precision, leaf batches over 4 CUDA
    streams; oracle on 10^4 sampled targets (golden)."""
    import bench
    import torch
    cfg = workloads.CONFIGS[5]
    pos, mass = workloads.make(cfg)
    tgt, ref, _ = _golden(5, pos)
    dpos = torch.from_numpy(pos.astype(np.float32)).cuda()       # flavour F: exact in fp32
    out = torch.empty((cfg.n, 3), dtype=torch.float64, device="cuda")
    with B.Photons(**bench.headline_params(cfg, precision="mixed", n_streams=4)) as ph:
        ph.set_particles(dpos, None)
        ph.build_leaves()
        st = ph.short_range_acc(out)
    a = out[torch.from_numpy(tgt).cuda()].cpu().numpy()
    _cut_flip_report(pos, tgt, a, ref, cfg, "config 5 mixed/poly, 4 streams", top=4)
    assert _err(a, ref) <= TOL_FP32
    assert st["n_leaves"] == cfg.n // 32 and bool(torch.isfinite(out).all())


def test_full_size_config4_golden_10k(B):
    """BASELINE config 4 (N = 256^3 clustered, MAXLEAF 32) exactly as bench.py times it (fp32, poly g, device-resident
    input), and north_star's two named variants (direct special functions, interpolation table) plus mixed and fp64,
    on the golden's 10^4 targets."""
    import bench
    import torch
    cfg = workloads.CONFIGS[4]
    pos, mass = workloads.make(cfg)
    tgt, ref, _ = _golden(4, pos)
    dpos = torch.from_numpy(pos).cuda()
    out = torch.empty((cfg.n, 3), dtype=torch.float64, device="cuda")
    d_tgt = torch.from_numpy(tgt).cuda()
    runs = [(bench.headline_params(cfg), TOL_FP32), (bench.headline_params(cfg, g_mode="direct"), TOL_FP32),
            (bench.headline_params(cfg, g_mode="fused"), TOL_FP32),
            (bench.headline_params(cfg, g_mode="table", table_nodes=512, table_level=2), TOL_TABLE),
            (bench.headline_params(cfg, precision="mixed"), TOL_FP32), (bench.headline_params(cfg, maxleaf=16), TOL_FP32),
            (bench.headline_params(cfg, mass_path=1), TOL_FP32),       # G m_j per pair (the equal-mass kernels are the default here)
            (bench.headline_params(cfg, precision="fp64", g_mode="table", table_nodes=4096, table_level=3), TOL_FP64)]
    for i, (params, tol) in enumerate(runs):
        with B.Photons(**params) as ph:
            ph.set_particles(dpos, None)
            ph.build_leaves()
            st = ph.short_range_acc(out)
            a = out[d_tgt].cpu().numpy()
            _cut_flip_report(pos, tgt, a, ref, cfg, f"config 4 {params['precision']}/{params['g_mode']}/maxleaf {params['maxleaf']}")
            assert _err(a, ref) <= tol, params
            if i == 0:
                # properties that hold at any size: finite everywhere, Newton's third law to fp32 accuracy
                assert bool(torch.isfinite(out).all())
                tot = out.sum(dim=0).abs().max().item()
                scale = out.norm(dim=1).sum().item()
                assert tot / scale < 1e-6
                assert st["n_leaves"] == cfg.n // 32
                assert 4e3 < st["pairs_evaluated"] / cfg.n < 4e4
