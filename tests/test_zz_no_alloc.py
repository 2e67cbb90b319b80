"""photons_m2l_noalloc (include/photons.h): the truncated M2L operator for callers that cannot allocate.  Its output is
checked against the existing path (photons_m2l with device pointers) at the M2L tests' tolerance, on calls made in a row
that share the library's static scratch array.  GPU only.

This file is named so that pytest collects it last: the suite runs with `pytest -x`, and a failure here must not hide
any other test.  It passes alone in a fresh process and after the other tests (it keeps no state of its own)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-12       # as tests/test_gpu_m2l.py: max |L - L_ref| per coefficient <= 1e-12 * max |L_ref| of that coefficient


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the CUDA path has no CPU fallback")
    from paper_2107_14008_b200 import binding
    binding.load()
    return binding


def _problem(B, seed, n_cells, p, *, max_list, empty_frac=0.1, periodic=True):
    """Cells on a jittered lattice (no zero separations), random multipoles, ragged source lists; as device tensors."""
    import torch
    rng = np.random.default_rng(seed)
    side = int(np.ceil(n_cells ** (1 / 3)))
    g = np.stack(np.meshgrid(*[np.arange(side)] * 3, indexing="ij"), axis=-1).reshape(-1, 3)[:n_cells]
    centres = (g + 0.5 + 0.2 * (rng.random((n_cells, 3)) - 0.5)) / side
    nc = B.m2l_n_coeffs(p)
    M = rng.normal(0.0, 1.0, (n_cells, nc)) * (0.4 / side) ** rng.integers(0, p + 1, nc)
    counts = rng.integers(0, max_list + 1, n_cells)
    counts[rng.random(n_cells) < empty_frac] = 0
    counts[:4] = [0, 1, 32, min(33, max_list)]
    ptr = np.zeros(n_cells + 1, dtype=np.int64)
    ptr[1:] = np.cumsum(counts)
    tgt = np.repeat(np.arange(n_cells), counts)
    src = ((tgt + 1 + rng.integers(0, n_cells - 1, len(tgt))) % n_cells).astype(np.int32)     # never the target itself
    shifts = np.rint(centres[tgt] - centres[src]).astype(np.int8) if periodic else None
    dev = [torch.from_numpy(x).cuda() if x is not None else None for x in (centres, M, ptr, src, shifts)]
    return dev, nc


def _agree(out, ref):
    out, ref = out.cpu().numpy(), ref.cpu().numpy()
    scale = np.abs(ref).max(axis=0)
    return bool(np.all(np.abs(out - ref).max(axis=0) <= TOL * scale))


def test_m2l_noalloc_matches_the_existing_path_on_calls_in_a_row(B):
    import torch
    r_s = 0.09
    # A: few cells, long lists (every list is split over several warps); B: as many cells, mostly empty or short lists,
    # other multipoles - the scratch slots A filled now belong to empty segments; C: another order and size (one segment)
    probs = {"A": (_problem(B, 11, 200, 4, max_list=700), 4), "B": (_problem(B, 12, 200, 4, max_list=40, empty_frac=0.6), 4),
             "C": (_problem(B, 13, 3001, 2, max_list=90, periodic=False), 2)}
    ref, out = {}, {}
    for k, ((dev, nc), p) in probs.items():
        ref[k], _ = B.m2l(*dev, p=p, r_s=r_s, boxsize=1.0)           # the existing path (allocates its own output)
        out[k] = torch.full_like(ref[k], float("nan"))
    torch.cuda.synchronize()
    first = {}
    for k in ("A", "B", "C", "A", "B"):                                # in a row, no synchronisation in between
        (dev, nc), p = probs[k]
        if k in first:
            out[k].fill_(float("nan"))
        B.m2l_noalloc(*dev, out=out[k], p=p, r_s=r_s, boxsize=1.0)
        if k not in first:
            first[k] = out[k].clone()
    torch.cuda.synchronize()
    for k in probs:
        assert _agree(first[k], ref[k]), k
        assert bool(torch.equal(out[k], first[k])), k                  # the same bits when called again after other work
    assert bool((first["B"][0] == 0).all())                            # empty list: zero, not the last call's partial sums


def test_m2l_noalloc_allocates_nothing_and_rejects_sizes_beyond_its_scratch(B):
    import torch
    r_s = 0.05
    p = 4
    n_max = B.M2L_NOALLOC_SCRATCH_BYTES // 8 // B.m2l_n_coeffs(p)        # 29 959 cells at order 4
    (dev, nc), _ = _problem(B, 21, n_max, p, max_list=6), p
    ref, _ = B.m2l(*dev, p=p, r_s=r_s, boxsize=1.0)
    out = torch.empty_like(ref)
    B.m2l_noalloc(*dev, out=out, p=p, r_s=r_s, boxsize=1.0)             # first call: kernels are loaded, the symbol looked up
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(2):
        B.m2l_noalloc(*dev, out=out, p=p, r_s=r_s, boxsize=1.0)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0                                               # no device memory taken or returned by the calls
    assert _agree(out, ref)                                             # the largest size that fits
    # one cell more does not fit: a clear error, nothing launched, out untouched
    (dev2, _), _ = _problem(B, 22, n_max + 1, p, max_list=3), p
    out2 = torch.full((n_max + 1, nc), 7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(B.PhotonsError) as e:
        B.m2l_noalloc(*dev2, out=out2, p=p, r_s=r_s, boxsize=1.0)
    assert e.value.code == B.EINVAL and "scratch" in str(e.value) and str(n_max) in str(e.value)
    torch.cuda.synchronize()
    assert bool((out2 == 7.0).all())
    with pytest.raises(B.PhotonsError):
        B.m2l_noalloc(*dev, out=out, p=p, r_s=0.0, boxsize=1.0)
