"""Parity of the CUDA truncated-M2L kernel (photons_m2l, through the C ABI) against the CPU oracle (oracle/m2l.py):
element by element on the same seeded inputs.  GPU only."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-12       # fp64: max |L_gpu - L_ref| per coefficient <= 1e-12 * max |L_ref| of that coefficient


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the CUDA path has no CPU fallback")
    from paper_2107_14008_b200 import binding
    binding.load()
    return binding


def _cells(seed, n_cells, p, *, max_list=90, periodic=False):
    """Cells on a jittered lattice (well separated: no zero separations), random multipoles with the magnitudes of a
    cell of extent ~0.4 spacing, ragged source lists (empty, one, many; several multiples of the warp size)."""
    rng = np.random.default_rng(seed)
    side = int(np.ceil(n_cells ** (1 / 3)))
    g = np.stack(np.meshgrid(*[np.arange(side)] * 3, indexing="ij"), axis=-1).reshape(-1, 3)[:n_cells]
    centres = (g + 0.5 + 0.2 * (rng.random((n_cells, 3)) - 0.5)) / side
    from oracle import m2l as om
    nc = om.n_coeffs(p)
    ext = 0.4 / side
    M = np.empty((n_cells, nc))
    for c, n in enumerate(om.multi_indices(p)):
        M[:, c] = rng.normal(0.0, 1.0, n_cells) * ext ** sum(n)
    counts = rng.integers(0, max_list, n_cells)
    counts[rng.integers(0, n_cells, n_cells // 10)] = 0
    counts[:4] = [0, 1, 32, 33]
    ptr = np.zeros(n_cells + 1, dtype=np.int64)
    ptr[1:] = np.cumsum(counts)
    src = np.empty(ptr[-1], dtype=np.int32)
    tgt = np.repeat(np.arange(n_cells), counts)
    src[:] = (tgt + 1 + rng.integers(0, n_cells - 1, len(tgt))) % n_cells        # never the target itself
    shifts = None
    if periodic:
        d = centres[tgt] - centres[src]
        shifts = np.rint(d).astype(np.int8)            # minimum image: move the source by s box lengths
    return centres, M, ptr, src, tgt, shifts


@pytest.mark.parametrize("p", [0, 1, 2, 3, 4])
@pytest.mark.parametrize("periodic", [False, True])
def test_m2l_parity(B, p, periodic):
    from oracle import m2l as om
    n_cells = 3001
    r_s = 0.09
    centres, M, ptr, src, tgt, shifts = _cells(40 + p, n_cells, p, periodic=periodic)
    ref = om.m2l(centres, M, np.stack([tgt, src], axis=1), p, r_s, boxsize=1.0, shifts=shifts)
    out, ms = B.m2l(centres, M, ptr, src, shifts, p=p, r_s=r_s, boxsize=1.0)
    scale = np.abs(ref).max(axis=0)
    assert np.all(np.abs(out - ref).max(axis=0) <= TOL * scale)
    assert np.all(out[0] == 0.0)                      # empty list: zero, not garbage
    assert ms > 0


def test_m2l_device_pointers_and_end_to_end(B):
    """Device-resident arrays through the same call, and the chain P2M (oracle) -> M2L (GPU) -> L2P (oracle) against the
    direct sum over particles: what the operator is for."""
    import math
    import torch
    from oracle import m2l as om
    p, r_s = 4, 0.3
    rng = np.random.default_rng(9)
    zA, zB = np.array([0.2, 0.3, 0.25]), np.array([0.62, 0.05, 0.61])
    ya = zA + 0.08 * (rng.random((50, 3)) - 0.5)
    ma = rng.uniform(0.5, 1.5, 50)
    xb = zB + 0.08 * (rng.random((20, 3)) - 0.5)
    M = np.stack([om.p2m(ya, ma, zA, p), np.zeros(om.n_coeffs(p))])
    centres = np.stack([zA, zB])
    ptr = np.array([0, 0, 1], dtype=np.int64)
    src = np.array([0], dtype=np.int32)
    out, _ = B.m2l(torch.from_numpy(centres).cuda(), torch.from_numpy(M).cuda(), torch.from_numpy(ptr).cuda(),
                   torch.from_numpy(src).cuda(), None, p=p, r_s=r_s)
    L = out.cpu().numpy()
    assert np.array_equal(L, B.m2l(centres, M, ptr, src, None, p=p, r_s=r_s)[0])      # host path: same bits
    phi, acc = om.l2p(L[1], zB, xb, p)
    ref = np.zeros((20, 3))
    for i, xv in enumerate(xb):
        d = ya - xv
        r = np.sqrt((d * d).sum(axis=1))
        u = r / (2 * r_s)
        T = np.array([math.erfc(v) for v in u]) + 2 * u / math.sqrt(math.pi) * np.exp(-u * u)
        ref[i] = ((ma * T / r ** 3)[:, None] * d).sum(axis=0)
    assert np.abs(acc - ref).max() <= 2e-3 * np.abs(ref).max()       # truncation error of the acceleration at order p = 4, size/sep ~ 0.13
