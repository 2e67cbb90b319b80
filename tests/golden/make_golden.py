#!/usr/bin/env python
"""Writes tests/golden/c{2,3,4,5}_acc_10k.npz: the CPU oracle's accelerations of 10^4 seeded targets of BASELINE
configs 2-5 at FULL size (north_star: "oracle on 10^4 sampled targets"; PAPER.md L202 is the paper's own
"fiducial direct P2P" check).  The full-size GPU parity tests load these files instead of running the oracle
inline on a few hundred targets.

    python tests/golden/make_golden.py [2 3 4 5]          # from the repo root; config 5 is ~1.3e12 pair tests

Imports ONLY ``oracle`` and ``paper_2107_14008_b200.workloads`` (the seeded input generators, which hold none
of the method's arithmetic).  Nothing here comes from the CUDA path.

Each file holds
    targets   int64[10^4]     workloads.sample_targets(N, 10^4, seed)  (sorted particle indices, caller order)
    pos_tgt   float64[10^4,3] the generated positions of those targets: the loader checks them against its own
                              workloads.make(cfg) so that a change of the generator cannot go unnoticed
    acc       float64[10^4,3] oracle.p2p_sampled(...) — fp64 minimum-image direct sum over all N sources
    pair_tests, pairs_in_cut  the oracle's counters
    n, n_pm, seed, r_s, r_cut, G, boxsize, flavour ("F": positions on the fp32 grid, A20)
"""
from __future__ import annotations

import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_2107_14008_b200 import workloads  # noqa: E402

N_TARGETS = 10_000


def path(cfg_id: int) -> str:
    return os.path.join(HERE, f"c{cfg_id}_acc_10k.npz")


def make(cfg_id: int) -> str:
    cfg = workloads.CONFIGS[cfg_id]
    t0 = time.time()
    pos, mass = workloads.make(cfg)                      # flavour F
    r_s = 1.2 * cfg.boxsize / cfg.n_pm
    r_cut = 6.0 * r_s                                    # north_star
    tgt = workloads.sample_targets(cfg.n, N_TARGETS, cfg.seed)
    t1 = time.time()
    acc, cnt = oracle.p2p_sampled(pos, mass, tgt, boxsize=cfg.boxsize, r_s=r_s, r_cut=r_cut, G=cfg.G)
    t2 = time.time()
    out = path(cfg_id)
    np.savez_compressed(out, targets=tgt, pos_tgt=pos[tgt], acc=acc, pair_tests=cnt["pair_tests"],
                        pairs_in_cut=cnt["pairs_in_cut"], n=cfg.n, n_pm=cfg.n_pm, seed=cfg.seed, r_s=r_s,
                        r_cut=r_cut, G=cfg.G, boxsize=cfg.boxsize, flavour="F")
    print(f"config {cfg_id}: {len(tgt)} targets x {cfg.n} sources, generate {t1 - t0:.0f} s, oracle {t2 - t1:.0f} s "
          f"on {oracle.num_threads()} threads -> {out}", flush=True)
    return out


if __name__ == "__main__":
    for c in [int(a) for a in sys.argv[1:]] or [2, 3, 4, 5]:
        make(c)
