"""Host-side logic of bench.py that needs no GPU: the multi-rank aggregation (world size 2 over gloo), the
replica seeding, the flop convention, and the polynomial behind PHOTONS_G_POLY against the oracle's g."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        # rank r took (10 + 5 r) ms for (1000 + r) units
        ms, units = bench.aggregate(10.0 + 5.0 * rank, 1000.0 + rank, dist)
        q.put((rank, ms, units))
    finally:
        dist.destroy_process_group()


def test_aggregate_is_max_time_sum_units_gloo_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, units in out:
        assert ms == 15.0            # MAX over ranks
        assert units == 2001.0       # SUM over ranks


def test_aggregate_single_process_is_identity():
    import bench
    assert bench.aggregate(3.5, 7.0, None) == (3.5, 7.0)


def test_replicas_have_their_own_seed():
    import bench
    from paper_2107_14008_b200 import workloads
    cfg = workloads.CONFIGS[4]
    assert bench.rank_config(cfg, 0) is cfg
    seeds = {bench.rank_config(cfg, r).seed for r in range(8)}
    assert len(seeds) == 8
    assert all(bench.rank_config(cfg, r).n == cfg.n for r in range(8))


def test_flop_convention_matches_design():
    import bench
    assert bench.flops_per_pair("fp32", "poly", poly_degree=12) == 46.0   # (8+12) FFMA x 2 + 3 FADD + 2 FMUL + 1 MUFU
    assert bench.flops_per_pair("mixed", "poly", poly_degree=13) == 48.0
    assert bench.flops_per_pair("fp32", "table") == 35.0                  # 512 nodes / T[2]
    assert bench.flops_per_pair("fp64", "table", table_level=4, table_layout="coef") == 42.0
    assert bench.flops_per_pair("fp64", "table", table_level=4) == 56.0
    assert bench.PAPER_FLOPS_PER_PAIR == 51.0
    # peak = SMs x lanes x 2 x clock
    assert bench.peak_tflops("fp32", 1965.0) == pytest.approx(74.45, rel=1e-4)
    assert bench.peak_tflops("fp64", 1965.0) == pytest.approx(37.2, rel=1e-3)
    # roofline.traffic comes from a committed ncu summary or is null, never a constant in bench.py
    t, src = bench.ncu_traffic("no_such_workload", 32, "fp32", "poly")
    assert t is None and src is None


def test_headline_params_follow_the_config():
    import bench
    from paper_2107_14008_b200 import workloads
    p = bench.headline_params(workloads.CONFIGS[4])
    assert (p["n_pm"], p["maxleaf"], p["precision"], p["g_mode"]) == (256, 32, "fp32", "poly")
    assert p["close_pair_radius"] == pytest.approx(5e-4 * 6 * 1.2 / 256)
    p1 = bench.headline_params(workloads.CONFIGS[1])
    assert p1["close_pair_radius"] == pytest.approx(0.02 * 6 * 1.2 / 32)


@pytest.mark.parametrize("degree,bound", [(10, 3e-6), (11, 5e-7), (12, 8e-8), (13, 1.2e-8), (14, 2e-9)])
def test_poly_g_against_oracle_T(oracle, degree, bound):
    """The FMA-pipe polynomial (host-only hook of the library) reproduces Eq. 1 as the oracle evaluates it:
    g(r) = 1 - s^(3/2) Q(t), s = (r/2r_s)^2, t = 2 s/9 - 1."""
    from paper_2107_14008_b200 import build, binding
    build.build()
    coeffs, err = binding.poly_fit(degree, 6.0)
    x = np.linspace(0.0, 3.0, 6001)
    s = x * x
    t = 2.0 * s / 9.0 - 1.0
    g = 1.0 - s ** 1.5 * np.polyval(coeffs[::-1], t)
    dev = np.abs(g - oracle.oracle_T(x)).max()
    assert dev <= bound
    assert err == pytest.approx(dev, rel=0.05, abs=1e-12)     # the library's own error estimate is honest
    # Newtonian limit and the value at the cut
    assert g[0] == 1.0
    assert g[-1] == pytest.approx(4.39849652838829e-4, abs=bound)


@pytest.mark.parametrize("degree,bound", [(9, 6e-7), (10, 1.5e-7), (11, 4e-8)])
def test_fused_g_against_oracle_T(oracle, degree, bound):
    """The hand-fused direct evaluation (host-only hook of the library): g(r) = exp(-x^2) H(t), H ~ erfcx(x) + 2x/sqrt(pi),
    t = 2x/3 - 1, against Eq. 1 as the oracle evaluates it."""
    from paper_2107_14008_b200 import build, binding
    build.build()
    coeffs, err = binding.fused_fit(degree, 6.0)
    x = np.linspace(0.0, 3.0, 6001)
    g = np.exp(-x * x) * np.polyval(coeffs[::-1], 2.0 * x / 3.0 - 1.0)
    dev = np.abs(g - oracle.oracle_T(x)).max()
    assert dev <= bound
    assert err == pytest.approx(dev, rel=0.05, abs=1e-12)
    assert g[0] == pytest.approx(1.0, abs=bound)
    assert g[-1] == pytest.approx(4.39849652838829e-4, abs=bound)


def test_poly_fit_rejects_bad_arguments():
    from paper_2107_14008_b200 import build, binding
    build.build()
    for deg, rc in ((0, 6.0), (21, 6.0), (12, 0.0), (12, 6.5)):
        with pytest.raises(binding.PhotonsError):
            binding.poly_fit(deg, rc)


def test_reference_arm_json_line_on_cpu(capsys):
    """`bench.py --impl reference` (the oracle arm) needs no GPU: run it on config 1 and check the contract keys."""
    import json
    import bench
    rc = bench.main(["--impl", "reference", "--config", "1", "--steps", "1", "--warmup", "0"])
    assert rc == 0
    line = json.loads(capsys.readouterr().out.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "pairs/s" and line["higher_is_better"] is True
    assert line["n_gpus"] == 1 and line["steps"] == 1 and line["warmup"] == 0 and line["vs_baseline"] is None
    assert line["value"] > 0 and line["ms_per_step"] > 0 and line["dtype"] == "f64" and line["data"] == "synthetic"
    assert line["config"]["workload"] == "c1_uniform_32"
    cb = line["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] == line["value"] and "targets" in cb["sample"]
    assert line["e2e"] == {"value": line["value"], "unit": "pairs/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    # all 32^3 targets against all sources: 2^30 pair tests, 1563.5 neighbours per particle on average
    assert cb["within_cut_pairs_per_s"] / cb["value"] == pytest.approx(1563.5 / 32768, rel=0.01)


def test_reference_arm_is_silent_on_other_ranks(capsys, monkeypatch):
    import bench
    monkeypatch.setenv("RANK", "1")
    assert bench.main(["--impl", "reference", "--config", "1", "--steps", "1", "--warmup", "0"]) == 0
    assert capsys.readouterr().out.strip() == ""
