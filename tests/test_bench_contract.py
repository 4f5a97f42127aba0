"""Host-side checks of the measurement contract (no GPU): the roofline bookkeeping of bench.py and the committed ncu
traffic numbers it reports beside every bench line."""
import json
import os

import pytest

import bench
from paper_1901_09266_b200 import synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_traffic_is_committed_for_every_bench_workload():
    """`roofline.traffic` must not be null on the default sweep or on the other dense / sparse workloads: every
    (workload, minibatch) that bench.py times has its dram bytes per pass in profiles/traffic.json."""
    cases = [("large_dense", b) for b in bench.LARGE_DENSE_SWEEP]
    cases += [(w, synth.CONFIGS[w].b) for w in ("corridor", "multiyear", "large_sparse")]
    for w, b in cases:
        for kind in ("forward", "gradient_update"):
            t = bench.traffic_from_profiles(w, b, kind)
            assert t is not None and t > 0, (w, b, kind)


def test_traffic_is_not_below_the_algorithmic_bytes():
    """a pass reads the operator once and the minibatch's state; measured DRAM traffic below that
    would mean a wrong key or a capture of another kernel."""
    t = json.load(open(os.path.join(ROOT, "profiles", "traffic.json")))
    for w, b in [("large_dense", 1), ("large_dense", 8), ("large_dense", 64), ("large_dense", 256), ("corridor", 32), ("multiyear", 64)]:
        cfg = synth.CONFIGS[w]
        f_b, g_b, _ = bench.algorithmic(cfg, b)
        e = t[f"{w}_b{b}"]
        assert e["forward"] >= 0.98 * f_b and e["gradient_update"] >= 0.98 * g_b, (w, b, e, f_b, g_b)
        assert e["forward"] <= 2.0 * f_b and e["gradient_update"] <= 2.0 * g_b, (w, b, e, f_b, g_b)


def test_algorithmic_bytes_and_flops_formula():
    """forward bytes = 4 nb L N + 4 n T (N + L), gradient = 4 nb L N + 4 n T N, flops = 2 nb L N n per
    pass, nb = T (H + 1) - H (H + 1) / 2 valid blocks."""
    cfg = synth.CONFIGS["corridor"]
    nb = cfg.T * (cfg.H + 1) - cfg.H * (cfg.H + 1) // 2
    f_b, g_b, fl = bench.algorithmic(cfg, 32)
    assert f_b == pytest.approx(4.0 * nb * cfg.L * cfg.N + 4.0 * 32 * cfg.T * (cfg.N + cfg.L))
    assert g_b == pytest.approx(4.0 * nb * cfg.L * cfg.N + 4.0 * 32 * cfg.T * cfg.N)
    assert fl == pytest.approx(2.0 * nb * cfg.L * cfg.N * 32)
