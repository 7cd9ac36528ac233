"""CPU-only: the host-side pieces of bench.py that the JSON line depends on (no GPU, no timing)."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def test_algorithmic_ops_per_evaluation_match_design_section_9():
    # A = 3 + (1 + [caps] (1 + B)) / L
    want = {1: 3.25, 2: 4.0, 3: 7.0, 4: 3.625}
    for cfg, a in want.items():
        w = bench.make_workload(cfg, 0, 2)
        assert abs(bench.alg_ops_per_eval(w) - a) < 1e-12, cfg


def test_every_bench_leg_has_a_committed_traffic_row():
    # roofline.traffic comes from profiles/r2_scorer_dram_bytes.csv: one row per workload the default line reports
    tags = [bench.workload_tag(c, False) for c in (1, 2, 3, 4)] + [bench.workload_tag(1, True), bench.workload_tag(1, "int32"), "linear_cfg1"]
    for t in tags:
        b, src = bench.committed_traffic(t)
        assert b is not None and b > 0 and "captured at commit" in src, t
    assert bench.committed_traffic("cfg0") == (None, None)      # latency-bound: no scorer row


def test_bench_variants_of_configs_1():
    base = bench.make_workload(1, 0, 3)
    wide = bench.make_workload(1, 0, 3, True)
    assert np.array_equal(wide.batch.lat_us, base.batch.lat_us.astype(np.int64) * bench.WIDE_FACTOR)
    assert np.array_equal(wide.batch.slo_us, base.batch.slo_us.astype(np.int64) * bench.WIDE_FACTOR)
    z = bench.make_workload(1, 0, 3, "int32")
    b = z.batch
    for r in range(b.R):       # one option per request with factor 1 - v (1 - a) = 0
        n = int(b.node_off[r]) + (r % b.n_nodes(r))
        assert b.vuln[n] == 1.0 and b.acc[int(b.opt_off[n])] == 0.0
    assert z.n_plans_total() == base.n_plans_total()


def test_oracle_sample_is_bounded_and_named():
    for cfg in (0, 1, 4):
        w = bench.make_workload(cfg, 0, None)
        sub, what = bench.oracle_sample(w)
        assert sub.n_plans_total() * sub.L <= 2 * bench.ORACLE_SAMPLE_EVALS + w.subset([0]).n_plans_total() * w.L
        assert "request" in what
    sub, what = bench.oracle_sample(bench.make_workload(4, 0, None))
    assert sub.batch.R == 1 and sub.L == 1 and "level 0" in what
