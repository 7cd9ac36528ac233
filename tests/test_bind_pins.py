"""Pins of oracle/bind_oracle.py (coefficient construction, Eq.(2), Alg. 1 l.1-8) against the
paper's text: the stage structures of the policy catalogue (Table 4 / App. A), the worked durations
of Fig. 7(a) ("27B + V [10 + 4]", "9B + V [4 + 3]") and the properties Section 4.2 states."""
from __future__ import annotations

import numpy as np
import pytest

from oracle import bind_oracle as bo


def test_fig7_durations_are_base_plus_verification():
    # "[.]: nominal time units": 27B + V = 10 + 4, 27B = 10, 9B + V = 4 + 3, 9B = 4, 9B (CodeGen) = 6; one token per unit
    th = 1e6                                  # tokens per second = one token per microsecond
    assert bo.bind_option([[10], [4]], th, 0.0, 1.0)[0] == 14
    assert bo.bind_option([[10]], th, 0.0, 1.0)[0] == 10
    assert bo.bind_option([[4], [3]], th, 0.0, 1.0)[0] == 7
    assert bo.bind_option([[4]], th, 0.0, 1.0)[0] == 4 and bo.bind_option([[6]], th, 0.0, 1.0)[0] == 6


def test_table4_stage_structures():
    th, pre = 2e6, 30.0                       # 2 tokens/us, 30 us prefill correction
    base, fb, rw = 400.0, 120.0, 380.0
    # none: "with no verification, only the base-call stage remains"
    assert bo.bind_option([[base]], th, pre, 1000.0) == (230, 0.4, 400.0)
    # self_refine: "separate base, feedback, and rewrite calls form three serial stages"
    t, c, tot = bo.bind_option([[base], [fb], [rw]], th, pre, 1000.0)
    assert (t, tot) == (int(np.rint((base + fb + rw) / 2 + pre)), 900.0) and c == pytest.approx(0.9)
    # advanced_refine: "Critique stage -> rewrite"; "A policy with multiple critiques may execute them in parallel before
    # a final revision": the stage contributes its longest call, the cost counts every call
    crit = [100.0, 160.0, 90.0]
    t, c, tot = bo.bind_option([[base], crit, [rw]], th, pre, 1000.0)
    assert t == int(np.rint((base + 160.0 + rw) / 2 + pre)) and tot == base + sum(crit) + rw
    # self_consistency: "Parallel samples -> selection"
    samples = [410.0, 395.0, 402.0, 388.0]
    t, c, tot = bo.bind_option([[base], samples, [50.0]], th, pre, 1000.0)
    assert t == int(np.rint((base + 410.0 + 50.0) / 2 + pre)) and tot == base + sum(samples) + 50.0
    # an absent call (0 tokens) changes nothing
    assert bo.bind_option([[base, 0.0], [0.0, 0.0], [rw, 0.0]], th, pre, 1000.0) == bo.bind_option([[base], [rw]], th, pre, 1000.0)


def test_parallel_calls_add_cost_but_not_latency_beyond_the_longest():
    a = bo.bind_option([[300.0], [200.0]], 1e6, 0.0, 100.0)
    b = bo.bind_option([[300.0], [200.0, 150.0, 199.0]], 1e6, 0.0, 100.0)
    assert a[0] == b[0] == 500 and b[1] > a[1] and b[2] == a[2] + 349.0


def test_retargeting_hardware_changes_only_the_service_terms():
    # "adapting to new hardware requires only calibrating per-model decode throughput and prefill latency"
    stages = [[640.0], [128.0, 256.0], [512.0]]
    t1, c1, _ = bo.bind_option(stages, 1e6, 40.0, 2048.0)
    t2, c2, _ = bo.bind_option(stages, 2e6, 40.0, 2048.0)
    assert c1 == c2 and (t1 - 40) == 2 * (t2 - 40)
    t3, _, _ = bo.bind_option(stages, 1e6, 140.0, 2048.0)
    assert t3 - t1 == 100


def test_batch_binding_gathers_by_skill_model_policy_backend_and_fan_in():
    dims = dict(S=2, M=2, P=2, D=2, A=2, J=2, ROLES=2, F=3)
    rng = np.random.default_rng(0)
    quality = rng.uniform(0.5, 1.0, size=(2, 2, 2)).astype(np.float32)
    tokens = rng.integers(0, 500, size=(2, 2, 2, 2, 2)).astype(np.float32)
    theta = np.array([[1e6, 2e6], [3e6, 0.0]], np.float32)        # (model 1, backend 1) is not calibrated
    pre = np.array([[10, 20], [30, 40]], np.float32)
    psi = rng.uniform(0, 1, size=(2, 2, 3)).astype(np.float32)
    # two nodes: node 0 (skill 1, role 0, no predecessor), node 1 (skill 0, role 1, two predecessors)... and a third with fan-in 5
    opt_off = [0, 2, 4, 5]
    out = bo.bind(dims, quality, tokens, theta, pre, psi, 1000.0, opt_off, [0, 0b01, 0b11111], [1, 0, 0], [0, 1, 1],
                  model=[0, 1, 1, 0, 7], backend=[1, 0, 1, 0, 0], policy=[0, 1, 1, 1, 0])
    assert out["vuln"].tolist() == [psi[0, 1, 0], psi[1, 0, 1], psi[1, 0, 2]]         # fan-in 5 falls in the last bucket
    assert out["acc"][0] == quality[1, 0, 0] and out["acc"][1] == quality[1, 1, 1] and out["acc"][3] == quality[0, 0, 1]
    g = tokens[1, 0, 0]
    assert out["lat_us"][0] == int(np.rint(1e6 * (g[0].max() + g[1].max()) / 2e6 + 20))
    assert out["cost"][0] == np.float32(g.sum() / 1000.0) and out["demand"][0] == int(g.sum())
    assert out["lat_us"][2] == -1 and np.isnan(out["acc"][2])                          # uncalibrated pair
    assert out["lat_us"][4] == -1 and np.isnan(out["cost"][4])                         # model id out of range
