"""-m gpu: BASELINE.json configs[1..4] at FULL size, in the launch configuration bench.py times (binding.launch on the
default context), checked on what the oracle can afford:

  * every record of every request: the oracle's score of the GPU's chosen plan (one plan, microseconds) must be
    bit-identical in T, feasibility, D_b, dominant model and canonical index, and within 1e-5 in C (P2);
  * sampled requests: the full brute-force oracle on a few requests, all matching rules P1-P4;
  * cfg4 (2.18e9 plans per request: brute force needs core-hours): the optimum C of sampled (request, level) pairs
    from the independent MILP of PIN13 (HiGHS), P3/P4-style.
"""
from __future__ import annotations

import numpy as np
import pytest

from paper_2607_02942_b200 import workloads as wl

from parity import REL, check_records

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def dy():
    import torch
    assert torch.cuda.is_available(), "-m gpu tests need a CUDA device"
    from paper_2607_02942_b200 import binding
    ctx = binding.Context(0)
    yield binding, ctx
    ctx.close()


def gpu_run(dy, w):
    import torch
    binding, ctx = dy
    dw = binding.upload(w, "cuda:0", True)
    binding.launch(ctx, dw)
    torch.cuda.synchronize()
    st = ctx.dyplan_last_stats()
    assert st["plans"] == w.n_plans_total()
    return dw.out.host(), st


def check_own_plan(orc, w, g, recs):
    """P2 on the records `recs`: the GPU's plan re-scored by the oracle."""
    b = w.batch
    L, B = w.L, b.B
    ch = g["choice"].reshape(-1, 16)
    dem = g["dem"].reshape(-1, B)
    n_ok = 0
    for rec in recs:
        r, l = divmod(int(rec), L)
        st = int(g["status"][rec])
        assert st in (0, 1), (rec, st)
        if st != 0:
            assert g["plan_idx"][rec] == np.iinfo(np.uint64).max
            continue
        n_ok += 1
        if w.kind == "compile":
            mult, skip = np.asarray(w.mult_pm).reshape(L, B)[l], 0
        else:
            mult = np.asarray(w.live_mult_pm).reshape(b.R, B)[r]
            skip = int(w.dispatched_mask[r]) if (w.flags & 1) else 0
        s = orc.score(b, r, mult, ch[rec].copy(), skip)
        assert s["status"] == 0 and s["feasible"], rec
        assert s["plan_idx"] == int(g["plan_idx"][rec]), rec
        assert s["lat"] == int(g["lat"][rec]), rec
        assert (s["dem"] == dem[rec]).all(), rec
        assert s["dom_model"] == int(g["dom_model"][rec]), rec
        assert abs(float(g["corr"][rec]) - s["corr"]) <= REL * s["corr"], rec
        assert abs(float(g["corr64"][rec]) - s["corr"]) <= 1e-12 * s["corr"], rec
    return n_ok


def check_sampled_requests(orc, w, g, rows, where):
    """Brute-force oracle on the requests `rows`; all matching rules on their records."""
    sub = w.subset(rows)
    ref = orc.run(sub)
    L, B = w.L, w.batch.B
    gs = {}
    for k, v in g.items():
        per = v.size // (w.batch.R * L)
        gs[k] = v.reshape(w.batch.R, L * per)[rows].reshape(-1)
    return check_records(orc, sub, gs, ref, where=where)


def test_cfg1_full(dy, orc):
    w = wl.make_config(1)                      # 256 requests x 8^8 plans x 4 levels
    g, st = gpu_run(dy, w)
    assert st["fast_requests"] == 256
    assert check_own_plan(orc, w, g, range(256 * 4)) > 900
    c = check_sampled_requests(orc, w, g, [0, 101, 255], "cfg1-full")
    assert c["records"] == 12


def test_cfg2_full(dy, orc):
    w = wl.make_config(2)                      # 4096 requests x 8^7 plans x 4 levels, caps
    g, st = gpu_run(dy, w)
    assert st["fast_requests"] == 4096
    rng = np.random.default_rng(2)
    assert check_own_plan(orc, w, g, rng.choice(4096 * 4, size=3000, replace=False)) > 2000
    rows = sorted(int(x) for x in rng.choice(4096, size=24, replace=False))
    check_sampled_requests(orc, w, g, rows, "cfg2-full")


def test_cfg3_full(dy, orc):
    w = wl.make_config(3)                      # 16384 replan queries, 12 options, caps, one live vector each
    g, st = gpu_run(dy, w)
    assert st["fast_requests"] == 16384
    rng = np.random.default_rng(3)
    assert check_own_plan(orc, w, g, rng.choice(16384, size=3000, replace=False)) > 1500
    nd = np.array([bin(int(m)).count("1") for m in w.dispatched_mask])
    rows = [int(r) for r in np.nonzero(nd >= 4)[0][:40]] + [int(r) for r in np.nonzero(nd == 3)[0][:6]]
    check_sampled_requests(orc, w, g, sorted(rows), "cfg3-full")
    # committed bindings are never replaced, on every query
    ch = g["choice"].reshape(-1, 16)
    b = w.batch
    for r in range(b.R):
        if g["status"][r] != 0:
            continue
        n0 = int(b.node_off[r])
        m = int(w.dispatched_mask[r])
        for i in range(b.n_nodes(r)):
            if (m >> i) & 1:
                assert ch[r, i] == w.fixed_choice[n0 + i]


def test_cfg4_full_against_the_milp(dy, orc):
    from test_oracle_pins import milp_best_corr
    w = wl.make_config(4)                      # 16 requests x 6^12 plans x 8 levels, B = 3, caps
    g, st = gpu_run(dy, w)
    assert st["fast_requests"] == 16
    assert check_own_plan(orc, w, g, range(16 * 8)) >= 1
    L, B = 8, 3
    mult = np.asarray(w.mult_pm).reshape(L, B)
    for rec in (0, 13, 42, 77, 127):
        r, l = divmod(rec, L)
        cstar = milp_best_corr(w.batch, r, mult[l])
        if cstar is None:
            assert g["status"][rec] == 1, rec
            continue
        assert g["status"][rec] == 0, rec
        c64 = float(g["corr64"][rec])
        assert c64 >= cstar * (1.0 - REL), (rec, c64, cstar)          # P3 against the MILP optimum
        assert c64 <= cstar * (1.0 + 1e-6), (rec, c64, cstar)         # and nothing beats a true optimum
