"""-m gpu: BASELINE.json configs[1..4] at FULL size, in the launch configuration bench.py times (binding.launch on the
default context), checked on what the oracle can afford:

  * every record of every request: the oracle's score of the GPU's chosen plan (one plan, microseconds) must be
    bit-identical in T, feasibility, D_b, dominant model and canonical index, and within 1e-5 in C (P2);
  * sampled requests: the full brute-force oracle on a few requests, all matching rules P1-P4;
  * cfg4 (2.18e9 plans per request): requests 0 and 1 against the brute-force oracle's stored records
    (tests/golden/cfg4_requests_0_1_oracle.txt, written by tests/golden/make_cfg4_oracle_golden.py from oracle/ alone),
    all matching rules; every one of the 128 records against the independent MILP of PIN13 (HiGHS);
  * cfg3's queries once more with non-prefix (down-set) dispatched sets, both replan semantics;
  * cfg1 once more with every duration x 3000 (the approx class of the fp32 scorer), same checks.
"""
from __future__ import annotations

import numpy as np
import pytest

from support import workloads as wl

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


def test_cfg1_full_with_second_scale_latencies(dy, orc):
    # configs[1] with every duration and SLO x 3000 (seconds to minutes): the requests leave the fp32
    # scorer's exact range and run on its verified instantiation (conservative fp32 screen, int32 check of every
    # candidate) -- at full size, in the launch configuration bench.py times for its x 3000 leg
    w = wl.make_config(1)
    w.batch.lat_us = (w.batch.lat_us.astype(np.int64) * 3000).astype(np.int32)
    w.batch.slo_us = (w.batch.slo_us.astype(np.int64) * 3000).astype(np.int32)
    g, st = gpu_run(dy, w)
    assert st["fast_requests"] == 256 and st["approx_requests"] == 256
    assert check_own_plan(orc, w, g, range(256 * 4)) > 900
    c = check_sampled_requests(orc, w, g, [0, 101, 255], "cfg1-full-x3000")
    assert c["records"] == 12
    # scaling every duration and the SLO by the same factor scales T and leaves the optimum's plan alone
    # (floor(tau * 3000 * m / 1000) = 3 * tau * m exactly, and floor(tau * m / 1000) * 3000 <= it: the feasible set can
    # only shrink by plans within one microsecond-rounding of the SLO), so most records keep their plan
    g1, _ = gpu_run(dy, wl.make_config(1))
    assert (g1["plan_idx"] == g["plan_idx"]).mean() > 0.9


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


def load_cfg4_golden(w_sub):
    """tests/golden/cfg4_requests_0_1_oracle.txt -> the dict oracle.run() returns, after checking that the file was
    written for exactly these inputs (digest over every input array)."""
    import importlib.util
    import os
    here = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    spec = importlib.util.spec_from_file_location("make_cfg4_oracle_golden", os.path.join(here, "make_cfg4_oracle_golden.py"))
    mk = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mk)
    from conftest import read_golden
    rows = read_golden("cfg4_requests_0_1_oracle.txt")
    assert rows[0][0] == "digest" and rows[0][1] == mk.input_digest(w_sub), \
        "cfg4 golden was written for other inputs: rerun tests/golden/make_cfg4_oracle_golden.py"
    rows = rows[1:]
    n, B = len(rows), w_sub.batch.B
    ref = dict(status=np.zeros(n, np.uint8), plan_idx=np.zeros(n, np.uint64), corr=np.zeros(n), lat=np.zeros(n, np.int64),
               dem=np.zeros((n, B), np.int64), dom_model=np.zeros(n, np.uint8), runner_idx=np.zeros(n, np.uint64),
               runner_corr=np.zeros(n), n_feasible=np.zeros(n, np.uint64), choice=np.zeros((n, 16), np.uint8))
    for i, c in enumerate(rows):
        assert int(c[0]) == i
        ref["status"][i] = int(c[1]); ref["plan_idx"][i] = int(c[2]); ref["corr"][i] = float.fromhex(c[3])
        ref["lat"][i] = int(c[4]); ref["dem"][i] = [int(x) for x in c[5].split()]; ref["dom_model"][i] = int(c[6])
        ref["runner_idx"][i] = int(c[7]); ref["runner_corr"][i] = float.fromhex(c[8]); ref["n_feasible"][i] = int(c[9])
        ref["choice"][i] = [int(x) for x in c[10].split()]
    return ref


def test_cfg4_full_brute_force_on_requests_0_and_1_milp_on_all(dy, orc):
    """BASELINE.json configs[4]: "oracle run on 2 of the 16 requests"; the MILP on all 16."""
    from test_oracle_pins import milp_best_corr
    w = wl.make_config(4)                      # 16 requests x 6^12 plans x 8 levels, B = 3, caps
    g, st = gpu_run(dy, w)
    assert st["fast_requests"] == 16
    assert check_own_plan(orc, w, g, range(16 * 8)) >= 1
    L, B = 8, 3
    # (a) requests 0 and 1 against the brute-force oracle: the full protocol P1-P6 on their 16 records
    rows = [0, 1]
    sub = w.subset(rows)
    ref = load_cfg4_golden(sub)
    gs = {}
    for k, v in g.items():
        per = v.size // (w.batch.R * L)
        gs[k] = v.reshape(w.batch.R, L * per)[rows].reshape(-1)
    c = check_records(orc, sub, gs, ref, where="cfg4-full[0,1]")
    assert c["records"] == 16
    print("cfg4 requests 0,1 vs brute force:", c)
    # (b) every (request, level) against the independent MILP optimum (PIN13): P1 (existence) and P3
    mult = np.asarray(w.mult_pm).reshape(L, B)
    n_ok = 0
    for rec in range(16 * L):
        r, l = divmod(rec, L)
        cstar = milp_best_corr(w.batch, r, mult[l])
        if cstar is None:
            assert g["status"][rec] == 1, rec
            continue
        n_ok += 1
        assert g["status"][rec] == 0, rec
        c64 = float(g["corr64"][rec])
        assert c64 >= cstar * (1.0 - REL), (rec, c64, cstar)          # P3 against the MILP optimum
        assert c64 <= cstar * (1.0 + 1e-6), (rec, c64, cstar)         # and nothing beats a true optimum
    assert n_ok >= 16
    # the MILP and the brute force agree on the records both cover (keeps the two references honest)
    for rec in range(16):
        cstar = milp_best_corr(sub.batch, rec // L, mult[rec % L])
        if cstar is None:
            assert ref["status"][rec] == 1
        else:
            assert abs(cstar - ref["corr"][rec]) <= 1e-6 * ref["corr"][rec]


def test_cfg3_full_size_with_non_prefix_dispatched_sets(dy, orc):
    """configs[3]'s 16 384 queries with every dispatched set redrawn as a random down-set of the DAG (predecessor-
    closed, in general not a prefix: App. D commits a SET of bindings), both replan semantics."""
    base = wl.make_config(3)
    for flags in (wl.FLAG_FIXED_IN_PLACE, wl.FLAG_RESIDUAL):
        w = wl.with_down_set_dispatch(base, seed=303, flags=flags)
        m = w.dispatched_mask.astype(np.int64)
        assert ((m & (m + 1)) != 0).sum() > 4000          # most sets are not prefixes
        g, st = gpu_run(dy, w)
        rng = np.random.default_rng(33)
        assert check_own_plan(orc, w, g, rng.choice(16384, size=2000, replace=False)) > 1000
        # brute force on queries the oracle finishes quickly (<= 12^5 free plans), non-prefix ones first
        free = np.array([w.subset([r]).n_plans_total() for r in range(600)])
        nonpre = (m[:600] & (m[:600] + 1)) != 0
        rows = [int(r) for r in np.nonzero((free <= 12 ** 5) & nonpre)[0][:40]]
        assert len(rows) >= 20
        c = check_sampled_requests(orc, w, g, rows, f"cfg3-downsets(flags={flags})")
        print("cfg3 down-sets:", c)
        ch = g["choice"].reshape(-1, 16)
        b = w.batch
        for r in range(0, b.R, 7):
            if g["status"][r] != 0:
                continue
            n0 = int(b.node_off[r])
            for i in range(b.n_nodes(r)):
                if (int(m[r]) >> i) & 1:
                    assert ch[r, i] == w.fixed_choice[n0 + i]      # committed bindings are never replaced
