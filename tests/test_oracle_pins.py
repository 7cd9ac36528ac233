"""Pins for the fp64 brute-force oracle (oracle/dyplan_oracle.c) -- CPU only.

Each test checks the oracle against something OTHER than itself: values the paper prints
(tests/golden/), closed forms, library routines (networkx longest path, scipy/HiGHS MILP), an
independent recursive solver written differently, and invariants.  Pin numbers follow SURVEY.md
section 8(c) C.5 / DESIGN.md section 4.
"""
import itertools
import math

import networkx as nx
import numpy as np
import pytest

from conftest import read_golden
from support import workloads as wl

U64MAX = np.iinfo(np.uint64).max


def mk(reqs, B=1, M=1, caps=False):
    return wl.batch_from_requests(reqs, B, M, caps)


def simple_req(pred_mask, lat, *, vuln=None, acc=None, demand=None, backend=None, model=None, slo=10**9, cap=None):
    n = len(pred_mask)
    return dict(
        pred_mask=pred_mask,
        vuln=[0.5] * n if vuln is None else vuln,
        lat=lat,
        acc=[[0.9] * len(x) for x in lat] if acc is None else acc,
        demand=[[0] * len(x) for x in lat] if demand is None else demand,
        backend=[[0] * len(x) for x in lat] if backend is None else backend,
        model=[[0] * len(x) for x in lat] if model is None else model,
        slo=slo, cap=cap)


def all_plans(rad):
    """All digit tuples in canonical-index order (node 0 least significant)."""
    for idx in range(int(np.prod(rad))):
        j, ks = idx, []
        for k in rad:
            ks.append(j % int(k)); j //= int(k)
        yield idx, ks


# ---------------------------------------------------------------- PIN1 / PIN2 closed forms
def test_pin1_chain_latency_is_sum(orc):
    rng = np.random.default_rng(1)
    n = 5
    pm = [0] + [1 << (i - 1) for i in range(1, n)]
    lat = [[int(x) for x in rng.integers(1, 5000, size=3)] for _ in range(n)]
    b = mk([simple_req(pm, lat)])
    for idx, ks in all_plans(b.radices(0)):
        s = orc.score(b, 0, [1000], ks)
        assert s["lat"] == sum(lat[i][ks[i]] for i in range(n))
        assert s["plan_idx"] == idx


def test_pin2_edgeless_latency_is_max(orc):
    rng = np.random.default_rng(2)
    n = 5
    lat = [[int(x) for x in rng.integers(1, 5000, size=3)] for _ in range(n)]
    b = mk([simple_req([0] * n, lat)])
    for idx, ks in all_plans(b.radices(0)):
        assert orc.score(b, 0, [1000], ks)["lat"] == max(lat[i][ks[i]] for i in range(n))


def test_scaled_duration_floor_rule(orc):
    # definition 2 / reading Q4: floor(tau*mult/1000); 1000 is the identity, 2000 doubles exactly.
    b = mk([simple_req([0], [[1, 999, 1001, 123457]])])
    for k, tau in enumerate([1, 999, 1001, 123457]):
        assert orc.score(b, 0, [1000], [k])["lat"] == tau
        assert orc.score(b, 0, [2000], [k])["lat"] == 2 * tau
    assert orc.score(b, 0, [1500], [0])["lat"] == 1      # floor(1.5)
    assert orc.score(b, 0, [1999], [0])["lat"] == 1      # floor(1.999)
    assert orc.score(b, 0, [1001], [1])["lat"] == 999    # floor(999.999)
    assert orc.score(b, 0, [1001], [2])["lat"] == 1002   # floor(1002.001)
    assert orc.score(b, 0, [2718], [3])["lat"] == (123457 * 2718) // 1000


def test_per_backend_multiplier_is_applied_per_option(orc):
    # two options on different backends, multipliers differ per backend
    b = mk([simple_req([0, 1], [[100, 100], [10, 10]], backend=[[0, 1], [1, 0]])], B=2)
    assert orc.score(b, 0, [1000, 3000], [0, 0])["lat"] == 100 + 30
    assert orc.score(b, 0, [1000, 3000], [1, 1])["lat"] == 300 + 10
    assert orc.score(b, 0, [1000, 3000], [1, 0])["lat"] == 300 + 30


# ---------------------------------------------------------------- PIN3 all v = 0
def test_pin3_zero_vulnerability(orc):
    rng = np.random.default_rng(3)
    n = 4
    lat = [[int(x) for x in rng.integers(1, 4000, size=4)] for _ in range(n)]
    acc = [[float(x) for x in rng.uniform(0.5, 1, size=4)] for _ in range(n)]
    pm = [0, 1, 1, 0b110]
    slo = 6000
    b = mk([simple_req(pm, lat, vuln=[0.0] * n, acc=acc, slo=slo)])
    ts = {}
    for idx, ks in all_plans(b.radices(0)):
        s = orc.score(b, 0, [1000], ks)
        assert s["corr"] == 1.0                       # exactly one
        ts[idx] = s["lat"]
    out = orc.compile(b, 1, [1000])
    feas = {i: t for i, t in ts.items() if t <= slo}
    assert feas, "pick an slo that leaves something feasible"
    want = min(feas.items(), key=lambda it: (it[1], it[0]))     # min T then min idx
    assert out["status"][0] == 0 and out["corr"][0] == 1.0
    assert (int(out["plan_idx"][0]), int(out["lat"][0])) == want
    assert int(out["n_feasible"][0]) == len(feas)


# ---------------------------------------------------------------- PIN4 single node by hand
def test_pin4_single_node_argmax_by_hand(orc):
    # v = 0.5; f = 1 - 0.5(1-a): a = .6,.9,.9,.95 -> f = .8,.95,.95,.975 ; lat 100,300,200,900 ; slo 500
    r = simple_req([0], [[100, 300, 200, 900]], vuln=[0.5], acc=[[0.6, 0.9, 0.9, 0.95]], slo=500,
                   demand=[[7, 8, 9, 10]], model=[[0, 1, 1, 0]])
    b = mk([r], M=2)
    out = orc.compile(b, 1, [1000])
    # option 3 has the best f but is too slow; options 1 and 2 tie in C, option 2 is faster
    assert int(out["plan_idx"][0]) == 2 and int(out["lat"][0]) == 200
    assert out["corr"][0] == pytest.approx(1 - float(np.float32(0.5)) * (1 - float(np.float32(0.9))), rel=1e-15)
    assert int(out["n_feasible"][0]) == 3 and int(out["runner_idx"][0]) == 1
    assert int(out["dem"][0, 0]) == 9 and int(out["dom_model"][0]) == 1
    # slo = 900 admits option 3
    b.slo_us[0] = 900
    assert int(orc.compile(b, 1, [1000])["plan_idx"][0]) == 3
    # equal C and equal T -> lowest idx
    r2 = simple_req([0], [[200, 200, 200]], acc=[[0.9, 0.9, 0.9]])
    assert int(orc.compile(mk([r2]), 1, [1000])["plan_idx"][0]) == 0


# ---------------------------------------------------------------- PIN5 library longest path
def _nx_longest(pm, d):
    """Node weights -> edge weights: split each node into in/out joined by an edge of weight d."""
    g = nx.DiGraph()
    n = len(pm)
    for v in range(n):
        g.add_edge(("i", v), ("o", v), weight=d[v])
        for u in range(v):
            if (pm[v] >> u) & 1:
                g.add_edge(("o", u), ("i", v), weight=0)
    return nx.dag_longest_path_length(g, weight="weight")


def _enum_paths_longest(pm, d):
    n = len(pm)
    succ = {u: [v for v in range(n) if (pm[v] >> u) & 1] for u in range(n)}
    best = 0
    def walk(u, acc):
        nonlocal best
        acc += d[u]
        best = max(best, acc)
        for v in succ[u]:
            walk(v, acc)
    for s in range(n):
        walk(s, 0)
    return best


def test_pin5_latency_matches_networkx_and_path_enumeration(orc):
    rng = np.random.default_rng(5)
    for trial in range(30):
        n = int(rng.integers(1, 9))
        pm = wl.random_pred_masks(rng, n, float(rng.uniform(0.1, 0.8)))
        lat = [[int(x) for x in rng.integers(0, 3000, size=int(rng.integers(1, 4)))] for _ in range(n)]
        be = [[int(x) for x in rng.integers(0, 2, size=len(l))] for l in lat]
        mult = [int(x) for x in rng.integers(1000, 3001, size=2)]
        b = mk([simple_req(pm, lat, backend=be)], B=2)
        for _ in range(10):
            ks = [int(rng.integers(0, len(l))) for l in lat]
            d = [(lat[i][ks[i]] * mult[be[i][ks[i]]]) // 1000 for i in range(n)]
            t = orc.score(b, 0, mult, ks)["lat"]
            assert t == _nx_longest(pm, d) == _enum_paths_longest(pm, d)


# ---------------------------------------------------------------- PIN6 the paper's worked numbers
def _walkthrough_batch(slo=10**6):
    # P -> {C, D} -> R -> A; P, R, A carry 0 ("common stages omitted").
    # C options: 27B+V [10+4], 27B [10], 9B [6];  D options: 9B+V [4+3], 9B [4].  One time unit = 1000 us.
    # demand := nominal duration in units, so sum_b D_b reproduces the "duration sum (C,D)" column.
    pm = [0, 0b1, 0b1, 0b110, 0b1000]
    lat = [[0], [14000, 10000, 6000], [7000, 4000], [0], [0]]
    dem = [[0], [14, 10, 6], [7, 4], [0], [0]]
    return mk([simple_req(pm, lat, demand=dem, slo=slo)])


def test_pin6_paper_fig7_fork_latency_and_duration_sum(orc):
    b = _walkthrough_batch()
    c_opt = {14: 0, 10: 1, 6: 2}
    d_opt = {7: 0, 4: 1}
    for name, dC, dD, fork, dsum, _acc in read_golden("paper_fig7_forkjoin.txt"):
        s = orc.score(b, 0, [1000], [0, c_opt[int(dC)], d_opt[int(dD)], 0, 0])
        assert s["lat"] == int(fork) * 1000, name
        assert int(s["dem"].sum()) == int(dsum), name


def test_pin6_paper_fig3a_verification_delta(orc):
    b = _walkthrough_batch()
    c_opt = {10: 1, 6: 2}
    d_opt = {7: 0, 4: 1}
    for name, dC, d_plain, d_ver, delta in read_golden("paper_fig3a_verification_delta.txt"):
        t1 = orc.score(b, 0, [1000], [0, c_opt[int(dC)], d_opt[int(d_ver)], 0, 0])["lat"]
        t0 = orc.score(b, 0, [1000], [0, c_opt[int(dC)], d_opt[int(d_plain)], 0, 0])["lat"]
        assert t1 - t0 == int(delta) * 1000, name


# ---------------------------------------------------------------- PIN8 / PIN9 separable closed form
def test_pin8_pin9_unconstrained_and_slo_edges(orc):
    rng = np.random.default_rng(8)
    w = wl.random_workload(8, R=6, nmin=2, nmax=5, kmin=2, kmax=4, L=2, caps=False, tool_p=0.2)
    b = w.batch
    big = b.subset(range(b.R)); big.slo_us[:] = 2**31 - 1
    out = orc.compile(big, w.L, w.mult_pm)
    for r in range(b.R):
        a, e = b.node_off[r], b.node_off[r + 1]
        want = 1.0
        for n in range(a, e):
            fs = [1.0 - float(b.vuln[n]) * (1.0 - float(b.acc[o])) for o in range(b.opt_off[n], b.opt_off[n + 1])]
            want *= max(fs)
        for l in range(w.L):
            assert out["status"][r * w.L + l] == 0
            assert out["corr"][r * w.L + l] == pytest.approx(want, rel=1e-14)
            assert int(out["n_feasible"][r * w.L + l]) == b.n_plans(r)
    # SLO below the smallest possible T (a lower bound: the smallest scaled duration of node 0) -> INFEASIBLE
    tiny = b.subset(range(b.R))
    mult = np.asarray(w.mult_pm).reshape(w.L, b.B)
    for r in range(b.R):
        n0 = b.node_off[r]
        ds = [(int(b.lat_us[o]) * int(mult[l, b.backend[o]])) // 1000 for o in range(b.opt_off[n0], b.opt_off[n0 + 1])
              for l in range(w.L)]
        tiny.slo_us[r] = max(0, min(ds) - 1)
    out = orc.compile(tiny, w.L, w.mult_pm)
    for r in range(b.R):
        if tiny.slo_us[r] < min(
                (int(b.lat_us[o]) * int(mult[l, b.backend[o]])) // 1000
                for o in range(b.opt_off[b.node_off[r]], b.opt_off[b.node_off[r] + 1]) for l in range(w.L)):
            for l in range(w.L):
                rec = r * w.L + l
                assert out["status"][rec] == 1 and out["plan_idx"][rec] == U64MAX and out["corr"][rec] == -1.0
                assert out["lat"][rec] == 2**31 - 1 and (out["choice"][rec] == 0xFF).all()


# ---------------------------------------------------------------- PIN10 invariants
def test_pin10_invariants(orc):
    w = wl.random_workload(10, R=8, nmin=2, nmax=5, kmin=2, kmax=4, L=2, caps=True, tool_p=0.1)
    b = w.batch
    base = orc.compile(b, w.L, w.mult_pm)
    # sum_b D_b = sum_n demand[n][k_n] for the winner
    for r in range(b.R):
        for l in range(w.L):
            rec = r * w.L + l
            if base["status"][rec] != 0:
                continue
            ks = base["choice"][rec][: b.n_nodes(r)]
            tot = sum(int(b.demand[b.opt_off[b.node_off[r] + i] + int(k)]) for i, k in enumerate(ks))
            assert int(base["dem"][rec].sum()) == tot
    # best C is non-decreasing in SLO and in caps
    loose = b.subset(range(b.R)); loose.slo_us[:] = (loose.slo_us.astype(np.int64) * 3 // 2).astype(np.int32)
    o2 = orc.compile(loose, w.L, w.mult_pm)
    loose2 = b.subset(range(b.R)); loose2.cap[:] = loose2.cap * 2
    o3 = orc.compile(loose2, w.L, w.mult_pm)
    # ... and non-increasing when every multiplier grows
    o4 = orc.compile(b, w.L, (np.asarray(w.mult_pm) * 2).astype(np.int32))
    for rec in range(b.R * w.L):
        c = base["corr"][rec]
        assert o2["corr"][rec] >= c and o3["corr"][rec] >= c and o4["corr"][rec] <= c
        assert o2["n_feasible"][rec] >= base["n_feasible"][rec] >= o4["n_feasible"][rec]
    # mult == 1000 -> T equals the unscaled longest path (checked against networkx)
    o5 = orc.compile(loose, 1, [1000] * b.B)
    for r in range(b.R):
        if o5["status"][r] != 0:
            continue
        n = b.n_nodes(r)
        ks = o5["choice"][r][:n]
        d = [int(b.lat_us[b.opt_off[b.node_off[r] + i] + int(k)]) for i, k in enumerate(ks)]
        pm = [int(x) for x in b.pred_mask[b.node_off[r]: b.node_off[r + 1]]]
        assert int(o5["lat"][r]) == _nx_longest(pm, d)


def test_pin10_relabelling_by_another_topological_order(orc):
    rng = np.random.default_rng(100)
    for trial in range(8):
        n = int(rng.integers(3, 6))
        q = wl.random_request(rng, n, 2, 3, 2, 2, edge_p=0.35, cap_frac=0.7)
        pm = q["pred_mask"]
        # random other topological order: repeatedly pick a random ready node
        order, done = [], set()
        while len(order) < n:
            ready = [v for v in range(n) if v not in done and all(((pm[v] >> u) & 1) == 0 or u in done for u in range(n))]
            v = ready[int(rng.integers(0, len(ready)))]
            order.append(v); done.add(v)
        pos = {v: i for i, v in enumerate(order)}
        q2 = dict(q)
        q2["pred_mask"] = [sum(1 << pos[u] for u in range(n) if (pm[v] >> u) & 1) for v in order]
        for key in ("lat", "acc", "demand", "backend", "model"):
            q2[key] = [q[key][v] for v in order]
        q2["vuln"] = [q["vuln"][v] for v in order]
        o1 = orc.compile(mk([q], 2, 2, True), 1, [1300, 2100])
        o2 = orc.compile(mk([q2], 2, 2, True), 1, [1300, 2100])
        assert o1["status"][0] == o2["status"][0]
        assert int(o1["n_feasible"][0]) == int(o2["n_feasible"][0])
        if o1["status"][0] == 0:
            assert o1["corr"][0] == pytest.approx(o2["corr"][0], rel=1e-12)
            # T* may differ only if two plans tie in C to the last bit; then compare via re-scoring
            ch1 = [int(o1["choice"][0][v]) for v in range(n)]
            ch2 = [int(o2["choice"][0][pos[v]]) for v in range(n)]
            if ch1 == ch2:
                assert int(o1["lat"][0]) == int(o2["lat"][0])
                assert (np.sort(o1["dem"][0]) == np.sort(o2["dem"][0])).all()


# ---------------------------------------------------------------- PIN11 independent recursive solver
class RecSolver:
    """Written differently on purpose: depth-first assignment node by node; latency by memoised
    top-down recursion from the sinks; C by exp(sum log1p(-v(1-a)))."""

    def __init__(self, b, r, mult, fixed=None, residual=False):
        self.b, self.r, self.mult = b, r, [int(m) for m in mult]
        self.n0 = int(b.node_off[r]); self.n = b.n_nodes(r)
        self.fixed = fixed or {}
        self.residual = residual
        self.cands = []

    def opt(self, i, k):
        return int(self.b.opt_off[self.n0 + i]) + k

    def solve(self):
        self._assign(0, [])
        return self.cands

    def _assign(self, i, ks):
        if i == self.n:
            self._leaf(list(ks)); return
        b = self.b
        K = int(b.opt_off[self.n0 + i + 1] - b.opt_off[self.n0 + i])
        for k in ([self.fixed[i]] if i in self.fixed else range(K)):
            ks.append(k); self._assign(i + 1, ks); ks.pop()

    def _leaf(self, ks):
        b = self.b
        skip = set(self.fixed) if self.residual else set()
        memo = {}
        def finish(v):
            if v not in memo:
                o = self.opt(v, ks[v])
                d = 0 if v in skip else (int(b.lat_us[o]) * self.mult[int(b.backend[o])]) // 1000
                preds = [u for u in range(self.n) if (int(b.pred_mask[self.n0 + v]) >> u) & 1]
                memo[v] = d + max([finish(u) for u in preds], default=0)
            return memo[v]
        has_succ = set(u for v in range(self.n) for u in range(self.n) if (int(b.pred_mask[self.n0 + v]) >> u) & 1)
        T = max(finish(v) for v in range(self.n) if v not in has_succ)
        logc = 0.0
        D = [0] * b.B
        for v in range(self.n):
            if v in skip:
                continue
            o = self.opt(v, ks[v])
            logc += math.log1p(-float(b.vuln[self.n0 + v]) * (1.0 - float(b.acc[o])))
            D[int(b.backend[o])] += int(b.demand[o])
        feas = T <= int(b.slo_us[self.r]) and (b.cap is None or all(D[x] <= int(b.cap[self.r * b.B + x]) for x in range(b.B)))
        stride, idx = 1, 0
        for v in range(self.n):
            idx += ks[v] * stride
            stride *= int(b.opt_off[self.n0 + v + 1] - b.opt_off[self.n0 + v])
        if feas:
            self.cands.append((math.exp(logc), T, idx, D))


def _check_against_rec(orc_out, rec, cands, tol=1e-12):
    if not cands:
        assert orc_out["status"][rec] == 1
        return
    assert orc_out["status"][rec] == 0
    assert int(orc_out["n_feasible"][rec]) == len(cands)
    cstar = max(c[0] for c in cands)
    assert orc_out["corr"][rec] == pytest.approx(cstar, rel=tol)
    # among candidates whose C is within tol of the best: min T, then min idx
    near = [c for c in cands if c[0] >= cstar * (1 - 1e-9)]
    others = [c for c in cands if c[0] < cstar * (1 - 1e-9)]
    # only decidable when the near-set is an exact-tie class (same factors): they are, for backend-only variants
    want = min(near, key=lambda c: (c[1], c[2]))
    got = (int(orc_out["lat"][rec]), int(orc_out["plan_idx"][rec]))
    if len(set(round(c[0] / cstar, 13) for c in near)) == 1:
        assert got == (want[1], want[2])
        assert [int(x) for x in orc_out["dem"][rec]] == want[3]
    if others and len(near) == 1:
        second = max(o[0] for o in others)
        assert orc_out["runner_corr"][rec] == pytest.approx(second, rel=tol)


def test_pin11_recursive_solver_tiny_instances(orc):
    w = wl.random_workload(11, R=40, nmin=1, nmax=5, kmin=1, kmax=4, L=3, caps=True, tool_p=0.15, slo_q=0.6)
    out = orc.compile(w.batch, w.L, w.mult_pm)
    mult = np.asarray(w.mult_pm).reshape(w.L, w.batch.B)
    assert (out["status"] <= 1).all()
    assert (out["status"] == 0).sum() > 40 and (out["status"] == 1).sum() > 0  # both outcomes exercised
    for r in range(w.batch.R):
        for l in range(w.L):
            _check_against_rec(out, r * w.L + l, RecSolver(w.batch, r, mult[l]).solve())


def test_diamond_cfg0_shape_vs_recursive_solver(orc):
    # BASELINE.json configs[0] shape at reduced radix: the diamond with 4 options per node
    w = wl.make_config(0)
    b = w.batch
    # keep options {0,1,4,5}: 2 models x verifier none x 2 backends ... any 4 of the 8
    keep = [0, 1, 4, 5]
    reqs = [dict(pred_mask=[int(x) for x in b.pred_mask], vuln=[float(x) for x in b.vuln],
                 lat=[[int(b.lat_us[b.opt_off[i] + k]) for k in keep] for i in range(6)],
                 acc=[[float(b.acc[b.opt_off[i] + k]) for k in keep] for i in range(6)],
                 demand=[[int(b.demand[b.opt_off[i] + k]) for k in keep] for i in range(6)],
                 backend=[[int(b.backend[b.opt_off[i] + k]) for k in keep] for i in range(6)],
                 model=[[int(b.model[b.opt_off[i] + k]) for k in keep] for i in range(6)],
                 slo=int(b.slo_us[0]))]
    sb = mk(reqs, 2, 2, False)
    out = orc.compile(sb, w.L, w.mult_pm)
    mult = np.asarray(w.mult_pm).reshape(w.L, 2)
    for l in range(w.L):
        _check_against_rec(out, l, RecSolver(sb, 0, mult[l]).solve())


# ---------------------------------------------------------------- PIN12 replan consistency
# The dispatched set is any predecessor-closed node set (dispatch needs finished predecessors;
# PAPER.md:521-530 App. D: the committed bindings are a set), so each pin runs on prefixes and on general down-sets.
@pytest.mark.parametrize("shape", ["prefix", "downset"])
def test_pin12_replan_consistency(orc, shape):
    w = wl.random_replan_workload(12, R=30, nmin=2, nmax=5, kmin=2, kmax=4, caps=True, shape=shape)
    b = w.batch
    live = w.live_mult_pm.reshape(b.R, b.B)
    out = orc.replan(b, w.dispatched_mask, w.fixed_choice, w.live_mult_pm, wl.FLAG_FIXED_IN_PLACE)
    non_prefix = 0
    for r in range(b.R):
        n = b.n_nodes(r)
        m = int(w.dispatched_mask[r])
        non_prefix += (m & (m + 1)) != 0
        fixed = {i: int(w.fixed_choice[b.node_off[r] + i]) for i in range(n) if (m >> i) & 1}
        # fixed set == compile's enumeration filtered to plans agreeing with the fixed bindings (independent solver)
        _check_against_rec(out, r, RecSolver(b, r, live[r], fixed=fixed).solve())
        if out["status"][r] == 0:
            for i in fixed:      # "the merge rejects overlap instead of replacing a committed binding" PAPER.md:528
                assert int(out["choice"][r][i]) == fixed[i]
        if len(fixed) == n:      # "If U_t is empty, there are no remaining choices" PAPER.md:528
            s = orc.score(b, r, live[r], [fixed[i] for i in range(n)])
            assert (out["status"][r] == 0) == s["feasible"]
            if s["feasible"]:
                assert int(out["plan_idx"][r]) == s["plan_idx"] and out["corr"][r] == s["corr"]
                assert int(out["lat"][r]) == s["lat"] and int(out["n_feasible"][r]) == 1
    assert (non_prefix >= 5) == (shape == "downset")
    # no node dispatched == compile at that single level
    zero = np.zeros(b.R, np.uint32)
    o0 = orc.replan(b, zero, w.fixed_choice, w.live_mult_pm, 0)
    for r in range(b.R):
        oc = orc.compile(b.subset([r]), 1, live[r])
        for key in ("plan_idx", "corr", "lat", "status", "n_feasible"):
            assert o0[key][r] == oc[key][0], key


@pytest.mark.parametrize("shape", ["prefix", "downset"])
def test_pin12_residual_equals_compile_on_induced_subdag(orc, shape):
    w = wl.random_replan_workload(13, R=25, nmin=2, nmax=5, kmin=2, kmax=4, caps=True, flags=wl.FLAG_RESIDUAL, shape=shape)
    b = w.batch
    live = w.live_mult_pm.reshape(b.R, b.B)
    out = orc.replan(b, w.dispatched_mask, w.fixed_choice, w.live_mult_pm, wl.FLAG_RESIDUAL)
    for r in range(b.R):
        n = b.n_nodes(r)
        m = int(w.dispatched_mask[r])
        n0 = int(b.node_off[r])
        U = [v for v in range(n) if not (m >> v) & 1]      # undispatched nodes, in order
        # G[U_t]: the sub-DAG induced by the undispatched nodes; predecessor bits renumbered
        pos = {v: i for i, v in enumerate(U)}
        sub = dict(pred_mask=[sum(1 << pos[u] for u in U if (int(b.pred_mask[n0 + v]) >> u) & 1) for v in U],
                   vuln=[float(b.vuln[n0 + v]) for v in U], slo=int(b.slo_us[r]),
                   cap=[int(x) for x in b.cap[r * b.B:(r + 1) * b.B]])
        for key, arr in (("lat", b.lat_us), ("acc", b.acc), ("demand", b.demand), ("backend", b.backend), ("model", b.model)):
            sub[key] = [[arr[o].item() for o in range(b.opt_off[n0 + v], b.opt_off[n0 + v + 1])] for v in U]
        if not U:
            assert out["status"][r] == 0 and out["corr"][r] == 1.0 and out["lat"][r] == 0
            continue
        oc = orc.compile(mk([sub], b.B, b.M, True), 1, live[r])
        assert out["status"][r] == oc["status"][0]
        assert int(out["n_feasible"][r]) == int(oc["n_feasible"][0])
        if oc["status"][0] == 0:
            assert out["corr"][r] == oc["corr"][0] and int(out["lat"][r]) == int(oc["lat"][0])
            assert (out["dem"][r] == oc["dem"][0]).all()
            assert [int(out["choice"][r][v]) for v in U] == [int(x) for x in oc["choice"][0][: len(U)]]


def test_replan_rejects_non_predecessor_closed_dispatch(orc):
    # node 1 depends on node 0; dispatching node 1 but not node 0 is invalid (reading Q11)
    b = mk([simple_req([0, 1], [[10, 20], [10, 20]])])
    out = orc.replan(b, np.array([0b10], np.uint32), np.array([0, 1], np.uint8), np.array([1000], np.int32), 0)
    assert out["status"][0] == 2
    out = orc.replan(b, np.array([0b01], np.uint32), np.array([5, 1], np.uint8), np.array([1000], np.int32), 0)
    assert out["status"][0] == 2   # fixed_choice >= K_n


# ---------------------------------------------------------------- PIN13 independent MILP, the paper's own style
def milp_best_corr(b, r, mult):
    """Eq.(3) as a MILP: binaries y[n,k]; sum_k y = 1; a_n >= a_u + d(u); T >= a_n + d(n);
    T <= SLO; sum demand*y <= cap_b; maximise sum log f * y.  HiGHS via scipy."""
    from scipy.optimize import Bounds, LinearConstraint, milp
    n0, n = int(b.node_off[r]), b.n_nodes(r)
    offs = [int(b.opt_off[n0 + i]) for i in range(n + 1)]
    ny = offs[n] - offs[0]
    nv = ny + n  # y..., a_0..a_{n-1}
    col = lambda i, k: offs[i] - offs[0] + k
    cobj = np.zeros(nv)
    rows, lo, hi = [], [], []
    for i in range(n):
        row = np.zeros(nv)
        for k in range(offs[i + 1] - offs[i]):
            o = offs[i] + k
            f = 1.0 - float(b.vuln[n0 + i]) * (1.0 - float(b.acc[o]))
            cobj[col(i, k)] = -math.log(max(f, 1e-300))
            row[col(i, k)] = 1
        rows.append(row); lo.append(1); hi.append(1)
    dcoef = lambda i: {col(i, k): (int(b.lat_us[offs[i] + k]) * int(mult[int(b.backend[offs[i] + k])])) // 1000
                       for k in range(offs[i + 1] - offs[i])}
    slo = int(b.slo_us[r])
    for v in range(n):
        for u in range(v):
            if (int(b.pred_mask[n0 + v]) >> u) & 1:      # a_v - a_u - d(u) >= 0
                row = np.zeros(nv); row[ny + v] = 1; row[ny + u] = -1
                for c, d in dcoef(u).items():
                    row[c] = -d
                rows.append(row); lo.append(0); hi.append(np.inf)
        row = np.zeros(nv); row[ny + v] = 1                # a_v + d(v) <= SLO  (T eliminated: T <= SLO)
        for c, d in dcoef(v).items():
            row[c] = d
        rows.append(row); lo.append(-np.inf); hi.append(slo)
    if b.cap is not None:
        for bb in range(b.B):
            row = np.zeros(nv)
            for i in range(n):
                for k in range(offs[i + 1] - offs[i]):
                    if int(b.backend[offs[i] + k]) == bb:
                        row[col(i, k)] = int(b.demand[offs[i] + k])
            rows.append(row); lo.append(-np.inf); hi.append(int(b.cap[r * b.B + bb]))
    integrality = np.concatenate([np.ones(ny), np.zeros(n)])
    bounds = Bounds(np.zeros(nv), np.concatenate([np.ones(ny), np.full(n, np.inf)]))
    res = milp(cobj, constraints=LinearConstraint(np.asarray(rows), lo, hi), integrality=integrality, bounds=bounds,
               options=dict(mip_rel_gap=0.0))
    if res.status == 2 or res.x is None:
        return None
    return math.exp(-res.fun)


def test_pin13_milp_agrees_with_brute_force(orc):
    w = wl.random_workload(1313, R=12, nmin=3, nmax=6, kmin=2, kmax=4, L=2, caps=True, tool_p=0.1, slo_q=0.4)
    out = orc.compile(w.batch, w.L, w.mult_pm)
    mult = np.asarray(w.mult_pm).reshape(w.L, w.batch.B)
    seen_ok = 0
    for r in range(w.batch.R):
        for l in range(w.L):
            c = milp_best_corr(w.batch, r, mult[l])
            rec = r * w.L + l
            if c is None:
                assert out["status"][rec] == 1
            else:
                assert out["status"][rec] == 0
                assert out["corr"][rec] == pytest.approx(c, rel=1e-7)
                seen_ok += 1
    assert seen_ok >= 10


def test_pin13_milp_on_cfg0_diamond_full_size(orc):
    w = wl.make_config(0)
    out = orc.compile(w.batch, w.L, w.mult_pm)
    mult = np.asarray(w.mult_pm).reshape(w.L, w.batch.B)
    for l in range(w.L):
        c = milp_best_corr(w.batch, 0, mult[l])
        assert (c is None) == (out["status"][l] == 1)
        if c is not None:
            assert out["corr"][l] == pytest.approx(c, rel=1e-7)


# ---------------------------------------------------------------- PIN14 select
def test_pin14_select(orc):
    w = wl.random_workload(14, R=20, nmin=2, nmax=5, kmin=2, kmax=4, L=3, caps=True, tool_p=0.1, slo_q=0.5)
    b = w.batch
    out = orc.compile(b, w.L, w.mult_pm)
    mult = np.asarray(w.mult_pm).reshape(w.L, b.B)
    for l in range(w.L):
        sel = orc.select(b, w.L, out["choice"], out["status"], mult[l])
        for r in range(b.R):
            recs = [r * w.L + x for x in range(w.L) if out["status"][r * w.L + x] == 0]
            if not recs:
                assert sel["variant"][r] == -1
                continue
            v = int(sel["variant"][r])
            assert out["status"][r * w.L + v] == 0
            if out["status"][r * w.L + l] == 0:
                # variant l re-scores to its stored T under its own multipliers and is feasible
                s = orc.score(b, r, mult[l], out["choice"][r * w.L + l][: b.n_nodes(r)])
                assert s["lat"] == out["lat"][r * w.L + l] and s["feasible"]
                assert sel["feasible"][r] == 1
                assert sel["corr"][r] >= out["corr"][r * w.L + l]
    # hand case: two stored variants, live vector makes the high-C one miss the SLO
    r = simple_req([0], [[100, 400]], vuln=[1.0], acc=[[0.5, 0.9]], slo=500)
    b1 = mk([r])
    choice = np.full((2, 16), 0xFF, np.uint8); choice[0, 0] = 1; choice[1, 0] = 0
    st = np.zeros(2, np.uint8)
    assert orc.select(b1, 2, choice, st, [1000])["variant"][0] == 0      # both feasible -> higher C
    assert orc.select(b1, 2, choice, st, [2000])["variant"][0] == 1      # 800 > 500 -> the feasible one
    s = orc.select(b1, 2, choice, st, [9000])                            # none feasible -> min T'
    assert s["variant"][0] == 1 and s["feasible"][0] == 0 and s["lat"][0] == 900
    st[1] = 1
    assert orc.select(b1, 2, choice, st, [9000])["variant"][0] == 0      # only stored variant
    st[0] = 1
    assert orc.select(b1, 2, choice, st, [1000])["variant"][0] == -1     # empty bundle


# ---------------------------------------------------------------- validation, caps, tie order, threads
def test_validation_statuses(orc):
    good = simple_req([0, 1], [[10, 20], [10, 20]])
    def status_of(mut, B=1, M=1, caps=False, L=1, mult=(1000,)):
        q = {k: (list(map(list, v)) if isinstance(v, list) and v and isinstance(v[0], list) else (list(v) if isinstance(v, list) else v))
             for k, v in good.items()}
        mut(q)
        return int(orc.compile(mk([q], B, M, caps), L, list(mult))["status"][0])
    assert status_of(lambda q: None) == 0
    assert status_of(lambda q: q.__setitem__("pred_mask", [0, 0b10])) == 2          # self/forward edge
    assert status_of(lambda q: q.__setitem__("pred_mask", [1, 0])) == 2
    assert status_of(lambda q: q.__setitem__("vuln", [float("nan"), 0.5])) == 2
    assert status_of(lambda q: q.__setitem__("vuln", [1.5, 0.5])) == 2
    assert status_of(lambda q: q["acc"].__setitem__(0, [0.9, -0.1])) == 2
    assert status_of(lambda q: q["lat"].__setitem__(1, [10, -1])) == 2
    assert status_of(lambda q: q["demand"].__setitem__(1, [10, -1])) == 2
    assert status_of(lambda q: q["backend"].__setitem__(0, [0, 1])) == 2            # backend >= B
    assert status_of(lambda q: q["model"].__setitem__(0, [0, 3])) == 2
    assert status_of(lambda q: q["lat"].__setitem__(0, [2**31 - 1, 5]), mult=(3000,)) == 2   # overflow (Q19)
    assert status_of(lambda q: q.__setitem__("slo", -1)) == 2
    # other requests in the batch still compile
    bad = dict(good); bad["vuln"] = [2.0, 0.1]
    out = orc.compile(mk([bad, good]), 1, [1000])
    assert list(out["status"]) == [2, 0]


def test_caps_are_inclusive_and_per_backend(orc):
    r = simple_req([0, 0], [[10, 10], [10, 10]], vuln=[1.0, 1.0], acc=[[0.5, 0.9], [0.5, 0.9]],
                   demand=[[5, 50], [5, 50]], backend=[[0, 1], [0, 1]], slo=100, cap=[10, 50])
    out = orc.compile(mk([r], 2, 1, True), 1, [1000, 1000])
    # both on backend 1 would be best (0.81) but needs 100 > 50; exactly one on backend 1 is allowed (50 <= 50)
    assert out["corr"][0] == pytest.approx(float(np.float32(0.9)) * float(np.float32(0.5)))
    assert int(out["plan_idx"][0]) == 1 and [int(x) for x in out["dem"][0]] == [5, 50]
    assert int(out["n_feasible"][0]) == 3


def test_slo_is_inclusive(orc):
    r = simple_req([0], [[100, 101]], vuln=[1.0], acc=[[0.5, 0.9]], slo=101)
    assert int(orc.compile(mk([r]), 1, [1000])["plan_idx"][0]) == 1
    r["slo"] = 100
    assert int(orc.compile(mk([r]), 1, [1000])["plan_idx"][0]) == 0


def test_inner_and_outer_parallel_paths_agree(orc):
    # R >= 4*threads takes the parallel-over-requests path; subsets of one request take the
    # parallel-over-index-chunks path.  The order is total, so both must give identical records.
    w = wl.make_config(1, R=2)
    small = wl.random_workload(77, R=40, nmin=3, nmax=6, kmin=2, kmax=4, L=2)
    a = orc.compile(small.batch, small.L, small.mult_pm)
    for r in range(0, small.batch.R, 7):
        o = orc.compile(small.batch.subset([r]), small.L, small.mult_pm)
        for key in ("plan_idx", "corr", "lat", "status", "n_feasible", "runner_idx"):
            assert (o[key] == a[key][r * small.L:(r + 1) * small.L]).all(), key


def test_canonical_index_and_choice_are_consistent(orc):
    w = wl.random_workload(21, R=10, nmin=2, nmax=6, kmin=1, kmax=5, L=2, tool_p=0.2)
    out = orc.compile(w.batch, w.L, w.mult_pm)
    for r in range(w.batch.R):
        rad = w.batch.radices(r)
        for l in range(w.L):
            rec = r * w.L + l
            if out["status"][rec] != 0:
                continue
            idx, stride = 0, 1
            for i, k in enumerate(rad):
                idx += int(out["choice"][rec][i]) * stride; stride *= int(k)
            assert idx == int(out["plan_idx"][rec])
            assert (out["choice"][rec][len(rad):] == 0xFF).all()
