"""Pins of oracle/linear_oracle.c (the paper's linear objective, Eq.(4)/(5)) against what the paper
and the mathematics fix: the reach-weight formula and its special case, the worked fork-join numbers of
Fig. 7(a) and the preference flip of Fig. 7(b), the algebraic identity of
PAPER.md:199, an independent MILP in the paper's own formulation (HiGHS), an independent itertools + networkx brute
force, separable special cases and the parametric monotonicity of D_tau in the level."""
from __future__ import annotations

import itertools
import math

import numpy as np
import pytest

from conftest import read_golden
from oracle import linear as lo
from support import workloads as wl

P0 = dict(lambda_f=0.5, lambda_c=0.1, lambda_l=0.0005, lambda_ld=0.0002, beta=0.5, effort=1.0)


def rand_case(seed, R=6, nmin=2, nmax=5, kmin=2, kmax=4):
    w = wl.random_workload(seed, R=R, nmin=nmin, nmax=nmax, kmin=kmin, kmax=kmax, B=2, M=2, L=1, caps=False)
    rng = np.random.default_rng(seed + 1)
    cost = rng.uniform(0.0, 1.0, size=w.batch.lat_us.size).astype(np.float32)
    return w.batch, cost


# ---- L1: reach weights -----------------------------------------------------------------------------------------------
def test_reach_weight_formula_and_single_node_case():
    assert lo.reach_weights([0], 0.7, 1.0).tolist() == [1.0]                      # "for a single-node workflow rho = 1"
    # chain 0 -> 1 -> 2 -> 3: |R(n)| = 4 - n
    rho = lo.reach_weights([0, 0b1, 0b10, 0b100], 0.6, 0.5)
    assert np.allclose(rho, [1 + 0.3 * 3 / 3, 1 + 0.3 * 2 / 3, 1 + 0.3 * 1 / 3, 1.0])
    # diamond 0 -> {1, 2} -> 3
    rho = lo.reach_weights([0, 0b1, 0b1, 0b110], 1.0, 1.0)
    assert np.allclose(rho, [1 + 3 / 3, 1 + 1 / 3, 1 + 1 / 3, 1.0])
    # effort 0 or beta 0 switch the emphasis off
    assert np.allclose(lo.reach_weights([0, 1, 3], 0.9, 0.0), 1.0) and np.allclose(lo.reach_weights([0, 1, 3], 0.0, 1.0), 1.0)


def test_reach_sets_equal_networkx_descendants():
    import networkx as nx
    rng = np.random.default_rng(5)
    for _ in range(20):
        n = int(rng.integers(2, 12))
        pm = [int(rng.integers(0, 1 << i)) if i else 0 for i in range(n)]
        g = nx.DiGraph()
        g.add_nodes_from(range(n))
        for v in range(n):
            for u in range(v):
                if (pm[v] >> u) & 1:
                    g.add_edge(u, v)
        rho = lo.reach_weights(pm, 1.0, 1.0)
        for v in range(n):
            assert rho[v] == pytest.approx(1.0 + len(nx.descendants(g, v)) / (n - 1))


# ---- Fig. 7: the paper's worked example ----------------------------------------------------------------------------
def fig7_batch():
    """Nodes: C (CodeGen) and D (TestGen) in parallel, "common stages omitted" (Fig. 7(a)).  Options and nominal time
    units from the table: C in {27B+V [10+4], 27B [10], 9B [6]}, D in {9B+V [4+3], 9B [4]}."""
    reqs = [dict(pred_mask=[0, 0], vuln=np.array([0.5, 0.5], np.float32),
                 lat=[[14, 10, 6], [7, 4]], acc=[[0.93, 0.90, 0.80], [0.90, 0.78]], demand=[[1, 1, 1], [1, 1]],
                 backend=[[0, 0, 0], [0, 0]], model=[[0, 0, 1], [1, 1]], slo=100, cap=None)]
    return wl.batch_from_requests(reqs, 1, 2, False)


def test_fig7a_fork_latency_and_duration_sums():
    b = fig7_batch()
    cost = np.zeros(5, np.float32)
    rows = read_golden("paper_fig7_forkjoin.txt")
    opt_c = {14: 0, 10: 1, 6: 2}               # d(C): 27B+V [10+4], 27B [10], 9B [6]
    opt_d = {7: 0, 4: 1}                        # d(D): 9B+V [4+3], 9B [4]
    seen = 0
    for row in rows:
        c, d, fork, dsum = int(row[1]), int(row[2]), int(row[3]), int(row[4])
        s = lo.score(b, cost, P0, 0, 0.0, [opt_c[c], opt_d[d]] + [255] * 14)
        assert (s["T"], s["Dtau"]) == (fork, dsum), row
        seen += 1
    assert seen == 4


def test_fig7b_preference_flips_with_the_demand_penalty():
    # "pi(0) Preferred C: 27B . D: 9B + V -- avoid unnecessary verification";
    # "pi(1) Pressure variant C: 9B . D: 9B -- lower demand; quality trade-off"
    b = fig7_batch()
    cost = np.array([0.3, 0.2, 0.1, 0.15, 0.1], np.float32)
    p = dict(lambda_f=0.4, lambda_c=0.05, lambda_l=0.01, lambda_ld=0.02, beta=0.0, effort=0.0)
    out = lo.compile(b, cost, p, [0.0, 1.5, 3.0])
    ch = out["choice"].reshape(3, 16)
    assert ch[0, :2].tolist() == [1, 0]            # (27B, 9B+V) at L = 0: verifying C would add 4 units to T for +0.03 quality
    assert ch[2, :2].tolist() == [2, 1]            # (9B, 9B) at the highest level
    assert out["Dtau"].tolist()[0] == 17 and out["Dtau"].tolist()[2] == 10 and out["T"].tolist()[0] == 10
    # "verification that fits within branch slack leaves T unchanged but still adds calls"
    a = lo.score(b, cost, p, 0, 0.0, [1, 1] + [255] * 14)
    v = lo.score(b, cost, p, 0, 0.0, [1, 0] + [255] * 14)
    assert a["T"] == v["T"] == 10 and v["Dtau"] == a["Dtau"] + 3


# ---- algebra -------------------------------------------------------------------------------------------------------
def test_identity_quality_and_error_terms_weight_correctness_by_rho_plus_lambda_f_v():
    # "the quality and error terms equivalently weight local correctness by rho(n) + lambda_f v_n, up to a
    # plan-independent constant"
    b, cost = rand_case(3)
    for r in range(b.R):
        n0, N = int(b.node_off[r]), b.n_nodes(r)
        rho = lo.reach_weights(b.pred_mask[n0:n0 + N], P0["beta"], P0["effort"])
        Ks = [int(b.opt_off[n0 + n + 1] - b.opt_off[n0 + n]) for n in range(N)]
        consts = set()
        for plan in itertools.islice(itertools.product(*[range(k) for k in Ks]), 50):
            s = lo.score(b, cost, P0, r, 1.0, list(plan) + [255] * (16 - N))
            alt = 0.0
            for n, k in enumerate(plan):
                o = int(b.opt_off[n0 + n]) + k
                alt += (rho[n] + P0["lambda_f"] * float(b.vuln[n0 + n])) * float(b.acc[o]) - P0["lambda_c"] * float(cost[o])
            alt -= P0["lambda_l"] * s["T"] + P0["lambda_ld"] * 1.0 * s["Dtau"]
            consts.add(round(s["J"] - alt, 9))
        assert len(consts) == 1
        assert consts.pop() == pytest.approx(-P0["lambda_f"] * float(np.sum(b.vuln[n0:n0 + N].astype(np.float64))), abs=1e-8)


def test_separable_special_case_and_level_zero():
    # all penalties off: J = sum_n q  ->  each node takes its best-quality option, J* = sum of per-node maxima
    b, cost = rand_case(4)
    p = dict(lambda_f=0.0, lambda_c=0.0, lambda_l=0.0, lambda_ld=0.0, beta=0.0, effort=0.0)
    out = lo.compile(b, cost, p, [0.0])
    for r in range(b.R):
        n0, N = int(b.node_off[r]), b.n_nodes(r)
        best = sum(float(b.acc[int(b.opt_off[n0 + n]): int(b.opt_off[n0 + n + 1])].astype(np.float64).max()) for n in range(N))
        assert out["J"][r] == pytest.approx(best, abs=1e-12)
    # only the latency charge: the winner minimises T, then the canonical index
    p = dict(p, lambda_l=1.0)
    out = lo.compile(b, cost, p, [0.0])
    for r in range(b.R):
        n0, N = int(b.node_off[r]), b.n_nodes(r)
        Ks = [int(b.opt_off[n0 + n + 1] - b.opt_off[n0 + n]) for n in range(N)]
        bestT = min(lo.score(b, cost, p, r, 0.0, list(pl) + [255] * (16 - N))["T"] - sum(
            float(b.acc[int(b.opt_off[n0 + n]) + k]) for n, k in enumerate(pl)) for pl in itertools.product(*[range(k) for k in Ks]))
        assert -out["J"][r] == pytest.approx(bestT, abs=1e-9)


def test_demand_of_the_chosen_plan_is_non_increasing_in_the_level():
    # parametric optimisation: raising the weight of D_tau can only lower the optimiser's D_tau
    b, cost = rand_case(6, R=10)
    out = lo.compile(b, cost, P0, [0.0, 0.5, 1.0, 2.0, 4.0, 8.0])
    D = out["Dtau"].reshape(b.R, 6)
    assert (np.diff(D, axis=1) <= 0).all()
    assert (np.diff(D, axis=1) < 0).any()


# ---- independent solvers -------------------------------------------------------------------------------------------
def brute_force(b, cost, p, r, level):
    import networkx as nx
    n0, N = int(b.node_off[r]), b.n_nodes(r)
    g = nx.DiGraph()
    g.add_nodes_from(range(N))
    for v in range(N):
        for u in range(v):
            if (int(b.pred_mask[n0 + v]) >> u) & 1:
                g.add_edge(u, v)
    rho = [1.0 + p["beta"] * p["effort"] * len(nx.descendants(g, v)) / (N - 1) if N > 1 else 1.0 for v in range(N)]
    Ks = [int(b.opt_off[n0 + n + 1] - b.opt_off[n0 + n]) for n in range(N)]
    best = None
    for plan in itertools.product(*[range(k) for k in Ks]):
        W, dur = 0.0, []
        for n, k in enumerate(plan):
            o = int(b.opt_off[n0 + n]) + k
            q, v = float(b.acc[o]), float(b.vuln[n0 + n])
            W += rho[n] * q - p["lambda_f"] * v * (1 - q) - p["lambda_c"] * float(cost[o])
            dur.append(int(b.lat_us[o]))
        h = nx.DiGraph()
        h.add_node("s")
        for v in range(N):
            h.add_edge("s", ("in", v), weight=0)
            h.add_edge(("in", v), ("out", v), weight=dur[v])
            for u in g.predecessors(v):
                h.add_edge(("out", u), ("in", v), weight=0)
        T = nx.dag_longest_path_length(h, weight="weight")
        J = W - p["lambda_l"] * T - p["lambda_ld"] * level * sum(dur)
        idx = sum(k * int(np.prod(Ks[:n])) for n, k in enumerate(plan))
        key = (-J, T, idx)
        if best is None or key < best[0]:
            best = (key, J, T, sum(dur), idx)
    return best[1:]


def test_against_itertools_and_networkx_brute_force():
    b, cost = rand_case(7, R=5, nmax=4, kmax=3)
    out = lo.compile(b, cost, P0, [0.0, 2.0])
    for r in range(b.R):
        for li, lv in enumerate((0.0, 2.0)):
            J, T, D, idx = brute_force(b, cost, P0, r, lv)
            rec = r * 2 + li
            assert out["J"][rec] == pytest.approx(J, abs=1e-9)
            assert (out["T"][rec], out["Dtau"][rec], int(out["plan_idx"][rec])) == (T, D, idx)


def milp_linear(b, cost, p, r, level):
    """Eq.(3)-(5) as the paper writes them: binaries y, start times a_n, completion T; HiGHS via scipy."""
    from scipy.optimize import Bounds, LinearConstraint, milp
    n0, N = int(b.node_off[r]), b.n_nodes(r)
    offs = [int(b.opt_off[n0 + i]) for i in range(N + 1)]
    ny = offs[N] - offs[0]
    nv = ny + N + 1                         # y..., a_0..a_{N-1}, T
    rho = lo.reach_weights(b.pred_mask[n0:n0 + N], p["beta"], p["effort"])
    c = np.zeros(nv)
    rows, lo_, hi_ = [], [], []
    for i in range(N):
        row = np.zeros(nv)
        for k in range(offs[i + 1] - offs[i]):
            o = offs[i] + k
            q, v = float(b.acc[o]), float(b.vuln[n0 + i])
            w = rho[i] * q - p["lambda_f"] * v * (1 - q) - p["lambda_c"] * float(cost[o])
            c[o - offs[0]] = -(w - p["lambda_ld"] * level * int(b.lat_us[o]))
            row[o - offs[0]] = 1
        rows.append(row); lo_.append(1); hi_.append(1)
    c[ny + N] = p["lambda_l"]
    for v in range(N):
        for u in range(v):
            if (int(b.pred_mask[n0 + v]) >> u) & 1:            # a_v >= a_u + d(u)
                row = np.zeros(nv); row[ny + v] = 1; row[ny + u] = -1
                for k in range(offs[u + 1] - offs[u]):
                    row[offs[u] + k - offs[0]] = -int(b.lat_us[offs[u] + k])
                rows.append(row); lo_.append(0); hi_.append(np.inf)
        row = np.zeros(nv); row[ny + N] = 1; row[ny + v] = -1    # T >= a_v + d(v)
        for k in range(offs[v + 1] - offs[v]):
            row[offs[v] + k - offs[0]] = -int(b.lat_us[offs[v] + k])
        rows.append(row); lo_.append(0); hi_.append(np.inf)
    integrality = np.concatenate([np.ones(ny), np.zeros(N + 1)])
    bounds = Bounds(np.zeros(nv), np.concatenate([np.ones(ny), np.full(N + 1, np.inf)]))
    res = milp(c, constraints=LinearConstraint(np.asarray(rows), lo_, hi_), integrality=integrality, bounds=bounds,
               options=dict(mip_rel_gap=0.0))
    assert res.status == 0
    return -res.fun


def test_against_the_papers_own_milp():
    b, cost = rand_case(8, R=6, nmin=3, nmax=6, kmax=4)
    levels = [0.0, 1.5, 3.0]
    out = lo.compile(b, cost, P0, levels)
    for r in range(b.R):
        for li, lv in enumerate(levels):
            assert out["J"][r * 3 + li] == pytest.approx(milp_linear(b, cost, P0, r, lv), abs=1e-6)


def test_invalid_requests_are_flagged():
    b, cost = rand_case(9)
    b.vuln[int(b.node_off[2])] = np.nan
    cost[int(b.opt_off[int(b.node_off[4])])] = -1.0
    out = lo.compile(b, cost, P0, [0.0])
    assert out["status"].tolist() == [0, 0, 2, 0, 2, 0]
