"""-m gpu: the CUDA path (through the C ABI of include/dyplan.h) against the fp64 oracle, record by record.

Sizes are chosen so the oracle finishes in seconds yet every case spans many work items, several inner
tiles and a ragged tail.  Full BASELINE.json sizes are covered in test_gpu_full_size.py.
"""
from __future__ import annotations

import numpy as np
import pytest

from support import workloads as wl

from parity import check_records

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def dy():
    import torch
    assert torch.cuda.is_available(), "-m gpu tests need a CUDA device"
    from paper_2607_02942_b200 import binding
    ctx = binding.Context(0)
    yield binding, ctx
    ctx.close()


RECORD_KEYS = ("status", "plan_idx", "choice", "corr", "corr64", "lat", "dem", "dom_model")


def gpu_run(dy, w, corr64=True):
    """One call through the C ABI.  A call of at most 32 requests runs twice: as it stands (small requests take the
    admission-path kernel k_small) and with DYPLAN_NO_SMALL_PATH (everything through the batched scorers); the two
    must agree bit for bit, and the batched result is returned (dyplan_last_stats then describes that call)."""
    import torch
    binding, ctx = dy
    dw = binding.upload(w, "cuda:0", corr64)
    binding.launch(ctx, dw)
    torch.cuda.synchronize()
    g = dw.out.host()
    if w.batch.R <= 32 and not (ctx.flags & binding.NO_SMALL_PATH):
        f0 = ctx.flags
        n_small = ctx.dyplan_last_stats()["small_requests"]
        ctx.dyplan_set_flags(f0 | binding.NO_SMALL_PATH)
        try:
            dw2 = binding.upload(w, "cuda:0", corr64)
            binding.launch(ctx, dw2)
            torch.cuda.synchronize()
            g2 = dw2.out.host()
        finally:
            ctx.dyplan_set_flags(f0)
        for k in RECORD_KEYS:
            if g[k] is not None:
                assert np.array_equal(g[k], g2[k]), f"{w.name}: {k} differs between the small path ({n_small} requests) and the batched scorers"
        return g2
    return g


def both(dy, orc, w, where):
    g = gpu_run(dy, w)
    ref = orc.run(w)
    c = check_records(orc, w, g, ref, where=where)
    return g, ref, c


# ---- BASELINE.json configs, down-scaled where the oracle needs it --------------------------------------------------
def test_cfg0_diamond_full(dy, orc):
    w = wl.make_config(0)
    g, ref, c = both(dy, orc, w, "cfg0")
    assert c["records"] == 3
    assert (ref["status"] == 0).any()


def test_cfg1_prefix(dy, orc):
    w = wl.make_config(1, R=3)      # 3 x 8^8 plans x 4 levels
    both(dy, orc, w, "cfg1[3]")


def test_cfg2_prefix(dy, orc):
    w = wl.make_config(2, R=24)     # 24 x 8^7 plans x 4 levels, caps
    both(dy, orc, w, "cfg2[24]")


def test_cfg3_prefix_both_flags(dy, orc):
    w = wl.make_config(3, R=96)
    # keep the oracle in seconds: drop the 12^7 queries (2 dispatched) from this case
    keep = [r for r in range(w.batch.R) if bin(int(w.dispatched_mask[r])).count("1") >= 3][:40]
    w = w.subset(keep)
    both(dy, orc, w, "cfg3[fixed-in-place]")
    w.flags = wl.FLAG_RESIDUAL
    both(dy, orc, w, "cfg3[residual]")


def test_cfg4_shape_reduced_nodes(dy, orc):
    # cfg4's option structure (3 models x 2 verifiers, backend = model, B = 3, 8 levels, caps) at N = 9
    full = wl.make_config(4, R=2)
    rng = np.random.default_rng(44)
    reqs = []
    for r in range(2):
        n = 9
        pm = wl.layered_pred_masks(rng, n, 4, 0.5)
        a, e = int(full.batch.node_off[r]), int(full.batch.node_off[r]) + n
        oa, oe = int(full.batch.opt_off[a]), int(full.batch.opt_off[e])
        K = 6
        reqs.append(dict(pred_mask=pm, vuln=full.batch.vuln[a:e],
                         lat=full.batch.lat_us[oa:oe].reshape(n, K), acc=full.batch.acc[oa:oe].reshape(n, K),
                         demand=full.batch.demand[oa:oe].reshape(n, K), backend=full.batch.backend[oa:oe].reshape(n, K),
                         model=full.batch.model[oa:oe].reshape(n, K), slo=int(full.batch.slo_us[r] * 0.8),
                         cap=(full.batch.cap.reshape(-1, 3)[r] * 0.8).astype(np.int32)))
    b = wl.batch_from_requests(reqs, 3, 3, True)
    w = wl.Workload(name="cfg4-n9", kind="compile", batch=b, L=8, mult_pm=full.mult_pm)
    both(dy, orc, w, "cfg4-n9")


# ---- ragged, free-form cases --------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed,L,B,caps", [(1, 1, 1, False), (2, 2, 2, True), (3, 3, 3, True), (4, 4, 2, False),
                                           (5, 5, 5, True), (6, 6, 2, True), (7, 7, 8, True), (8, 8, 4, False)])
def test_random_ragged(dy, orc, seed, L, B, caps):
    w = wl.random_workload(seed, R=40, nmin=1, nmax=7, kmin=1, kmax=7, B=B, M=min(B + 1, 8), L=L, caps=caps)
    both(dy, orc, w, f"ragged(seed={seed})")


@pytest.mark.parametrize("seed", [11, 12])
def test_random_wide_options(dy, orc, seed):
    # K up to 16 (every inner radix class), few nodes
    w = wl.random_workload(seed, R=24, nmin=2, nmax=5, kmin=9, kmax=16, B=2, M=3, L=3, caps=True, tool_p=0.0)
    both(dy, orc, w, f"wide(seed={seed})")


@pytest.mark.parametrize("seed", [21, 22])
def test_random_many_nodes_tool_nodes(dy, orc, seed):
    # up to 14 nodes, most of them tool nodes (K = 1), arbitrary DAGs
    w = wl.random_workload(seed, R=12, nmin=10, nmax=14, kmin=2, kmax=3, B=2, M=3, L=2, caps=True, tool_p=0.45,
                           edge_p=0.3)
    both(dy, orc, w, f"deep(seed={seed})")


@pytest.mark.parametrize("seed,flags", [(31, wl.FLAG_FIXED_IN_PLACE), (32, wl.FLAG_RESIDUAL),
                                        (33, wl.FLAG_FIXED_IN_PLACE), (34, wl.FLAG_RESIDUAL)])
def test_random_replan(dy, orc, seed, flags):
    w = wl.random_replan_workload(seed, R=48, nmin=1, nmax=8, kmin=1, kmax=6, B=3, M=3, caps=True, flags=flags)
    g, ref, c = both(dy, orc, w, f"replan(seed={seed})")
    # the cases the paper singles out: nothing left to choose / everything left to choose
    nd = np.array([bin(int(m)).count("1") for m in w.dispatched_mask])
    nn = np.array([w.batch.n_nodes(r) for r in range(w.batch.R)])
    assert (nd == nn).any() and (nd == 0).any()


@pytest.mark.parametrize("seed,flags", [(35, wl.FLAG_FIXED_IN_PLACE), (36, wl.FLAG_RESIDUAL), (37, wl.FLAG_FIXED_IN_PLACE)])
def test_random_replan_non_prefix_down_sets(dy, orc, seed, flags):
    """Dispatched sets that are predecessor-closed but NOT a prefix of the node order (nodes {0, 2} when 2 does not
    depend on 1): valid under include/dyplan.h and App. D; k_stage's orientation, pinned node 0
    and base_idx paths differ from the prefix case."""
    w = wl.random_replan_workload(seed, R=64, nmin=3, nmax=9, kmin=1, kmax=5, B=3, M=3, caps=(seed != 37), flags=flags,
                                  shape="downset")
    m = w.dispatched_mask.astype(np.int64)
    assert ((m & (m + 1)) != 0).sum() >= 16, "too few non-prefix sets drawn"
    # node 0 free while later nodes are pinned, and the last node pinned while earlier ones are free
    nn = np.array([w.batch.n_nodes(r) for r in range(w.batch.R)])
    assert (((m & 1) == 0) & (m != 0)).any() and (((m >> (nn - 1)) & 1 == 1) & (m != (1 << nn) - 1)).any()
    both(dy, orc, w, f"replan-downsets(seed={seed})")


def test_cfg3_shape_non_prefix_down_sets_both_flags(dy, orc):
    base = wl.make_config(3, R=160)
    for flags in (wl.FLAG_FIXED_IN_PLACE, wl.FLAG_RESIDUAL):
        w = wl.with_down_set_dispatch(base, seed=77, max_free_plans=12 ** 5, flags=flags)
        m = w.dispatched_mask.astype(np.int64)
        assert ((m & (m + 1)) != 0).sum() >= 60
        both(dy, orc, w, f"cfg3-downsets(flags={flags})")


def test_slo_sweep_monotone_and_infeasible(dy, orc):
    # SLO below the smallest possible T => INFEASIBLE at every level; huge SLO, no caps => separable optimum
    w = wl.random_workload(41, R=6, nmin=4, nmax=6, kmin=3, kmax=5, B=2, M=2, L=3, caps=False)
    w.batch.slo_us[:] = 0
    w.batch.lat_us[:] = np.maximum(w.batch.lat_us, 1)
    g, ref, _ = both(dy, orc, w, "slo=0")
    assert (g["status"] == 1).all()
    w.batch.slo_us[:] = 2**31 - 1
    g, ref, _ = both(dy, orc, w, "slo=max")
    assert (g["status"] == 0).all()
    for r in range(w.batch.R):
        a, e = w.batch.node_off[r], w.batch.node_off[r + 1]
        best = 1.0
        for n in range(a, e):
            f = 1.0 - float(w.batch.vuln[n]) * (1.0 - w.batch.acc[w.batch.opt_off[n]: w.batch.opt_off[n + 1]].astype(np.float64))
            best *= f.max()
        assert abs(g["corr64"][r * 3] - best) <= 1e-12 * best     # PIN8 on the GPU path


def test_all_vulnerabilities_zero_tie_break(dy, orc):
    # C == 1 for every plan: the winner is the (T asc, idx asc) minimum, bit-exact index (order 7)
    w = wl.random_workload(42, R=8, nmin=3, nmax=6, kmin=2, kmax=6, B=2, M=2, L=4, caps=True)
    w.batch.vuln[:] = 0.0
    g, ref, c = both(dy, orc, w, "v=0")
    assert c["within_tol"] == 0
    ok = ref["status"] == 0
    assert (g["plan_idx"][ok] == ref["plan_idx"][ok]).all()
    assert (g["corr"][ok] == 1.0).all()


def test_duplicate_options_exact_ties(dy, orc):
    # backend-only variants tie in C (quality does not depend on the backend): T then idx decides
    w = wl.make_config(1, R=2)
    b = w.batch
    b.acc[:] = np.round(b.acc * 8) / 8          # few distinct accuracies -> many exact C ties
    b.vuln[:] = np.round(b.vuln * 4) / 4
    g, ref, c = both(dy, orc, w, "ties")


# ---- the admission path: small calls (k_small) ------------------------------------------------------------------------
def test_small_call_path_takes_small_requests_only(dy, orc):
    import torch
    binding, ctx = dy
    # configs[0] alone: one launch pair (stage + small) through the host entry point, and through the device one too:
    # the sizes in the struct bound the plan count (max_n min(KK / n, 16)^n x L = 8^6 x 3 <= 2^21), so the batched scorers are not launched
    w = wl.make_config(0)
    dw = binding.upload(w)
    binding.launch(ctx, dw)
    torch.cuda.synchronize()
    st = ctx.dyplan_last_stats()
    assert st["small_requests"] == 1 and st["fast_requests"] == 0 and st["plans"] == w.n_plans_total() and st["launches"] == 2
    check_records(orc, w, dw.out.host(), orc.run(w), where="small cfg0")
    # the same shape with 8 levels: the bound x L = 2^21 exactly, which 20.99 bits do not cover -- the device call then
    # launches all six kernels although k_stage finds the request small (the bound is deliberately on the safe side)
    w8 = wl.random_workload(302, R=1, nmin=6, nmax=6, kmin=8, kmax=8, B=2, M=2, L=8, caps=False, tool_p=0.0)
    dw8 = binding.upload(w8)
    binding.launch(ctx, dw8)
    torch.cuda.synchronize()
    st = ctx.dyplan_last_stats()
    assert st["small_requests"] == 1 and st["launches"] == 6 and st["plans"] == 8**6
    check_records(orc, w8, dw8.out.host(), orc.run(w8), where="small 8^6 x 8")
    g, _, _ = binding.run_host(ctx, w)
    st = ctx.dyplan_last_stats()
    assert st["launches"] == 2 and st["small_requests"] == 1 and st["plans"] == w.n_plans_total()
    check_records(orc, w, g, orc.run(w), where="small cfg0 host")
    # a call that mixes one large request (8^8 x 4 evaluations: batched scorers) with small ones
    big = wl.make_config(1, R=1)
    small = wl.random_workload(301, R=5, nmin=1, nmax=5, kmin=1, kmax=6, B=2, M=2, L=4, caps=False)
    b1, b2 = big.batch, small.batch
    cat = lambda x, y: np.concatenate([x, y])
    batch = wl.Batch(R=6, B=2, M=2, node_off=cat(b2.node_off, b2.node_off[-1] + b1.node_off[1:]).astype(np.int32),
                     opt_off=cat(b2.opt_off, b2.opt_off[-1] + b1.opt_off[1:]).astype(np.int32),
                     pred_mask=cat(b2.pred_mask, b1.pred_mask), vuln=cat(b2.vuln, b1.vuln), lat_us=cat(b2.lat_us, b1.lat_us),
                     acc=cat(b2.acc, b1.acc), demand=cat(b2.demand, b1.demand), backend=cat(b2.backend, b1.backend),
                     model=cat(b2.model, b1.model), slo_us=cat(b2.slo_us, b1.slo_us), cap=None)
    reqs = wl.Workload(name="mixed-small", kind="compile", batch=batch, L=4, mult_pm=big.mult_pm.copy())
    dw = binding.upload(reqs)
    binding.launch(ctx, dw)
    torch.cuda.synchronize()
    st = ctx.dyplan_last_stats()
    assert st["small_requests"] == 5 and st["fast_requests"] == 1 and st["plans"] == reqs.n_plans_total()
    check_records(orc, reqs, dw.out.host(), orc.run(reqs), where="mixed small + large")
    g, _, _ = binding.run_host(ctx, reqs)
    assert ctx.dyplan_last_stats()["launches"] == 6           # not all small: the batched scorers run too
    check_records(orc, reqs, g, orc.run(reqs), where="mixed small + large, host")


@pytest.mark.parametrize("seed,L,B,caps", [(311, 1, 1, False), (312, 3, 2, True), (313, 8, 3, True), (314, 4, 8, True)])
def test_small_call_path_ragged(dy, orc, seed, L, B, caps):
    # everything k_small must get right on its own: ragged N and K, tool nodes, caps with up to 8 backends, invalid and
    # infeasible requests, replans in both modes (the helper compares with the batched scorers, then with the oracle)
    w = wl.random_workload(seed, R=30, nmin=1, nmax=6, kmin=1, kmax=7, B=B, M=3, L=L, caps=caps)
    w.batch.slo_us[3] = 0                      # infeasible
    w.batch.vuln[int(w.batch.node_off[5])] = np.nan     # invalid
    g = gpu_run(dy, w)
    check_records(orc, w, g, orc.run(w), where=f"small-ragged(seed={seed})")
    for flags in (wl.FLAG_FIXED_IN_PLACE, wl.FLAG_RESIDUAL):
        wr = wl.random_replan_workload(seed + 50, R=28, nmin=1, nmax=7, kmin=1, kmax=6, B=B, M=3, caps=caps, flags=flags)
        check_records(orc, wr, gpu_run(dy, wr), orc.run(wr), where=f"small-replan(seed={seed})")


@pytest.mark.parametrize("seed,L,B,caps,nmin,nmax", [(321, 2, 2, True, 9, 12), (322, 8, 3, False, 13, 16), (323, 3, 8, True, 9, 16)])
def test_small_call_path_many_nodes(dy, orc, seed, L, B, caps, nmin, nmax):
    # 9 to 16 nodes of one or two options: still at most 2^16 plans, so k_small takes them -- through the instantiations
    # of its walk that bound the node count by 12 and 16 (the ragged test above stops at 8 nodes)
    w = wl.random_workload(seed, R=20, nmin=nmin, nmax=nmax, kmin=1, kmax=2, B=B, M=3, L=L, caps=caps, tool_p=0.05, edge_p=0.3)
    g = gpu_run(dy, w)
    st = dy[1].dyplan_last_stats()
    check_records(orc, w, g, orc.run(w), where=f"small-many-nodes(seed={seed})")
    binding, ctx = dy
    import torch
    dw = binding.upload(w)
    binding.launch(ctx, dw)
    torch.cuda.synchronize()
    assert ctx.dyplan_last_stats()["small_requests"] == int((orc.run(w)["status"].reshape(-1, L)[:, 0] != 2).sum())
    wr = wl.random_replan_workload(seed + 50, R=20, nmin=nmin, nmax=nmax, kmin=1, kmax=3, B=B, M=3, caps=caps, flags=wl.FLAG_FIXED_IN_PLACE)
    check_records(orc, wr, gpu_run(dy, wr), orc.run(wr), where=f"small-many-nodes-replan(seed={seed})")


# ---- scorer classes: fp32 slack DP for small exact ranges, int32 slack DP for the rest ----------------
def gpu_run_stats(dy, w):
    g = gpu_run(dy, w)
    return g, dy[1].dyplan_last_stats()


def test_baseline_configs_take_the_fp32_scorer(dy):
    for cfg, R in ((0, 1), (1, 2), (2, 8), (3, 16), (4, 1)):
        w = wl.make_config(cfg, R=R)
        if cfg == 4:   # keep the run short: the class is decided per request, before any enumeration
            w.batch.slo_us[:] = 0
        _, st = gpu_run_stats(dy, w)
        assert st["fast_requests"] == w.batch.R, (cfg, st)


def _scale_latencies(w, rows, factor):
    b = w.batch
    for r in rows:
        a, e = int(b.opt_off[b.node_off[r]]), int(b.opt_off[b.node_off[r + 1]])
        b.lat_us[a:e] *= factor
        b.slo_us[r] = int(min(int(b.slo_us[r]) * factor, 2**31 - 1))


@pytest.mark.parametrize("seed,L,B,caps,factor", [(91, 2, 2, True, 3000), (92, 4, 3, False, 3000), (93, 5, 4, True, 3000),
                                                  (191, 3, 2, True, 40000), (192, 8, 3, False, 40000), (193, 1, 1, True, 40000)])
def test_large_latencies_take_the_verified_fp32_path(dy, orc, seed, L, B, caps, factor):
    # latency sums far above 2^22 us (the paper's own requests take 4 s ... 414 s): fp32 is no longer exact, so
    # the fp32 scorer runs as a conservative screen (slack upper bounds by directed rounding) and every candidate is
    # re-evaluated in int32 (ReqHdr.approx).  Factor 40000 puts durations near 2^27 (fp32 spacing 8-16 us): the SLO is
    # some sampled plan's exact T, so plans sit exactly on and next to the feasibility boundary.
    nmax = 7 if factor == 3000 else 5
    w = wl.random_workload(seed, R=24, nmin=2, nmax=nmax, kmin=1, kmax=6, B=B, M=3, L=L, caps=caps)
    _scale_latencies(w, range(w.batch.R), factor)
    if caps and factor != 3000:   # demand sums beyond 2^22 as well
        w.batch.demand[:] = w.batch.demand.astype(np.int64) * 5000
        w.batch.cap[:] = np.minimum(w.batch.cap.astype(np.int64) * 5000, 2**31 - 1).astype(np.int32)
    g = gpu_run(dy, w)
    st = dy[1].dyplan_last_stats()
    assert st["fast_requests"] == w.batch.R
    assert st["approx_requests"] >= w.batch.R - 2        # (a one- or two-node request can still fit under 2^22)
    ref = orc.run(w)
    assert (ref["status"] == 0).sum() > 10
    check_records(orc, w, g, ref, where=f"verified-fp32(seed={seed})")


def test_verified_fp32_path_on_the_feasibility_boundary(dy, orc):
    # SLO = T of the oracle's own optimum, SLO - 1 and SLO + 1, with durations around 2^28: the screen's rounded slacks
    # cannot tell these apart, the integer verification must
    w = wl.random_workload(194, R=12, nmin=3, nmax=5, kmin=2, kmax=5, B=2, M=2, L=2, caps=False, tool_p=0.0)
    _scale_latencies(w, range(w.batch.R), 60000)
    ref0 = orc.run(w)
    for delta in (0, -1, 1):
        for r in range(w.batch.R):
            if ref0["status"][r * 2] == 0:
                w.batch.slo_us[r] = int(ref0["lat"][r * 2]) + delta
        g = gpu_run(dy, w)
        assert dy[1].dyplan_last_stats()["approx_requests"] >= 10
        check_records(orc, w, g, orc.run(w), where=f"boundary(delta={delta})")


def test_mixed_classes_in_one_batch(dy, orc):
    w = wl.random_workload(94, R=40, nmin=2, nmax=7, kmin=1, kmax=6, B=2, M=3, L=3, caps=True)
    _scale_latencies(w, range(0, 40, 3), 3000)
    b = w.batch
    for r in range(1, 40, 6):      # and some requests only the int32 scorer takes (a zero factor)
        n = int(b.node_off[r])
        b.vuln[n] = 1.0
        b.acc[int(b.opt_off[n]): int(b.opt_off[n + 1])] = 0.0
    g = gpu_run(dy, w)
    st = dy[1].dyplan_last_stats()
    assert 0 < st["approx_requests"] < st["fast_requests"] < w.batch.R
    check_records(orc, w, g, orc.run(w), where="mixed-classes")


def test_int32_scorer_with_large_latencies(dy, orc):
    # the wide class proper: zero factors AND second-scale latencies
    w = wl.random_workload(195, R=16, nmin=2, nmax=6, kmin=2, kmax=5, B=2, M=2, L=3, caps=True, tool_p=0.0)
    _scale_latencies(w, range(w.batch.R), 3000)
    b = w.batch
    for r in range(16):
        n = int(b.node_off[r]) + (r % b.n_nodes(r))
        b.vuln[n] = 1.0
        b.acc[int(b.opt_off[n])] = 0.0          # one zero-factor option: the request leaves the fp32 scorer
    g = gpu_run(dy, w)
    assert dy[1].dyplan_last_stats()["fast_requests"] == 0
    check_records(orc, w, g, orc.run(w), where="int32-scorer")


def test_zero_factor_requests_go_to_the_int32_scorer(dy, orc):
    # f = 1 - v (1 - a) = 0 makes C32 = 0 for real plans; the fp32 screen needs C32 > 0, so k_stage routes them away
    w = wl.random_workload(95, R=16, nmin=2, nmax=5, kmin=2, kmax=5, B=2, M=2, L=2, caps=False, tool_p=0.0)
    b = w.batch
    for r in range(0, 16, 2):
        n = int(b.node_off[r])
        b.vuln[n] = 1.0
        b.acc[int(b.opt_off[n]): int(b.opt_off[n + 1])] = 0.0     # every option of that node: every plan has C = 0
    g = gpu_run(dy, w)
    st = dy[1].dyplan_last_stats()
    assert st["fast_requests"] == 8
    ref = orc.run(w)
    check_records(orc, w, g, ref, where="zero-factor")
    assert (g["corr"].reshape(16, 2)[0::2][g["status"].reshape(16, 2)[0::2] == 0] == 0.0).all()


@pytest.mark.parametrize("seed,B,kmax", [(96, 2, 16), (97, 3, 12), (98, 4, 16), (99, 8, 16), (100, 6, 9)])
def test_fast_class_backend_group_layouts(dy, orc, seed, B, kmax):
    # caps + many options: node 0's slots are grouped by backend (2/3/4/8 groups); shapes that do not fit go wide
    w = wl.random_workload(seed, R=20, nmin=2, nmax=4, kmin=2, kmax=kmax, B=B, M=3, L=2, caps=True, tool_p=0.0)
    both(dy, orc, w, f"groups(seed={seed})")


# ---- malformed inputs: per-request status, the rest of the batch still compiles ------------------------
def test_invalid_requests_are_isolated(dy, orc):
    w = wl.random_workload(51, R=12, nmin=3, nmax=6, kmin=2, kmax=5, B=2, M=3, L=2, caps=True, tool_p=0.0)
    b = w.batch
    n0 = b.node_off
    b.pred_mask[n0[1] + 1] |= np.uint32(1 << 2)            # predecessor with a larger index
    b.vuln[n0[3]] = np.nan                                 # missing vulnerability is not zero
    b.acc[b.opt_off[n0[5]]] = 1.5
    b.lat_us[b.opt_off[n0[7] + 1]] = -3
    b.backend[b.opt_off[n0[9]]] = 7                        # >= B
    b.slo_us[10] = -1
    g, ref, _ = both(dy, orc, w, "invalid")
    st = g["status"].reshape(b.R, 2)
    for r in (1, 3, 5, 7, 9, 10):
        assert (st[r] == 2).all(), r
    for r in (0, 2, 4, 6, 8, 11):
        assert (st[r] != 2).all(), r


def test_latency_overflow_is_invalid(dy, orc):
    w = wl.random_workload(52, R=3, nmin=4, nmax=5, kmin=2, kmax=3, B=2, M=2, L=2, caps=False, tool_p=0.0)
    o = w.batch.opt_off[w.batch.node_off[1]]
    w.batch.lat_us[o] = 2**31 - 1                           # x multiplier >= 1000 per mille, summed: > INT32_MAX
    g, ref, _ = both(dy, orc, w, "overflow")
    assert (g["status"].reshape(3, 2)[1] == 2).all()


def test_replan_dispatched_set_must_be_predecessor_closed(dy, orc):
    w = wl.random_replan_workload(53, R=6, nmin=5, nmax=6, kmin=2, kmax=4, B=2, M=2, caps=False, tool_p=0.0)
    b = w.batch
    # chain 0 -> 1 in request 2, dispatch node 1 but not node 0
    b.pred_mask[b.node_off[2] + 1] = 1
    w.dispatched_mask[2] = 0b10
    w.fixed_choice[b.node_off[4]] = 15                      # fixed choice >= K_n
    w.dispatched_mask[4] |= 1
    g, ref, _ = both(dy, orc, w, "replan-invalid")
    assert g["status"][2] == 2 and g["status"][4] == 2


def test_plan_space_too_large(dy, orc):
    # 16 nodes x 16 options = 2^64 plans: TOO_LARGE, not a hang
    n, K = 16, 16
    req = dict(pred_mask=[0] * n, vuln=np.full(n, 0.5, np.float32), lat=np.full((n, K), 10, np.int32),
               acc=np.full((n, K), 0.5, np.float32), demand=np.full((n, K), 1, np.int32),
               backend=np.zeros((n, K), np.uint8), model=np.zeros((n, K), np.uint8), slo=1000, cap=[100])
    small = dict(req)
    small.update(pred_mask=[0] * 2, vuln=req["vuln"][:2], lat=req["lat"][:2, :2], acc=req["acc"][:2, :2],
                 demand=req["demand"][:2, :2], backend=req["backend"][:2, :2], model=req["model"][:2, :2])
    b = wl.batch_from_requests([req, small], 1, 1, True)
    w = wl.Workload(name="huge", kind="compile", batch=b, L=1, mult_pm=np.array([1000], np.int32))
    g, ref, _ = both(dy, orc, w, "too-large")
    assert g["status"][0] == 3 and g["status"][1] == 0


def test_empty_batch_and_empty_request(dy, orc):
    import torch
    binding, ctx = dy
    w = wl.random_workload(54, R=3, nmin=2, nmax=3, kmin=2, kmax=3, B=2, M=2, L=2, caps=False)
    e = wl.Workload(name="empty", kind="compile", batch=wl.batch_from_requests([], 2, 2, False), L=2,
                    mult_pm=w.mult_pm)
    dw = binding.upload(e)
    binding.launch(ctx, dw)          # R = 0: a no-op that returns OK
    torch.cuda.synchronize()
    # a request with zero nodes has exactly one (empty) plan: C = 1, T = 0
    b = w.batch
    b2 = wl.Batch(R=2, B=b.B, M=b.M, node_off=np.array([0, 0, b.node_off[1]], np.int32),
                  opt_off=b.opt_off[: b.node_off[1] + 1].copy(), pred_mask=b.pred_mask[: b.node_off[1]].copy(),
                  vuln=b.vuln[: b.node_off[1]].copy(), lat_us=b.lat_us[: b.opt_off[b.node_off[1]]].copy(),
                  acc=b.acc[: b.opt_off[b.node_off[1]]].copy(), demand=b.demand[: b.opt_off[b.node_off[1]]].copy(),
                  backend=b.backend[: b.opt_off[b.node_off[1]]].copy(), model=b.model[: b.opt_off[b.node_off[1]]].copy(),
                  slo_us=np.array([5, b.slo_us[0]], np.int32), cap=None)
    w2 = wl.Workload(name="empty-req", kind="compile", batch=b2, L=2, mult_pm=w.mult_pm)
    g, ref, _ = both(dy, orc, w2, "empty-req")
    assert (g["status"][:2] == 0).all() and (g["corr"][:2] == 1.0).all() and (g["lat"][:2] == 0).all()


# ---- the *_host entry points and select ----------------------------------------------------------------------------
def test_host_calls_equal_device_calls(dy, orc):
    binding, ctx = dy
    for w in (wl.random_workload(61, R=30, nmin=2, nmax=6, kmin=2, kmax=6, B=3, M=3, L=3, caps=True),
              wl.random_replan_workload(62, R=30, nmin=2, nmax=7, kmin=2, kmax=5, B=2, M=3, caps=True)):
        g = gpu_run(dy, w)
        h, h2d, d2h = binding.run_host(ctx, w)
        for k in g:
            assert np.array_equal(g[k], h[k]), k
        assert h2d > 0 and d2h > 0


@pytest.mark.parametrize("seed", [71, 72, 73])
def test_select_parity(dy, orc, seed):
    import torch
    binding, ctx = dy
    L, B = 4, 3
    w = wl.random_workload(seed, R=200, nmin=1, nmax=8, kmin=1, kmax=4, B=B, M=3, L=L, caps=True, slo_q=0.3)
    w.batch.vuln[w.batch.node_off[5]] = np.nan     # one invalid request -> variant -1
    dw = binding.upload(w)
    binding.launch(ctx, dw)
    torch.cuda.synchronize()
    g = dw.out.host()
    rng = np.random.default_rng(seed)
    for trial in range(4):
        live = rng.integers(1000, 4001, size=B).astype(np.int32) if trial else np.asarray(w.mult_pm[:B], np.int32)
        dlive = torch.from_numpy(live).cuda()
        variant = torch.full((w.batch.R,), -7, dtype=torch.int32, device="cuda")
        res = binding.alloc_bundle(w.batch.R, 1, B, "cuda:0")
        ctx.dyplan_select(dw.batch, dw.out, L, dlive, variant, res)
        torch.cuda.synchronize()
        ref = orc.select(w.batch, L, g["choice"], g["status"], live)
        v = variant.cpu().numpy()
        assert np.array_equal(v, ref["variant"])
        rs = res.host()
        pick = v >= 0
        assert np.array_equal(rs["lat"][pick].astype(np.int64), ref["lat"][pick])
        assert np.allclose(rs["corr64"][pick], ref["corr"][pick], rtol=1e-12, atol=0)
        assert np.array_equal(rs["status"][pick] == 0, ref["feasible"][pick] == 1)
        assert (rs["status"][~pick] != 0).all() and v[5] == -1
        # the re-scored record is a consistent plan of the stored bundle
        for r in np.nonzero(pick)[0][:50]:
            rec = r * L + v[r]
            assert np.array_equal(rs["choice"].reshape(-1, 16)[r], g["choice"].reshape(-1, 16)[rec])
            assert rs["plan_idx"][r] == g["plan_idx"][rec]
            assert np.array_equal(rs["dem"].reshape(-1, B)[r], g["dem"].reshape(-1, B)[rec])
            assert rs["dom_model"][r] == g["dom_model"][rec]
        if trial == 0:
            # PIN14 on the GPU path: under level 0's own multipliers variant 0 re-scores to its stored T
            ok0 = g["status"].reshape(-1, L)[:, 0] == 0
            assert (v[ok0] >= 0).all()
        # host entry point gives the same answer
        vh = np.full(w.batch.R, -9, np.int32)
        hb = binding.make_batch(w.batch, None)
        hbundle = binding.bundle_from_host(g, w.batch.R, L, B, None)
        ctx.dyplan_select_host(hb, hbundle, L, live, vh, None)
        assert np.array_equal(vh, v)


# ---- the paper's stateful selector: dyplan_switch against oracle/switch_oracle.py ---------------
@pytest.mark.parametrize("seed", [111, 112, 113])
def test_switch_parity(dy, orc, seed):
    import torch
    from oracle import switch_oracle as so
    binding, ctx = dy
    L, B, M, R = 5, 3, 4, 300
    w = wl.random_workload(seed, R=R, nmin=1, nmax=8, kmin=1, kmax=4, B=B, M=M, L=L, caps=True, slo_q=0.35)
    w.batch.vuln[w.batch.node_off[7]] = np.nan                 # one request without any plan
    ref = orc.run(w)                                           # the bundle comes from the oracle, not from the GPU
    bundle_host = dict(plan_idx=ref["plan_idx"], choice=ref["choice"], corr=ref["corr"].astype(np.float32),
                       corr64=ref["corr"], lat=np.minimum(ref["lat"], 2**31 - 1).astype(np.int32), dem=ref["dem"],
                       dom_model=ref["dom_model"], status=ref["status"])
    dbundle = binding.bundle_from_host(bundle_host, R, L, B, "cuda:0")
    dbatch = binding.make_batch(w.batch, "cuda:0")
    rng = np.random.default_rng(seed)
    n_nodes = np.array([w.batch.n_nodes(r) for r in range(R)])
    f32 = lambda x: float(np.float32(x))
    seen = set()
    for trial in range(6):
        params = dict(hi_load=f32(rng.uniform(0.5, 0.9)), lo_load=f32(rng.uniform(0.1, 0.5)),
                      load_margin=f32(rng.uniform(0.0, 0.3)), quality_tol=f32(rng.uniform(0.0, 0.2)),
                      min_dwell=f32(rng.uniform(0.0, 5.0)))
        load = rng.uniform(0.0, 1.2, size=M).astype(np.float32)
        if trial == 4:
            load[1] = np.nan
        cur = rng.integers(-1, L, size=R).astype(np.int32)
        since = rng.uniform(0.0, 10.0, size=R).astype(np.float32)
        disp = np.array([rng.integers(0, 1 << n) if n else 0 for n in n_nodes], dtype=np.uint32)
        active = rng.integers(0, 4, size=R * 16).astype(np.uint8)
        exp = so.switch(R, L, n_nodes, ref["status"], ref["dom_model"], ref["corr"], ref["choice"], load, cur, since,
                        disp, active, params)
        t = lambda a: torch.from_numpy(a.view(np.int32) if a.dtype == np.uint32 else a).cuda()
        d_cur, d_act = t(cur.copy()), t(active.copy())
        d_sw = torch.full((R,), 77, dtype=torch.uint8, device="cuda")
        ctx.dyplan_switch(dbatch, dbundle, L, params, t(load), t(since), t(disp), d_cur, d_act, d_sw)
        torch.cuda.synchronize()
        assert np.array_equal(d_cur.cpu().numpy(), exp["variant"]), trial
        assert np.array_equal(d_sw.cpu().numpy(), exp["switched"]), trial
        assert np.array_equal(d_act.cpu().numpy(), exp["active"]), trial
        seen |= set(exp["switched"].tolist())
    assert seen == {0, 1, 2, 3}                                # every branch of the rule was reached
    # argument checks
    with pytest.raises(binding.DyplanError) as e:
        ctx.dyplan_switch(dbatch, dbundle, L, dict(params, hi_load=0.1, lo_load=0.5), t(load), t(since), t(disp), d_cur,
                          d_act, d_sw)
    assert e.value.code == binding.ERR_ARG


def test_calls_on_different_streams_of_one_ctx_are_ordered(dy, orc):
    # a ctx has one set of scratch: a call on another stream waits (on the device) for the previous call of the ctx
    import torch
    binding, ctx = dy
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    w1 = wl.make_config(2, R=96)
    w2 = wl.random_workload(88, R=40, nmin=2, nmax=7, kmin=1, kmax=6, B=2, M=3, L=3, caps=True)
    d1, d2 = binding.upload(w1), binding.upload(w2)
    torch.cuda.synchronize()
    for _ in range(3):
        binding.launch(ctx, d1, s1)
        binding.launch(ctx, d2, s2)        # would reset the counters the first call's scorers are pulling from
    torch.cuda.synchronize()
    check_records(orc, w2, d2.out.host(), orc.run(w2), where="two streams, second call")
    ref1 = orc.run(w1, 0, 12)
    g1 = d1.out.host()
    check_records(orc, w1, g1, ref1, records=range(12 * w1.L), where="two streams, first call")


def test_api_argument_errors(dy):
    binding, ctx = dy
    w = wl.random_workload(81, R=2, nmin=2, nmax=3, kmin=2, kmax=3, B=2, M=2, L=2, caps=False)
    dw = binding.upload(w)
    with pytest.raises(binding.DyplanError) as e:
        ctx.dyplan_compile(dw.batch, 9, dw.mult, dw.out)          # L over the limit
    assert e.value.code == binding.ERR_LIMIT
    with pytest.raises(binding.DyplanError) as e:
        ctx.dyplan_compile(dw.batch, 2, None, dw.out)             # NULL multipliers
    assert e.value.code == binding.ERR_NULL
    with pytest.raises(binding.DyplanError) as e:
        ctx.dyplan_replan(dw.batch, dw.mult, dw.mult, dw.mult, 2, dw.out)   # unknown flag
    assert e.value.code == binding.ERR_ARG


# ---- exact dominance pruning: same results, smaller enumerated space -------------
@pytest.fixture()
def pruning(dy):
    binding, ctx = dy
    ctx.dyplan_set_flags(binding.PRUNE_DOMINATED)
    yield
    ctx.dyplan_set_flags(0)


@pytest.mark.parametrize("seed,L,B,caps", [(121, 1, 1, False), (122, 3, 2, True), (123, 4, 3, True), (124, 8, 2, False)])
def test_pruned_enumeration_equals_the_full_oracle(dy, orc, pruning, seed, L, B, caps):
    w = wl.random_workload(seed, R=40, nmin=1, nmax=7, kmin=1, kmax=8, B=B, M=3, L=L, caps=caps)
    g = gpu_run(dy, w)
    st = dy[1].dyplan_last_stats()
    assert st["plans"] < w.n_plans_total()                      # something was pruned ...
    check_records(orc, w, g, orc.run(w), where=f"pruned(seed={seed})")   # ... and nothing changed


def test_pruned_configs_and_replan(dy, orc, pruning):
    for w in (wl.make_config(0), wl.make_config(1, R=2), wl.make_config(2, R=12)):
        g = gpu_run(dy, w)
        st = dy[1].dyplan_last_stats()
        c = check_records(orc, w, g, orc.run(w), where=f"pruned {w.name}")
        assert st["plans"] <= w.n_plans_total()
    w = wl.random_replan_workload(125, R=40, nmin=1, nmax=8, kmin=1, kmax=6, B=3, M=3, caps=True)
    check_records(orc, w, gpu_run(dy, w), orc.run(w), where="pruned replan")
    w.flags = wl.FLAG_RESIDUAL
    check_records(orc, w, gpu_run(dy, w), orc.run(w), where="pruned replan residual")


def test_pruning_with_exact_ties_keeps_the_tie_break(dy, orc, pruning):
    # duplicated options (equal f, equal durations): only the lower index may survive, and order 7 must still hold
    w = wl.make_config(1, R=2)
    b = w.batch
    b.acc[:] = np.round(b.acc * 4) / 4
    b.vuln[:] = np.round(b.vuln * 2) / 2
    b.lat_us[:] = (b.lat_us // 400 + 1) * 400
    g = gpu_run(dy, w)
    ref = orc.run(w)
    c = check_records(orc, w, g, ref, where="pruned ties")
    ok = ref["status"] == 0
    assert (g["plan_idx"][ok] == ref["plan_idx"][ok]).all()


def test_pruning_reaches_a_space_beyond_brute_force(dy, orc, pruning):
    # 11 nodes x 16 options = 1.8e13 plans: TOO_LARGE unpruned; dominance leaves a Pareto front per node.  Optimum from
    # the independent MILP of PIN13.
    from test_oracle_pins import milp_best_corr
    binding, ctx = dy
    w = wl.random_workload(126, R=3, nmin=11, nmax=11, kmin=16, kmax=16, B=2, M=3, L=2, caps=True, tool_p=0.0, slo_q=0.4)
    g = gpu_run(dy, w)
    st = ctx.dyplan_last_stats()
    assert (g["status"] != 3).all() and st["plans"] < 2**40
    mult = np.asarray(w.mult_pm).reshape(2, 2)
    for rec in range(6):
        r, l = divmod(rec, 2)
        cstar = milp_best_corr(w.batch, r, mult[l])
        if cstar is None:
            assert g["status"][rec] == 1
            continue
        assert g["status"][rec] == 0
        c64 = float(g["corr64"][rec])
        assert cstar * (1 - 1e-5) <= c64 <= cstar * (1 + 1e-6), (rec, c64, cstar)
    ctx.dyplan_set_flags(0)
    g0 = gpu_run(dy, w)
    assert (g0["status"] == 3).all()                             # the same batch without pruning: plan space too large


# ---- exact subtree bounds (second half): same results, fewer plans walked ----------
@pytest.fixture()
def bounding(dy):
    binding, ctx = dy
    ctx.dyplan_set_flags(binding.PRUNE_BOUNDS)
    yield
    ctx.dyplan_set_flags(0)


@pytest.mark.parametrize("seed,L,B,caps", [(131, 1, 1, False), (132, 3, 2, True), (133, 4, 3, True), (134, 8, 2, False),
                                           (135, 6, 2, True), (136, 2, 1, False)])
def test_bounded_enumeration_equals_the_full_oracle(dy, orc, bounding, seed, L, B, caps):
    w = wl.random_workload(seed, R=40, nmin=1, nmax=7, kmin=1, kmax=8, B=B, M=3, L=L, caps=caps)
    g = gpu_run(dy, w)
    st = dy[1].dyplan_last_stats()
    assert st["plans"] == w.n_plans_total()                     # the space is the whole space ...
    check_records(orc, w, g, orc.run(w), where=f"bounded(seed={seed})")   # ... and nothing changed


def test_bounded_configs_skip_subtrees_and_change_nothing(dy, orc, bounding):
    # large enough for lane-aligned work items (the bound votes warp-wide and is off for calls too small to fill the GPU)
    binding, ctx = dy
    for w in (wl.make_config(1, R=16), wl.make_config(2, R=96), wl.make_config(3, R=64)):
        g = gpu_run(dy, w)
        st = ctx.dyplan_last_stats()
        check_records(orc, w, g, orc.run(w), where=f"bounded {w.name}")
        assert st["bound_skipped"] > 0, w.name                  # the bound did cut something on the paper-shaped inputs
        assert st["plans"] == w.n_plans_total()
    for w in (wl.make_config(0), wl.make_config(1, R=2), wl.make_config(4, R=1)):   # small calls: bound off or on, same records
        if w.name.startswith("cfg4"):
            w.batch.slo_us[:] //= 3                              # mostly infeasible prefixes: the latency bound cuts
            ctx.dyplan_set_flags(0)
            ref = gpu_run(dy, w)                                 # 6^12 plans: the exhaustive GPU run is the comparison
            ctx.dyplan_set_flags(binding.PRUNE_BOUNDS)
            g = gpu_run(dy, w)
            for k in ("plan_idx", "lat", "dem", "status", "choice", "corr"):
                assert np.array_equal(g[k], ref[k]), k
        else:
            check_records(orc, w, gpu_run(dy, w), orc.run(w), where=f"bounded {w.name}")


def test_bounded_random_batches_large_enough_to_align(dy, orc, bounding):
    for seed, L, B, caps in [(141, 3, 2, True), (142, 2, 3, False)]:
        w = wl.random_workload(seed, R=300, nmin=6, nmax=7, kmin=5, kmax=8, B=B, M=3, L=L, caps=caps)
        g = gpu_run(dy, w)
        st = dy[1].dyplan_last_stats()
        check_records(orc, w, g, orc.run(w), where=f"bounded aligned(seed={seed})")
        assert st["bound_skipped"] > 0
    w = wl.random_replan_workload(137, R=40, nmin=1, nmax=8, kmin=1, kmax=6, B=3, M=3, caps=True)
    check_records(orc, w, gpu_run(dy, w), orc.run(w), where="bounded replan")
    w.flags = wl.FLAG_RESIDUAL
    check_records(orc, w, gpu_run(dy, w), orc.run(w), where="bounded replan residual")


def test_bounds_with_exact_ties_keep_the_tie_break(dy, orc, bounding):
    # many plans tie with the optimum in C: a subtree whose bound EQUALS the incumbent must still be walked (T, idx decide)
    w = wl.make_config(1, R=12)
    b = w.batch
    b.acc[:] = np.round(b.acc * 4) / 4
    b.vuln[:] = np.round(b.vuln * 2) / 2
    b.lat_us[:] = (b.lat_us // 400 + 1) * 400
    g = gpu_run(dy, w)
    ref = orc.run(w)
    check_records(orc, w, g, ref, where="bounded ties")
    ok = ref["status"] == 0
    assert (g["plan_idx"][ok] == ref["plan_idx"][ok]).all()


def test_bounds_and_dominance_pruning_together(dy, orc):
    binding, ctx = dy
    ctx.dyplan_set_flags(binding.PRUNE_BOUNDS | binding.PRUNE_DOMINATED)
    try:
        for seed, L, B, caps in [(138, 4, 2, True), (139, 3, 3, False)]:
            w = wl.random_workload(seed, R=40, nmin=1, nmax=7, kmin=1, kmax=8, B=B, M=3, L=L, caps=caps)
            check_records(orc, w, gpu_run(dy, w), orc.run(w), where=f"bounded+pruned(seed={seed})")
        with pytest.raises(binding.DyplanError) as e:
            ctx.dyplan_set_flags(1 << 10)                        # unknown bit
        assert e.value.code == binding.ERR_ARG
    finally:
        ctx.dyplan_set_flags(0)


# ---- both prunings: records identical BIT FOR BIT to the exhaustive GPU run (not only to the oracle within 1e-5) -----
def _near_tie_workload(seed, R=24, L=2, B=2, caps=False):
    """Tie-heavy inputs for the pruning A/B test: vulnerabilities around 1e-7 (every factor 1 - v(1 - a) lands within
    a few fp32 ulps of 1, so products of distinct factors round to equal C32) and few distinct durations (T ties),
    so the canonical-index tie-break decides most records."""
    rng = np.random.default_rng(seed)
    w = wl.random_workload(seed, R=R, nmin=2, nmax=6, kmin=2, kmax=8, B=B, M=3, L=L, caps=caps, tool_p=0.0)
    b = w.batch
    b.vuln[:] = rng.choice([0.0, 5e-8, 1e-7, 2e-7, 1e-6], size=b.vuln.size).astype(np.float32)
    half = rng.random(b.R) < 0.5
    for r in range(b.R):
        n0, n1 = int(b.node_off[r]), int(b.node_off[r + 1])
        o0, o1 = int(b.opt_off[n0]), int(b.opt_off[n1])
        if half[r]:
            b.lat_us[o0:o1] = 500                                   # all durations equal: T ties everywhere
        else:
            b.lat_us[o0:o1] = rng.choice([400, 500], size=o1 - o0)
        b.slo_us[r] = 500 * (n1 - n0) * 4
    return w


def _gpu_with_flags(dy, w, flags):
    binding, ctx = dy
    ctx.dyplan_set_flags(flags)
    try:
        g = gpu_run(dy, w)
        st = ctx.dyplan_last_stats()
    finally:
        ctx.dyplan_set_flags(0)
    return g, st


@pytest.mark.parametrize("seed,L,B,caps", [(141, 1, 1, False), (142, 2, 2, False), (143, 3, 2, True), (144, 4, 3, True)])
def test_prunings_are_bit_identical_to_the_exhaustive_run_on_near_ties(dy, orc, seed, L, B, caps):
    binding, _ = dy
    w = _near_tie_workload(seed, L=L, B=B, caps=caps)
    base, st0 = _gpu_with_flags(dy, w, 0)
    check_records(orc, w, base, orc.run(w), where=f"near-ties(seed={seed})")
    for flags in (binding.PRUNE_DOMINATED, binding.PRUNE_BOUNDS, binding.PRUNE_DOMINATED | binding.PRUNE_BOUNDS):
        g, st = _gpu_with_flags(dy, w, flags)
        for k in ("status", "plan_idx", "choice", "corr", "corr64", "lat", "dem", "dom_model"):
            assert np.array_equal(base[k], g[k]), f"flags={flags}: {k} differs from the exhaustive run"


@pytest.mark.parametrize("seed", [151, 152])
def test_prunings_are_bit_identical_on_ordinary_batches(dy, orc, seed):
    binding, _ = dy
    ws = [wl.random_workload(seed, R=40, nmin=1, nmax=7, kmin=1, kmax=8, B=3, M=3, L=4, caps=True),
          wl.make_config(2, R=16), wl.make_config(1, R=2)]
    ws.append(wl.random_replan_workload(seed, R=40, nmin=1, nmax=8, kmin=1, kmax=6, B=3, M=3, caps=True))
    for w in ws:
        base, _ = _gpu_with_flags(dy, w, 0)
        for flags in (binding.PRUNE_DOMINATED, binding.PRUNE_BOUNDS, binding.PRUNE_DOMINATED | binding.PRUNE_BOUNDS):
            g, _ = _gpu_with_flags(dy, w, flags)
            for k in ("status", "plan_idx", "choice", "corr", "corr64", "lat", "dem", "dom_model"):
                assert np.array_equal(base[k], g[k]), f"{w.name} flags={flags}: {k} differs from the exhaustive run"
