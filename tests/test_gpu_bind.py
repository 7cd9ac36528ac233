"""-m gpu: dyplan_bind (Alg. 1 l.1-8, Eq.(2)) against oracle/bind_oracle.py, bit-exact on every output, and the paper's
whole compile chain on the device: bind -> dyplan_compile_linear -> dyplan_switch, against the three oracles."""
from __future__ import annotations

import numpy as np
import pytest

from support import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def dy():
    import torch
    assert torch.cuda.is_available()
    from paper_2607_02942_b200 import binding
    ctx = binding.Context(0)
    yield binding, ctx
    ctx.close()


def profiles(rng, S=4, M=3, P=8, D=4, A=4, J=4, ROLES=3, F=4):
    """Synthetic profiles with the paper's shapes: 3 models x 8 policies, stage structures in the
    style of Table 4 (some stages parallel, some absent)."""
    dims = dict(S=S, M=M, P=P, D=D, A=A, J=J, ROLES=ROLES, F=F)
    quality = rng.uniform(0.4, 0.99, size=(S, M, P)).astype(np.float32)
    tokens = np.zeros((S, M, P, A, J), np.float32)
    for p in range(P):
        n_stage = 1 + p % A
        for a in range(n_stage):
            n_call = 1 if a in (0, n_stage - 1) else 1 + (p + a) % J
            tokens[:, :, p, a, :n_call] = rng.integers(20, 900, size=(S, M, n_call)).astype(np.float32)
    theta = rng.uniform(2e3, 2e4, size=(M, D)).astype(np.float32)          # tokens/s
    pre = rng.uniform(5e3, 5e4, size=(M, D)).astype(np.float32)           # us
    psi = rng.uniform(0.0, 1.0, size=(ROLES, S, F)).astype(np.float32)
    return dims, quality, tokens, theta, pre, psi


def graph_inputs(rng, dims, R=50):
    w = wl.random_workload(int(rng.integers(1, 10**6)), R=R, nmin=1, nmax=7, kmin=1, kmax=6, B=dims["D"], M=dims["M"], L=1, caps=False)
    b = w.batch
    skill = rng.integers(0, dims["S"], size=b.NN).astype(np.uint8)
    role = rng.integers(0, dims["ROLES"], size=b.NN).astype(np.uint8)
    policy = rng.integers(0, dims["P"], size=b.KK).astype(np.uint8)
    return b, skill, role, policy


def gpu_bind(dy, dims, quality, tokens, theta, pre, psi, norm, b, skill, role, policy):
    import torch
    binding, ctx = dy
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a).view(np.int32) if a.dtype == np.uint32 else np.ascontiguousarray(a)).cuda()
    vuln = torch.full((b.NN,), -7.0, dtype=torch.float32, device="cuda")
    acc = torch.full((b.KK,), -7.0, dtype=torch.float32, device="cuda")
    lat = torch.full((b.KK,), -7, dtype=torch.int32, device="cuda")
    cost = torch.full((b.KK,), -7.0, dtype=torch.float32, device="cuda")
    dem = torch.full((b.KK,), -7, dtype=torch.int32, device="cuda")
    keep = [t(quality), t(tokens), t(theta), t(pre), t(psi), t(b.opt_off), t(b.pred_mask), t(skill), t(role), t(b.model),
            t(b.backend), t(policy)]
    ctx.dyplan_bind(dims, keep[0], keep[1], keep[2], keep[3], keep[4], norm, b.NN, b.KK, keep[5], keep[6], keep[7], keep[8],
                    keep[9], keep[10], keep[11], vuln, acc, lat, cost, dem)
    torch.cuda.synchronize()
    return dict(vuln=vuln.cpu().numpy(), acc=acc.cpu().numpy(), lat_us=lat.cpu().numpy(), cost=cost.cpu().numpy(),
                demand=dem.cpu().numpy())


@pytest.mark.parametrize("seed", [301, 302, 303])
def test_bind_parity_bit_exact(dy, seed):
    from oracle import bind_oracle as bo
    rng = np.random.default_rng(seed)
    dims, quality, tokens, theta, pre, psi = profiles(rng)
    if seed == 303:
        theta[1, 2] = 0.0                                     # an uncalibrated (model, backend) pair
    b, skill, role, policy = graph_inputs(rng, dims)
    if seed == 302:
        skill[3] = 200                                        # out-of-range skill tag
        policy[5] = 99
    norm = float(np.float32(4096.0))
    g = gpu_bind(dy, dims, quality, tokens, theta, pre, psi, norm, b, skill, role, policy)
    ref = bo.bind(dims, quality, tokens, theta, pre, psi, norm, b.opt_off, b.pred_mask, skill, role, b.model, b.backend, policy)
    for k in ("lat_us", "demand"):
        assert np.array_equal(g[k], ref[k]), k
    for k in ("vuln", "acc", "cost"):
        assert np.array_equal(g[k], ref[k], equal_nan=True), k
    assert (g["lat_us"] >= -1).all() and (g["lat_us"] > 0).any()


def test_paper_chain_bind_compile_switch_on_the_device(dy):
    """Algorithm 1 end to end: coefficients from the profiles, one variant per level under Eq.(5), then Section 5.1's
    switch when the dominant model of the preferred plan is congested."""
    import torch
    from oracle import bind_oracle as bo, linear as lo, switch_oracle as so
    binding, ctx = dy
    rng = np.random.default_rng(304)
    dims, quality, tokens, theta, pre, psi = profiles(rng, D=3)
    b, skill, role, policy = graph_inputs(rng, dims, R=30)
    norm = float(np.float32(2048.0))
    g = gpu_bind(dy, dims, quality, tokens, theta, pre, psi, norm, b, skill, role, policy)
    ref = bo.bind(dims, quality, tokens, theta, pre, psi, norm, b.opt_off, b.pred_mask, skill, role, b.model, b.backend, policy)
    assert np.array_equal(g["lat_us"], ref["lat_us"])
    # compile on the bound coefficients (the oracle side binds with the oracle's own outputs)
    b.vuln[:], b.acc[:], b.lat_us[:], b.demand[:] = ref["vuln"], ref["acc"], ref["lat_us"], ref["demand"]
    params = {k: float(np.float32(v)) for k, v in dict(lambda_f=0.5, lambda_c=0.2, lambda_l=2e-6, lambda_ld=1e-6, beta=0.5, effort=1.0).items()}
    levels = [0.0, 1.5, 3.0]
    L, R, B = 3, b.R, b.B
    db = binding.make_batch(b, "cuda:0")
    out = binding.alloc_bundle(R, L, B, "cuda:0", True)
    dcost = torch.from_numpy(ref["cost"]).cuda()
    qual = torch.zeros(R * L, dtype=torch.float64, device="cuda")
    ctx.dyplan_compile_linear(db, dcost, params, levels, out, None, qual)
    torch.cuda.synchronize()
    gb = out.host()
    rl = lo.compile(b, ref["cost"], params, levels)
    ok = rl["status"] == 0
    assert ok.any() and np.array_equal(gb["status"] == 0, ok)
    same = (gb["plan_idx"][ok] == rl["plan_idx"][ok]).mean()
    assert same >= 0.9
    # the switch consumes the bundle's annotations: dominant model and quality estimate
    M = b.M
    p = dict(hi_load=0.75, lo_load=0.25, load_margin=0.125, quality_tol=0.5, min_dwell=1.0)
    load = np.array([0.9, 0.1, 0.3][:M] + [0.2] * max(0, M - 3), np.float32)
    cur = np.zeros(R, np.int32)
    since = np.full(R, 2.0, np.float32)
    disp = np.array([1 if b.n_nodes(r) > 1 else 0 for r in range(R)], np.uint32)     # the first node is dispatched
    active = gb["choice"].reshape(R, L, 16)[:, 0, :].copy().reshape(-1)
    qh = qual.cpu().numpy()
    exp = so.switch(R, L, [b.n_nodes(r) for r in range(R)], gb["status"], gb["dom_model"], qh, gb["choice"], load, cur, since,
                    disp, active, p)
    bundle = binding.Buffers(dict(out.arrays, corr64=qual), binding.CBundle(*[binding._ptr(dict(out.arrays, corr64=qual)[n]) for n, _, _ in binding._BUNDLE_FIELDS]), R, B, L)
    t = lambda a: torch.from_numpy(a.view(np.int32) if a.dtype == np.uint32 else a).cuda()
    d_cur, d_act, d_sw = t(cur.copy()), t(active.copy()), torch.zeros(R, dtype=torch.uint8, device="cuda")
    ctx.dyplan_switch(db, bundle, L, p, t(load), t(since), t(disp), d_cur, d_act, d_sw)
    torch.cuda.synchronize()
    assert np.array_equal(d_cur.cpu().numpy(), exp["variant"]) and np.array_equal(d_act.cpu().numpy(), exp["active"])
    assert np.array_equal(d_sw.cpu().numpy(), exp["switched"])
    moved = exp["switched"] == 1
    assert moved.any()                                          # some request left its congested dominant model
    dm = gb["dom_model"].reshape(R, L)
    assert (dm[moved, 0] == 0).all() and (dm[np.arange(R)[moved], exp["variant"][moved]] != 0).all()
