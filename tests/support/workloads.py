"""Seeded synthetic inputs for the dyplan hot path (numpy only).

This module is the ONE thing the oracle-side tests and the CUDA-side tests /
bench / smoke share (test support: it is not part of the shipped package).  It produces flat little-endian arrays in exactly the layout of
``include/dyplan.h`` (``dyplan_batch``) and nothing else: it contains no
enumeration, no arg-best, no correctness product and no demand accounting --
i.e. none of the method's arithmetic.  The one piece of workload *recipe* that
needs a DAG walk (``BASELINE.json`` configs: "SLO = median latency of 1000
random plans") is done by ``_sampled_latency_quantile`` below with a private
numpy helper; it only decides the VALUE of an input (``slo_us``) and is used by
neither the oracle nor the kernels (DESIGN.md section "Input recipe").

The paper's own workload for this path -- 92 frozen Flow/GPT-5.4 workflows with
at most 11 nodes, 3 models x 8 policies x replicas
-- is not available; the five configurations of ``BASELINE.json`` stand in for
it, with the shapes of section 6's walkthrough (planner -> parallel branches ->
aggregator).  Readings Q14-Q18 of SURVEY.md section 8(c) apply
and are restated in DESIGN.md.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Optional

import numpy as np

MAX_NODES = 16
MAX_OPTS = 16
MAX_BACKENDS = 8
MAX_MODELS = 8
MAX_LEVELS = 8

FLAG_FIXED_IN_PLACE = 0
FLAG_RESIDUAL = 1


@dataclass
class Batch:
    """Host-side mirror of ``dyplan_batch`` (include/dyplan.h)."""

    R: int
    B: int
    M: int
    node_off: np.ndarray  # int32 [R+1]
    opt_off: np.ndarray  # int32 [NN+1]
    pred_mask: np.ndarray  # uint32 [NN]
    vuln: np.ndarray  # float32 [NN]
    lat_us: np.ndarray  # int32 [KK]
    acc: np.ndarray  # float32 [KK]
    demand: np.ndarray  # int32 [KK]
    backend: np.ndarray  # uint8 [KK]
    model: np.ndarray  # uint8 [KK]
    slo_us: np.ndarray  # int32 [R]
    cap: Optional[np.ndarray] = None  # int32 [R*B] or None

    @property
    def NN(self) -> int:
        return int(self.node_off[-1])

    @property
    def KK(self) -> int:
        return int(self.opt_off[-1])

    def n_nodes(self, r: int) -> int:
        return int(self.node_off[r + 1] - self.node_off[r])

    def radices(self, r: int) -> np.ndarray:
        a, b = int(self.node_off[r]), int(self.node_off[r + 1])
        return (self.opt_off[a + 1 : b + 1] - self.opt_off[a:b]).astype(np.int64)

    def n_plans(self, r: int) -> int:
        return int(np.prod(self.radices(r), dtype=object)) if self.n_nodes(r) else 1

    def subset(self, rs) -> "Batch":
        """A new batch holding requests ``rs`` (in that order)."""
        rs = [int(r) for r in rs]
        node_off = [0]
        opt_off = [0]
        nsel = []
        ksel = []
        for r in rs:
            a, b = int(self.node_off[r]), int(self.node_off[r + 1])
            for n in range(a, b):
                ka, kb = int(self.opt_off[n]), int(self.opt_off[n + 1])
                ksel.extend(range(ka, kb))
                opt_off.append(opt_off[-1] + (kb - ka))
            nsel.extend(range(a, b))
            node_off.append(node_off[-1] + (b - a))
        nsel = np.asarray(nsel, dtype=np.int64)
        ksel = np.asarray(ksel, dtype=np.int64)
        cap = None
        if self.cap is not None:
            cap = np.ascontiguousarray(self.cap.reshape(self.R, self.B)[rs].reshape(-1))
        return Batch(
            R=len(rs), B=self.B, M=self.M,
            node_off=np.asarray(node_off, dtype=np.int32),
            opt_off=np.asarray(opt_off, dtype=np.int32),
            pred_mask=np.ascontiguousarray(self.pred_mask[nsel]),
            vuln=np.ascontiguousarray(self.vuln[nsel]),
            lat_us=np.ascontiguousarray(self.lat_us[ksel]),
            acc=np.ascontiguousarray(self.acc[ksel]),
            demand=np.ascontiguousarray(self.demand[ksel]),
            backend=np.ascontiguousarray(self.backend[ksel]),
            model=np.ascontiguousarray(self.model[ksel]),
            slo_us=np.ascontiguousarray(self.slo_us[rs]),
            cap=cap,
        )


@dataclass
class Workload:
    """One benchmark / test case: a batch plus the call arguments."""

    name: str
    kind: str  # "compile" | "replan"
    batch: Batch
    L: int
    mult_pm: Optional[np.ndarray] = None  # int32 [L*B]          (compile)
    dispatched_mask: Optional[np.ndarray] = None  # uint32 [R]   (replan)
    fixed_choice: Optional[np.ndarray] = None  # uint8 [NN]      (replan)
    live_mult_pm: Optional[np.ndarray] = None  # int32 [R*B]     (replan)
    flags: int = FLAG_FIXED_IN_PLACE
    meta: dict = field(default_factory=dict)

    def subset(self, rs) -> "Workload":
        rs = [int(r) for r in rs]
        b = self.batch
        w = replace(self, batch=b.subset(rs), name=f"{self.name}[{len(rs)}]")
        if self.kind == "replan":
            w.dispatched_mask = np.ascontiguousarray(self.dispatched_mask[rs])
            w.live_mult_pm = np.ascontiguousarray(self.live_mult_pm.reshape(b.R, b.B)[rs].reshape(-1))
            nsel = np.concatenate([np.arange(b.node_off[r], b.node_off[r + 1]) for r in rs]).astype(np.int64)
            w.fixed_choice = np.ascontiguousarray(self.fixed_choice[nsel])
        return w

    def n_plans_total(self) -> int:
        """Plans the call has to score (replan: undispatched nodes only)."""
        b = self.batch
        total = 0
        for r in range(b.R):
            rad = b.radices(r)
            if self.kind == "replan":
                m = int(self.dispatched_mask[r])
                rad = np.array([1 if (m >> n) & 1 else int(k) for n, k in enumerate(rad)], dtype=object)
            total += int(np.prod(rad, dtype=object)) if len(rad) else 1
        return total


# --------------------------------------------------------------------------
# DAG shapes
# --------------------------------------------------------------------------

def diamond_pred_masks() -> list[int]:
    """cfg0: 0 -> {1 -> 2, 3 -> 4} -> 5 (planner, two 2-node branches, aggregator)."""
    edges = [(0, 1), (1, 2), (0, 3), (3, 4), (2, 5), (4, 5)]
    pm = [0] * 6
    for u, v in edges:
        pm[v] |= 1 << u
    return pm


def layered_pred_masks(rng: np.random.Generator, n: int, width: int, p: float = 0.5) -> list[int]:
    """Random layered DAG(N, W, p): draw layer widths U{1..W} until N nodes
    (truncate the last), number nodes layer by layer; each node of layer j>0
    takes each node of layer j-1 as predecessor with probability p, and one
    uniformly chosen predecessor if it got none."""
    layers = []
    used = 0
    while used < n:
        w = int(rng.integers(1, width + 1))
        w = min(w, n - used)
        layers.append(list(range(used, used + w)))
        used += w
    pm = [0] * n
    for j in range(1, len(layers)):
        prev = layers[j - 1]
        for v in layers[j]:
            m = 0
            for u in prev:
                if rng.random() < p:
                    m |= 1 << u
            if m == 0:
                m = 1 << prev[int(rng.integers(0, len(prev)))]
            pm[v] = m
    return pm


# --------------------------------------------------------------------------
# private helper for the SLO recipe only (see module docstring)
# --------------------------------------------------------------------------

def _scaled(lat: np.ndarray, mult: np.ndarray) -> np.ndarray:
    return (lat.astype(np.int64) * mult.astype(np.int64)) // 1000


def _sampled_latency_quantile(rng, pred_masks, lat, backend, mults, q, n_draws=1000, fixed=None):
    """SLO recipe (readings Q14/Q15): ``n_draws`` draws of (uniform plan,
    uniform level); sort the critical-path latencies ascending; return element
    floor(q*n_draws).  ``lat``/``backend`` are [N][K]; ``mults`` is [L][B];
    ``fixed`` optionally pins the first nodes' options (cfg3)."""
    n, k = lat.shape
    ks = rng.integers(0, k, size=(n_draws, n))
    if fixed is not None:
        for node, opt in fixed.items():
            ks[:, node] = opt
    ls = rng.integers(0, mults.shape[0], size=n_draws)
    sel_lat = np.take_along_axis(np.broadcast_to(lat, (n_draws, n, k)), ks[:, :, None], axis=2)[:, :, 0]
    sel_be = np.take_along_axis(np.broadcast_to(backend, (n_draws, n, k)), ks[:, :, None], axis=2)[:, :, 0]
    m = mults[ls[:, None], sel_be]
    d = _scaled(sel_lat, m)
    fin = np.zeros((n_draws, n), dtype=np.int64)
    for v in range(n):
        start = np.zeros(n_draws, dtype=np.int64)
        for u in range(v):
            if (pred_masks[v] >> u) & 1:
                start = np.maximum(start, fin[:, u])
        fin[:, v] = start + d[:, v]
    t = np.sort(fin.max(axis=1))
    return int(t[min(n_draws - 1, int(np.floor(q * n_draws)))])


# --------------------------------------------------------------------------
# option tables
# --------------------------------------------------------------------------

def _option_tables(rng, n, n_models, n_backend_slots, backend_is_model):
    """Per-node option tables, k = model*(2*B') + verifier*B' + backend_slot
    (cfg4: k = model*2 + verifier, backend = model).  Readings Q18."""
    bs = 1 if backend_is_model else n_backend_slots
    base = np.maximum(1, np.rint(rng.lognormal(np.log(800.0), 0.5, size=(n, n_models, bs)))).astype(np.int64)
    extra = np.maximum(1, np.rint(rng.lognormal(np.log(400.0), 0.4, size=(n, n_models, bs)))).astype(np.int64)
    a0 = rng.uniform(0.6, 0.95, size=(n, n_models))
    rr = rng.uniform(0.3, 0.7, size=(n, n_models))
    averif = 1.0 - (1.0 - a0) * (1.0 - rr)
    K = n_models * 2 * bs
    lat = np.zeros((n, K), dtype=np.int64)
    acc = np.zeros((n, K), dtype=np.float64)
    backend = np.zeros((n, K), dtype=np.uint8)
    model = np.zeros((n, K), dtype=np.uint8)
    for m in range(n_models):
        for ver in range(2):
            for b in range(bs):
                k = m * (2 * bs) + ver * bs + b
                lat[:, k] = base[:, m, b] + (extra[:, m, b] if ver else 0)
                acc[:, k] = averif[:, m] if ver else a0[:, m]
                backend[:, k] = m if backend_is_model else b
                model[:, k] = m
    demand = rng.integers(200, 4001, size=(n, K)).astype(np.int64)
    return lat, acc.astype(np.float32), demand, backend, model


_CFG = {
    0: dict(R=1, N=6, W=None, models=2, slots=2, L=3, q=0.5, caps=False, tasks=False, be_is_model=False),
    1: dict(R=256, N=8, W=3, models=2, slots=2, L=4, q=0.4, caps=False, tasks=False, be_is_model=False),
    2: dict(R=4096, N=7, W=3, models=2, slots=2, L=4, q=0.4, caps=True, tasks=True, be_is_model=False),
    3: dict(R=16384, N=9, W=3, models=3, slots=2, L=1, q=0.4, caps=True, tasks=True, be_is_model=False),
    4: dict(R=16, N=12, W=4, models=3, slots=1, L=8, q=0.4, caps=True, tasks=True, be_is_model=True),
}


def make_config(cfg: int, R: Optional[int] = None, seed: Optional[int] = None) -> Workload:
    """``BASELINE.json: configs[cfg]``.  ``R`` overrides the request count (the
    first R requests of the stream are identical for any R, so a down-scaled
    case is a prefix of the full one); ``seed`` defaults to the config index."""
    c = _CFG[cfg]
    R = c["R"] if R is None else int(R)
    seed = cfg if seed is None else int(seed)
    n, L = c["N"], c["L"]
    B = c["models"] if c["be_is_model"] else c["slots"]
    M = c["models"]
    root = np.random.default_rng(seed)
    # config-wide draws first, then one child stream per request so that request r does not
    # depend on R.
    task_w = root.uniform(0.5, 1.5, size=4)
    mult = root.integers(1000, 3001, size=(L, B)).astype(np.int32)
    children = root.spawn(R) if hasattr(root, "spawn") else [np.random.default_rng([seed, r]) for r in range(R)]

    node_off = [0]
    opt_off = [0]
    pred_mask, vuln, lat_us, acc_l, dem_l, be_l, mo_l = [], [], [], [], [], [], []
    slo = np.zeros(R, dtype=np.int32)
    cap = np.zeros((R, B), dtype=np.int32) if c["caps"] else None
    disp = np.zeros(R, dtype=np.uint32)
    fixed_choice = []
    live = np.zeros((R, B), dtype=np.int32)
    for r in range(R):
        rng = children[r]
        pm = diamond_pred_masks() if c["W"] is None else layered_pred_masks(rng, n, c["W"], 0.5)
        lat, acc, dem, be, mo = _option_tables(rng, n, c["models"], c["slots"], c["be_is_model"])
        K = lat.shape[1]
        if c["tasks"]:
            pos = rng.uniform(0.2, 1.0, size=n)
            typ = rng.integers(0, 4, size=n)
            v = np.clip(pos * task_w[typ], 0.0, 1.0)
        else:
            v = rng.uniform(0.0, 1.0, size=n)
        fixed = None
        if cfg == 3:
            d = int(rng.integers(2, 6))  # 2..5 topologically-first nodes already dispatched
            fc = np.full(n, 0, dtype=np.uint8)
            fc[:d] = rng.integers(0, K, size=d)
            fixed = {i: int(fc[i]) for i in range(d)}
            disp[r] = (1 << d) - 1
            fixed_choice.append(fc)
            live[r] = rng.integers(1000, 4001, size=B)
            mults_r = live[r][None, :].astype(np.int64)
        else:
            mults_r = mult.astype(np.int64)
        slo[r] = _sampled_latency_quantile(rng, pm, lat, be, mults_r, c["q"], fixed=fixed)
        if c["caps"]:
            for b in range(B):
                on_b = np.where(be == b, dem, 0)
                cap[r, b] = int(np.floor(0.6 * on_b.max(axis=1).sum()))  # reading Q16
        node_off.append(node_off[-1] + n)
        for i in range(n):
            opt_off.append(opt_off[-1] + K)
        pred_mask.extend(pm)
        vuln.append(v.astype(np.float32))
        lat_us.append(lat.reshape(-1))
        acc_l.append(acc.reshape(-1))
        dem_l.append(dem.reshape(-1))
        be_l.append(be.reshape(-1))
        mo_l.append(mo.reshape(-1))

    batch = Batch(
        R=R, B=B, M=M,
        node_off=np.asarray(node_off, dtype=np.int32),
        opt_off=np.asarray(opt_off, dtype=np.int32),
        pred_mask=np.asarray(pred_mask, dtype=np.uint32),
        vuln=np.concatenate(vuln).astype(np.float32),
        lat_us=np.concatenate(lat_us).astype(np.int32),
        acc=np.concatenate(acc_l).astype(np.float32),
        demand=np.concatenate(dem_l).astype(np.int32),
        backend=np.concatenate(be_l).astype(np.uint8),
        model=np.concatenate(mo_l).astype(np.uint8),
        slo_us=slo,
        cap=None if cap is None else np.ascontiguousarray(cap.reshape(-1)),
    )
    if cfg == 3:
        return Workload(
            name=f"cfg3(R={R})", kind="replan", batch=batch, L=1,
            dispatched_mask=disp, fixed_choice=np.concatenate(fixed_choice).astype(np.uint8),
            live_mult_pm=np.ascontiguousarray(live.reshape(-1)), flags=FLAG_FIXED_IN_PLACE,
            meta=dict(cfg=3, seed=seed),
        )
    return Workload(name=f"cfg{cfg}(R={R})", kind="compile", batch=batch, L=L,
                    mult_pm=np.ascontiguousarray(mult.reshape(-1)), meta=dict(cfg=cfg, seed=seed))


# --------------------------------------------------------------------------
# free-form small cases for tests (ragged N, ragged K, tool nodes, arbitrary DAGs)
# --------------------------------------------------------------------------

def batch_from_requests(reqs: list[dict], B: int, M: int, with_caps: bool) -> Batch:
    """Assemble a Batch from per-request dicts with keys pred_mask [N], vuln [N],
    and per-node lists lat/acc/demand/backend/model (ragged), slo, cap [B]."""
    node_off = [0]
    opt_off = [0]
    pm, vu, la, ac, de, be, mo, slo, cap = [], [], [], [], [], [], [], [], []
    for q in reqs:
        n = len(q["pred_mask"])
        node_off.append(node_off[-1] + n)
        pm.extend(int(x) for x in q["pred_mask"])
        vu.extend(float(x) for x in q["vuln"])
        for i in range(n):
            k = len(q["lat"][i])
            opt_off.append(opt_off[-1] + k)
            la.extend(q["lat"][i])
            ac.extend(q["acc"][i])
            de.extend(q["demand"][i])
            be.extend(q["backend"][i])
            mo.extend(q["model"][i])
        slo.append(int(q["slo"]))
        if with_caps:
            cap.extend(int(x) for x in q["cap"])
    return Batch(
        R=len(reqs), B=B, M=M,
        node_off=np.asarray(node_off, dtype=np.int32), opt_off=np.asarray(opt_off, dtype=np.int32),
        pred_mask=np.asarray(pm, dtype=np.uint32), vuln=np.asarray(vu, dtype=np.float32),
        lat_us=np.asarray(la, dtype=np.int32), acc=np.asarray(ac, dtype=np.float32),
        demand=np.asarray(de, dtype=np.int32), backend=np.asarray(be, dtype=np.uint8),
        model=np.asarray(mo, dtype=np.uint8), slo_us=np.asarray(slo, dtype=np.int32),
        cap=np.asarray(cap, dtype=np.int32) if with_caps else None,
    )


def random_pred_masks(rng, n: int, p: float) -> list[int]:
    """Arbitrary DAG on a fixed topological order: each pair u<v is an edge with prob p."""
    pm = [0] * n
    for v in range(n):
        for u in range(v):
            if rng.random() < p:
                pm[v] |= 1 << u
    return pm


def random_request(rng, n: int, kmin: int, kmax: int, B: int, M: int, *, edge_p: float = 0.4,
                   tool_p: float = 0.0, slo_q: float = 0.5, cap_frac: Optional[float] = 0.6,
                   lat_hi: int = 3000, mults: Optional[np.ndarray] = None) -> dict:
    """A ragged random request: node n has K_n ~ U{kmin..kmax} options (a tool node,
    K_n = 1 with acc = 1 and demand 0, with probability ``tool_p``; reading Q8)."""
    pm = random_pred_masks(rng, n, edge_p)
    q = dict(pred_mask=pm, vuln=rng.uniform(0, 1, size=n).astype(np.float32), lat=[], acc=[], demand=[],
             backend=[], model=[])
    for i in range(n):
        if rng.random() < tool_p:
            q["lat"].append([int(rng.integers(1, lat_hi))]); q["acc"].append([1.0]); q["demand"].append([0])
            q["backend"].append([int(rng.integers(0, B))]); q["model"].append([int(rng.integers(0, M))])
            continue
        k = int(rng.integers(kmin, kmax + 1))
        q["lat"].append([int(x) for x in rng.integers(1, lat_hi, size=k)])
        q["acc"].append([float(np.float32(x)) for x in rng.uniform(0.5, 1.0, size=k)])
        q["demand"].append([int(x) for x in rng.integers(0, 4001, size=k)])
        q["backend"].append([int(x) for x in rng.integers(0, B, size=k)])
        q["model"].append([int(x) for x in rng.integers(0, M, size=k)])
    if mults is None:
        mults = np.full((1, B), 1000, dtype=np.int64)
    # SLO from the same sampled-quantile recipe on a padded rectangular copy of the ragged tables
    kmx = max(len(x) for x in q["lat"])
    lat = np.zeros((n, kmx), dtype=np.int64); be = np.zeros((n, kmx), dtype=np.uint8)
    for i in range(n):
        k = len(q["lat"][i])
        reps = -(-kmx // k)
        lat[i] = (q["lat"][i] * reps)[:kmx]
        be[i] = (q["backend"][i] * reps)[:kmx]
    q["slo"] = _sampled_latency_quantile(rng, pm, lat, be, np.asarray(mults, dtype=np.int64), slo_q, n_draws=200)
    if cap_frac is not None:
        q["cap"] = []
        for b in range(B):
            tot = 0
            for i in range(n):
                on_b = [d for d, bb in zip(q["demand"][i], q["backend"][i]) if bb == b]
                tot += max(on_b) if on_b else 0
            q["cap"].append(int(np.floor(cap_frac * tot)))
    return q


def random_workload(seed: int, R: int, nmin: int, nmax: int, kmin: int, kmax: int, B: int = 2, M: int = 3,
                    L: int = 3, *, caps: bool = True, tool_p: float = 0.15, edge_p: float = 0.4,
                    slo_q: float = 0.5) -> Workload:
    rng = np.random.default_rng(seed)
    mult = rng.integers(1000, 3001, size=(L, B)).astype(np.int32)
    reqs = [random_request(rng, int(rng.integers(nmin, nmax + 1)), kmin, kmax, B, M, edge_p=edge_p, tool_p=tool_p,
                           slo_q=slo_q, cap_frac=0.6 if caps else None, mults=mult) for _ in range(R)]
    batch = batch_from_requests(reqs, B, M, caps)
    return Workload(name=f"random(seed={seed},R={R})", kind="compile", batch=batch, L=L,
                    mult_pm=np.ascontiguousarray(mult.reshape(-1)), meta=dict(seed=seed))


def random_down_set(rng, pred_masks, p: float) -> int:
    """A random predecessor-closed node set (a down-set of the DAG): visit the nodes in topological order and take
    a node with probability ``p`` if all its predecessors were taken.  PAPER.md:129: a node is dispatched only after
    its predecessors finished; PAPER.md:521-530 (App. D): the committed bindings are a set, not a prefix."""
    m = 0
    for v, pm in enumerate(pred_masks):
        if (int(pm) & ~m) == 0 and rng.random() < p:
            m |= 1 << v
    return m


def random_replan_workload(seed: int, R: int, nmin: int, nmax: int, kmin: int, kmax: int, B: int = 2, M: int = 3,
                           *, caps: bool = True, flags: int = FLAG_FIXED_IN_PLACE, tool_p: float = 0.1,
                           shape: str = "mixed") -> Workload:
    """Replan queries with a predecessor-closed dispatched set.  ``shape``: "prefix" = a random prefix of the node
    order (any prefix of a topological order is predecessor-closed); "downset" = a random down-set of the DAG, in
    general NOT a prefix (nodes {0, 2} when 2 does not depend on 1); "mixed" = either, per query."""
    w = random_workload(seed, R, nmin, nmax, kmin, kmax, B, M, L=1, caps=caps, tool_p=tool_p)
    rng = np.random.default_rng(seed + 7919)
    b = w.batch
    disp = np.zeros(R, dtype=np.uint32)
    fc = np.zeros(b.NN, dtype=np.uint8)
    for r in range(R):
        n = b.n_nodes(r)
        d = int(rng.integers(0, n + 1))
        disp[r] = (1 << d) - 1
        rad = b.radices(r)
        for i in range(n):
            fc[b.node_off[r] + i] = int(rng.integers(0, rad[i]))
    if shape != "prefix":
        rng2 = np.random.default_rng(seed + 104729)
        for r in range(R):
            if shape == "mixed" and rng2.random() < 0.35:
                continue
            pm = b.pred_mask[b.node_off[r]: b.node_off[r + 1]]
            disp[r] = random_down_set(rng2, pm, float(rng2.uniform(0.3, 0.9)))
    live = rng.integers(1000, 4001, size=(R, B)).astype(np.int32)
    return Workload(name=f"random_replan(seed={seed},R={R},{shape})", kind="replan", batch=b, L=1,
                    dispatched_mask=disp, fixed_choice=fc, live_mult_pm=np.ascontiguousarray(live.reshape(-1)),
                    flags=flags, meta=dict(seed=seed))


def with_down_set_dispatch(w: Workload, seed: int, p_lo: float = 0.3, p_hi: float = 0.8, max_free_plans: int = 1 << 26,
                           flags: Optional[int] = None) -> Workload:
    """The replan workload ``w`` (e.g. configs[3]) with every query's dispatched set redrawn as a random down-set of
    its DAG (not a prefix) and a uniformly drawn fixed option on every node; all other inputs unchanged.  A draw that
    leaves more than ``max_free_plans`` plans to enumerate is redrawn (keeps the oracle affordable)."""
    assert w.kind == "replan"
    rng = np.random.default_rng(seed)
    b = w.batch
    disp = np.zeros(b.R, dtype=np.uint32)
    fc = np.zeros(b.NN, dtype=np.uint8)
    for r in range(b.R):
        n0, n1 = int(b.node_off[r]), int(b.node_off[r + 1])
        rad = b.radices(r)
        fc[n0:n1] = [int(rng.integers(0, k)) for k in rad]
        for _ in range(64):
            m = random_down_set(rng, b.pred_mask[n0:n1], float(rng.uniform(p_lo, p_hi)))
            free = 1
            for i, k in enumerate(rad):
                if not (m >> i) & 1:
                    free *= int(k)
            if free <= max_free_plans:
                break
        disp[r] = m
    return replace(w, name=w.name + "+downsets", dispatched_mask=disp, fixed_choice=fc,
                   flags=w.flags if flags is None else flags)
