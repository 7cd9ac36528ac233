"""The plan-bundle cache (variants reused across requests with the same workflow) is host logic:
tested on CPU with the oracle standing in for the compile call."""
from __future__ import annotations

import numpy as np

from support import workloads as wl
from paper_2607_02942_b200.cache import BundleCache, request_key

FIELDS = ("plan_idx", "choice", "corr", "lat", "dem", "dom_model", "status")


def make(seed, R=12, L=3):
    return wl.random_workload(seed, R=R, nmin=2, nmax=5, kmin=2, kmax=4, B=2, M=2, L=L, caps=True)


def test_cache_returns_the_compile_results_and_compiles_each_workflow_once(orc):
    w = make(1)
    calls = []

    def compile_fn(batch, rows):
        calls.append(list(rows))
        res = orc.run(w.subset(rows))
        return {k: np.asarray(res[k]) for k in FIELDS}

    ref = orc.run(w)
    c = BundleCache(capacity=64)
    out = c.compile(w.batch, w.L, w.mult_pm, compile_fn)
    for k in FIELDS:
        assert np.array_equal(out[k], np.asarray(ref[k]).reshape(-1)), k
    assert (c.hits, c.misses, calls) == (0, 12, [list(range(12))])
    out2 = c.compile(w.batch, w.L, w.mult_pm, compile_fn)             # same workflows again: nothing is compiled
    assert (c.hits, c.misses, len(calls)) == (12, 12, 1)
    for k in FIELDS:
        assert np.array_equal(out2[k], out[k]), k


def test_duplicates_inside_a_batch_and_partial_hits(orc):
    w = make(2, R=6)
    dup = w.subset([0, 1, 0, 2, 1, 0])                                 # three distinct workflows
    calls = []

    def compile_fn(batch, rows):
        calls.append(list(rows))
        res = orc.run(dup.subset(rows))
        return {k: np.asarray(res[k]) for k in FIELDS}

    c = BundleCache()
    out = c.compile(dup.batch, dup.L, dup.mult_pm, compile_fn)
    assert calls == [[0, 1, 3]] and (c.hits, c.misses) == (3, 3)
    ref = orc.run(dup)
    for k in FIELDS:
        assert np.array_equal(out[k], np.asarray(ref[k]).reshape(-1)), k
    # a different level set is a different bundle
    m2 = np.asarray(dup.mult_pm).copy()
    m2[0] += 7
    c.compile(dup.batch, dup.L, m2, lambda b, rows: {k: np.asarray(orc.compile(dup.subset(rows).batch, dup.L, m2)[k]) for k in FIELDS})
    assert c.misses == 6


def test_key_covers_everything_the_compile_reads_and_nothing_else():
    w = make(3, R=4)
    b = w.batch
    k0 = [request_key(b, r) for r in range(4)]
    assert len(set(k0)) == 4
    b.slo_us[1] += 1
    b.acc[int(b.opt_off[int(b.node_off[2])])] = np.float32(0.123)
    k1 = [request_key(b, r) for r in range(4)]
    assert k1[0] == k0[0] and k1[3] == k0[3] and k1[1] != k0[1] and k1[2] != k0[2]
    # the key does not depend on where the request sits in the batch
    s = w.subset([3, 0])
    assert request_key(s.batch, 0) == k1[3] and request_key(s.batch, 1) == k1[0]


def test_lru_eviction():
    w = make(4, R=8)
    c = BundleCache(capacity=3)
    fake = lambda b, rows: {"status": np.zeros(len(rows) * w.L, np.uint8), "lat": np.arange(len(rows) * w.L, dtype=np.int32)}
    c.compile(w.batch, w.L, w.mult_pm, fake)
    assert len(c) == 3
    c.compile(w.subset([7]).batch, w.L, w.mult_pm, fake)              # the most recent one is still there
    assert c.hits == 1
    c.compile(w.subset([0]).batch, w.L, w.mult_pm, fake)              # the oldest was evicted
    assert c.misses == 9
