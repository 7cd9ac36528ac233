"""The N > 1 host logic on CPU: two processes, torch.distributed with the gloo backend (127.0.0.1).

What is exercised is what bench.py --gpus N and a request-sharded compile rely on: balanced request shards, distinct
per-rank batches, the max-over-ranks of the timings, whole-job throughput, and gathering per-request records in rank
order.  There is no data-path collective to test: the records of a shard come from a local
solver -- here the oracle, because no GPU exists on this box -- and must equal the single-process result."""
from __future__ import annotations

import os
import socket

import numpy as np
import pytest

from paper_2607_02942_b200 import multi
from support import workloads as wl


def test_shard_requests_is_a_balanced_partition():
    for R in (0, 1, 5, 16, 4096, 16385):
        for world in (1, 2, 3, 8):
            sh = multi.shard_requests(R, world)
            assert len(sh) == world and sh[0][0] == 0 and sh[-1][1] == R
            assert all(sh[i][1] == sh[i + 1][0] for i in range(world - 1))
            sizes = [e - b for b, e in sh]
            assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        multi.shard_requests(4, 0)


def test_rank_seeds_give_distinct_batches_of_the_same_shape():
    a = wl.make_config(2, R=4, seed=multi.rank_seed(2, 0))
    b = wl.make_config(2, R=4, seed=multi.rank_seed(2, 1))
    ref = wl.make_config(2, R=4)
    assert np.array_equal(a.batch.lat_us, ref.batch.lat_us)             # rank 0 runs the config's own seed
    assert a.batch.lat_us.shape == b.batch.lat_us.shape and not np.array_equal(a.batch.lat_us, b.batch.lat_us)
    assert a.n_plans_total() == b.n_plans_total()


def test_whole_job_rate():
    assert multi.whole_job_rate(100.0, 4, 10, 2000.0) == pytest.approx(2000.0)
    assert multi.max_over_ranks([1.0, 2.5]) == [1.0, 2.5]               # no process group: identity


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, q):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import oracle
        w = wl.random_workload(7, R=9, nmin=2, nmax=5, kmin=2, kmax=4, B=2, M=2, L=2, caps=True)
        b, e = multi.shard_requests(w.batch.R, world)[rank]
        local = oracle.run(w.subset(list(range(b, e))))
        rec = {k: np.asarray(local[k]) for k in ("plan_idx", "lat", "status", "corr")}
        # fake timings: rank r took (r + 1) ms per step and 10 * (r + 1) ms end to end
        t = multi.max_over_ranks([float(rank + 1), 10.0 * (rank + 1)])
        dist.barrier()
        full = multi.gather_records(rec, world, rank)
        if rank == 0:
            q.put(("ok", t, {k: v.tolist() for k, v in full.items()}))
    except Exception as ex:  # pragma: no cover
        q.put(("error", repr(ex), None))
        raise
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo_shard_reduce_gather(orc):
    import torch.multiprocessing as mp
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    status, t, full = q.get(timeout=180)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert status == "ok", t
    assert t == [2.0, 20.0]                                             # max over ranks of each timing
    w = wl.random_workload(7, R=9, nmin=2, nmax=5, kmin=2, kmax=4, B=2, M=2, L=2, caps=True)
    ref = orc.run(w)
    for k in ("plan_idx", "lat", "status"):
        assert np.array_equal(np.asarray(full[k], dtype=np.asarray(ref[k]).dtype), np.asarray(ref[k])), k
    assert np.allclose(np.asarray(full["corr"]), np.asarray(ref["corr"]), rtol=0, atol=0)
