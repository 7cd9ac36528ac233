"""Host-side logic of the N > 1 path: requests are independent, so they shard across ranks
with NO data-path collective.  What the ranks exchange is bookkeeping only -- a barrier and the max over ranks of
the device timings -- through torch.distributed (NCCL on GPUs, gloo in the CPU tests).

Two ways to use N GPUs:
  * weak scaling (bench.py --gpus N): every rank compiles its own batch of the configured shape (`rank_seed`);
  * one batch split across ranks (`shard_requests` / `gather_records`): rank r compiles a contiguous slice of the
    requests and rank 0 collects the records, which are independent per request.
"""
from __future__ import annotations

from typing import Dict, List, Sequence, Tuple

import numpy as np


def rank_seed(cfg: int, rank: int) -> int:
    """Seed of the batch rank `rank` generates for BASELINE.json configs[cfg]: rank 0 runs the config's own seed."""
    return cfg + 1000 * rank


def shard_requests(R: int, world: int) -> List[Tuple[int, int]]:
    """Contiguous, balanced [begin, end) request ranges, one per rank; the first R % world ranks get one more."""
    if world < 1 or R < 0:
        raise ValueError("world >= 1 and R >= 0 required")
    base, extra = divmod(R, world)
    out, b = [], 0
    for r in range(world):
        e = b + base + (1 if r < extra else 0)
        out.append((b, e))
        b = e
    return out


def max_over_ranks(values: Sequence[float], device=None) -> List[float]:
    """Element-wise max over ranks of a few floats (the device timings of one measurement).  No-op when
    torch.distributed is not initialised."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.cpu()]


def whole_job_rate(units_per_rank: float, world: int, steps: int, max_ms: float) -> float:
    """Whole-job throughput: the units all ranks processed divided by the slowest rank's time."""
    return world * units_per_rank * steps / (max_ms * 1e-3)


def gather_records(local: Dict[str, np.ndarray], world: int, rank: int) -> Dict[str, np.ndarray] | None:
    """Concatenate per-rank record arrays (one batch sharded by `shard_requests`) on rank 0, in rank order.
    Records are independent per request, so this is pure bookkeeping (gather_object; not on the timed path)."""
    import torch.distributed as dist
    if world == 1:
        return local
    bucket = [None] * world if rank == 0 else None
    dist.gather_object(local, bucket, dst=0)
    if rank != 0:
        return None
    return {k: np.concatenate([b[k] for b in bucket]) for k in local}
