"""Plan-bundle cache ("prepared variants reused across requests with the same workflow";
SURVEY.md 2.1 A12 / 8(f) NEXT-4, second half).  Host-side memoisation above the C ABI: no arithmetic of the method
lives here.  A request's key is a digest of everything the compile reads for that request -- DAG, vulnerabilities,
per-option tables, SLO, caps -- plus the call-wide levels; equal keys give bit-identical records, so a hit returns the
stored records and only the misses are sent to `compile_fn` (which runs the CUDA path on a sub-batch).

    cache = BundleCache(capacity=4096)
    records = cache.compile(batch, L, mult_pm, compile_fn)      # compile_fn(sub_batch) -> dict of per-record arrays
"""
from __future__ import annotations

import hashlib
from collections import OrderedDict
from typing import Callable, Dict, List

import numpy as np

_NODE_FIELDS = ("pred_mask", "vuln")
_OPT_FIELDS = ("lat_us", "acc", "demand", "backend", "model")


def request_key(batch, r: int, extra: bytes = b"") -> bytes:
    """Digest of request r's inputs (and `extra`: the levels / multipliers / flags of the call)."""
    n0, n1 = int(batch.node_off[r]), int(batch.node_off[r + 1])
    o0, o1 = int(batch.opt_off[n0]), int(batch.opt_off[n1])
    h = hashlib.blake2b(digest_size=20)
    h.update(np.asarray([batch.B, batch.M, n1 - n0], np.int32).tobytes())
    h.update((np.asarray(batch.opt_off[n0:n1 + 1], np.int64) - o0).tobytes())
    for f in _NODE_FIELDS:
        h.update(np.ascontiguousarray(getattr(batch, f)[n0:n1]).tobytes())
    for f in _OPT_FIELDS:
        h.update(np.ascontiguousarray(getattr(batch, f)[o0:o1]).tobytes())
    h.update(np.asarray([batch.slo_us[r]], np.int32).tobytes())
    if batch.cap is not None:
        h.update(np.ascontiguousarray(np.asarray(batch.cap).reshape(batch.R, batch.B)[r]).tobytes())
    else:
        h.update(b"nocap")
    h.update(extra)
    return h.digest()


class BundleCache:
    """LRU cache of per-request record blocks (L records each)."""

    def __init__(self, capacity: int = 4096):
        self.capacity = int(capacity)
        self._d: "OrderedDict[bytes, Dict[str, np.ndarray]]" = OrderedDict()
        self.hits = 0
        self.misses = 0

    def __len__(self):
        return len(self._d)

    def compile(self, batch, L: int, mult_pm, compile_fn: Callable[[object, List[int]], Dict[str, np.ndarray]]):
        """Records of every request of `batch` ([R*L*w] arrays like dyplan_bundle's), compiling only the misses.
        compile_fn(batch, rows) must return the records of batch.subset(rows), in that order."""
        extra = np.asarray([L], np.int32).tobytes() + np.ascontiguousarray(mult_pm, np.int32).tobytes()
        keys = [request_key(batch, r, extra) for r in range(batch.R)]
        miss_rows, seen = [], {}
        for r, k in enumerate(keys):
            if k in self._d:
                self._d.move_to_end(k)
                self.hits += 1
            elif k in seen:
                self.hits += 1                      # a duplicate inside this batch: compiled once
            else:
                seen[k] = len(miss_rows)
                miss_rows.append(r)
                self.misses += 1
        fresh = compile_fn(batch, miss_rows) if miss_rows else {}
        blocks = {}
        for k, j in seen.items():
            blocks[k] = {name: np.array(a.reshape(len(miss_rows), -1)[j]) for name, a in fresh.items()}
        out: Dict[str, List[np.ndarray]] = {}
        for k in keys:
            blk = blocks.get(k) or self._d[k]
            for name, a in blk.items():
                out.setdefault(name, []).append(a)
        for k, blk in blocks.items():
            self._d[k] = blk
            while len(self._d) > self.capacity:
                self._d.popitem(last=False)
        return {name: np.concatenate(v) if v else np.zeros(0) for name, v in out.items()}
