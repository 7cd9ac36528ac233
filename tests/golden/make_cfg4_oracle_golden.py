#!/usr/bin/env python
"""Writes tests/golden/cfg4_requests_0_1_oracle.txt: the brute-force oracle's records for requests 0 and 1 of
BASELINE.json configs[4] ("16 large requests ... 6^12 ~ 2.18e9 plans per request ... oracle run on 2 of the 16
requests only"; "oracle on requests 0 and 1 only").

Calls ONLY oracle/ (the fp64 brute force) and the seeded input generator tests/support/workloads.py; nothing from the
CUDA path.  The two requests cost the oracle 3.5e10 (plan, level) evaluations (minutes on 8-16 host threads), which is
why the -m gpu test reads this file instead of re-running it.  The file carries a digest of every input array of the
two requests, so a change of the generator invalidates it loudly (tests/test_gpu_full_size.py checks the digest).

    python tests/golden/make_cfg4_oracle_golden.py          # rewrites the file
"""
from __future__ import annotations

import hashlib
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)
sys.path.insert(1, os.path.join(ROOT, "tests"))
OUT = os.path.join(HERE, "cfg4_requests_0_1_oracle.txt")
ROWS = [0, 1]


def input_digest(w) -> str:
    """sha256 over every input array of the workload, in a fixed order."""
    b = w.batch
    h = hashlib.sha256()
    for a in (b.node_off, b.opt_off, b.pred_mask, b.vuln, b.lat_us, b.acc, b.demand, b.backend, b.model, b.slo_us,
              b.cap, w.mult_pm):
        a = np.ascontiguousarray(a)
        h.update(str(a.dtype).encode() + b"|" + str(a.shape).encode() + b"|")
        h.update(a.tobytes())
    h.update(f"R={b.R} B={b.B} M={b.M} L={w.L}".encode())
    return h.hexdigest()


def main():
    from oracle import oracle
    from support import workloads as wl
    oracle.build()
    w = wl.make_config(4).subset(ROWS)
    t0 = time.time()
    ref = oracle.run(w)
    dt = time.time() - t0
    L, B = w.L, w.batch.B
    with open(OUT, "w") as f:
        f.write("# Brute-force oracle (oracle/dyplan_oracle.c, fp64 / int64) on requests 0 and 1 of BASELINE.json configs[4]\n")
        f.write("# (seed 4, 12-node layered DAGs, 6 options per node, 8 pressure levels, 3 backends, caps): 2 x 6^12 plans x 8 levels.\n")
        f.write("# Source of the values: tests/golden/make_cfg4_oracle_golden.py, which calls only oracle/ and the input generator.\n")
        f.write("# Citation for the case: BASELINE.json configs[4]; SURVEY.md 8(d) D.2; the objective: PAPER.md:186-193 Eq.(3), Alg. 1 l.10-13.\n")
        f.write(f"# oracle wall time when written: {dt:.0f} s on {oracle.num_threads()} threads\n")
        f.write("# floats are C99 hex floats (exact)\n")
        f.write(f"digest | {input_digest(w)}\n")
        f.write("# rec | status | plan_idx | corr | lat | dem[0..B) | dom_model | runner_idx | runner_corr | n_feasible | choice[0..16)\n")
        for rec in range(len(ROWS) * L):
            row = [rec, int(ref["status"][rec]), int(ref["plan_idx"][rec]), float(ref["corr"][rec]).hex(), int(ref["lat"][rec]),
                   " ".join(str(int(x)) for x in ref["dem"][rec]), int(ref["dom_model"][rec]), int(ref["runner_idx"][rec]),
                   float(ref["runner_corr"][rec]).hex(), int(ref["n_feasible"][rec]),
                   " ".join(str(int(x)) for x in ref["choice"][rec])]
            f.write(" | ".join(str(x) for x in row) + "\n")
    print(f"wrote {OUT} ({dt:.0f} s)")


if __name__ == "__main__":
    main()
