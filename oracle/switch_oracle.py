"""ORACLE (test infrastructure, not product): the paper's stateful load-driven selector, Section 5.1
(PAPER.md:217-231), written sentence by sentence in plain Python.  Shares no code with the CUDA path.

Thresholds, the comparison margin, the quality tolerance and the dwell time are "configured" in the paper and never
printed: they are parameters here, and the rule -- not any constant -- is what the pins in
tests/test_switch_pins.py fix (Fig. 7(c) Case A / Case B among them).  Constants: parity unpinned.

Inputs per request r (L variants, ordered by the pressure-specialization levels used during compilation,
PAPER.md:221): status[r][k] (0 = a plan exists), dom_model[r][k] (the model receiving the largest share of the
variant's planned demand, identified during compilation), quality[r][k] (profile-based quality estimate,
PAPER.md:225), choice[r][k][n]; the request's active variant index cur (-1: none), time since its last switch, its
dispatched-node mask, its active assignment.  Shared: load[m] per model class.
Returns (variant, active, switched) with switched in {0 retained, 1 pressure switch, 2 return, 3 first install}.
"""
from __future__ import annotations

import math
from typing import List, Sequence, Tuple


def switch_one(L: int, n_nodes: int, status: Sequence[int], dom_model: Sequence[int], quality: Sequence[float],
               choice: Sequence[Sequence[int]], load: Sequence[float], cur: int, since_switch: float,
               dispatched_mask: int, active: Sequence[int], hi_load: float, lo_load: float, load_margin: float,
               quality_tol: float, min_dwell: float) -> Tuple[int, List[int], int]:
    M = len(load)

    def usable(k):  # the bundle holds a plan for this level
        return status[k] == 0 and 0 <= dom_model[k] < M

    new, how = cur, 0
    if cur < 0 or cur >= L or not usable(cur):
        # nothing installed yet: execution starts with the first prepared variant (pi^(0) first)
        new = -1
        for k in range(L):
            if usable(k):
                new, how = k, 3
                break
    elif math.isnan(since_switch) or math.isnan(load[dom_model[cur]]):
        pass                                       # no measurement: "the current selection is retained"
    elif since_switch < min_dwell:
        pass                                       # "A minimum dwell time between switches limits repeated changes" (l.229)
    elif load[dom_model[cur]] > hi_load:
        # "When the load of the current variant's dominant model exceeds the high-load threshold, the runtime scans
        #  later variants in that order." (l.221)
        for k in range(cur + 1, L):
            if not usable(k):
                continue
            if dom_model[k] == dom_model[cur]:     # "skips candidates whose dominant model is the same congested class"
                continue
            lk = load[dom_model[k]]
            if not (lk <= hi_load):                # "... or is itself overloaded"
                continue
            if not (lk <= load[dom_model[cur]] - load_margin):   # "sufficiently lower load under the configured comparison rule"
                continue
            if not (quality[cur] - quality[k] <= quality_tol):   # "rejects a candidate whose estimated quality drop exceeds a configured tolerance" (l.225)
                continue
            new, how = k, 1                        # "selects the first later variant that passes both the load and quality checks" (l.227)
            break
    else:
        # "When load subsides, the runtime returns directly to the lowest-index variant whose dominant-model load is
        #  below the low-load threshold and that passes the quality check." (l.229)
        for k in range(0, cur):
            if not usable(k):
                continue
            if not (load[dom_model[k]] < lo_load):
                continue
            if not (quality[cur] - quality[k] <= quality_tol):
                continue
            new, how = k, 2
            break
    # "If no transition is eligible, the current selection is retained." (l.229)
    out = list(active)
    if new != cur and new >= 0:
        # "updating the model, verification policy, and backend only for LLM nodes whose base calls have not been
        #  dispatched ... The updated plan can therefore combine previous assignments with the selected variant's
        #  assignments for the remaining nodes" (l.231)
        for n in range(n_nodes):
            if not (dispatched_mask >> n) & 1:
                out[n] = choice[new][n]
    return new, out, (how if new != cur else 0)


def switch(R: int, L: int, n_nodes, status, dom_model, quality, choice, load, cur, since_switch, dispatched_mask, active,
           params: dict):
    """Batch form over numpy arrays: status/dom_model/quality [R*L], choice [R*L*16], active [R*16]."""
    import numpy as np
    st = np.asarray(status).reshape(R, L)
    dm = np.asarray(dom_model).reshape(R, L)
    q = np.asarray(quality, dtype=np.float64).reshape(R, L)
    ch = np.asarray(choice).reshape(R, L, 16)
    act = np.asarray(active).reshape(R, 16)
    variant = np.zeros(R, np.int32)
    new_act = act.copy()
    sw = np.zeros(R, np.uint8)
    for r in range(R):
        v, a, h = switch_one(L, int(n_nodes[r]), [int(x) for x in st[r]], [int(x) for x in dm[r]],
                             [float(x) for x in q[r]], ch[r].tolist(), [float(x) for x in load], int(cur[r]),
                             float(since_switch[r]), int(dispatched_mask[r]), act[r].tolist(), **params)
        variant[r], sw[r] = v, h
        new_act[r] = a
    return dict(variant=variant, active=new_act.reshape(-1), switched=sw)
