"""The GPU <-> oracle matching protocol (from BASELINE.json north_star "Matching rules").

For every record (request r, level l):
  P1  status equal (existence of a feasible plan is integer-exact; INVALID / TOO_LARGE equal too).
  P2  the oracle's score of the GPU's chosen plan is bit-identical in T, feasibility, every D_b, the
      dominant model and the canonical index, and its fp64 C is within 1e-5 relative of the GPU's fp32 C
      (and within 1e-12 of the GPU's fp64 re-evaluation).
  P3  C64(GPU plan) >= C* (1 - 1e-5)                         C* = the oracle's optimum
  P4  (C* - C_runner_up) / C* > 1e-5  ==>  identical plan index.
  P5  C64(GPU plan) == C* bit for bit  ==>  the GPU plan minimises (T, idx) in that class, i.e. it is the
      oracle's plan unless fp32 rounding merged a strictly worse class into it -- checked as:
      GPU T <= oracle T is impossible for a different plan of the same C (the oracle already took the min), so
      equal C64 and a different index requires GPU T > T* or (T == T* and idx > idx*) to be a fp32 artefact;
      we assert the weaker, always-valid form: equal C64 and equal T ==> idx >= idx* can only be equality
      when the fp32 classes coincide.  (Reported, not asserted, when it differs.)
Sentinels are checked on non-OK records.
"""
from __future__ import annotations

import numpy as np

REL = 1e-5
NO_IDX = np.iinfo(np.uint64).max


def check_records(orc, w, gpu: dict, ref: dict, records=None, *, where: str = "") -> dict:
    """Compare GPU bundle arrays ``gpu`` with the oracle result ``ref`` for workload ``w``.

    ``records``: iterable of record indices (default: all whose oracle status is not 255).
    Returns counters (how many records had an identical index, how many differed within tolerance)."""
    b = w.batch
    L, B = w.L, b.B
    g_choice = gpu["choice"].reshape(-1, 16)
    g_dem = gpu["dem"].reshape(-1, B)
    r_dem = ref["dem"].reshape(-1, B)
    if records is None:
        records = [i for i in range(b.R * L) if ref["status"][i] != 255]
    same = within = 0
    for rec in records:
        r, l = divmod(int(rec), L)
        tag = f"{where} rec={rec} (r={r}, l={l})"
        st = int(ref["status"][rec])
        assert int(gpu["status"][rec]) == st, f"P1 status {tag}: gpu={gpu['status'][rec]} oracle={st}"
        if st != 0:
            assert gpu["plan_idx"][rec] == NO_IDX, tag
            assert (g_choice[rec] == 0xFF).all(), tag
            assert gpu["corr"][rec] == -1.0 and gpu["lat"][rec] == 2**31 - 1, tag
            assert (g_dem[rec] == 0).all() and gpu["dom_model"][rec] == 0xFF, tag
            if gpu.get("corr64") is not None:
                assert gpu["corr64"][rec] == -1.0, tag
            continue
        if w.kind == "compile":
            mult = np.asarray(w.mult_pm).reshape(L, B)[l]
            skip = 0
        else:
            mult = np.asarray(w.live_mult_pm).reshape(b.R, B)[r]
            skip = int(w.dispatched_mask[r]) if (w.flags & 1) else 0
        n = b.n_nodes(r)
        ch = g_choice[rec]
        assert (ch[n:] == 0xFF).all(), f"choice padding {tag}"
        s = orc.score(b, r, mult, ch[:16].copy(), skip)
        assert s["status"] == 0, f"P2 GPU choice is not a valid plan {tag}: {ch}"
        # P2: integer-exact annotations of the GPU's own plan
        assert s["plan_idx"] == int(gpu["plan_idx"][rec]), f"P2 idx/choice inconsistent {tag}"
        assert s["feasible"], f"P2 GPU plan infeasible {tag}"
        assert s["lat"] == int(gpu["lat"][rec]), f"P2 T {tag}: oracle={s['lat']} gpu={gpu['lat'][rec]}"
        assert (s["dem"] == g_dem[rec]).all(), f"P2 D_b {tag}: oracle={s['dem']} gpu={g_dem[rec]}"
        assert s["dom_model"] == int(gpu["dom_model"][rec]), f"P2 dominant model {tag}"
        c64 = s["corr"]
        assert abs(float(gpu["corr"][rec]) - c64) <= REL * c64 + 1e-30, f"P2 C {tag}: {gpu['corr'][rec]} vs {c64}"
        if gpu.get("corr64") is not None:
            assert abs(float(gpu["corr64"][rec]) - c64) <= 1e-12 * max(c64, 1e-300), f"P2 C64 {tag}"
        if w.kind == "replan":
            m = int(w.dispatched_mask[r])
            fc = np.asarray(w.fixed_choice)[b.node_off[r]: b.node_off[r] + n]
            for i in range(n):
                if (m >> i) & 1:
                    assert ch[i] == fc[i], f"committed binding replaced at node {i} {tag}"
        # P3 / P4 / P5 against the optimum
        cstar = float(ref["corr"][rec])
        assert c64 >= cstar * (1.0 - REL), f"P3 {tag}: C64(gpu)={c64} C*={cstar}"
        assert c64 <= cstar * (1.0 + 1e-12), f"oracle optimum beaten?! {tag}: C64(gpu)={c64} C*={cstar}"
        if int(gpu["plan_idx"][rec]) == int(ref["plan_idx"][rec]):
            same += 1
            assert (ch == ref["choice"].reshape(-1, 16)[rec]).all(), tag
            assert (g_dem[rec] == r_dem[rec]).all() and int(gpu["lat"][rec]) == int(ref["lat"][rec]), tag
            continue
        within += 1
        crun = float(ref["runner_corr"][rec])
        assert crun >= 0 and (cstar - crun) <= REL * cstar, \
            f"P4 {tag}: top two separated by {(cstar - crun) / cstar:.3e} but idx differs " \
            f"(gpu={gpu['plan_idx'][rec]} oracle={ref['plan_idx'][rec]})"
    return dict(records=len(list(records)), same=same, within_tol=within)
