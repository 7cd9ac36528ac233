"""Pins of oracle/switch_oracle.py (the paper's stateful selector) against what the paper fixes:
the worked Case A / Case B of Fig. 7(c) (tests/golden/paper_fig7c_switch_cases.txt) and each sentence of Section 5.1
as a scenario whose outcome can be read off the sentence.  Thresholds themselves are never printed in the paper
(parity unpinned for constants); every scenario below depends on the ORDER relations only."""
from __future__ import annotations

import math

from conftest import read_golden
from oracle import switch_oracle as so

P = dict(hi_load=0.8, lo_load=0.3, load_margin=0.1, quality_tol=0.15, min_dwell=5.0)

# option encoding of the Fig. 7 example: per node, option index -> label
OPT = {"27B": 0, "27B+V": 1, "9B": 2, "9B+V": 3}
M27, M9 = 0, 1


def fig7_bundle():
    """pi(0) = (P: 27B, C: 27B, D: 9B+V, A: 27B) dominant 27B, accuracy 90; pi(1) = (.., C: 9B, D: 9B, ..) dominant 9B,
    accuracy 80 (Fig. 7(a): 'Illustrative accuracy' 90 / 80)."""
    choice = [[OPT["27B"], OPT["27B"], OPT["9B+V"], OPT["27B"]] + [255] * 12,
              [OPT["27B"], OPT["9B"], OPT["9B"], OPT["27B"]] + [255] * 12]
    return dict(L=2, n_nodes=4, status=[0, 0], dom_model=[M27, M9], quality=[0.90, 0.80], choice=choice)


def test_fig7c_case_a_and_b_from_the_paper():
    rows = read_golden("paper_fig7c_switch_cases.txt")
    assert [r[0] for r in rows] == ["A", "B"]
    names = {"P": 0, "C": 1, "D": 2, "A": 3}
    b = fig7_bundle()
    for case, disp, c_tr, d_tr, _ in rows:
        mask = 0
        for nm in disp.split(","):
            mask |= 1 << names[nm.strip()]
        c_before, c_after = [x.strip() for x in c_tr.split("->")]
        d_before, d_after = [x.strip() for x in d_tr.split("->")]
        active = list(b["choice"][0])
        assert active[1] == OPT[c_before] and active[2] == OPT[d_before]
        # "27B load > threshold; dwell met"
        v, act, how = so.switch_one(load=[0.95, 0.2], cur=0, since_switch=10.0, dispatched_mask=mask, active=active,
                                    **b, **{**P, "quality_tol": 0.15})
        assert (v, how) == (1, 1), case                      # "Select precompiled pi(1) . No solver"
        assert act[1] == OPT[c_after] and act[2] == OPT[d_after], case
        assert act[0] == active[0]                           # P is done in both cases: never touched


def test_dwell_blocks_a_switch_in_either_direction():
    b = fig7_bundle()
    a = list(b["choice"][0])
    assert so.switch_one(load=[0.95, 0.2], cur=0, since_switch=4.9, dispatched_mask=0, active=a, **b, **P)[0] == 0
    a1 = list(b["choice"][1])
    assert so.switch_one(load=[0.1, 0.2], cur=1, since_switch=4.9, dispatched_mask=0, active=a1, **b, **P)[0] == 1
    assert so.switch_one(load=[0.1, 0.2], cur=1, since_switch=5.0, dispatched_mask=0, active=a1, **b, **P)[::2] == (0, 2)


def test_same_congested_class_is_skipped_even_with_less_verification():
    # "Reducing verification while retaining the congested dominant model is therefore insufficient."
    ch = [[1] + [255] * 15, [0] + [255] * 15, [2] + [255] * 15]
    b = dict(L=3, n_nodes=1, status=[0, 0, 0], dom_model=[M27, M27, M9], quality=[0.9, 0.88, 0.85], choice=ch)
    v, act, how = so.switch_one(load=[0.9, 0.1], cur=0, since_switch=9.0, dispatched_mask=0, active=[1] + [255] * 15, **b, **P)
    assert (v, how, act[0]) == (2, 1, 2)


def test_overloaded_or_not_sufficiently_lower_candidates_are_skipped():
    ch = [[0] + [255] * 15, [1] + [255] * 15, [2] + [255] * 15]
    b = dict(L=3, n_nodes=1, status=[0, 0, 0], dom_model=[0, 1, 2], quality=[0.9, 0.9, 0.9], choice=ch)
    a = [0] + [255] * 15
    # candidate 1 itself overloaded -> 2
    assert so.switch_one(load=[0.95, 0.85, 0.2], cur=0, since_switch=9.0, dispatched_mask=0, active=a, **b, **P)[0] == 2
    # candidate 1 below hi but not by the margin (0.95 - 0.1 = 0.85 < 0.8? no: 0.8 <= 0.85 passes) -> 1
    assert so.switch_one(load=[0.95, 0.8, 0.2], cur=0, since_switch=9.0, dispatched_mask=0, active=a, **b, **P)[0] == 1
    # cur just above hi: candidate at 0.78 is within the margin (0.81 - 0.1 = 0.71) -> skipped, 2 taken
    assert so.switch_one(load=[0.81, 0.78, 0.2], cur=0, since_switch=9.0, dispatched_mask=0, active=a, **b, **P)[0] == 2
    # everyone overloaded: retained
    assert so.switch_one(load=[0.95, 0.9, 0.9], cur=0, since_switch=9.0, dispatched_mask=0, active=a, **b, **P)[::2] == (0, 0)


def test_quality_tolerance_rejects_even_an_idle_backend():
    # "It rejects a candidate whose estimated quality drop exceeds a configured tolerance, even if the candidate's backend is idle."
    b = fig7_bundle()
    a = list(b["choice"][0])
    tight = {**P, "quality_tol": 0.05}
    assert so.switch_one(load=[0.95, 0.0], cur=0, since_switch=9.0, dispatched_mask=0, active=a, **b, **tight)[::2] == (0, 0)
    assert so.switch_one(load=[0.95, 0.0], cur=0, since_switch=9.0, dispatched_mask=0, active=a, **b, **P)[0] == 1


def test_return_goes_directly_to_the_lowest_index_variant_below_the_low_threshold():
    ch = [[k] + [255] * 15 for k in range(4)]
    b = dict(L=4, n_nodes=1, status=[0, 0, 0, 0], dom_model=[0, 1, 2, 3], quality=[0.9, 0.88, 0.86, 0.84], choice=ch)
    a = [3] + [255] * 15
    # model 0 still warm (0.5 >= lo), model 1 cool -> variant 1, not 2
    assert so.switch_one(load=[0.5, 0.2, 0.1, 0.4], cur=3, since_switch=9.0, dispatched_mask=0, active=a, **b, **P)[::2] == (1, 2)
    # everything cool -> straight to variant 0
    assert so.switch_one(load=[0.1, 0.2, 0.1, 0.4], cur=3, since_switch=9.0, dispatched_mask=0, active=a, **b, **P)[::2] == (0, 2)
    # nothing below lo -> retained (between lo and hi is the hysteresis band)
    assert so.switch_one(load=[0.5, 0.5, 0.5, 0.5], cur=3, since_switch=9.0, dispatched_mask=0, active=a, **b, **P)[::2] == (3, 0)


def test_missing_variants_and_first_install_and_nan():
    ch = [[k] + [255] * 15 for k in range(3)]
    b = dict(L=3, n_nodes=1, status=[1, 0, 0], dom_model=[255, 0, 1], quality=[-1.0, 0.9, 0.85], choice=ch)
    a = [255] * 16
    v, act, how = so.switch_one(load=[0.1, 0.1], cur=-1, since_switch=0.0, dispatched_mask=0, active=a, **b, **P)
    assert (v, how, act[0]) == (1, 3, 1)                     # variant 0 holds no plan: first usable one is installed
    a = [1] + [255] * 15
    assert so.switch_one(load=[math.nan, 0.1], cur=1, since_switch=9.0, dispatched_mask=0, active=a, **b, **P)[::2] == (1, 0)
    assert so.switch_one(load=[0.95, math.nan], cur=1, since_switch=9.0, dispatched_mask=0, active=a, **b, **P)[::2] == (1, 0)
    none = dict(b, status=[1, 1, 1])
    assert so.switch_one(load=[0.1, 0.1], cur=-1, since_switch=0.0, dispatched_mask=0, active=[255] * 16, **none, **P)[::2] == (-1, 0)


def test_a_second_call_with_the_same_load_is_a_fixed_point():
    b = fig7_bundle()
    a = list(b["choice"][0])
    v, act, _ = so.switch_one(load=[0.95, 0.2], cur=0, since_switch=10.0, dispatched_mask=0b0001, active=a, **b, **P)
    v2, act2, how2 = so.switch_one(load=[0.95, 0.2], cur=v, since_switch=10.0, dispatched_mask=0b0001, active=act, **b, **P)
    assert (v2, how2, act2) == (v, 0, act)
