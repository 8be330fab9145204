"""Pins for NEXT row N2 (R39): the embedded HU assignment of PAPER.md:L190 ("tours with minimum
and maximum completion times ... decreased and increased by one HU ... until the maximum completion time over all
tours cannot be further reduced") and L203 (non-uniform HUs: classes "sorted according to rising in-field
working rates")."""
from dataclasses import replace
import numpy as np
import pytest
from oracle import lgo
from paper_1909_10286_b200 import workloads as wl

Q = 1024
HU_BALANCE = 2        # lgx_instance_desc.flags bit 1


def test_trace_uniform_units_three_tours():
    """Worked by hand.  road 1 h each, areas (100, 40, 10) ha, five HUs of 2 ha/h on tours (0, 1, 2, 2, 2):
    T = (51, 21, 2.67).  Iter 1: g_max 0, g_2nd 1, donor 2; u2, u3 give T_0 = 26 (not < 21), u4 is the last ->
    moved; max 51 -> 26 kept.  Iter 2: u2 gives T_0 = 1 + 100/6 = 17.67 < 21 -> moved; max 26 -> 21 kept.
    Iter 3: the donor has one HU -> stop."""
    m, hu, T = lgo.hu_balance([1.0, 1.0, 1.0], [100 * Q, 40 * Q, 10 * Q], [2 * Q] * 5, [0, 1, 2, 2, 2])
    assert m == 2 and list(hu) == [0, 1, 0, 2, 0]
    assert T[0] == 1.0 + 100.0 / 6.0 and T[1] == 21.0 and T[2] == 6.0


def test_trace_mixed_rates_two_tours_with_undo():
    """Worked by hand.  No road time, areas (60, 12) ha, rates (1 | 1, 2, 3) ha/h: T = (60, 2).  Iter 1: u1 -> 30,
    u2 -> 20 (neither < 2), u3 is the fastest -> moved: T = (15, 4) kept.  Iter 2: u1 -> 12 (not < 4), u2 last ->
    moved: T = (10, 12) kept (12 < 15).  Iter 3: g_max = 1; donor tour 0 by rising rate: u0 -> T_1 = 6 < 10
    accepted, but then T_0 = 12 = the old maximum: not a strict decrease -> undone, stop."""
    m, hu, T = lgo.hu_balance([0.0, 0.0], [60 * Q, 12 * Q], [1 * Q, 1 * Q, 2 * Q, 3 * Q], [0, 1, 1, 1])
    assert m == 2 and list(hu) == [0, 1, 0, 0]
    assert list(T) == [10.0, 12.0]


def test_degenerate_cases():
    # one tour: nothing to do; a tour keeps >= 1 HU; an inactive tour (no fields, T = 0) gives its spare HUs away
    m, hu, T = lgo.hu_balance([2.0], [10 * Q], [Q, Q], [0, 0])
    assert m == 0 and list(hu) == [0, 0] and T[0] == 7.0
    m, hu, T = lgo.hu_balance([0.0, 0.0], [100 * Q, 1 * Q], [Q, Q], [0, 1])
    assert m == 0 and list(hu) == [0, 1]
    m, hu, T = lgo.hu_balance([0.0, 0.0, 0.0], [0, 30 * Q, 29 * Q], [Q] * 5, [0, 0, 0, 1, 2])
    assert m == 2 and list(hu) == [1, 2, 0, 1, 2] and list(T) == [0.0, 15.0, 14.5]
    # a tie for the maximum blocks the step: moving a HU to tour 0 leaves tour 1 at the old maximum -> undone (strict decrease)
    m, hu, T = lgo.hu_balance([0.0, 0.0, 0.0], [40 * Q, 40 * Q, 4 * Q], [Q] * 5, [0, 1, 2, 2, 2])
    assert m == 0 and list(hu) == [0, 1, 2, 2, 2] and T[0] == 40.0 and T[1] == 40.0


@pytest.mark.parametrize("name", ["toy", "small", "medium", "large", "paper_scale"])
def test_embedded_in_score(name):
    inst = wl.make(name); o = lgo.Oracle(inst)
    for pid in range(40):
        p = o.decode(inst.seed, pid)
        r0, r1 = o.score(p), o.score(p, hu_balance=True)
        assert r0["feasible"] == r1["feasible"]
        if not r0["feasible"]:
            assert np.array_equal(r1["hu_tour_final"], p["hu_tour"])
            continue
        assert np.array_equal(r0["hu_tour_final"], p["hu_tour"])              # off: the candidate's sets (R20)
        hu = r1["hu_tour_final"]
        cnt = np.bincount(hu, minlength=o.n_t)
        assert cnt.min() >= 1 and cnt.sum() == o.n_hu
        assert r1["makespan"] <= r0["makespan"]                                  # the maximum never increases
        assert np.array_equal(r1["route"], r0["route"])                          # geometry untouched
        # the plan with the balanced sets scores the same without the embedded step, and is a fixed point of it
        p2 = dict(p); p2["hu_tour"] = hu
        r2 = o.score(p2)
        assert r2["cost"] == r1["cost"] and r2["makespan"] == r1["makespan"] and r2["L_HU"] == r1["L_HU"]
        r3 = o.score(p2, hu_balance=True)
        assert np.array_equal(r3["hu_tour_final"], hu) and r3["cost"] == r1["cost"]
        # L_HU = sum_g n_HU(g) L_tour(g) (L106)
        assert r1["L_HU"] == pytest.approx(float((cnt * r1["route"]).sum()), rel=1e-12)


def test_workers_and_search_honour_the_flag():
    base = wl.make("small")
    inst = replace(base, flags=HU_BALANCE)
    o0, o1 = lgo.Oracle(base), lgo.Oracle(inst)
    p0 = o0.init_plan()
    c0, _, m0, f0 = o0.move_eval_batch(p0, 7, 0, 512)
    c1, _, m1, f1 = o1.move_eval_batch(p0, 7, 0, 512)
    assert np.array_equal(f0, f1)
    fin = f0.astype(bool)
    assert np.all(m1[fin] <= m0[fin]) and np.any(m1[fin] < m0[fin])
    # a worker = move, then score with the embedded step
    blk = lgo.philox4x32_10([5, 0, 5, 0], [7, 0])
    r = o1.score(o1.apply_move(p0, int(blk[0]), int(blk[1]), int(blk[2])), hu_balance=True)
    assert (r["cost"] == c1[5]) or (np.isinf(c1[5]) and not r["feasible"])
    # eval_batch / search sample plans with fixed HU sets (R20): unaffected by the flag
    assert np.array_equal(o0.eval_batch(0, first_id=0, n=256)[0], o1.eval_batch(0, first_id=0, n=256)[0])
    # the loop: x* carries the balanced sets and re-scores to C* with no further HU or SU move
    best, c, hc, hi = o1.local_search(p0, 3, 40, 256, 0x66666666)
    r = o1.score(best, hu_balance=True)
    assert r["cost"] == c and r["moves"] == 0 and np.array_equal(r["hu_tour_final"], best["hu_tour"])
    assert c < o1.score(p0, hu_balance=True)["cost"]
