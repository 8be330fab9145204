"""Pin P8 of DESIGN.md: exhaustive enumeration on the N_B=2, N_F=6 sub-instance of Toy
(BASELINE.json config 0).  The search's best must never beat the true optimum over all
feasible plans and must equal it once the budget covers the space (north_star)."""
import itertools
import numpy as np
from oracle import lgo
from paper_1909_10286_b200 import workloads as wl


def brute_force(o):
    """All plans: BP->tour (2) x ordered field partitions (6! x 7) x HU splits (3) x SU splits (7).
    Units are homogeneous on Toy, so a split is fixed by its counts (R30)."""
    best = np.inf; n_plans = 0; n_feas = 0
    sc = np.zeros(8)
    bp_pos = np.zeros(2, np.uint8)
    fb = np.zeros(6, np.uint16); fp = np.zeros(6, np.uint16)
    hu_splits = [np.array([0] * a + [1] * (4 - a), np.uint8) for a in (1, 2, 3)]
    su_splits = [np.array([0] * a + [1] * (8 - a), np.uint8) for a in range(1, 8)]
    for bp_first in (0, 1):                       # which BP is on tour 0
        bp_tour = np.array([0, 1] if bp_first == 0 else [1, 0], np.uint8)
        for perm in itertools.permutations(range(6)):
            for cut in range(7):
                for q, f in enumerate(perm):
                    if q < cut: fb[f] = bp_first; fp[f] = q
                    else:       fb[f] = 1 - bp_first; fp[f] = q - cut
                # eq. (2) does not depend on the unit splits: test it once per field plan
                splits = [(hu, su) for hu in hu_splits for su in su_splits]
                n_plans += len(splits)
                for n_done, (hu, su) in enumerate(splits):
                    assert o.score_fast(bp_tour, bp_pos, fb, fp, hu, su, sc) == 0
                    if sc[0] == 0.0:
                        assert n_done == 0
                        break
                    n_feas += 1
                    best = min(best, sc[6])
    return best, n_plans, n_feas


def test_search_reaches_bruteforce_optimum():
    inst = wl.make("toy_brute")
    o = lgo.Oracle(inst)
    opt, n_plans, n_feas = brute_force(o)
    assert n_plans == 2 * 5040 * 21 and n_feas > 0 and np.isfinite(opt)
    prev = np.inf
    for budget in (1 << 10, 1 << 16, 1 << 22):
        c, i = o.search(inst.seed, budget)
        assert c >= opt                      # never better than the true optimum
        assert c <= prev; prev = c           # monotone in the budget (prefix property)
        # the winner re-scores to the same cost through decode + score
        assert o.score(o.decode(inst.seed, i))["cost"] == c
    assert c == opt                          # budget 2^22 covers the space for seed 0


def test_search_is_ordered_min_of_eval_batch_and_ties_take_lowest_id():
    inst = wl.make("toy"); o = lgo.Oracle(inst)
    cost, _, _, feas = o.eval_batch(0, first_id=0, n=1 << 14)
    c, i = o.search(0, 1 << 14)
    assert c == cost.min() and i == int(np.argmin(cost))       # argmin returns the first minimum
    # shifted window
    c2, i2 = o.search(0, 1000, first_id=5000)
    assert c2 == cost[5000:6000].min() and i2 == 5000 + int(np.argmin(cost[5000:6000]))
    # all candidates identical (1 tour, 1 BP, 1 field, 1 HU, 1 SU) => lowest id wins (R29)
    from helpers import mk_instance
    one = lgo.Oracle(mk_instance((0, 0), [(3, 4, 25, 1)], [(6, 0, 10)], [2.0], [10.0], 1))
    c3, i3 = one.search(0, 500, first_id=77)
    assert i3 == 77 and c3 == (1 + 1) * 10 + 2 * 3 * 5 + (10 / 40 + 0.5)
    # no feasible candidate at all => +inf and the lowest id
    none = lgo.Oracle(mk_instance((0, 0), [(3, 4, 25, 1)], [(6, 0, 26)], [2.0], [10.0], 1))
    c4, i4 = none.search(0, 100, first_id=9)
    assert np.isinf(c4) and i4 == 9
