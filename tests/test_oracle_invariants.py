"""Pins P4/P5 of DESIGN.md: structural invariants the paper's model fixes
(PAPER.md:L21 each BP on one tour / each field on one BP; eq. (1); eq. (2);
L190 makespan >= every tour time; L106 path = HU + eSU + lSU lengths) and statistical
pins of the decoder's random process (uniform Fisher-Yates, geometric extras)."""
import numpy as np
import pytest
from oracle import lgo
from paper_1909_10286_b200 import workloads as wl

CFGS = ["toy", "small", "medium", "large", "sweep"]
N_IDS = {"toy": 400, "small": 300, "medium": 200, "large": 60, "sweep": 30}


def plan_lists(o, p):
    """tours -> ordered BP lists; BPs -> ordered field lists (validates positions)."""
    tours = [[] for _ in range(o.n_t)]
    for b in np.lexsort((p["bp_pos"], p["bp_tour"])):
        tours[p["bp_tour"][b]].append(int(b))
    for g, lst in enumerate(tours):
        assert [p["bp_pos"][b] for b in lst] == list(range(len(lst)))
    fl = [[] for _ in range(o.n_b)]
    for f in np.lexsort((p["field_pos"], p["field_bp"])):
        fl[p["field_bp"][f]].append(int(f))
    for b, lst in enumerate(fl):
        assert [p["field_pos"][f] for f in lst] == list(range(len(lst)))
    return tours, fl


@pytest.mark.parametrize("name", CFGS)
def test_decoder_and_score_invariants(name):
    inst = wl.make(name)
    o = lgo.Oracle(inst)
    s_q, d_q, c_q = o.quanta(0), o.quanta(2), o.quanta(4)
    ids = np.concatenate([np.arange(N_IDS[name] // 2, dtype=np.uint64),
                          wl.sample_ids(inst.budget, N_IDS[name] // 2)])
    n_feas = 0
    for id_ in ids:
        p = o.decode(inst.seed, int(id_))
        tours, fl = plan_lists(o, p)
        # every BP on exactly one tour, every tour >= 1 BP / HU / SU (R22), eq. (1)
        assert sorted(b for t in tours for b in t) == list(range(o.n_b))
        assert all(len(t) >= 1 for t in tours)
        assert sorted(f for l in fl for f in l) == list(range(o.n_f))       # each field once
        nhu = np.bincount(p["hu_tour"], minlength=o.n_t); nsu = np.bincount(p["su_tour"], minlength=o.n_t)
        assert nhu.min() >= 1 and nsu.min() >= 1 and nhu.sum() == o.n_hu and nsu.sum() == o.n_su
        # non-last BPs in plan order: minimal demand-meeting prefix (+ extras), unless the
        # field stream ran dry (then every later BP is empty)
        order = [b for t in tours for b in t]
        dry = False
        for b in order[:-1]:
            cs = np.cumsum(s_q[fl[b]]) if fl[b] else np.array([], dtype=np.int64)
            if dry:
                assert len(fl[b]) == 0
            elif len(cs) == 0 or cs[-1] < d_q[b]:
                if d_q[b] > 0:
                    dry = True
            else:
                m = int(np.searchsorted(cs, d_q[b], side="left")) + 1 if d_q[b] > 0 else 0
                assert len(fl[b]) >= m
        r = o.score(p)
        Sq = np.array([s_q[l].sum() for l in fl])
        assert list(r["bp_supply_q"]) == list(Sq)
        assert r["feasible"] == bool(np.all(Sq >= d_q))                     # eq. (2)
        # eq. (2) recomputed in FP64 from the raw inputs agrees away from quantisation ties
        raw = np.array([inst.field_supply_t[l].sum() for l in fl])
        margin = np.abs(raw - inst.bp_demand_t)
        if margin.min() > (o.n_f + 1) / 1024.0:
            assert r["feasible"] == bool(np.all(raw >= inst.bp_demand_t))
        if not r["feasible"]:
            assert np.isinf(r["cost"]) and np.isinf(r["path"]) and np.isinf(r["makespan"])
            continue
        n_feas += 1
        assert r["makespan"] == r["T"].max() and np.all(r["makespan"] >= r["T"])
        assert r["path"] == pytest.approx(r["L_HU"] + r["L_eSU"] + r["L_lSU"], rel=1e-13)
        assert r["path"] == pytest.approx(r["L"].sum(), rel=1e-13)
        assert r["cost"] == pytest.approx(inst.w_path * r["path"] + inst.w_time * r["makespan"], rel=1e-15)
        # Alg. 2 preserves the unit set and every tour keeps >= 1 SU (R15)
        nsf = np.bincount(r["su_tour_final"], minlength=o.n_t)
        assert nsf.sum() == o.n_su and nsf.min() >= 1
        # shuttle counts: eq. (4) with the tour's mean capacity, real-number check
        for g, t in enumerate(tours):
            C = c_q[r["su_tour_final"] == g].sum(); n = nsf[g]
            for b in t:
                for f in fl[b]:
                    N = r["shuttles"][f]
                    assert (N - 1) * C < s_q[f] * n <= N * C
        # Alg. 2 never increases the maximum wait: re-run it from the final state -> 0 moves
        # is not guaranteed, but the final max wait must be <= the initial one
        nhu_l = [int(x) for x in nhu]
        _, _, W0 = lgo.su_local_min(r["E"], nhu_l, c_q, p["su_tour"], inst.su_fill_h_per_t)
        assert list(W0) == list(r["wait"])
    assert n_feas > 0


def wait_of(E, nhu, c_q, su, kappa, n_t):
    W = []
    for g in range(n_t):
        c = c_q[su == g]
        W.append(E[g] - kappa * ((c.sum() - c.max()) / 1024.0) / nhu[g])
    return np.array(W)


@pytest.mark.parametrize("name", ["small", "medium", "large"])
def test_alg2_monotone_on_configs(name):
    """Alg. 2 keeps a move only while max_g T_wait strictly decreases."""
    inst = wl.make(name); o = lgo.Oracle(inst); c_q = o.quanta(4)
    moved = 0
    for id_ in range(150):
        p = o.decode(0, id_); r = o.score(p)
        if not r["feasible"]:
            continue
        nhu = np.bincount(p["hu_tour"], minlength=o.n_t)
        w_init = wait_of(r["E"], nhu, c_q, p["su_tour"], inst.su_fill_h_per_t, o.n_t)
        w_fin = wait_of(r["E"], nhu, c_q, r["su_tour_final"], inst.su_fill_h_per_t, o.n_t)
        assert w_fin == pytest.approx(r["wait"], rel=1e-12, abs=1e-12)
        if r["moves"] > 0:
            assert w_fin.max() < w_init.max(); moved += 1
        else:
            assert list(r["su_tour_final"]) == list(p["su_tour"])
        assert c_q[r["su_tour_final"] >= 0].sum() == c_q.sum()
    assert moved > 10


def test_scaling_coordinates_scales_lengths():
    """Scaling all coordinates by 2 (exact in FP64) doubles every length and the road part
    of every completion time; shuttle counts, feasibility and Alg. 2's E scale with it."""
    inst = wl.make("small"); o1 = lgo.Oracle(inst)
    inst2 = wl.make("small"); inst2.field_xy = inst2.field_xy * 2.0; inst2.bp_xy = inst2.bp_xy * 2.0
    o2 = lgo.Oracle(inst2)
    for id_ in range(40):
        p = o1.decode(0, id_)
        r1, r2 = o1.score(p), o2.score(p)
        assert r1["feasible"] == r2["feasible"]
        assert list(r2["route"]) == list(2.0 * r1["route"])
        assert list(r2["E"]) == list(2.0 * r1["E"])
        if r1["feasible"] and list(r1["su_tour_final"]) == list(r2["su_tour_final"]):
            assert r2["path"] == 2.0 * r1["path"]


def test_fisher_yates_is_uniform():
    """3 BPs on 1 tour: the 6 visiting orders must be equally likely (chi-square), and the
    11 fields of a 1-BP instance must each be first with probability 1/11."""
    inst = wl.make("toy"); inst.n_tours = 1
    o = lgo.Oracle(inst)
    n = 12000
    d = o.decode_batch(0, first_id=0, n=n)
    key = np.argsort(d["bp_pos"], axis=1)            # visiting order of the 3 BPs
    code = key[:, 0] * 9 + key[:, 1] * 3 + key[:, 2]
    cnt = np.array([np.sum(code == c) for c in np.unique(code)])
    assert len(cnt) == 6
    chi2 = ((cnt - n / 6) ** 2 / (n / 6)).sum()
    assert chi2 < 25.7                                # p = 1e-4 at 5 dof
    # first field of the first BP in plan order: uniform over the 11 fields
    first_bp = key[:, 0]
    ff = np.array([np.where((d["field_bp"][i] == first_bp[i]) & (d["field_pos"][i] == 0))[0][0]
                   if np.any(d["field_bp"][i] == first_bp[i]) else -1 for i in range(n)])
    cnt = np.bincount(ff[ff >= 0], minlength=11)
    m = (ff >= 0).sum()
    assert ((cnt - m / 11) ** 2 / (m / 11)).sum() < 35.6   # p = 1e-4 at 10 dof


def test_partition_first_k_then_uniform_bins():
    """ordered_partition: bins are never empty, and tour sizes of the extra items are
    uniform: E[count of tour g] = 1 + (n-k)/k for every g."""
    inst = wl.make("medium"); o = lgo.Oracle(inst)
    d = o.decode_batch(0, first_id=0, n=4000)
    for key, n_items in (("hu_tour", o.n_hu), ("su_tour_init", o.n_su), ("bp_tour", o.n_b)):
        cnt = np.stack([np.sum(d[key] == g, axis=1) for g in range(o.n_t)], axis=1)
        assert cnt.min() >= 1
        assert cnt.mean(axis=0) == pytest.approx(np.full(o.n_t, n_items / o.n_t), rel=0.04)
        # each unit is equally likely on each tour
        per_unit = np.stack([np.mean(d[key] == g, axis=0) for g in range(o.n_t)])
        assert np.abs(per_unit - 1 / o.n_t).max() < 0.035


def test_extras_are_geometric():
    """Non-last BPs take extra fields while draw < thresh: P(extra) = thresh / 2^32."""
    inst = wl.make("small"); o = lgo.Oracle(inst)
    s_q, d_q = o.quanta(0), o.quanta(2)
    ext = []
    for id_ in range(1500):
        p = o.decode(0, id_)
        tours, fl = plan_lists(o, p)
        order = [b for t in tours for b in t]
        left = o.n_f
        for b in order[:-1]:
            cs = np.cumsum(s_q[fl[b]])
            left -= len(fl[b])
            if len(cs) and cs[-1] >= d_q[b] and left > 3:
                m = int(np.searchsorted(cs, d_q[b], side="left")) + 1
                ext.append(len(fl[b]) - m)
    ext = np.array(ext)
    assert len(ext) > 1000
    assert ext.mean() == pytest.approx(0.25 / 0.75, rel=0.15)
    assert np.mean(ext == 0) == pytest.approx(0.75, abs=0.03)
    # thresh = 0: never an extra; thresh = 2^32-1: (almost) always => first BP takes everything
    inst0 = wl.make("small"); inst0.extra_field_thresh = 0
    o0 = lgo.Oracle(inst0)
    for id_ in range(50):
        p = o0.decode(0, id_); tours, fl = plan_lists(o0, p)
        for b in [b for t in tours for b in t][:-1]:
            cs = np.cumsum(s_q[fl[b]])
            assert len(cs) == 0 or cs[-1] < d_q[b] or (len(cs) == 1 or cs[-2] < d_q[b])
    inst1 = wl.make("small"); inst1.extra_field_thresh = 0xFFFFFFFF
    o1 = lgo.Oracle(inst1)
    p = o1.decode(0, 3); tours, fl = plan_lists(o1, p)
    assert len(fl[tours[0][0]]) == o1.n_f
