"""GPU parity (-m gpu) for the NEXT rows N1 / N3: Algorithm 1's nearest-neighbour
initialisation, the remove/reinsert workers (L158-165, L184) and the whole
iteration with eq. (5) (L133-169, L177), through the C ABI against the oracle: plans bit-exact,
costs bit-equal (bar: 1e-9 relative), identical winners in every iteration."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import lgo
from paper_1909_10286_b200 import binding, workloads as wl
from helpers import mk_instance

RTOL = 1e-9
PLAN = ("bp_tour", "bp_pos", "field_bp", "field_pos", "hu_tour", "su_tour")


@pytest.fixture(scope="module")
def ctxs():
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the product path must fail loudly, not fall back")
    cache = {}
    def get(name):
        if name not in cache:
            inst = wl.make(name)
            cache[name] = (inst, lgo.Oracle(inst), binding.Instance(inst))
        return cache[name]
    return get


def hand_instance():
    fields = [(11, 1, 30, 1), (9, -1, 30, 1), (29, 2, 40, 1), (1, 19, 10, 1), (12, 0, 5, 1), (2, 21, 50, 1)]
    bps = [(10, 0, 50), (0, 20, 40), (30, 0, 40)]
    return mk_instance((0, 0), fields, bps, [2.0, 2.0, 2.0], [20, 10, 10, 20], 2)


def assert_plan_equal(got, want, what):
    for k in PLAN:
        assert np.array_equal(np.asarray(got[k]), np.asarray(want[k])), f"{what}: plan array {k} differs"


def assert_costs(got, want, what):
    got = np.asarray(got); want = np.asarray(want)
    fin = np.isfinite(want)
    assert np.array_equal(np.isfinite(got), fin), what
    if not np.array_equal(got[fin], want[fin]):
        rel = np.abs(got[fin] - want[fin]) / np.abs(want[fin])
        assert rel.max() <= RTOL, f"{what}: max rel err {rel.max():.3e}"
        pytest.fail(f"{what}: within {RTOL} (max rel {rel.max():.3e}) but not bit-equal — operation order drifted")


def check_move_eval(o, g, plan, seed, first_id, n, what):
    want = o.move_eval_batch(plan, seed, first_id, n)
    got = [t.cpu().numpy() for t in g.move_eval_batch(plan, seed, first_id, n)]
    assert np.array_equal(got[3], want[3]), f"{what}: feasibility flags differ"
    for k, nm in enumerate(("cost", "path_km", "makespan_h")):
        assert_costs(got[k], want[k], f"{what}/{nm}")
    return want


def test_init_plan_hand_example_and_configs(ctxs):
    h = hand_instance()
    g, o = binding.Instance(h), lgo.Oracle(h)
    p = g.init_plan()
    assert list(p["bp_tour"]) == [0, 1, 1] and list(p["field_bp"]) == [0, 0, 2, 1, 1, 1] and list(p["field_pos"]) == [1, 0, 0, 1, 0, 2]
    assert_plan_equal(p, o.init_plan(), "hand")
    for name in ("toy", "small", "medium", "large", "sweep", "paper_scale"):
        inst, o, g = ctxs(name)
        assert_plan_equal(g.init_plan(), o.init_plan(), name)


@pytest.mark.parametrize("name,n", [("toy", 4096), ("small", 8192), ("medium", 8192), ("large", 4096), ("sweep", 2048),
                                    ("paper_scale", 2048)])
def test_move_eval_batch_matches_oracle(ctxs, name, n):
    inst, o, g = ctxs(name)
    p = o.init_plan()
    w = check_move_eval(o, g, p, 7, 0, n, f"{name}/init")
    if name != "toy":
        assert 0 < w[3].mean() <= 1.0
    check_move_eval(o, g, p, 0xDEADBEEFCAFEF00D, (1 << 40) + 11, 513, f"{name}/bigid")
    # from a sampled plan (random field order, SU sets not yet at Alg. 2's fixed point)
    check_move_eval(o, g, o.decode(inst.seed, 12345), 3, 100, min(n, 2048), f"{name}/sampled")


def test_move_eval_degenerate_plans(ctxs):
    """Inactive tours (L184), BPs without fields, every vertex kind: plans reached by explicit moves."""
    def w_for(v, n): return -(-(v << 32) // n)
    h = hand_instance(); o, g = lgo.Oracle(h), binding.Instance(h)
    p = o.init_plan()
    nf, nb, nt = 6, 3, 2
    plans = [p,
             o.apply_move(p, w_for(nf + 0, nf + nb), w_for(1, nt), w_for(2, 3)),       # tour 0 inactive
             o.apply_move(p, w_for(2, nf + nb), w_for(0, nb), w_for(0, 3))]            # BP 2 without fields
    plans.append(o.apply_move(plans[2], w_for(nf + 2, nf + nb), w_for(0, nt), w_for(0, 2)))   # the empty BP moves
    for k, q in enumerate(plans):
        check_move_eval(o, g, q, 11 + k, 0, 4096, f"hand/plan{k}")
    # zero-demand BPs: an emptied BP stays feasible
    z = wl.make("small"); z.bp_demand_t = z.bp_demand_t.copy(); z.bp_demand_t[[1, 3]] = 0.0
    oz, gz = lgo.Oracle(z), binding.Instance(z)
    q = oz.init_plan()
    rng = np.random.default_rng(9)
    for _ in range(3):       # drift away from the initial plan with a few random moves
        w = rng.integers(0, 2**32, 3)
        q = oz.apply_move(q, int(w[0]), int(w[1]), int(w[2]))
    check_move_eval(oz, gz, q, 5, 0, 8192, "small/zero-demand")
    # N_T = 1 and N_T = N_B = N_HU = N_SU
    for nt_ in (1, 5):
        z = wl.make("small"); z.n_tours = nt_
        if nt_ == 5:
            z.hu_rate_ha_per_h = z.hu_rate_ha_per_h[:5].copy(); z.su_capacity_t = z.su_capacity_t[:5].copy()
        oz, gz = lgo.Oracle(z), binding.Instance(z)
        check_move_eval(oz, gz, oz.init_plan(), 2, 0, 4096, f"small/nt{nt_}")
    # ragged worker counts around the block / grid granularity
    inst, om, gm = ctxs("medium")
    pm = om.init_plan()
    for n in (1, 31, 33, 511, 513):
        check_move_eval(om, gm, pm, 1, 3, n, f"medium/n{n}")
    for n in (148 * 512 + 1, 148 * 512 * 8 + 700):           # two rounds; more rounds than one sorted super-round
        got = gm.move_eval_batch(pm, 1, 3, n)[0].cpu().numpy()
        want = om.move_eval_batch(pm, 1, 3 + n - 64, 64)[0]
        assert np.array_equal(got[-64:], want)
        mid = n // 2
        want = om.move_eval_batch(pm, 1, 3 + mid, 64)[0]
        assert np.array_equal(got[mid:mid + 64], want)


def test_invalid_plans_are_rejected(ctxs):
    inst, o, g = ctxs("small")
    p = o.init_plan()
    for key, idx, val in (("bp_tour", 0, 200), ("field_bp", 3, 99), ("field_pos", 3, 39), ("bp_pos", 1, 4), ("su_tour", 0, 9)):
        q = {k: v.copy() for k, v in p.items()}
        q[key][idx] = val
        with pytest.raises(binding.LgxError):
            g.move_eval_batch(q, 0, 0, 16)
        with pytest.raises(binding.LgxError):
            g.local_search(q, 0, 1, 16, 0)
    q = {k: v.copy() for k, v in p.items()}
    q["hu_tour"][:] = 0                                     # tours 1, 2 without an HU
    with pytest.raises(binding.LgxError):
        g.move_eval_batch(q, 0, 0, 16)
    with pytest.raises(binding.LgxError):
        g.local_search(p, 0, 1, 0, 0)                       # no workers


@pytest.mark.parametrize("name,n_iters,n_workers", [("toy", 40, 100), ("small", 60, 256), ("medium", 25, 1000),
                                                    ("large", 6, 700), ("paper_scale", 4, 600)])
@pytest.mark.parametrize("eps", [0, 0x66666666, 0xFFFFFFFF])
def test_local_search_matches_oracle(ctxs, name, n_iters, n_workers, eps):
    inst, o, g = ctxs(name)
    p0 = o.init_plan()
    want_p, want_c, want_hc, want_hi = o.local_search(p0, 3, n_iters, n_workers, eps)
    got_p, got_c, got_hc, got_hi = g.local_search(p0, 3, n_iters, n_workers, eps)
    assert np.array_equal(got_hi, want_hi), f"{name}: winners differ (first at iteration {int(np.argmax(got_hi != want_hi))})"
    assert_costs(got_hc, want_hc, f"{name}/hist_cost")
    assert got_c == want_c
    assert_plan_equal(got_p, want_p, name)
    if name != "toy":
        assert want_c < o.score(p0)["cost"]


def test_local_search_edge_cases(ctxs):
    inst, o, g = ctxs("small")
    p0 = o.init_plan()
    # n_iters = 0 scores x_0 and gives it Alg. 2's SU sets (R37)
    got_p, got_c, _, _ = g.local_search(p0, 1, 0, 64, 0)
    r = o.score(p0)
    assert got_c == r["cost"] and np.array_equal(got_p["su_tour"], r["su_tour_final"])
    # more workers than one grid round; a single worker; an infeasible start (toy's tight instance)
    for n_iters, n_workers in ((3, 148 * 512 + 77), (50, 1)):
        want = o.local_search(p0, 5, n_iters, n_workers, 0x80000000)
        got = g.local_search(p0, 5, n_iters, n_workers, 0x80000000)
        assert np.array_equal(got[3], want[3]) and np.array_equal(got[2], want[2]) and got[1] == want[1]
        assert_plan_equal(got[0], want[0], f"small/{n_workers}")
    it, ot, gt = ctxs("toy")
    pt = ot.init_plan()
    assert not ot.score(pt)["feasible"]
    want = ot.local_search(pt, 2, 30, 64, 0x40000000)
    got = gt.local_search(pt, 2, 30, 64, 0x40000000)
    assert np.array_equal(got[3], want[3]) and np.array_equal(got[2], want[2]) and got[1] == want[1]
    assert_plan_equal(got[0], want[0], "toy/infeasible start")


@pytest.mark.parametrize("name,n,n_iters,n_workers", [("toy", 4096, 30, 100), ("small", 8192, 40, 300), ("medium", 8192, 20, 1000),
                                                      ("sweep", 1024, 3, 400), ("paper_scale", 2048, 4, 600)])
def test_embedded_hu_assignment_matches_oracle(name, n, n_iters, n_workers):
    """NEXT row N2 (R39): with LGX_FLAG_HU_BALANCE the workers rebalance the HUs before
    Algorithm 2; x_{i*} carries the HU sets it was scored with."""
    from dataclasses import replace
    inst = replace(wl.make(name), flags=2)
    o, g = lgo.Oracle(inst), binding.Instance(inst)
    p0 = o.init_plan()
    w = check_move_eval(o, g, p0, 7, 0, n, f"{name}/hb/init")
    check_move_eval(o, g, o.decode(inst.seed, 4242), 9, 1 << 33, min(n, 2048), f"{name}/hb/sampled")
    base = lgo.Oracle(wl.make(name)).move_eval_batch(p0, 7, 0, n)
    if name != "toy" and o.n_hu > o.n_t:                            # (paper_scale has one HU per tour: nothing can move)
        assert not np.array_equal(base[2], w[2])                    # the flag changes makespans
    for eps in (0, 0x66666666):
        want_p, want_c, want_hc, want_hi = o.local_search(p0, 3, n_iters, n_workers, eps)
        got_p, got_c, got_hc, got_hi = g.local_search(p0, 3, n_iters, n_workers, eps)
        assert np.array_equal(got_hi, want_hi), f"{name}: winners differ (first at iteration {int(np.argmax(got_hi != want_hi))})"
        assert_costs(got_hc, want_hc, f"{name}/hb/hist_cost")
        assert got_c == want_c
        assert_plan_equal(got_p, want_p, f"{name}/hb")
    # n_iters = 0: x_0 takes the balanced HU sets
    got_p, got_c, _, _ = g.local_search(p0, 1, 0, 64, 0)
    r = o.score(p0, hu_balance=True)
    assert (got_c == r["cost"] or (np.isinf(got_c) and not r["feasible"])) and np.array_equal(got_p["hu_tour"], r["hu_tour_final"])
    g.close()


def test_local_search_at_bench_scale_is_self_consistent(ctxs):
    """Beyond the oracle's reach (bench.py's launch configuration: 8 grid rounds of workers per iteration on the
    paper's problem shape): x* re-scores in the oracle to exactly C* with no further Algorithm-2 move, C* is the
    best winner of the history, every winner is one of its iteration's workers, and the run is reproducible."""
    inst, o, g = ctxs("paper_scale")
    p0 = o.init_plan()
    n_workers = g.query(6) * g.query(15) * 8
    n_iters = 30
    best, c, hc, hi = g.local_search(p0, inst.seed, n_iters, n_workers, int(0.4 * 2**32))
    r = o.score(best)
    assert r["feasible"] and r["cost"] == c and r["moves"] == 0
    c0 = o.score(p0)["cost"]
    assert c == min(c0, hc.min()) and c < c0
    assert np.all(hi // n_workers == np.arange(n_iters))
    # the first iteration's winner, replayed by the oracle from x_0 (one worker)
    p0s = dict(p0); p0s["su_tour"] = o.score(p0)["su_tour_final"]
    w = o.move_eval_batch(p0s, inst.seed, int(hi[0]), 1)
    assert w[0][0] == hc[0]
    # sampled workers of iteration 0 are never better than its winner
    ids = np.random.default_rng(1).integers(0, n_workers, 200)
    for i in ids[:50]:
        assert not (o.move_eval_batch(p0s, inst.seed, int(i), 1)[0][0] < hc[0])
    again = g.local_search(p0, inst.seed, n_iters, n_workers, int(0.4 * 2**32))
    assert again[1] == c and np.array_equal(again[3], hi) and np.array_equal(again[2], hc)


def test_search_winner_seeds_the_local_search(ctxs):
    """The two halves compose through the C ABI: lgx_search's winner, decoded by lgx_decode_batch, is a valid x_0
    whose score is the search's best cost, and Algorithm 1 improves on it (same result as the oracle's loop)."""
    inst, o, g = ctxs("medium")
    c, i = g.search(inst.seed, 1 << 20)
    p = g.plan_of(inst.seed, i)
    want = o.decode(inst.seed, i)
    assert_plan_equal(p, want, "plan_of")
    assert o.score(p)["cost"] == c
    got = g.local_search(p, 5, 20, 2000, 0x66666666)
    ref = o.local_search(p, 5, 20, 2000, 0x66666666)
    assert got[1] == ref[1] and np.array_equal(got[3], ref[3]) and got[1] < c
    assert_plan_equal(got[0], ref[0], "search -> local search")


@pytest.mark.parametrize("name,flags", [("small", 4), ("medium", 4), ("large", 6), ("paper_scale", 4)])
def test_makespan_filter_matches_oracle(name, flags):
    """The paper's selection rule (R38): rank by path length (w_time = 0), discard workers whose
    makespan exceeds the best-so-far one; alone and together with the embedded HU assignment."""
    from dataclasses import replace
    inst = replace(wl.make(name), flags=flags, w_time=0.0)
    o, g = lgo.Oracle(inst), binding.Instance(inst)
    p0 = o.init_plan()
    w = check_move_eval(o, g, p0, 7, 0, 4096, f"{name}/filter")
    assert np.isinf(w[0][w[3] == 1]).any()                       # some feasible workers are discarded
    for eps, n_iters, n_workers in ((0x66666666, 12, 700), (0xFFFFFFFF, 6, 1500)):
        want = o.local_search(p0, 3, n_iters, n_workers, eps)
        got = g.local_search(p0, 3, n_iters, n_workers, eps)
        assert np.array_equal(got[3], want[3]) and got[1] == want[1]
        assert_costs(got[2], want[2], f"{name}/filter/hist")
        assert_plan_equal(got[0], want[0], f"{name}/filter")
    g.close()


@pytest.mark.parametrize("name,flags", [("small", 8), ("medium", 8 | 2), ("paper_scale", 8 | 4)])
def test_fixed_field_bp_assignment_matches_oracle(name, flags):
    """PAPER.md §2.6 (L249), Cases 2-3: a moved field is reinserted into its own BP."""
    from dataclasses import replace
    inst = replace(wl.make(name), flags=flags)
    o, g = lgo.Oracle(inst), binding.Instance(inst)
    p0 = o.init_plan()
    check_move_eval(o, g, p0, 7, 0, 4096, f"{name}/fixbp")
    want = o.local_search(p0, 3, 10, 900, 0x66666666)
    got = g.local_search(p0, 3, 10, 900, 0x66666666)
    assert np.array_equal(got[3], want[3]) and got[1] == want[1]
    assert_plan_equal(got[0], want[0], f"{name}/fixbp")
    assert np.array_equal(got[0]["field_bp"], p0["field_bp"])
    g.close()


def test_results_do_not_depend_on_the_launch_shape(ctxs):
    """Which thread scores which worker is free (sorted rounds, warps drawing chunks): the winners must not depend on it."""
    inst, o, g = ctxs("medium")
    p0 = o.init_plan()
    ref = g.local_search(p0, 9, 15, 20000, 0x66666666)
    refb = g.move_eval_batch(p0, 9, 0, 50000)[0].cpu().numpy()
    for threads in (64, 160, 384):
        g2 = binding.Instance(inst)
        g2.set_option(binding.LGX_OPT_THREADS_MV, threads)
        assert g2.query(15) == threads
        got = g2.local_search(p0, 9, 15, 20000, 0x66666666)
        assert got[1] == ref[1] and np.array_equal(got[3], ref[3]) and np.array_equal(got[2], ref[2])
        assert_plan_equal(got[0], ref[0], f"threads {threads}")
        assert np.array_equal(g2.move_eval_batch(p0, 9, 0, 50000)[0].cpu().numpy(), refb)
        g2.close()
