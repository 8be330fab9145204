"""GPU parity (-m gpu): the CUDA path through the C ABI against the oracle, element by
element on the same seeded inputs.  Bar (BASELINE.json north_star): decoded plans and
feasibility flags bit-exact, FP64 costs within 1e-9 relative (the kernels reproduce the
oracle's operation order, so the tests first assert bit equality and report the relative
error if that ever fails), identical argmin id."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import lgo
from paper_1909_10286_b200 import binding, workloads as wl
from helpers import mk_instance, oracle_eval_mp, oracle_search_mp

RTOL = 1e-9
# SURVEY s8(d) parity protocol: 2^16 ids per id set on every config (2^12 on paper_scale); the oracle runs as it is,
# one process per host core over disjoint chunks of the ids (helpers.oracle_eval_mp)
N_ORACLE = {"toy": 1 << 16, "small": 1 << 16, "medium": 1 << 16, "large": 1 << 16, "sweep": 1 << 16, "paper_scale": 1 << 12}


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


def id_sets(inst, n):
    """first n ids, n ids sampled over the whole budget (incl. >= 2^31 for the big configs),
    and the last n ids of the budget."""
    yield "first", None, 0
    yield "sampled", wl.sample_ids(inst.budget, n), 0
    yield "last", None, inst.budget - n


def assert_costs(got, want, what):
    got = np.asarray(got); want = np.asarray(want)
    fin = np.isfinite(want)
    assert np.array_equal(np.isfinite(got), fin), what
    if not np.array_equal(got[fin], want[fin]):
        rel = np.abs(got[fin] - want[fin]) / np.abs(want[fin])
        assert rel.max() <= RTOL, f"{what}: max rel err {rel.max():.3e}"
        pytest.fail(f"{what}: within {RTOL} (max rel {rel.max():.3e}) but not bit-equal — operation order drifted")


@pytest.mark.parametrize("name", ["toy", "small", "medium", "large", "sweep"])
def test_eval_batch_matches_oracle(ctxs, name):
    inst, o, g = ctxs(name)
    n = N_ORACLE[name]
    for label, ids, first in id_sets(inst, n):
        want = oracle_eval_mp(name, inst.seed, ids=ids, first_id=first, n=n)
        d_ids = torch.from_numpy(ids.astype(np.int64)).cuda() if ids is not None else None
        got = [t.cpu().numpy() for t in g.eval_batch(inst.seed, ids=d_ids, first_id=first, n=n)]
        assert np.array_equal(got[3], want[3]), f"{name}/{label}: feasibility flags differ"
        for k, nm in enumerate(("cost", "path_km", "makespan_h")):
            assert_costs(got[k], want[k], f"{name}/{label}/{nm}")
        assert 0 < want[3].mean() <= 1.0


@pytest.mark.parametrize("name", ["toy", "small", "medium", "large", "sweep"])
def test_decode_batch_matches_oracle(ctxs, name):
    inst, o, g = ctxs(name)
    n = 2048 if name in ("toy", "small", "medium") else 512
    for label, ids, first in id_sets(inst, n):
        want = o.decode_batch(inst.seed, ids=ids, first_id=first, n=n)
        d_ids = torch.from_numpy(ids.astype(np.int64)).cuda() if ids is not None else None
        got = g.decode_batch(inst.seed, ids=d_ids, first_id=first, n=n)
        torch.cuda.synchronize()
        for key in want:
            a = got[key].cpu().numpy()
            if a.dtype == np.int16: a = a.view(np.uint16)
            assert np.array_equal(a, want[key]), f"{name}/{label}: plan array {key} differs"


@pytest.mark.parametrize("name,budget", [("toy", 1 << 16), ("small", 1 << 24), ("medium", 1 << 24),
                                         ("large", 1 << 20), ("sweep", 1 << 20), ("paper_scale", 1 << 17)])
def test_search_matches_oracle_argmin(ctxs, name, budget):
    """lgx_search against the oracle's full scan of Toy and Small (2^24) and of id prefixes of the
    others (Medium 2^24, Large / Sweep 2^20), the oracle spread over the host cores."""
    inst, o, g = ctxs(name)
    want_c, want_i = oracle_search_mp(name, inst.seed, budget)
    got_c, got_i = g.search(inst.seed, budget)
    assert got_i == want_i and got_c == want_c
    # a window that does not start at 0 (multi-GPU shards use these)
    first = inst.budget - budget // 16
    want_c, want_i = oracle_search_mp(name, inst.seed, budget // 16, first_id=first)
    got_c, got_i = g.search(inst.seed, budget // 16, first_id=first)
    assert got_i == want_i and got_c == want_c


def test_eight_shard_windows_combine_to_one_search(ctxs):
    """SURVEY s4 / s8(e) on one GPU: eight disjoint lgx_search_range windows (sharding.split_range), min-combined by
    sharding.combine, equal one lgx_search over the whole range — ties and all."""
    from paper_1909_10286_b200 import sharding
    for name, budget in (("medium", (1 << 24) + 12345), ("toy", 1 << 16), ("sweep", 1 << 18)):
        inst, o, g = ctxs(name)
        whole = g.search(inst.seed, budget, first_id=77)
        parts = []
        for r in range(8):
            first, n = sharding.split_range(budget, 8, r, first_id=77)
            parts.append(g.search(inst.seed, n, first_id=first) if n else None)
        assert sharding.combine(parts) == whole


def test_search_equals_min_of_eval_batch_at_scale(ctxs):
    """Self-consistency beyond the oracle's reach: search over 2^22 ids of Medium equals the
    ordered min of eval_batch outputs, and the winner re-scores to the same cost in the oracle."""
    inst, o, g = ctxs("medium")
    n = 1 << 22
    cost = g.eval_batch(inst.seed, first_id=0, n=n)[0]
    c, i = g.search(inst.seed, n)
    cmin = cost.min().item()
    assert c == cmin and i == int((cost == cmin).nonzero()[0].item())
    assert o.score(o.decode(inst.seed, i))["cost"] == c


def test_full_budget_tail_ids_sampled(ctxs):
    """At the full budgets (2^30, 2^32) single sampled ids near the top of the range decode
    and score identically (64-bit id handling)."""
    for name in ("large", "sweep"):
        inst, o, g = ctxs(name)
        ids = np.array([inst.budget - 1, inst.budget - 2, (1 << 31) + 5, (1 << 31) - 1, inst.budget // 2 + 1], dtype=np.uint64)
        want = o.eval_batch(inst.seed, ids=ids)
        got = [t.cpu().numpy() for t in g.eval_batch(inst.seed, ids=torch.from_numpy(ids.astype(np.int64)).cuda())]
        assert np.array_equal(got[3], want[3])
        assert np.array_equal(got[0], want[0])
    # ids beyond 2^32 and a non-zero seed
    inst, o, g = ctxs("small")
    ids = np.array([(1 << 40) + 3, (1 << 63) + 11, 2**64 - 1], dtype=np.uint64)
    seed = 0xDEADBEEFCAFEF00D
    want = o.eval_batch(seed, ids=ids)
    got = [t.cpu().numpy() for t in g.eval_batch(seed, ids=torch.from_numpy(ids.view(np.int64)).cuda())]
    assert np.array_equal(got[3], want[3]) and np.array_equal(got[0], want[0])


def test_edge_cases(ctxs):
    # hand toy A through the CUDA path: every candidate is the same plan up to field order
    a = mk_instance((0, 0), [(3, 4, 25, 1), (6, 8, 40, 2)], [(6, 0, 60)], [2.0], [10.0, 10.0], 1)
    g = binding.Instance(a); o = lgo.Oracle(a)
    cost, path, mk, fe = [t.cpu().numpy() for t in g.eval_batch(0, first_id=0, n=100)]
    assert np.all(fe == 1) and np.all(path == 154.0) and np.all(mk == 2.0) and np.all(cost == 156.0)
    assert g.search(0, 100, first_id=7) == (156.0, 7)          # ties: lowest id
    # all infeasible: +inf and the lowest id
    b = mk_instance((0, 0), [(3, 4, 25, 1), (6, 8, 40, 2)], [(6, 0, 66)], [2.0], [10.0, 10.0], 1)
    gb = binding.Instance(b)
    c, i = gb.search(0, 1000, first_id=5)
    assert np.isinf(c) and i == 5
    out = [t.cpu().numpy() for t in gb.eval_batch(0, first_id=0, n=33)]
    assert np.all(out[3] == 0) and np.all(np.isinf(out[0])) and np.all(np.isinf(out[1])) and np.all(np.isinf(out[2]))
    # n = 0 is a no-op; budget 0 is an error
    g.eval_batch(0, first_id=0, n=0)
    with pytest.raises(binding.LgxError):
        g.search(0, 0)
    # ragged sizes around the block/grid granularity
    inst, om, gm = ctxs("medium")
    for n in (1, 31, 33, 511, 513, 148 * 512 + 1):
        want = om.eval_batch(0, first_id=3, n=min(n, 2000))
        got = [t.cpu().numpy() for t in gm.eval_batch(0, first_id=3, n=n)]
        assert np.array_equal(got[0][:2000], want[0]) and np.array_equal(got[3][:2000], want[3])
    # zero-demand BPs and thresh extremes (decoder degenerate paths)
    for thresh in (0, 0xFFFFFFFF, 0x40000000):
        z = wl.make("small"); z.bp_demand_t = z.bp_demand_t.copy(); z.bp_demand_t[[1, 3]] = 0.0
        z.extra_field_thresh = thresh
        oz, gz = lgo.Oracle(z), binding.Instance(z)
        want = oz.eval_batch(1, first_id=0, n=4096)
        got = [t.cpu().numpy() for t in gz.eval_batch(1, first_id=0, n=4096)]
        assert np.array_equal(got[3], want[3]) and np.array_equal(got[0], want[0])
        wd = oz.decode_batch(1, first_id=0, n=512); gd = gz.decode_batch(1, first_id=0, n=512)
        for key in wd:
            a_ = gd[key].cpu().numpy()
            if a_.dtype == np.int16: a_ = a_.view(np.uint16)
            assert np.array_equal(a_, wd[key]), key
    # N_T = N_B = N_HU = N_SU (every bin exactly one item) and N_T = 1
    for nt in (1, 5):
        z = wl.make("small"); z.n_tours = nt
        if nt == 5:
            z.hu_rate_ha_per_h = z.hu_rate_ha_per_h[:5].copy(); z.su_capacity_t = z.su_capacity_t[:5].copy()
        oz, gz = lgo.Oracle(z), binding.Instance(z)
        want = oz.eval_batch(2, first_id=0, n=2048)
        got = [t.cpu().numpy() for t in gz.eval_batch(2, first_id=0, n=2048)]
        assert np.array_equal(got[3], want[3]) and np.array_equal(got[0], want[0])


def test_eval_batch_host_buffers(ctxs):
    inst, o, g = ctxs("small")
    ids = wl.sample_ids(inst.budget, 5000)
    want = o.eval_batch(inst.seed, ids=ids)
    got = g.eval_batch_host(inst.seed, ids=ids)
    assert np.array_equal(got[3], want[3]) and np.array_equal(got[0], want[0])
    got = g.eval_batch_host(inst.seed, first_id=10, n=(1 << 22) + 17)       # crosses a chunk boundary
    want = o.eval_batch(inst.seed, first_id=10 + (1 << 22) - 8, n=25)
    assert np.array_equal(got[0][(1 << 22) - 8:], want[0])
    # page-locked buffers (copies overlap the next chunk's kernels), five chunks on two streams, explicit ids: every
    # element equal to the device-buffer call
    n = (1 << 23) + 4099
    ids = torch.arange(n, dtype=torch.int64) * 3 + 7
    pinned = tuple(torch.empty(n, dtype=dt, pin_memory=True) for dt in (torch.float64, torch.float64, torch.float64, torch.uint8))
    g.eval_batch_host(inst.seed, ids=ids.numpy().astype(np.uint64), out=tuple(t.numpy() for t in pinned))
    dev = g.eval_batch(inst.seed, ids=ids.cuda())
    torch.cuda.synchronize()
    for a, b in zip(pinned, dev):
        assert torch.equal(a, b.cpu())
    for k in (1 << 21) - 1, 1 << 21, (1 << 22) + 5, n - 1:               # chunk seams against the oracle
        w = o.eval_batch(inst.seed, ids=np.array([3 * k + 7], dtype=np.uint64))
        assert pinned[0][k].item() == w[0][0] or (np.isinf(w[0][0]) and np.isinf(pinned[0][k].item()))
        assert pinned[3][k].item() == w[3][0]


def test_paper_scale_workload(ctxs):
    """NEXT row N4: the paper's own problem shape (1200 fields, 20 BPs, 7 tours; L267)."""
    inst, o, g = ctxs("paper_scale")
    n = N_ORACLE["paper_scale"]
    for label, ids, first in id_sets(inst, n):
        want = oracle_eval_mp("paper_scale", inst.seed, ids=ids, first_id=first, n=n)
        d_ids = torch.from_numpy(ids.astype(np.int64)).cuda() if ids is not None else None
        got = [t.cpu().numpy() for t in g.eval_batch(inst.seed, ids=d_ids, first_id=first, n=n)]
        assert np.array_equal(got[3], want[3]), label
        for k in range(3):
            assert np.array_equal(got[k], want[k]), (label, k)
    wd = o.decode_batch(inst.seed, first_id=0, n=128); gd = g.decode_batch(inst.seed, first_id=0, n=128)
    for key in wd:
        a_ = gd[key].cpu().numpy()
        if a_.dtype == np.int16: a_ = a_.view(np.uint16)
        assert np.array_equal(a_, wd[key]), key


def test_timing_hook_and_query(ctxs):
    inst, o, g = ctxs("small")
    info = g.info()
    assert info["threads"] % 32 == 0 and info["threads_finish"] % 32 == 0 and info["grid"] == info["sm_count"]
    assert info["smem_bytes"] <= 227 * 1024 and info["smem_bytes_finish"] <= 227 * 1024 and info["record_bytes"] > 0 and info["chunk"] % 32 == 0
    l0 = g.query(7)
    g.set_timing(True)
    want = g.search(inst.seed, 3 * info["chunk"] + 5)
    ns_a, ns_c, pairs = g.kernel_times()
    assert pairs == 4 and ns_a > 0 and ns_c > 0 and g.query(7) - l0 == 8      # 4 chunks x 2 kernels
    g.set_timing(False)
    assert g.kernel_times() == (0, 0, 0)
    assert g.search(inst.seed, 3 * info["chunk"] + 5) == want                 # timing does not change results


@pytest.mark.parametrize("name", ["toy", "small", "medium", "large", "sweep", "paper_scale"])
def test_results_do_not_depend_on_the_launch_shape(ctxs, name):
    """Threads per block of both kernels, candidates per kernel pair and the s_q replication are launch configuration
    only (include/lgx.h).  The per-candidate state rows are laid out by blockDim (lgx_image.h): a thread that touches
    another thread's cells — a race between warps in different phases of the kernel — shows up here as a result that
    changes with the shape.  (compute-sanitizer's racecheck is closed on the GPU pool.)"""
    inst, o, g = ctxs(name)
    n = (1 << 15) if inst.n_fields <= 250 else (1 << 13)
    ref = [t.cpu().numpy() for t in g.eval_batch(inst.seed, first_id=11, n=n)]
    want = oracle_eval_mp(name, inst.seed, first_id=11, n=n)
    for k in range(4):
        assert np.array_equal(ref[k], want[k])
    ref_best = g.search(inst.seed, n, first_id=11)
    ta_max, tb_max = g.query(1), g.query(8)
    shapes = [(32, 32, 10, 0), (64, 64, 12, 1), (ta_max, 64, 11, 2), (32, tb_max, 13, 3), (min(96, ta_max), min(96, tb_max), 14, 5),
              (ta_max, max(32, tb_max // 2 // 32 * 32), 12, 4)]
    for ta, tb, chunk, sq in shapes:
        g2 = binding.Instance(inst)
        g2.set_option(binding.LGX_OPT_SQ_SHIFT, min(sq, g2.query(17)))
        g2.set_option(binding.LGX_OPT_THREADS_A, min(ta, g2.query(1))); g2.set_option(binding.LGX_OPT_THREADS_B, tb)
        g2.set_option(binding.LGX_OPT_CHUNK_LOG2, chunk)
        for rep in range(2):                             # twice: a race need not show on the first pass
            got = [t.cpu().numpy() for t in g2.eval_batch(inst.seed, first_id=11, n=n)]
            for k in range(4):
                assert np.array_equal(got[k], ref[k]), f"{name}: output {k} changes with the launch shape {(ta, tb, chunk, sq)}"
        assert g2.search(inst.seed, n, first_id=11) == ref_best
        g2.close()


def test_concurrent_streams_share_an_instance(ctxs):
    """The instance is immutable and every call owns its workspace: calls on different
    streams may overlap (include/lgx.h)."""
    inst, o, g = ctxs("small")
    n = 1 << 18
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    with torch.cuda.stream(s1):
        a = g.eval_batch(inst.seed, first_id=0, n=n, stream=s1)
    with torch.cuda.stream(s2):
        b = g.eval_batch(inst.seed, first_id=n, n=n, stream=s2)
    torch.cuda.synchronize()
    ref = g.eval_batch(inst.seed, first_id=0, n=2 * n)
    torch.cuda.synchronize()
    assert torch.equal(torch.cat([a[0], b[0]]), ref[0]) and torch.equal(torch.cat([a[3], b[3]]), ref[3])
    want = o.eval_batch(inst.seed, first_id=n - 100, n=200)
    got = ref[0][n - 100:n + 100].cpu().numpy()
    assert np.array_equal(got, want[0])


def test_inline_sqrt_equals_library_sqrt():
    """The walk/finish kernel's in-line square root (two independent chains per field instead of two subroutine
    calls) must be __dsqrt_rn bit for bit: 2^26 arguments per seed, structured and random (include/lgx.h)."""
    for seed in (0, 0xC0FFEE, 2**63 + 17):
        checked, bad = binding.selftest(0, 1 << 26, seed)
        assert checked > (1 << 25) and bad == 0, (seed, checked, bad)


@pytest.mark.parametrize("mode", [1, 2])
def test_distance_modes_agree(ctxs, mode):
    """The three distance modes (tables / coordinates / mixed; tuning flags of the descriptor) compute the same
    D(u,v) bit for bit."""
    from dataclasses import replace
    for name in ("small", "large"):
        inst = replace(wl.make(name), flags=binding.LGX_FLAG_DIST_COORDS if mode == 1 else binding.LGX_FLAG_DIST_MIXED)
        g2 = binding.Instance(inst)
        assert g2.info()["coords"] == mode
        _, o, _ = ctxs(name)
        want = o.eval_batch(inst.seed, first_id=0, n=4096)
        got = [t.cpu().numpy() for t in g2.eval_batch(inst.seed, first_id=0, n=4096)]
        assert np.array_equal(got[3], want[3]) and np.array_equal(got[0], want[0])
        assert g2.search(inst.seed, 4096) == o.search(inst.seed, 4096)


def test_workspace_pool_is_shared_and_trimmable(ctxs):
    """The queue of feasible candidates comes from ONE cached pool per device (include/lgx.h, Conventions): a second
    instance, an instance created after the first was destroyed, and calls after lgx_workspace_trim all give the same
    results; trimming is legal whenever no call is in flight."""
    inst, o, g = ctxs("small")
    n = 1 << 16
    ref = g.search(inst.seed, n)
    assert ref == o.search(inst.seed, n)
    g2 = binding.Instance(inst)
    assert g2.search(inst.seed, n) == ref
    g2.close()
    torch.cuda.synchronize()
    binding.workspace_trim()
    g3 = binding.Instance(inst)
    assert g3.search(inst.seed, n) == ref and g.search(inst.seed, n) == ref
    g3.close()
    binding.workspace_trim(); binding.workspace_trim()
    got = g.eval_batch(inst.seed, first_id=5, n=1000)
    want = o.eval_batch(inst.seed, first_id=5, n=1000)
    assert np.array_equal(got[3].cpu().numpy(), want[3]) and np.array_equal(got[0].cpu().numpy(), want[0])


@pytest.mark.parametrize("nf", [253, 255, 256, 257, 258, 259, 510, 511, 512, 513, 1022, 1023, 1024, 1025, 1026, 1027])
def test_field_count_boundaries(nf):
    """Field counts around the 8-bit / 16-bit switch of the Fisher-Yates array (255 | 256) and around 512 and 1024, for
    every padding of the right-aligned words (and every length of the last, partial block of four steps): plans,
    flags, costs and the argmin against the oracle."""
    from dataclasses import replace
    z = wl.make("paper_scale")
    z = replace(z, field_xy=z.field_xy[:nf].copy(), field_supply_t=z.field_supply_t[:nf].copy(), field_area_ha=z.field_area_ha[:nf].copy(),
                bp_demand_t=z.bp_demand_t * (0.9 * z.field_supply_t[:nf].sum() / z.bp_demand_t.sum()))
    o, g = lgo.Oracle(z), binding.Instance(z)
    n = 512
    want = o.eval_batch(6, first_id=0, n=n)
    got = [t.cpu().numpy() for t in g.eval_batch(6, first_id=0, n=n)]
    assert np.array_equal(got[3], want[3])
    for k in range(3):
        assert_costs(got[k], want[k], f"nf={nf} output {k}")
    wd = o.decode_batch(6, first_id=0, n=128); gd = g.decode_batch(6, first_id=0, n=128)
    for key in wd:
        a_ = gd[key].cpu().numpy()
        if a_.dtype == np.int16: a_ = a_.view(np.uint16)
        assert np.array_equal(a_, wd[key]), key
    fin = np.isfinite(want[0])
    best = (float(want[0][fin].min()), int(np.flatnonzero(want[0] == want[0][fin].min())[0])) if fin.any() else (float("inf"), 0)
    assert g.search(6, n) == best == o.search(6, n)
    g.close()




@pytest.mark.parametrize("name", ["small", "large", "sweep", "paper_scale"])
def test_walk_lockstep_does_not_change_results(ctxs, name):
    """LGX_OPT_WALK_LOCKSTEP only changes how the warps of a walk/finish block draw their records: same bits either way,
    also when the last batch of a launch is ragged and when a block's batch is larger than the queue."""
    inst, o, g = ctxs(name)
    default = g.query(24)
    assert default == (1 if g.query(4) != 0 and inst.n_fields < 1024 else 0)      # coordinates and N_F < 1024: on by default
    outs = []
    for mode in (0, 1):
        g.set_option(binding.LGX_OPT_WALK_LOCKSTEP, mode)
        assert g.query(24) == mode
        r = [t.clone() for t in g.eval_batch(inst.seed, first_id=9, n=100003)] + [g.search(inst.seed, 70001, first_id=3), g.search(inst.seed, 17)]
        outs.append(r)
    g.set_option(binding.LGX_OPT_WALK_LOCKSTEP, default)
    assert all(torch.equal(a, b) for a, b in zip(outs[0][:4], outs[1][:4])) and outs[0][4:] == outs[1][4:]
    want = o.eval_batch(inst.seed, first_id=9, n=512)
    assert np.array_equal(outs[1][0][:512].cpu().numpy(), want[0]) and np.array_equal(outs[1][3][:512].cpu().numpy(), want[3])


def test_pipe_microbenchmarks_report_plausible_rates():
    """lgx_selftest what = 1..5 (include/lgx.h): sustained warp-instructions per clock per SM of five pipes.  No pipe
    can beat the four schedulers of an SM, and each of these is known to be a fraction of that; the bounds are wide
    (they guard the counting and the clock arithmetic, not a particular GPU)."""
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    for what, lo, hi in ((1, 0.4, 2.1), (2, 0.9, 4.01), (3, 0.4, 2.1), (4, 0.02, 2.1), (5, 0.1, 1.1)):
        n_inst, cycles = binding.selftest(what, 1 << 13)
        assert n_inst == 2 * sms * 32 * (1 << 13) * 4 * 8 * (2 if what in (2, 3) else 1) and cycles > 0
        rate = n_inst / cycles / sms
        assert lo <= rate <= hi, (what, rate)
    with pytest.raises(binding.LgxError):
        binding.selftest(6, 1 << 10)
