"""GPU parity on RANDOM instance shapes (-m gpu): seeded draws of N_F, N_B, N_T, N_HU, N_SU, demand tightness,
extra-field threshold, weights and velocities — shapes the five configs never hit (N_T = N_B, one HU per tour, more
tours than the move kernels take, 129..255-field byte arrays next to 16-bit ones, BPs with zero demand) — each through
every launch variant the instance allows (distance modes, lock-step work fetch, the per-warp decode/cut kernel).
Flags and plans bit-exact, costs bit-equal (bar: 1e-9 relative), identical argmin."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import lgo
from paper_1909_10286_b200 import binding, workloads as wl


def random_instance(k):
    rng = np.random.default_rng(7700 + k)
    nf = int(rng.choice([1, 2, 3, 7, 31, 32, 33, 64, 129, 200, 255, 256, 300, 640, 1100])) if k % 3 else int(rng.integers(1, 420))
    nb = int(min(nf, rng.integers(1, 24))) if nf > 1 else 1
    nt = int(rng.integers(1, nb + 1))
    nhu = int(rng.integers(nt, nt + 12))
    nsu = int(rng.integers(nt, min(128, nt + 70) + 1))
    side = float(rng.uniform(5.0, 300.0))
    field_xy = rng.uniform(0, side, (nf, 2))
    if k % 5 == 0 and nf > 2:
        field_xy[1] = field_xy[0]                                  # coincident fields: a zero-length leg
    bp_xy = rng.uniform(0, side, (nb, 2))
    area = rng.uniform(0.5, 40.0, nf)
    supply = area * rng.uniform(20.0, 60.0, nf)
    tight = float(rng.choice([0.3, 0.8, 0.95, 1.02]))
    demand = tight * supply.sum() * rng.dirichlet(np.ones(nb))
    if k % 4 == 1 and nb > 2:
        demand[int(rng.integers(0, nb))] = 0.0                     # a BP that wants nothing (R21: the general cut step)
    hu = rng.uniform(1.0, 4.0, nhu) if k % 2 else np.full(nhu, 2.5)
    su = rng.uniform(10.0, 40.0, nsu) if k % 2 else np.full(nsu, 16.5)
    return wl.Instance(name=f"fuzz{k}", hq=(float(rng.uniform(0, side)), 0.0), field_xy=field_xy, field_supply_t=supply,
                       field_area_ha=area, bp_xy=bp_xy, bp_demand_t=demand, hu_rate_ha_per_h=hu, su_capacity_t=su, n_tours=nt,
                       v_hu_road_kmh=float(rng.uniform(10, 60)), v_su_road_kmh=float(rng.uniform(10, 60)),
                       su_fill_h_per_t=float(rng.choice([0.0, 0.008, 0.05])), w_path=float(rng.uniform(0, 2)), w_time=float(rng.uniform(0, 50)),
                       extra_field_thresh=int(rng.choice([0, 0x20000000, 0x40000000, 0xC0000000, 0xFFFFFFFF])), budget=1 << 20, seed=int(rng.integers(0, 2**63)))


def variants(inst):
    """(flags, options) of every launch variant that exists for this instance."""
    from dataclasses import replace
    out = []
    for fl in (0, binding.LGX_FLAG_DIST_COORDS, binding.LGX_FLAG_DIST_MIXED):
        try:
            g = binding.Instance(replace(inst, flags=fl))
        except binding.LgxError:
            continue
        out.append((g, f"flags={fl}"))
    return out


@pytest.mark.parametrize("k", range(60))
def test_random_instance(k):
    inst = random_instance(k)
    try:
        o = lgo.Oracle(inst)
    except Exception:
        pytest.fail("the fuzz generator drew an instance outside the documented ranges: every seeded shape must run (no skips)")
    n = 700 if inst.n_fields <= 300 else 260
    first = [0, (1 << 33) + 7, 2**64 - n][k % 3]
    want = o.eval_batch(inst.seed, first_id=first, n=n)
    wplan = o.decode_batch(inst.seed, first_id=first, n=64)
    wbest = o.search(inst.seed, n, first_id=first)
    for g, tag in variants(inst):
        modes = [(None, None)]
        if g.query(4) != 0:
            modes.append((binding.LGX_OPT_WALK_LOCKSTEP, 1 - g.query(24)))
        for key, val in modes:
            if key is not None:
                g.set_option(key, val)
            got = [t.cpu().numpy() for t in g.eval_batch(inst.seed, first_id=first, n=n)]
            what = f"fuzz {k} N_F={inst.n_fields} N_B={inst.n_bps} N_T={inst.n_tours} {tag} opt={key}:{val}"
            assert np.array_equal(got[3], want[3]), what
            for j in range(3):
                fin = np.isfinite(want[j])
                assert np.array_equal(np.isfinite(got[j]), fin), what
                assert np.array_equal(got[j][fin], want[j][fin]), what + f" output {j}: max rel {np.max(np.abs(got[j][fin] - want[j][fin]) / np.abs(want[j][fin])):.3e}"
            assert g.search(inst.seed, n, first_id=first) == wbest, what
        gd = g.decode_batch(inst.seed, first_id=first, n=64)
        for key in wplan:
            a = gd[key].cpu().numpy()
            if a.dtype == np.int16: a = a.view(np.uint16)
            assert np.array_equal(a, wplan[key]), f"fuzz {k} {tag} plan array {key}"
        g.close()


@pytest.mark.parametrize("k", range(40))
def test_random_instance_algorithm1(k):
    """The paper's own loop on the same random shapes: start plan, one batch of workers (ids >= 2^40), six iterations of
    lgx_local_search with each flag combination — identical to the oracle, plan arrays included."""
    from dataclasses import replace
    base = random_instance(100 + k)
    flags = [0, binding.LGX_FLAG_HU_BALANCE, binding.LGX_FLAG_MAKESPAN_FILTER, binding.LGX_FLAG_FIX_FIELD_BP,
             binding.LGX_FLAG_HU_BALANCE | binding.LGX_FLAG_MAKESPAN_FILTER | binding.LGX_FLAG_FIX_FIELD_BP][k % 5]
    inst = replace(base, flags=flags)
    try:
        o = lgo.Oracle(inst)
    except Exception:
        pytest.fail("the fuzz generator drew an instance outside the documented ranges: every seeded shape must run (no skips)")
    g = binding.Instance(inst)
    if g.query(15) == 0:
        g.close(); pytest.fail("the move kernels do not fit a seeded fuzz shape: every shape must run (no skips)")
    p0, q0 = g.init_plan(), o.init_plan()
    for key in q0:
        assert np.array_equal(p0[key], q0[key]), f"fuzz {k}: start plan array {key}"
    n = 1500
    got = [t.cpu().numpy() for t in g.move_eval_batch(p0, inst.seed, (1 << 40) + 3, n)]
    want = o.move_eval_batch(p0, inst.seed, (1 << 40) + 3, n)
    assert np.array_equal(got[3], want[3])
    for j in range(3):
        fin = np.isfinite(want[j])
        assert np.array_equal(np.isfinite(got[j]), fin) and np.array_equal(got[j][fin], want[j][fin]), f"fuzz {k} flags={flags} worker output {j}"
    g.set_option(binding.LGX_OPT_THREADS_MV, 64)
    nw = g.query(6) * 64 + 77                                  # more than one grid round, ragged
    gp, gc, ghc, ghi = g.local_search(p0, inst.seed, 6, nw, 0x66666666)
    op, oc, ohc, ohi = o.local_search(p0, inst.seed, 6, nw, 0x66666666)
    assert np.array_equal(ghi, ohi) and np.array_equal(ghc, ohc) and gc == oc, f"fuzz {k} flags={flags}: search history"
    for key in op:
        assert np.array_equal(gp[key], op[key]), f"fuzz {k} flags={flags}: x* array {key}"
    g.close()
