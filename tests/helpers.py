"""Small helpers shared by tests (no method arithmetic)."""
from types import SimpleNamespace
import numpy as np


def mk_instance(hq, fields, bps, hu, su, n_tours, **kw):
    """fields: [(x,y,supply_t,area_ha)], bps: [(x,y,demand_t)]."""
    f = np.asarray(fields, dtype=np.float64).reshape(-1, 4)
    b = np.asarray(bps, dtype=np.float64).reshape(-1, 3)
    d = dict(name="hand", hq=tuple(hq), field_xy=f[:, :2].copy(), field_supply_t=f[:, 2].copy(),
             field_area_ha=f[:, 3].copy(), bp_xy=b[:, :2].copy(), bp_demand_t=b[:, 2].copy(),
             hu_rate_ha_per_h=np.asarray(hu, dtype=np.float64), su_capacity_t=np.asarray(su, dtype=np.float64),
             n_tours=n_tours, v_hu_road_kmh=40.0, v_su_road_kmh=40.0, v_infield_kmh=15.0,
             su_fill_h_per_t=0.008, w_path=1.0, w_time=1.0, extra_field_thresh=0x40000000, flags=0)
    d.update(kw)
    ns = SimpleNamespace(**d)
    ns.n_fields, ns.n_bps = f.shape[0], b.shape[0]
    ns.n_hu, ns.n_su = len(ns.hu_rate_ha_per_h), len(ns.su_capacity_t)
    return ns


# ---- the oracle on all host cores: one single-threaded oracle process per core over disjoint chunks of the SAME
# request (the oracle itself stays as it is; this only spreads the ids)

def _mp_eval_chunk(name, seed, ids, first, n):
    from oracle import lgo
    from paper_1909_10286_b200 import workloads as wl
    o = lgo.Oracle(wl.make(name))
    return o.eval_batch(seed, ids=ids, first_id=first, n=n)


def _mp_search_chunk(name, seed, first, n):
    from oracle import lgo
    from paper_1909_10286_b200 import workloads as wl
    o = lgo.Oracle(wl.make(name))
    return o.search(seed, n, first_id=first)


def _chunks(n, parts):
    base, rem = divmod(n, parts)
    out, at = [], 0
    for r in range(parts):
        k = base + (1 if r < rem else 0)
        if k:
            out.append((at, k))
        at += k
    return out


def oracle_eval_mp(name, seed, ids=None, first_id=0, n=None, procs=None):
    """lgo_eval_batch of workloads.make(name) over `procs` processes; same outputs as Oracle.eval_batch."""
    import multiprocessing as mp, os
    procs = procs or os.cpu_count() or 1
    if ids is not None:
        n = len(ids)
    jobs = [(name, seed, None if ids is None else ids[a:a + k], first_id + a if ids is None else 0, k) for a, k in _chunks(n, procs)]
    with mp.get_context("fork").Pool(len(jobs)) as pool:
        res = pool.starmap(_mp_eval_chunk, jobs)
    return tuple(np.concatenate([r[j] for r in res]) for j in range(4))


def oracle_search_mp(name, seed, budget, first_id=0, procs=None):
    """Ordered minimum of (cost bits, id) over [first_id, first_id + budget): per-process lgo_search over contiguous
    id ranges, combined in id order (lowest id on equal cost)."""
    import multiprocessing as mp, os, struct
    procs = procs or os.cpu_count() or 1
    jobs = [(name, seed, first_id + a, k) for a, k in _chunks(budget, procs)]
    with mp.get_context("fork").Pool(len(jobs)) as pool:
        res = pool.starmap(_mp_search_chunk, jobs)
    bits = lambda c: struct.unpack("<Q", struct.pack("<d", c))[0]
    return min(res, key=lambda p: (bits(p[0]), p[1]))
