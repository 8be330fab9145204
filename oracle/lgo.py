"""ctypes binding of the ORACLE (oracle/lgo.c).  Test infrastructure, not product code:
only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this module.  It imports nothing from the product package."""
from __future__ import annotations
import ctypes as C
import numpy as np
from . import build as _build

_lib = C.CDLL(_build.build())

_dp = C.POINTER(C.c_double)


class _Desc(C.Structure):
    _fields_ = [("hq_x", C.c_double), ("hq_y", C.c_double),
                ("n_fields", C.c_int32), ("field_x", _dp), ("field_y", _dp),
                ("field_supply_t", _dp), ("field_area_ha", _dp),
                ("n_bps", C.c_int32), ("bp_x", _dp), ("bp_y", _dp), ("bp_demand_t", _dp),
                ("n_hu_total", C.c_int32), ("hu_rate_ha_per_h", _dp),
                ("n_su_total", C.c_int32), ("su_capacity_t", _dp),
                ("n_tours", C.c_int32),
                ("v_hu_road_kmh", C.c_double), ("v_su_road_kmh", C.c_double),
                ("v_infield_kmh", C.c_double), ("su_fill_h_per_t", C.c_double),
                ("w_path", C.c_double), ("w_time", C.c_double),
                ("extra_field_thresh", C.c_uint32), ("flags", C.c_uint32)]


def _f64(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t)) if a is not None else None


_lib.lgo_instance_create.argtypes = [C.POINTER(_Desc), C.POINTER(C.c_void_p)]
_lib.lgo_instance_destroy.argtypes = [C.c_void_p]
_lib.lgo_draw.restype = C.c_uint32
_lib.lgo_draw.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32]
_lib.lgo_distance.restype = C.c_double
_lib.lgo_distance.argtypes = [C.c_void_p, C.c_int32, C.c_int32]
_lib.lgo_quantum.restype = C.c_int64
_lib.lgo_quantum.argtypes = [C.c_void_p, C.c_int, C.c_int32]
_lib.lgo_decode.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64] + [C.c_void_p] * 6
_lib.lgo_score.argtypes = [C.c_void_p] + [C.c_void_p] * 15
_lib.lgo_score_ex.argtypes = [C.c_void_p] + [C.c_void_p] * 6 + [C.c_int] + [C.c_void_p] * 10
_lib.lgo_hu_balance.argtypes = [C.c_int32, C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]
_lib.lgo_su_local_min.argtypes = [C.c_int32, C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p,
                                  C.c_void_p, C.c_double, C.c_void_p]
_lib.lgo_eval_batch.argtypes = [C.c_void_p, C.c_uint64, C.c_void_p, C.c_uint64, C.c_uint64] + [C.c_void_p] * 4
_lib.lgo_decode_batch.argtypes = [C.c_void_p, C.c_uint64, C.c_void_p, C.c_uint64, C.c_uint64] + [C.c_void_p] * 7
_lib.lgo_search.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64, C.c_uint64, C.POINTER(C.c_double),
                            C.POINTER(C.c_uint64)]
_lib.lgo_philox4x32_10.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
_lib.lgo_init_plan.argtypes = [C.c_void_p] + [C.c_void_p] * 6
_lib.lgo_apply_move.argtypes = [C.c_void_p, C.c_uint32, C.c_uint32, C.c_uint32] + [C.c_void_p] * 4
_lib.lgo_move_eval_batch.argtypes = [C.c_void_p] + [C.c_void_p] * 6 + [C.c_uint64, C.c_uint64, C.c_uint64] + [C.c_void_p] * 4
_lib.lgo_local_search.argtypes = [C.c_void_p] + [C.c_void_p] * 6 + [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32,
                                                                    C.POINTER(C.c_double), C.c_void_p, C.c_void_p]

PLAN_KEYS = (("bp_tour", np.uint8), ("bp_pos", np.uint8), ("field_bp", np.uint16), ("field_pos", np.uint16),
             ("hu_tour", np.uint8), ("su_tour", np.uint8))


def _plan_arrays(plan):
    return [np.ascontiguousarray(plan[k], dtype=t).copy() for k, t in PLAN_KEYS]


class OracleError(RuntimeError):
    def __init__(self, code):
        super().__init__(f"lgo error {code}")
        self.code = code


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32); k = np.asarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    _lib.lgo_philox4x32_10(c.ctypes.data, k.ctypes.data, out.ctypes.data)
    return out


def draw(seed, id_, stream, d):
    return int(_lib.lgo_draw(seed, id_, stream, d))


def su_local_min(E_h, n_hu, cap_q, su_tour, kappa):
    E = _f64(E_h); nh = np.ascontiguousarray(n_hu, dtype=np.int32)
    cq = np.ascontiguousarray(cap_q, dtype=np.int64)
    st = np.ascontiguousarray(su_tour, dtype=np.uint8).copy()
    W = np.zeros(len(E), dtype=np.float64)
    moves = _lib.lgo_su_local_min(len(E), E.ctypes.data, nh.ctypes.data, len(cq), cq.ctypes.data,
                                  st.ctypes.data, float(kappa), W.ctypes.data)
    return moves, st, W


class Oracle:
    """One oracle instance (lgo_instance_create .. lgo_instance_destroy)."""

    def __init__(self, inst):
        """inst: any object with the attributes of workloads.Instance."""
        self.n_f, self.n_b = inst.n_fields, inst.n_bps
        self.n_hu, self.n_su, self.n_t = inst.n_hu, inst.n_su, inst.n_tours
        fx, fy = _f64(inst.field_xy[:, 0]), _f64(inst.field_xy[:, 1])
        bx, by = _f64(inst.bp_xy[:, 0]), _f64(inst.bp_xy[:, 1])
        keep = [fx, fy, bx, by, _f64(inst.field_supply_t), _f64(inst.field_area_ha),
                _f64(inst.bp_demand_t), _f64(inst.hu_rate_ha_per_h), _f64(inst.su_capacity_t)]
        d = _Desc(inst.hq[0], inst.hq[1], self.n_f, _p(fx, C.c_double), _p(fy, C.c_double),
                  _p(keep[4], C.c_double), _p(keep[5], C.c_double),
                  self.n_b, _p(bx, C.c_double), _p(by, C.c_double), _p(keep[6], C.c_double),
                  self.n_hu, _p(keep[7], C.c_double), self.n_su, _p(keep[8], C.c_double),
                  self.n_t, inst.v_hu_road_kmh, inst.v_su_road_kmh, inst.v_infield_kmh,
                  inst.su_fill_h_per_t, inst.w_path, inst.w_time,
                  inst.extra_field_thresh, inst.flags)
        h = C.c_void_p()
        rc = _lib.lgo_instance_create(C.byref(d), C.byref(h))
        if rc != 0:
            raise OracleError(rc)
        self._h = h

    def close(self):
        if getattr(self, "_h", None):
            _lib.lgo_instance_destroy(self._h); self._h = None

    __del__ = close

    def distance(self, u, v):
        return float(_lib.lgo_distance(self._h, u, v))

    def quanta(self, what):
        n = {0: self.n_f, 1: self.n_f, 2: self.n_b, 3: self.n_hu, 4: self.n_su}[what]
        return np.array([_lib.lgo_quantum(self._h, what, i) for i in range(n)], dtype=np.int64)

    def decode(self, seed, id_):
        bt = np.zeros(self.n_b, np.uint8); bp = np.zeros(self.n_b, np.uint8)
        fb = np.zeros(self.n_f, np.uint16); fp = np.zeros(self.n_f, np.uint16)
        hu = np.zeros(self.n_hu, np.uint8); su = np.zeros(self.n_su, np.uint8)
        rc = _lib.lgo_decode(self._h, seed, id_, bt.ctypes.data, bp.ctypes.data, fb.ctypes.data,
                             fp.ctypes.data, hu.ctypes.data, su.ctypes.data)
        if rc: raise OracleError(rc)
        return dict(bp_tour=bt, bp_pos=bp, field_bp=fb, field_pos=fp, hu_tour=hu, su_tour=su)

    def score(self, plan, hu_balance=False):
        a = lambda k, t: np.ascontiguousarray(plan[k], dtype=t)
        bt, bp = a("bp_tour", np.uint8), a("bp_pos", np.uint8)
        fb, fp = a("field_bp", np.uint16), a("field_pos", np.uint16)
        hu, su = a("hu_tour", np.uint8), a("su_tour", np.uint8)
        sc = np.zeros(8); nt = self.n_t
        route, time_h, E, W, Lg = (np.zeros(nt) for _ in range(5))
        Sq = np.zeros(self.n_b, np.int64); sh = np.zeros(self.n_f, np.int64)
        suf = np.zeros(self.n_su, np.uint8); huf = np.zeros(self.n_hu, np.uint8)
        rc = _lib.lgo_score_ex(self._h, bt.ctypes.data, bp.ctypes.data, fb.ctypes.data, fp.ctypes.data,
                               hu.ctypes.data, su.ctypes.data, 1 if hu_balance else 0, sc.ctypes.data, route.ctypes.data,
                               time_h.ctypes.data, E.ctypes.data, W.ctypes.data, Lg.ctypes.data,
                               Sq.ctypes.data, sh.ctypes.data, suf.ctypes.data, huf.ctypes.data)
        if rc: raise OracleError(rc)
        return dict(feasible=bool(sc[0]), L_HU=sc[1], L_eSU=sc[2], L_lSU=sc[3], path=sc[4],
                    makespan=sc[5], cost=sc[6], moves=int(sc[7]), route=route, T=time_h, E=E,
                    wait=W, L=Lg, bp_supply_q=Sq, shuttles=sh, su_tour_final=suf, hu_tour_final=huf)

    def score_fast(self, bt, bp, fb, fp, hu, su, sc):
        """score() without array outputs, on pre-typed contiguous arrays (brute force)."""
        return _lib.lgo_score(self._h, bt.ctypes.data, bp.ctypes.data, fb.ctypes.data, fp.ctypes.data,
                              hu.ctypes.data, su.ctypes.data, sc.ctypes.data,
                              None, None, None, None, None, None, None, None)

    def eval_batch(self, seed, ids=None, first_id=0, n=None):
        if ids is not None:
            ids = np.ascontiguousarray(ids, dtype=np.uint64); n = len(ids)
        cost = np.zeros(n); path = np.zeros(n); mk = np.zeros(n); fe = np.zeros(n, np.uint8)
        rc = _lib.lgo_eval_batch(self._h, seed, ids.ctypes.data if ids is not None else None,
                                 first_id, n, cost.ctypes.data, path.ctypes.data, mk.ctypes.data,
                                 fe.ctypes.data)
        if rc: raise OracleError(rc)
        return cost, path, mk, fe

    def decode_batch(self, seed, ids=None, first_id=0, n=None):
        if ids is not None:
            ids = np.ascontiguousarray(ids, dtype=np.uint64); n = len(ids)
        bt = np.zeros((n, self.n_b), np.uint8); bp = np.zeros((n, self.n_b), np.uint8)
        fb = np.zeros((n, self.n_f), np.uint16); fp = np.zeros((n, self.n_f), np.uint16)
        hu = np.zeros((n, self.n_hu), np.uint8)
        si = np.zeros((n, self.n_su), np.uint8); sf = np.zeros((n, self.n_su), np.uint8)
        rc = _lib.lgo_decode_batch(self._h, seed, ids.ctypes.data if ids is not None else None,
                                   first_id, n, bt.ctypes.data, bp.ctypes.data, fb.ctypes.data,
                                   fp.ctypes.data, hu.ctypes.data, si.ctypes.data, sf.ctypes.data)
        if rc: raise OracleError(rc)
        return dict(bp_tour=bt, bp_pos=bp, field_bp=fb, field_pos=fp, hu_tour=hu,
                    su_tour_init=si, su_tour_final=sf)

    def search(self, seed, budget, first_id=0):
        c = C.c_double(); i = C.c_uint64()
        rc = _lib.lgo_search(self._h, seed, first_id, budget, C.byref(c), C.byref(i))
        if rc: raise OracleError(rc)
        return c.value, i.value

    # ---- NEXT rows: Algorithm 1 (initialisation, moves, local search)
    def init_plan(self):
        bt = np.zeros(self.n_b, np.uint8); bp = np.zeros(self.n_b, np.uint8)
        fb = np.zeros(self.n_f, np.uint16); fp = np.zeros(self.n_f, np.uint16)
        hu = np.zeros(self.n_hu, np.uint8); su = np.zeros(self.n_su, np.uint8)
        rc = _lib.lgo_init_plan(self._h, bt.ctypes.data, bp.ctypes.data, fb.ctypes.data, fp.ctypes.data,
                                hu.ctypes.data, su.ctypes.data)
        if rc: raise OracleError(rc)
        return dict(bp_tour=bt, bp_pos=bp, field_bp=fb, field_pos=fp, hu_tour=hu, su_tour=su)

    def apply_move(self, plan, w0, w1, w2):
        a = _plan_arrays(plan)
        rc = _lib.lgo_apply_move(self._h, w0, w1, w2, *[x.ctypes.data for x in a[:4]])
        if rc: raise OracleError(rc)
        return dict(zip([k for k, _ in PLAN_KEYS], a))

    def move_eval_batch(self, plan, seed, first_id, n):
        a = _plan_arrays(plan)
        cost = np.zeros(n); path = np.zeros(n); mk = np.zeros(n); fe = np.zeros(n, np.uint8)
        rc = _lib.lgo_move_eval_batch(self._h, *[x.ctypes.data for x in a], seed, first_id, n,
                                      cost.ctypes.data, path.ctypes.data, mk.ctypes.data, fe.ctypes.data)
        if rc: raise OracleError(rc)
        return cost, path, mk, fe

    def local_search(self, plan, seed, n_iters, n_workers, eps_thresh):
        a = _plan_arrays(plan)
        c = C.c_double(); hc = np.zeros(n_iters); hi = np.zeros(n_iters, np.uint64)
        rc = _lib.lgo_local_search(self._h, *[x.ctypes.data for x in a], seed, n_iters, n_workers, eps_thresh,
                                   C.byref(c), hc.ctypes.data, hi.ctypes.data)
        if rc: raise OracleError(rc)
        return dict(zip([k for k, _ in PLAN_KEYS], a)), c.value, hc, hi


def hu_balance(road_h, area_q, rate_q, hu_tour):
    """The embedded HU assignment alone (R39) on explicit numbers.
    Returns (moves, hu_tour, T)."""
    road = np.ascontiguousarray(road_h, dtype=np.float64); nt = len(road)
    aq = np.ascontiguousarray(area_q, dtype=np.int64); rq = np.ascontiguousarray(rate_q, dtype=np.int64)
    hu = np.array(hu_tour, dtype=np.uint8, copy=True); T = np.zeros(nt)
    m = _lib.lgo_hu_balance(nt, road.ctypes.data, aq.ctypes.data, len(rq), rq.ctypes.data, hu.ctypes.data, T.ctypes.data)
    return m, hu, T
