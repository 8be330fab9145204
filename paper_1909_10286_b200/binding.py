"""Thin ctypes binding of liblgx.so (include/lgx.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI.  torch is used for
device memory and streams only.  There is no CPU fallback: if the library cannot be loaded
or there is no CUDA device, calls raise LgxError.
"""
from __future__ import annotations
import ctypes as C
import os
import numpy as np

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liblgx.so")

LGX_OK, LGX_EINVAL, LGX_ETOOBIG, LGX_ECUDA, LGX_ENOMEM, LGX_ESTATIC = 0, -1, -2, -3, -4, -5
LGX_STATIC_SCRATCH_BYTES = 16 << 20
# include/lgx.h: descriptor flags and lgx_instance_set_option keys
LGX_FLAG_HU_BALANCE, LGX_FLAG_MAKESPAN_FILTER, LGX_FLAG_FIX_FIELD_BP = 2, 4, 8
LGX_FLAG_DIST_COORDS, LGX_FLAG_DIST_MIXED = 16, 32
LGX_OPT_THREADS_A, LGX_OPT_THREADS_B, LGX_OPT_THREADS_MV, LGX_OPT_CHUNK_LOG2, LGX_OPT_SQ_SHIFT, LGX_OPT_WALK_LOCKSTEP = 1, 2, 3, 4, 5, 7
LGX_MAX_BPS, LGX_MAX_SUS, LGX_MAX_MOVE_TOURS, LGX_MAX_MOVE_HUS = 127, 128, 64, 64

_dp = C.POINTER(C.c_double)


class lgx_instance_desc(C.Structure):
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


EXPORTS = ("lgx_instance_create", "lgx_instance_destroy", "lgx_eval_batch", "lgx_eval_batch_host",
           "lgx_eval_batch_static", "lgx_eval_batch_static_max",
           "lgx_search_range", "lgx_search", "lgx_decode_batch", "lgx_instance_query", "lgx_instance_set_timing",
           "lgx_instance_set_option", "lgx_selftest", "lgx_workspace_trim",
           "lgx_init_plan", "lgx_move_eval_batch", "lgx_local_search", "lgx_strerror")

_lib = None


def load(rebuild_if_stale: bool = True):
    """Load liblgx.so (building it in-tree with nvcc if missing or stale)."""
    global _lib
    if _lib is not None:
        return _lib
    if rebuild_if_stale and _build.is_stale():
        _build.build()
    if not os.path.exists(LIB_PATH):
        raise LgxError(LGX_ECUDA, "liblgx.so is missing: run `python -m paper_1909_10286_b200.build`")
    lib = C.CDLL(LIB_PATH)
    vp, u64, i32 = C.c_void_p, C.c_uint64, C.c_int
    lib.lgx_instance_create.argtypes = [C.POINTER(lgx_instance_desc), C.POINTER(vp)]
    lib.lgx_instance_destroy.argtypes = [vp]
    lib.lgx_eval_batch.argtypes = [vp, u64, vp, u64, u64, vp, vp, vp, vp, vp]
    lib.lgx_eval_batch_host.argtypes = [vp, u64, vp, u64, u64, vp, vp, vp, vp]
    lib.lgx_eval_batch_static.argtypes = [vp, u64, vp, u64, u64, vp, vp, vp, vp, vp]
    lib.lgx_eval_batch_static_max.argtypes = [vp, C.POINTER(u64)]
    lib.lgx_search_range.argtypes = [vp, u64, u64, u64, C.POINTER(C.c_double), C.POINTER(u64), vp]
    lib.lgx_search.argtypes = [vp, u64, u64, C.POINTER(C.c_double), C.POINTER(u64), vp]
    lib.lgx_decode_batch.argtypes = [vp, u64, vp, u64, u64] + [vp] * 7 + [vp]
    lib.lgx_instance_query.argtypes = [vp, i32, C.POINTER(C.c_int64)]
    lib.lgx_instance_set_timing.argtypes = [vp, i32]
    lib.lgx_instance_set_option.argtypes = [vp, i32, C.c_int64]
    lib.lgx_selftest.argtypes = [i32, u64, u64, C.POINTER(u64)]
    lib.lgx_init_plan.argtypes = [vp] + [vp] * 6 + [vp]
    lib.lgx_move_eval_batch.argtypes = [vp] + [vp] * 6 + [u64, u64, u64, vp, vp, vp, vp, vp]
    lib.lgx_local_search.argtypes = [vp] + [vp] * 6 + [u64, C.c_uint32, C.c_uint32, C.c_uint32,
                                                      C.POINTER(C.c_double), vp, vp, vp]
    lib.lgx_strerror.argtypes = [i32]
    lib.lgx_strerror.restype = C.c_char_p
    for f in EXPORTS:
        if f != "lgx_strerror":
            getattr(lib, f).restype = C.c_int
    _lib = lib
    return lib


class LgxError(RuntimeError):
    def __init__(self, code, msg=None):
        if msg is None:
            try:
                msg = load(False).lgx_strerror(code).decode()
            except Exception:      # noqa: BLE001
                msg = "lgx error"
        super().__init__(f"lgx error {code}: {msg}")
        self.code = code


def _check(rc):
    if rc != LGX_OK:
        raise LgxError(rc)


def _f64(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def _ptr(t):
    """data_ptr of a torch tensor (device or host) or None."""
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream_ptr(stream):
    if stream is None:
        import torch
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def make_desc(inst):
    """Marshal a workloads.Instance-like object into (lgx_instance_desc, keepalive)."""
    fx, fy = _f64(inst.field_xy[:, 0]), _f64(inst.field_xy[:, 1])
    bx, by = _f64(inst.bp_xy[:, 0]), _f64(inst.bp_xy[:, 1])
    sup, area, dem = _f64(inst.field_supply_t), _f64(inst.field_area_ha), _f64(inst.bp_demand_t)
    hu, su = _f64(inst.hu_rate_ha_per_h), _f64(inst.su_capacity_t)
    p = lambda a: a.ctypes.data_as(_dp)
    d = lgx_instance_desc(inst.hq[0], inst.hq[1], len(fx), p(fx), p(fy), p(sup), p(area),
                          len(bx), p(bx), p(by), p(dem), len(hu), p(hu), len(su), p(su),
                          inst.n_tours, inst.v_hu_road_kmh, inst.v_su_road_kmh, inst.v_infield_kmh,
                          inst.su_fill_h_per_t, inst.w_path, inst.w_time,
                          inst.extra_field_thresh, inst.flags)
    return d, (fx, fy, bx, by, sup, area, dem, hu, su)


PLAN_KEYS = (("bp_tour", np.uint8), ("bp_pos", np.uint8), ("field_bp", np.uint16), ("field_pos", np.uint16),
             ("hu_tour", np.uint8), ("su_tour", np.uint8))


def _plan_arrays(plan):
    """The six host arrays of a plan (copies, contiguous, typed) in the C ABI's order."""
    return [np.array(plan[k], dtype=dt, order="C", copy=True) for k, dt in PLAN_KEYS]


def selftest(what: int, n: int, seed: int = 0):
    """lgx_selftest: (arguments checked, mismatches) of a device routine against its library counterpart."""
    out = (C.c_uint64 * 2)()
    _check(load().lgx_selftest(what, n, seed, out))
    return int(out[0]), int(out[1])


def workspace_trim():
    """lgx_workspace_trim: release the workspace memory the library caches per device."""
    _check(load().lgx_workspace_trim())


class Instance:
    """lgx_instance_create .. lgx_instance_destroy, with the C calls as methods."""

    def __init__(self, inst):
        self._lib = load()
        self.n_f, self.n_b = len(inst.field_supply_t), len(inst.bp_demand_t)
        self.n_hu, self.n_su, self.n_t = len(inst.hu_rate_ha_per_h), len(inst.su_capacity_t), inst.n_tours
        d, keep = make_desc(inst)
        h = C.c_void_p()
        _check(self._lib.lgx_instance_create(C.byref(d), C.byref(h)))
        self._h = h

    def close(self):
        if getattr(self, "_h", None):
            self._lib.lgx_instance_destroy(self._h)
            self._h = None

    __del__ = close

    def query(self, what: int) -> int:
        v = C.c_int64()
        _check(self._lib.lgx_instance_query(self._h, what, C.byref(v)))
        return v.value

    def set_timing(self, enable: bool):
        _check(self._lib.lgx_instance_set_timing(self._h, 1 if enable else 0))

    def set_option(self, key: int, value: int):
        """lgx_instance_set_option: launch configuration only (LGX_OPT_*), never results."""
        _check(self._lib.lgx_instance_set_option(self._h, key, value))

    def kernel_times(self):
        """(ns in lgx_decode_cut, ns in lgx_walk_finish, kernel pairs timed) since set_timing(True)."""
        return self.query(12), self.query(13), self.query(14)

    def info(self):
        keys = ["image_bytes", "threads", "grid", "smem_bytes", "coords", "state_bytes", "sm_count", "launches",
                "threads_finish", "smem_bytes_finish", "chunk", "record_bytes"]
        d = {k: self.query(i) for i, k in enumerate(keys)}
        d.update(threads_mv=self.query(15), sq_shift=self.query(17), threads_decode=self.query(18),
                 state_bytes_finish=self.query(19), device=self.query(20))
        return d

    # -- lgx_eval_batch: device tensors in/out (torch), asynchronous on `stream`
    def eval_batch(self, seed, ids=None, first_id=0, n=None, out=None, stream=None):
        import torch
        if ids is not None:
            assert ids.is_cuda and ids.dtype in (torch.int64, torch.uint64) and ids.is_contiguous()
            n = ids.numel()
        dev = torch.device("cuda", torch.cuda.current_device())
        if out is None:
            out = (torch.empty(n, dtype=torch.float64, device=dev), torch.empty(n, dtype=torch.float64, device=dev),
                   torch.empty(n, dtype=torch.float64, device=dev), torch.empty(n, dtype=torch.uint8, device=dev))
        cost, path, mk, feas = out
        _check(self._lib.lgx_eval_batch(self._h, seed, _ptr(ids), first_id, n, _ptr(cost), _ptr(path),
                                        _ptr(mk), _ptr(feas), _stream_ptr(stream)))
        return out

    # -- lgx_eval_batch_static: lgx_eval_batch without any allocation inside the library (fixed 16 MiB device array)
    def eval_batch_static_max(self) -> int:
        """Largest n eval_batch_static takes for this instance (lgx_eval_batch_static_max)."""
        v = C.c_uint64()
        _check(self._lib.lgx_eval_batch_static_max(self._h, C.byref(v)))
        return v.value

    def eval_batch_static(self, seed, out, ids=None, first_id=0, n=None, stream=None):
        """lgx_eval_batch_static.  `out` = the caller's (cost, path_km, makespan_h, feasible) device tensors: unlike
        eval_batch this wrapper creates none, because the callers it is for cannot allocate.  One call at a time per
        device: every call shares the library's one scratch array (include/lgx.h)."""
        if ids is not None:
            n = ids.numel()
        cost, path, mk, feas = out
        _check(self._lib.lgx_eval_batch_static(self._h, seed, _ptr(ids), first_id, n, _ptr(cost), _ptr(path),
                                               _ptr(mk), _ptr(feas), _stream_ptr(stream)))
        return out

    # -- lgx_eval_batch_host: numpy host buffers in/out
    def eval_batch_host(self, seed, ids=None, first_id=0, n=None, out=None):
        if ids is not None:
            ids = np.ascontiguousarray(ids, dtype=np.uint64); n = len(ids)
        if out is None:
            out = (np.empty(n), np.empty(n), np.empty(n), np.empty(n, np.uint8))
        cost, path, mk, feas = out
        _check(self._lib.lgx_eval_batch_host(self._h, seed, ids.ctypes.data if ids is not None else None,
                                             first_id, n, cost.ctypes.data, path.ctypes.data,
                                             mk.ctypes.data, feas.ctypes.data))
        return out

    # -- lgx_search / lgx_search_range: returns (best_cost, best_id) on the host
    def search(self, seed, budget, first_id=0, stream=None):
        c = C.c_double(); i = C.c_uint64()
        _check(self._lib.lgx_search_range(self._h, seed, first_id, budget, C.byref(c), C.byref(i),
                                          _stream_ptr(stream)))
        return c.value, i.value

    # -- lgx_decode_batch: diagnostic plan export (device tensors)
    def decode_batch(self, seed, ids=None, first_id=0, n=None, stream=None):
        import torch
        if ids is not None:
            n = ids.numel()
        dev = torch.device("cuda", torch.cuda.current_device())
        z8 = lambda m: torch.zeros((n, m), dtype=torch.uint8, device=dev)
        z16 = lambda m: torch.zeros((n, m), dtype=torch.int16, device=dev)
        o = dict(bp_tour=z8(self.n_b), bp_pos=z8(self.n_b), field_bp=z16(self.n_f), field_pos=z16(self.n_f),
                 hu_tour=z8(self.n_hu), su_tour_init=z8(self.n_su), su_tour_final=z8(self.n_su))
        _check(self._lib.lgx_decode_batch(self._h, seed, _ptr(ids), first_id, n, _ptr(o["bp_tour"]),
                                          _ptr(o["bp_pos"]), _ptr(o["field_bp"]), _ptr(o["field_pos"]),
                                          _ptr(o["hu_tour"]), _ptr(o["su_tour_init"]), _ptr(o["su_tour_final"]),
                                          _stream_ptr(stream)))
        return o

    # -- Algorithm 1 (lgx_init_plan, lgx_move_eval_batch, lgx_local_search); plans are dicts of host arrays
    def init_plan(self, stream=None):
        a = [np.zeros(n, dt) for n, dt in ((self.n_b, np.uint8), (self.n_b, np.uint8), (self.n_f, np.uint16),
                                           (self.n_f, np.uint16), (self.n_hu, np.uint8), (self.n_su, np.uint8))]
        _check(self._lib.lgx_init_plan(self._h, *[x.ctypes.data for x in a], _stream_ptr(stream)))
        return dict(zip([k for k, _ in PLAN_KEYS], a))

    def move_eval_batch(self, plan, seed, first_id, n, out=None, stream=None):
        import torch
        a = _plan_arrays(plan)
        dev = torch.device("cuda", torch.cuda.current_device())
        if out is None:
            out = (torch.empty(n, dtype=torch.float64, device=dev), torch.empty(n, dtype=torch.float64, device=dev),
                   torch.empty(n, dtype=torch.float64, device=dev), torch.empty(n, dtype=torch.uint8, device=dev))
        cost, path, mk, feas = out
        _check(self._lib.lgx_move_eval_batch(self._h, *[x.ctypes.data for x in a], seed, first_id, n,
                                             _ptr(cost), _ptr(path), _ptr(mk), _ptr(feas), _stream_ptr(stream)))
        return out

    def local_search(self, plan, seed, n_iters, n_workers, eps_thresh, history=True, stream=None):
        """Returns (x*, C*, hist_cost, hist_id)."""
        a = _plan_arrays(plan)
        c = C.c_double()
        hc = np.zeros(n_iters) if history else None
        hi = np.zeros(n_iters, np.uint64) if history else None
        _check(self._lib.lgx_local_search(self._h, *[x.ctypes.data for x in a], seed, n_iters, n_workers, eps_thresh,
                                          C.byref(c), hc.ctypes.data if history else None,
                                          hi.ctypes.data if history else None, _stream_ptr(stream)))
        return dict(zip([k for k, _ in PLAN_KEYS], a)), c.value, hc, hi

    def plan_of(self, seed, cand_id, stream=None):
        """The plan of one sampled candidate (lgx_decode_batch, one row) as a dict of host arrays: the bridge from
        lgx_search's winner to lgx_local_search's x_0 (SU sets as sampled; Algorithm 2 runs when x_0 is scored)."""
        import torch
        ids = torch.tensor([cand_id - (1 << 64) if cand_id >= (1 << 63) else cand_id], dtype=torch.int64, device="cuda")
        d = self.decode_batch(seed, ids=ids, stream=stream)
        torch.cuda.synchronize()
        h = {k: v[0].cpu().numpy() for k, v in d.items()}
        return dict(bp_tour=h["bp_tour"], bp_pos=h["bp_pos"], field_bp=h["field_bp"].view(np.uint16),
                    field_pos=h["field_pos"].view(np.uint16), hu_tour=h["hu_tour"], su_tour=h["su_tour_init"])
