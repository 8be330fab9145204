"""CPU-side checks of the boundary: liblgx.so builds, loads and exports every symbol
include/lgx.h declares; host-side validation in lgx_instance_create returns the documented
codes before any CUDA call (no compute without a GPU)."""
import os, re
import numpy as np
import pytest
from paper_1909_10286_b200 import binding, workloads as wl
from helpers import mk_instance

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_header_symbols_are_exported():
    hdr = open(os.path.join(ROOT, "include", "lgx.h")).read()
    declared = set(re.findall(r"\b(lgx_[a-z_]+)\s*\(", hdr))
    assert declared == set(binding.EXPORTS)
    lib = binding.load()
    for name in declared:
        assert getattr(lib, name) is not None
    assert lib.lgx_strerror(0) == b"ok"
    assert b"argument" in lib.lgx_strerror(-1)


def test_desc_layout_matches_header():
    # 8-byte alignment of every pointer/double; same field order as include/lgx.h
    hdr = open(os.path.join(ROOT, "include", "lgx.h")).read()
    body = hdr[hdr.index("typedef struct {"):hdr.index("} lgx_instance_desc;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = re.findall(r"\*?\s*([a-z_]+[a-z0-9_]*)\s*[,;]", body)
    assert names == [f[0] for f in binding.lgx_instance_desc._fields_]
    assert binding.lgx_instance_desc.hq_y.offset == 8 and binding.lgx_instance_desc.field_x.offset == 24


def _create(inst):
    import ctypes as C
    lib = binding.load()
    d, keep = binding.make_desc(inst)
    h = C.c_void_p()
    rc = lib.lgx_instance_create(C.byref(d), C.byref(h))
    if rc == 0:
        lib.lgx_instance_destroy(h)
    return rc


def toy(**kw):
    nt = kw.pop("n_tours", 1)
    return mk_instance((0, 0), [(3, 4, 25, 1), (6, 8, 40, 2)], [(6, 0, 60)], [2.0], [10.0, 10.0], nt, **kw)


def test_create_validation_codes():
    for bad in (dict(n_tours=2), dict(n_tours=0), dict(v_hu_road_kmh=0.0), dict(v_su_road_kmh=float("inf")),
                dict(su_fill_h_per_t=-1.0), dict(w_path=float("nan")), dict(flags=1)):
        assert _create(toy(**bad)) == binding.LGX_EINVAL
    i = toy(); i.su_capacity_t[0] = 0.0
    assert _create(i) == binding.LGX_EINVAL
    i = toy(); i.hu_rate_ha_per_h[0] = 1e-5        # quantises to 0
    assert _create(i) == binding.LGX_EINVAL
    i = toy(); i.field_supply_t[1] = float("nan")
    assert _create(i) == binding.LGX_EINVAL
    i = toy(); i.field_supply_t[0] = 3e6            # s_q*N_SU + sum c_q >= 2^32
    assert _create(i) == binding.LGX_ETOOBIG
    i = toy(); i.bp_demand_t[0] = 5e6               # d_q >= 2^32
    assert _create(i) == binding.LGX_ETOOBIG
    assert _create(toy(flags=binding.LGX_FLAG_DIST_COORDS | binding.LGX_FLAG_DIST_MIXED)) == binding.LGX_EINVAL
    assert _create(toy(flags=64)) == binding.LGX_EINVAL
    # a valid instance reaches the device step: OK on a GPU box, LGX_ECUDA (never a CPU
    # fallback) without one
    import torch
    rc = _create(toy())
    assert rc == (binding.LGX_OK if torch.cuda.is_available() else binding.LGX_ECUDA)


def _sized(n_f, n_b, n_hu, n_su, n_t):
    rng = np.random.default_rng(5)
    fields = [(rng.uniform(0, 50), rng.uniform(0, 50), 10.0, 1.0) for _ in range(n_f)]
    bps = [(rng.uniform(0, 50), rng.uniform(0, 50), 1.0) for _ in range(n_b)]
    return mk_instance((0, 0), fields, bps, [2.0] * n_hu, [10.0] * n_su, n_t)


def test_documented_limits_return_documented_codes():
    """include/lgx.h: counts above 65535 fields / 255 BPs, tours, HUs, SUs are LGX_EINVAL; N_B > LGX_MAX_BPS and
    N_SU > LGX_MAX_SUS are LGX_ETOOBIG (kernel limits of this build); at the limits creation reaches the device step."""
    import torch
    hdr = open(os.path.join(ROOT, "include", "lgx.h")).read()
    lim = {k: int(v) for k, v in re.findall(r"#define (LGX_MAX_[A-Z_]+)\s+(\d+)", hdr)}
    assert lim == dict(LGX_MAX_BPS=binding.LGX_MAX_BPS, LGX_MAX_SUS=binding.LGX_MAX_SUS,
                       LGX_MAX_MOVE_TOURS=binding.LGX_MAX_MOVE_TOURS, LGX_MAX_MOVE_HUS=binding.LGX_MAX_MOVE_HUS)
    assert _create(_sized(300, 256, 4, 4, 2)) == binding.LGX_EINVAL
    assert _create(_sized(300, 8, 256, 4, 2)) == binding.LGX_EINVAL
    assert _create(_sized(300, 8, 4, 256, 2)) == binding.LGX_EINVAL
    assert _create(_sized(300, binding.LGX_MAX_BPS + 1, 4, 4, 2)) == binding.LGX_ETOOBIG
    assert _create(_sized(300, 8, 4, binding.LGX_MAX_SUS + 1, 2)) == binding.LGX_ETOOBIG
    ok = binding.LGX_OK if torch.cuda.is_available() else binding.LGX_ECUDA
    assert _create(_sized(300, binding.LGX_MAX_BPS, 4, 4, 2)) == ok
    assert _create(_sized(300, 8, 4, binding.LGX_MAX_SUS, 2)) == ok


def test_null_arguments():
    import ctypes as C
    lib = binding.load()
    assert lib.lgx_instance_create(None, None) == binding.LGX_EINVAL
    assert lib.lgx_instance_destroy(None) == binding.LGX_EINVAL
    c = C.c_double(); i = C.c_uint64()
    assert lib.lgx_search(None, 0, 10, C.byref(c), C.byref(i), None) == binding.LGX_EINVAL
    assert lib.lgx_eval_batch(None, 0, None, 0, 1, None, None, None, None, None) == binding.LGX_EINVAL
