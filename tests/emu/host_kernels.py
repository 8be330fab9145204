"""TEST INFRASTRUCTURE: the CUDA sources of the sampling path (lgx_decode_cut, lgx_walk_finish and the host code of
lgx_api.cu) compiled for the HOST through tests/emu/cuda_host_shim.h — one lane, every "device" buffer and every
launch's shared memory a heap block of the exact size — and driven through the same C ABI.  With
LGX_HOST_SANITIZE=1 the build uses -fsanitize=address,undefined (run python with LD_PRELOAD=libasan.so).
Used by tests/test_kernels_on_host.py; never imported by the package, bench.py or smoke()."""
from __future__ import annotations
import ctypes as C, os, subprocess, sys
from concurrent.futures import ThreadPoolExecutor
import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
CSRC = os.path.join(ROOT, "paper_1909_10286_b200", "csrc")
SANITIZE = os.environ.get("LGX_HOST_SANITIZE", "") not in ("", "0")
OBJ = os.path.join(HERE, "build", "san" if SANITIZE else "plain")
LIB = os.path.join(OBJ, "liblgx_host.so")
UNITS = [("api", os.path.join(CSRC, "lgx_api.cu"), []), ("decode", os.path.join(CSRC, "lgx_inst_decode.cu"), []),
         ("walk0", os.path.join(CSRC, "lgx_inst_walk.cu"), ["-DLGX_DM=0"]), ("walk1", os.path.join(CSRC, "lgx_inst_walk.cu"), ["-DLGX_DM=1"]),
         ("walk2", os.path.join(CSRC, "lgx_inst_walk.cu"), ["-DLGX_DM=2"]),
         ("moves1", os.path.join(CSRC, "lgx_inst_moves.cu"), ["-DLGX_MASKW=1"]), ("moves2", os.path.join(CSRC, "lgx_inst_moves.cu"), ["-DLGX_MASKW=2"]),
         ("params", os.path.join(HERE, "emu_params.cu"), [])]
FLAGS = ["-O1", "-g", "-std=c++17", "-ffp-contract=off", "-fPIC", "-fno-strict-aliasing", "-Wno-attributes", "-Wno-unused",
         "-I", os.path.join(HERE, "fake"), "-include", os.path.join(HERE, "cuda_host_shim.h"), "-x", "c++"]
SAN_FLAGS = ["-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"]


def build(force: bool = False) -> str:
    deps = [u[1] for u in UNITS] + [os.path.join(CSRC, f) for f in ("lgx_kernels.cuh", "lgx_moves.cuh", "lgx_image.h", "lgx_dispatch.h")] + \
           [os.path.join(HERE, "cuda_host_shim.h"), os.path.join(ROOT, "include", "lgx.h")]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(d) <= os.path.getmtime(LIB) for d in deps):
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    extra = SAN_FLAGS if SANITIZE else []

    def cc(u):
        obj = os.path.join(OBJ, u[0] + ".o")
        r = subprocess.run(["g++"] + FLAGS + extra + u[2] + ["-c", u[1], "-o", obj], capture_output=True, text=True)
        if r.returncode:
            raise RuntimeError("host build of %s failed:\n%s" % (u[1], r.stderr[-3000:]))
        return obj

    with ThreadPoolExecutor(max_workers=os.cpu_count() or 1) as ex:
        objs = list(ex.map(cc, UNITS))
    subprocess.run(["g++", "-shared", "-o", LIB] + extra + objs, check=True)
    return LIB


class HostKernels:
    """One lgx instance inside the host build (the C ABI of include/lgx.h, host pointers everywhere)."""
    _lib = None

    def __init__(self, inst):
        from paper_1909_10286_b200 import binding as B      # argument marshalling only; the CUDA library is not loaded
        if HostKernels._lib is None:
            lib = C.CDLL(build())
            vp, u64 = C.c_void_p, C.c_uint64
            lib.lgx_instance_create.argtypes = [C.POINTER(B.lgx_instance_desc), C.POINTER(vp)]
            lib.lgx_instance_destroy.argtypes = [vp]
            lib.lgx_eval_batch.argtypes = [vp, u64, vp, u64, u64, vp, vp, vp, vp, vp]
            lib.lgx_search_range.argtypes = [vp, u64, u64, u64, C.POINTER(C.c_double), C.POINTER(u64), vp]
            lib.lgx_decode_batch.argtypes = [vp, u64, vp, u64, u64] + [vp] * 7 + [vp]
            lib.lgx_instance_query.argtypes = [vp, C.c_int, C.POINTER(C.c_int64)]
            lib.lgx_instance_set_option.argtypes = [vp, C.c_int, C.c_int64]
            HostKernels._lib = lib
        self.lib = HostKernels._lib
        d, self.keep = B.make_desc(inst)
        h = C.c_void_p()
        rc = self.lib.lgx_instance_create(C.byref(d), C.byref(h))
        if rc:
            raise RuntimeError("lgx_instance_create (host build): %d" % rc)
        self.h = h
        self.n_f, self.n_b, self.n_hu, self.n_su = inst.n_fields, inst.n_bps, inst.n_hu, inst.n_su

    def close(self):
        if self.h:
            self.lib.lgx_instance_destroy(self.h); self.h = None

    def query(self, what):
        v = C.c_int64(); assert self.lib.lgx_instance_query(self.h, what, C.byref(v)) == 0; return v.value

    def set_option(self, key, value):
        return self.lib.lgx_instance_set_option(self.h, key, value)

    def eval_batch(self, seed, ids=None, first_id=0, n=None):
        if ids is not None:
            ids = np.ascontiguousarray(ids, np.uint64); n = len(ids)
        o = (np.zeros(n), np.zeros(n), np.zeros(n), np.zeros(n, np.uint8))
        rc = self.lib.lgx_eval_batch(self.h, seed, ids.ctypes.data if ids is not None else None, first_id, n, *[x.ctypes.data for x in o], None)
        assert rc == 0, rc
        return o

    def decode_batch(self, seed, ids=None, first_id=0, n=None):
        if ids is not None:
            ids = np.ascontiguousarray(ids, np.uint64); n = len(ids)
        o = dict(bp_tour=np.zeros((n, self.n_b), np.uint8), bp_pos=np.zeros((n, self.n_b), np.uint8),
                 field_bp=np.zeros((n, self.n_f), np.uint16), field_pos=np.zeros((n, self.n_f), np.uint16),
                 hu_tour=np.zeros((n, self.n_hu), np.uint8), su_tour_init=np.zeros((n, self.n_su), np.uint8),
                 su_tour_final=np.zeros((n, self.n_su), np.uint8))
        keys = ("bp_tour", "bp_pos", "field_bp", "field_pos", "hu_tour", "su_tour_init", "su_tour_final")
        rc = self.lib.lgx_decode_batch(self.h, seed, ids.ctypes.data if ids is not None else None, first_id, n, *[o[k].ctypes.data for k in keys], None)
        assert rc == 0, rc
        return o

    def search(self, seed, n, first_id=0):
        c = C.c_double(); i = C.c_uint64()
        rc = self.lib.lgx_search_range(self.h, seed, first_id, n, C.byref(c), C.byref(i), None)
        assert rc == 0, rc
        return c.value, i.value


def check(inst, n, label, seed=None, ids=None, first=0, decode=True, search=True):
    """Host build against the oracle: eval_batch element by element (bit-equal), decoded plans, argmin."""
    from oracle import lgo
    seed = inst.seed if seed is None else seed
    o, g = lgo.Oracle(inst), HostKernels(inst)
    g.set_option(4, 10)                                   # chunks of 1024 candidates: several chunks per call
    want = o.eval_batch(seed, ids=ids, first_id=first, n=n)
    got = g.eval_batch(seed, ids=ids, first_id=first, n=n)
    ok = all(np.array_equal(got[k], want[k]) for k in range(4))
    msg = f"{label}: eval {'OK' if ok else 'FAIL'} feasible={want[3].mean():.3f} mode={g.query(4)}"
    if decode:
        nd = min(n, 512)
        wd = o.decode_batch(seed, ids=None if ids is None else ids[:nd], first_id=first, n=nd)
        gd = g.decode_batch(seed, ids=None if ids is None else ids[:nd], first_id=first, n=nd)
        for k in wd:
            if not np.array_equal(gd[k], wd[k]):
                msg += f" DECODE {k} FAIL"; ok = False
    if search and ids is None:
        if o.search(seed, n, first_id=first) != g.search(seed, n, first_id=first):
            msg += " SEARCH FAIL"; ok = False
    print(msg, flush=True)
    g.close(); o.close()
    return ok


def main():
    """All configs (three distance modes each) and the degenerate cases of tests/test_gpu_parity.py::test_edge_cases."""
    sys.path.insert(0, ROOT); sys.path.insert(0, os.path.join(ROOT, "tests"))
    from dataclasses import replace
    from paper_1909_10286_b200 import workloads as wl
    from helpers import mk_instance
    N = {"toy": 8192, "small": 4096, "medium": 4096, "large": 1500, "sweep": 700, "paper_scale": 200}
    ok = True
    for nm in N:
        inst = wl.make(nm)
        ok &= check(inst, N[nm], nm)
        ok &= check(inst, N[nm] // 4, nm + "/sampled", ids=wl.sample_ids(inst.budget, N[nm] // 4))
        for fl, tag in ((16, "coords"), (32, "mixed")):
            ok &= check(replace(inst, flags=fl), N[nm] // 4, f"{nm}/{tag}", decode=False)
    a = mk_instance((0, 0), [(3, 4, 25, 1), (6, 8, 40, 2)], [(6, 0, 60)], [2.0], [10.0, 10.0], 1); a.seed = 0
    ok &= check(a, 100, "handA", first=7)
    b = mk_instance((0, 0), [(3, 4, 25, 1), (6, 8, 40, 2)], [(6, 0, 66)], [2.0], [10.0, 10.0], 1); b.seed = 0
    ok &= check(b, 100, "handA-infeasible", first=5)
    for thresh in (0, 0xFFFFFFFF, 0x40000000):
        z = wl.make("small"); z.bp_demand_t = z.bp_demand_t.copy(); z.bp_demand_t[[1, 3]] = 0.0; z.extra_field_thresh = thresh
        ok &= check(z, 2048, f"small/zero-demand/thresh={thresh:#x}", seed=1)
    for nm in ("small", "medium", "sweep"):
        for thresh in (0xC0000000, 0xFFFFFFFF, 0):
            z = wl.make(nm); z.extra_field_thresh = thresh
            ok &= check(z, 400, f"{nm}/thresh={thresh:#x}", seed=3, decode=(nm != "sweep"))
    for nt in (1, 5):
        z = wl.make("small"); z.n_tours = nt
        if nt == 5:
            z.hu_rate_ha_per_h = z.hu_rate_ha_per_h[:5].copy(); z.su_capacity_t = z.su_capacity_t[:5].copy()
        ok &= check(z, 1024, f"small/nt={nt}", seed=2)
    for nf in (253, 254, 255, 256, 257, 258, 259):        # both element widths around the 8/16-bit switch, every padding
        z = wl.make("sweep")
        z = replace(z, field_xy=z.field_xy[:nf].copy(), field_supply_t=z.field_supply_t[:nf].copy(), field_area_ha=z.field_area_ha[:nf].copy(),
                    bp_demand_t=z.bp_demand_t * (z.field_supply_t[:nf].sum() / z.field_supply_t.sum()))
        ok &= check(z, 128, f"sweep/nf={nf}", seed=5)
    for nf in (510, 511, 512, 513, 514, 515, 1022, 1023, 1024, 1025):     # 16-bit field ids around 512 and 1024, every padding and tail length of the blocked Fisher-Yates steps
        z = wl.make("paper_scale")
        z = replace(z, field_xy=z.field_xy[:nf].copy(), field_supply_t=z.field_supply_t[:nf].copy(), field_area_ha=z.field_area_ha[:nf].copy(),
                    bp_demand_t=z.bp_demand_t * (0.9 * z.field_supply_t[:nf].sum() / z.bp_demand_t.sum()))
        ok &= check(z, 96, f"paper_scale/nf={nf}", seed=6)
    inst = wl.make("small")
    ids = np.array([(1 << 40) + 3, (1 << 63) + 11, 2**64 - 1], dtype=np.uint64)
    ok &= check(inst, 3, "small/bigids", seed=0xDEADBEEFCAFEF00D, ids=ids)
    print("ALL OK" if ok else "FAILURES")
    return 0 if ok else 1


if __name__ == "__main__":
    sys.path.insert(0, ROOT)
    sys.exit(main())
