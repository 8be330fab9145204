"""Build paper_1909_10286_b200/liblgx.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

The kernel templates are instantiated in translation units of their own (csrc/lgx_inst_*.cu, see
csrc/lgx_dispatch.h) that are compiled in parallel, then linked with the host code of csrc/lgx_api.cu.

`-fmad=false` and `-Xcompiler -ffp-contract=off`: every FP64 operation of the cost path is
rounded once, in source order, on device and host (bit-identical costs).
"""
from __future__ import annotations
import os, subprocess, sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
ROOT = os.path.dirname(HERE)
LIB = os.path.join(HERE, "liblgx.so")
OBJDIR = os.path.join(HERE, "build")
# (object name, source, extra defines)
UNITS = [("api", "lgx_api.cu", []),
         ("pipes", "lgx_pipes.cu", []),
         ("decode", "lgx_inst_decode.cu", []),
         ("walk0", "lgx_inst_walk.cu", ["-DLGX_DM=0"]),
         ("walk1", "lgx_inst_walk.cu", ["-DLGX_DM=1"]),
         ("walk2", "lgx_inst_walk.cu", ["-DLGX_DM=2"]),
         ("moves1", "lgx_inst_moves.cu", ["-DLGX_MASKW=1"]),
         ("moves2", "lgx_inst_moves.cu", ["-DLGX_MASKW=2"])]
DEPS = [os.path.join(CSRC, f) for f in ("lgx_api.cu", "lgx_pipes.cu", "lgx_inst_decode.cu", "lgx_inst_walk.cu", "lgx_inst_moves.cu",
                                        "lgx_dispatch.h", "lgx_kernels.cuh", "lgx_moves.cuh", "lgx_image.h")] + \
       [os.path.join(ROOT, "include", "lgx.h")]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-fmad=false", "-Xcompiler", "-fPIC,-ffp-contract=off,-O2", "-Xptxas", "-v"]


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(p) > t for p in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or is_stale():
        nvcc = os.environ.get("NVCC", "nvcc")
        os.makedirs(OBJDIR, exist_ok=True)

        def compile_unit(u):
            name, src, defs = u
            obj = os.path.join(OBJDIR, name + ".o")
            cmd = [nvcc] + NVCC_FLAGS + defs + ["-c", os.path.join(CSRC, src), "-o", obj]
            r = subprocess.run(cmd, capture_output=True, text=True)
            return obj, cmd, r

        with ThreadPoolExecutor(max_workers=min(len(UNITS), os.cpu_count() or 1)) as ex:
            results = list(ex.map(compile_unit, UNITS))
        log = [" ".join(cmd) + "\n" + r.stdout + r.stderr for _, cmd, r in results]
        for _, cmd, r in results:
            if r.returncode != 0:
                raise RuntimeError("nvcc failed: " + " ".join(cmd) + "\n" + r.stderr[-4000:])
        link = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB] + [o for o, _, _ in results]
        r = subprocess.run(link, capture_output=True, text=True)
        log.append(" ".join(link) + "\n" + r.stdout + r.stderr)
        with open(os.path.join(HERE, "build.log"), "w") as fh:
            fh.write("\n".join(log))
        if verbose:
            print("\n".join(log))
        if r.returncode != 0:
            raise RuntimeError("link failed:\n" + r.stderr[-4000:])
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
