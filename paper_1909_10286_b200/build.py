"""Build paper_1909_10286_b200/liblgx.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

`-fmad=false` and `-Xcompiler -ffp-contract=off`: every FP64 operation of the cost path is
rounded once, in source order, on device and host (bit-identical costs).
"""
from __future__ import annotations
import os, subprocess, sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
ROOT = os.path.dirname(HERE)
LIB = os.path.join(HERE, "liblgx.so")
SOURCES = [os.path.join(CSRC, "lgx_api.cu")]
DEPS = SOURCES + [os.path.join(CSRC, "lgx_kernels.cuh"), os.path.join(CSRC, "lgx_moves.cuh"), os.path.join(CSRC, "lgx_image.h"),
                  os.path.join(ROOT, "include", "lgx.h")]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-fmad=false", "-Xcompiler", "-fPIC,-ffp-contract=off,-O2", "-shared",
              "-Xptxas", "-v"]


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(p) > t for p in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or is_stale():
        nvcc = os.environ.get("NVCC", "nvcc")
        cmd = [nvcc] + NVCC_FLAGS + ["-o", LIB] + SOURCES
        r = subprocess.run(cmd, capture_output=True, text=True)
        log = os.path.join(HERE, "build.log")
        with open(log, "w") as fh:
            fh.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
        if verbose:
            print(r.stdout + r.stderr)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed:\n" + r.stderr[-4000:])
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
