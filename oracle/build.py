"""Build oracle/liblgo.so from oracle/lgo.c (plain C, gcc).  ORACLE = test infrastructure.

Flags: -O2 -ffp-contract=off (no FMA contraction, no -ffast-math) so every FP64
operation is rounded exactly where lgo.c writes it.

LGO_SANITIZE=1 in the environment builds oracle/liblgo_san.so with -fsanitize=address,undefined instead (run the
CPU tests with LD_PRELOAD=$(gcc -print-file-name=libasan.so); profiles/r02_sanitizers.md has the command).
"""
from __future__ import annotations
import os, subprocess, sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "lgo.c")
HDR = os.path.join(HERE, "lgo.h")
SANITIZE = os.environ.get("LGO_SANITIZE", "") not in ("", "0")
LIB = os.path.join(HERE, "liblgo_san.so" if SANITIZE else "liblgo.so")


def build(force: bool = False) -> str:
    stale = (not os.path.exists(LIB) or
             os.path.getmtime(LIB) < max(os.path.getmtime(SRC), os.path.getmtime(HDR)))
    if force or stale:
        cmd = ["gcc", "-std=c11", "-O2", "-ffp-contract=off", "-fno-fast-math", "-Wall", "-Wextra",
               "-fPIC", "-shared", "-o", LIB, SRC, "-lm"]
        if SANITIZE:
            cmd[3:3] = ["-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined"]
        subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
