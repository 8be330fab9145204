"""The CUDA sources of the sampling path compiled for the host (tests/emu: one lane, heap blocks of the exact size for
every device buffer and every launch's shared memory) against the oracle, under AddressSanitizer + UBSan when gcc's
libasan is there: the index arithmetic, the shared-memory row layout, the queue records and the right-aligned
permutation words are checked on a CPU on every config, the three distance modes and the degenerate cases.
(It cannot see races between threads; compute-sanitizer is closed on the GPU pool, see profiles/r02_sanitizers.md.)"""
import os, subprocess, sys
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _libasan():
    try:
        p = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    except OSError:
        return None
    return p if p and os.path.isabs(p) and os.path.exists(p) else None


def test_sampling_kernels_on_host_match_the_oracle_under_sanitizers():
    env = dict(os.environ)
    asan = _libasan()
    if asan:
        env.update(LGX_HOST_SANITIZE="1", LD_PRELOAD=asan, ASAN_OPTIONS="detect_leaks=0", UBSAN_OPTIONS="print_stacktrace=1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "tests", "emu", "host_kernels.py")], env=env, capture_output=True, text=True, timeout=1500)
    tail = (r.stdout + r.stderr)[-4000:]
    assert r.returncode == 0 and "ALL OK" in r.stdout, tail
    assert "AddressSanitizer" not in r.stderr and "runtime error" not in r.stderr, tail
