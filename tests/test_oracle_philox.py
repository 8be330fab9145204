"""Pins for the oracle's random stream (S1).

1. Published Philox4x32-10 known-answer vectors (tests/golden/philox4x32_10_kat.txt).
2. NVIDIA's cuRAND header routine curand_Philox4x32_10, compiled for the HOST with nvcc
   (a library routine the oracle does not use), on random counters/keys.
3. The counter layout (id_lo, id_hi, stream, block) and word selection d%4 of block d//4.
"""
import os, shutil, subprocess, textwrap
import numpy as np
import pytest
from oracle import lgo

HERE = os.path.dirname(os.path.abspath(__file__))


def test_known_answer_vectors():
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "philox4x32_10_kat.txt"))
            if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        out = lgo.philox4x32_10(v[0:4], v[4:6])
        assert [int(x) for x in out] == v[6:10]


def test_draw_layout():
    seed, id_ = 0x0123456789ABCDEF, 0xFEDCBA9876543210
    key = [seed & 0xFFFFFFFF, seed >> 32]
    for stream in (0, 3, 4):
        for d in (0, 1, 5, 7, 130):
            blk = lgo.philox4x32_10([id_ & 0xFFFFFFFF, id_ >> 32, stream, d // 4], key)
            assert lgo.draw(seed, id_, stream, d) == int(blk[d % 4])


@pytest.mark.skipif(shutil.which("nvcc") is None, reason="nvcc not found")
def test_against_curand_header(tmp_path):
    src = tmp_path / "k.cu"
    src.write_text(textwrap.dedent(r'''
        #include <cstdio>
        #include <cstdlib>
        #include <cuda_runtime.h>
        #define QUALIFIERS static inline __host__ __device__
        #include <curand_philox4x32_x.h>
        int main(int argc, char** argv) {
          unsigned v[6];
          while (scanf("%x %x %x %x %x %x", v, v+1, v+2, v+3, v+4, v+5) == 6) {
            uint4 c = make_uint4(v[0], v[1], v[2], v[3]); uint2 k = make_uint2(v[4], v[5]);
            uint4 r = curand_Philox4x32_10(c, k);
            printf("%08x %08x %08x %08x\n", r.x, r.y, r.z, r.w);
          }
          return 0;
        }'''))
    exe = tmp_path / "k"
    r = subprocess.run(["nvcc", "-O1", "-o", str(exe), str(src)], capture_output=True, text=True)
    if r.returncode != 0:
        pytest.skip("cuRAND header does not compile for the host here: " + r.stderr[-300:])
    rng = np.random.default_rng(7)
    vecs = rng.integers(0, 2**32, (64, 6), dtype=np.uint64)
    inp = "\n".join(" ".join(f"{int(x):08x}" for x in row) for row in vecs) + "\n"
    out = subprocess.run([str(exe)], input=inp, capture_output=True, text=True, check=True).stdout.split("\n")
    for row, line in zip(vecs, out):
        want = [int(x, 16) for x in line.split()]
        got = [int(x) for x in lgo.philox4x32_10(row[:4], row[4:6])]
        assert got == want
