"""Pins for the oracle's RNG (readings C1, C2, C3 of DESIGN.md) -- no GPU."""
import os
import shutil
import subprocess
from fractions import Fraction

import numpy as np
import pytest

import oracle as O
import workloads as W

from conftest import GOLDEN, ROOT


def _lines(name):
    with open(os.path.join(GOLDEN, name)) as fh:
        return [ln.split() for ln in fh if ln.strip() and not ln.startswith("#")]


def test_c1_known_answer_vectors():
    rows = _lines("philox4x32_10_kat.txt")
    assert len(rows) == 3
    for t in rows:
        ctr = [int(v, 16) for v in t[0:4]]
        key = [int(v, 16) for v in t[4:6]]
        want = [int(v, 16) for v in t[6:10]]
        assert O.philox4x32_10(ctr, key).tolist() == want


def test_c2_layout_vectors():
    for t in _lines("philox_layout_c2.txt"):
        seed, it, ev, blk = (int(v) for v in t[0:4])
        want = [int(v, 16) for v in t[4:8]]
        got = [O.word(seed, it, ev, 4 * blk + i) for i in range(4)]
        assert got == want


def test_c2_high_bits_reach_counter_and_key():
    # event >= 2^32 goes to counter word 3, seed >= 2^32 to key word 1
    e = (7 << 32) | 5
    s = (9 << 32) | 3
    for j in (0, 5, 19):
        blk = O.philox4x32_10([j >> 2, 11, 5, 7], [3, 9])
        assert O.word(s, 11, e, j) == int(blk[j & 3])
    assert O.word(s, 11, e, 0) != O.word(s, 11, 5, 0)
    assert O.word(s, 11, e, 0) != O.word(3, 11, e, 0)


def test_c1_against_independent_python_integers():
    # workloads.parameter_uniforms is a separate restatement in Python ints (C10)
    for seed in (4, 5, (1 << 40) + 17):
        u = W.parameter_uniforms(seed, 23)
        for q in range(23):
            w = O.word(seed, 0xFFFFFFFF, 0, q)
            assert u[q] == (w + 0.5) / 4294967296.0


def test_c1_against_cuda_toolkit_header(tmp_path):
    """Library pin: curand_Philox4x32_10 from the toolkit header, compiled for the host."""
    inc = "/usr/local/cuda/include"
    if not (shutil.which("g++") and os.path.exists(os.path.join(inc, "curand_philox4x32_x.h"))):
        pytest.skip("g++ or the CUDA toolkit header is not available")
    exe = str(tmp_path / "curand_host_philox")
    subprocess.run(["g++", "-O1", "-I", inc, "-o", exe,
                    os.path.join(ROOT, "tests", "helpers", "curand_host_philox.cpp")], check=True)
    rng = np.random.default_rng(20021292)
    vec = rng.integers(0, 2**32, size=(2000, 6), dtype=np.uint64)
    vec[0] = 0
    vec[1] = 0xFFFFFFFF
    text = "\n".join(" ".join("%08x" % v for v in row) for row in vec) + "\n"
    out = subprocess.run([exe], input=text, capture_output=True, text=True, check=True).stdout
    got = [[int(v, 16) for v in ln.split()] for ln in out.strip().splitlines()]
    assert len(got) == len(vec)
    for row, g in zip(vec, got):
        assert O.philox4x32_10(row[:4], row[4:]).tolist() == g


@pytest.mark.parametrize("nb", [2, 3, 50, 100, 128, 255])
def test_c3_split_exact(nb):
    rng = np.random.default_rng(nb)
    words = [0, 1, 2**32 - 1, 2**31, 2**31 - 1] + rng.integers(0, 2**32, size=300).tolist()
    # the first and last word of every bin: ceil(b*2^32/nb) starts bin b
    for b in range(1, nb):
        start = -((-b * 2**32) // nb)
        words += [start - 1, start]
    for w in words:
        b, r = O.split(w, nb)
        P = w * nb
        assert b == P >> 32 and 0 <= b < nb
        assert Fraction(r) == Fraction(2 * (P & 0xFFFFFFFF) + 1, 2**33)   # exact in fp64
        assert 0.0 < r < 1.0
    for b in range(1, nb):
        start = -((-b * 2**32) // nb)
        assert O.split(start - 1, nb)[0] == b - 1 and O.split(start, nb)[0] == b


def test_c3_bin_populations_closed_form():
    # number of 32-bit words landing in bin b is ceil((b+1)2^32/nb) - ceil(b 2^32/nb):
    # floor(2^32/nb) or that + 1 (85899345/85899346 for nb=50).
    for nb, lo in ((50, 85899345), (100, 42949672)):
        counts = {-((-(b + 1) * 2**32) // nb) - (-((-b * 2**32) // nb)) for b in range(nb)}
        assert counts == {lo, lo + 1}
        assert sum(-((-(b + 1) * 2**32) // nb) - (-((-b * 2**32) // nb)) for b in range(nb)) == 2**32


def test_c3_mean_of_r_over_a_bin_is_half():
    # r runs over a midpoint lattice: averaging r over all words of one bin gives 1/2 up to
    # the lattice granularity (nb / 2^32)
    nb = 50
    b = 17
    start = -((-b * 2**32) // nb)
    stop = -((-(b + 1) * 2**32) // nb)
    step = 9973
    ws = range(start, stop, step)
    rs = [O.split(w, nb)[1] for w in ws]
    assert all(O.split(w, nb)[0] == b for w in (start, stop - 1))
    assert abs(np.mean(rs) - 0.5) < 1e-3
    # exact statement: r(word) is affine in word inside a bin with slope nb/2^32
    r0, r1 = O.split(start, nb)[1], O.split(start + 1, nb)[1]
    assert Fraction(r1) - Fraction(r0) == Fraction(nb, 2**32)
