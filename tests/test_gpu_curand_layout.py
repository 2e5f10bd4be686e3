"""C2 on the box: the counter/key layout against cuRAND's own device generator ("On the box:
equality with cuRAND's device curand4 under the mapping in C2"; PAPER.md:49-51 leaves the generator open).

tests/helpers/curand_device_words.cu runs curand_init(seed, subsequence = e, offset = 4 ((u64)iteration << 32 | j >> 2))
followed by curand4() -- toolkit code only.  Its four outputs must be the Philox words of dimensions 4(j>>2)..4(j>>2)+3
of event e that (a) the oracle computes (oracle_word: the pin of C2 that the host-compiled round function cannot give,
because it never sees curand_init's subsequence / offset arithmetic) and (b) the library's kernels draw
(vegas_debug_sample, both kernel paths), bit for bit -- including events beyond 2^32, iteration indices up to what
curand_init's 64-bit offset can express (2^30 - 1) and seeds with high key bits."""
import os
import shutil
import subprocess

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle as O
import workloads as W
from conftest import ROOT


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    from paper_2002_12921_b200 import build
    build.build()
    from paper_2002_12921_b200 import binding
    return binding


@pytest.fixture(scope="module")
def curand4(tmp_path_factory):
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    if not (os.path.exists(nvcc) or shutil.which(nvcc)):
        pytest.skip("nvcc is not available on this box")
    exe = str(tmp_path_factory.mktemp("curand") / "curand_device_words")
    subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O1", "-o", exe,
                    os.path.join(ROOT, "tests", "helpers", "curand_device_words.cu")], check=True)

    def run(queries):
        """queries: (seed, e, iteration, block) -> uint32 [n, 4]"""
        text = "".join("%x %x %x %x\n" % q for q in queries)
        out = subprocess.run([exe], input=text, capture_output=True, text=True, check=True).stdout
        got = np.array([[int(v, 16) for v in ln.split()] for ln in out.strip().splitlines()], dtype=np.uint32)
        assert got.shape == (len(queries), 4)
        return got
    return run


SEEDS = (1, 3, 0xA4093822299F31D0, 0xFFFFFFFFFFFFFFFF)
# (first event, iteration).  curand_init takes the offset as ONE 64-bit count of 32-bit outputs, so 4 (iteration << 32 | block)
# must stay below 2^64: the cross-check reaches iteration indices below 2^30 (the layout itself is pinned up to 0xFFFFFFFE
# by the oracle's own tests and by test_p1_p2_words_and_bins_bit_exact); event indices use all 64 bits of the subsequence
RANGES = ((0, 0), (123_456_789, 7), ((1 << 32) - 3, 1), ((5 << 32) + 17, 0x3FFFFFFF), ((1 << 63) + 5, 0x2AAAAAAA))


def test_layout_vectors_of_the_survey(curand4):
    # SURVEY.md:445, key = (1, 0): the four printed layout vectors come out of cuRAND's device API under the C2 mapping
    got = curand4([(1, 0, 0, 0), (1, 1, 0, 0), (1, 0, 0, 1), (1, 0, 1, 0)])
    want = ["e3e80670 e50a0ebc 95f222c0 b615aa27", "07071c12 428264b6 3909104b 6da2bda2",
            "ac08141b dfc5ccbe 79c07a47 a7f66093", "833ff8dc 225c963c 232b88b3 0b334b07"]
    assert [" ".join("%08x" % v for v in row) for row in got] == want


def test_oracle_words_equal_curand_device_words(curand4):
    queries = [(s, first + k, it, blk) for s in SEEDS for first, it in RANGES for k in range(6) for blk in range(8)]
    got = curand4(queries)
    for (s, e, it, blk), row in zip(queries, got):
        assert [O.word(s, it, e, 4 * blk + i) for i in range(4)] == row.tolist(), (hex(s), e, hex(it), blk)


@pytest.mark.parametrize("path", ["auto", "generic"])
def test_library_words_equal_curand_device_words(B, curand4, path):
    dim, nb, count = 30, 16, 64                     # 8 Philox blocks, the last one with 2 dimensions
    g = B.VegasGrid(dim, nb)
    if path == "generic":
        g.set_launch(0, 0, 1, 1)
    for seed in SEEDS[1:]:
        for first, it in RANGES[:4]:                # event indices the ABI's uint64 first_event + count can address
            words = g.debug_sample(first, count, seed, it, B.VEGAS_F_CONST, 64)[0]
            ref = curand4([(seed, first + k, it, blk) for k in range(count) for blk in range(8)]).reshape(count, 32)
            assert np.array_equal(words, ref[:, :dim]), (hex(seed), first, hex(it))
    g.close()
