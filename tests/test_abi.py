"""The C-ABI shared library loads without a GPU and exports every symbol include/*.h declares;
host-only entry points behave; compute entry points fail loudly without a device (no CPU fallback)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from conftest import ROOT


@pytest.fixture(scope="module")
def B():
    from paper_2002_12921_b200 import build
    build.build()
    from paper_2002_12921_b200 import binding
    return binding


def _declared_symbols():
    text = "".join(open(os.path.join(ROOT, "include", h)).read() for h in sorted(os.listdir(os.path.join(ROOT, "include"))) if h.endswith(".h"))
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(vegas_[a-z_0-9]+)\s*\(", text)))


def test_every_declared_symbol_is_exported_and_bound(B):
    names = _declared_symbols()
    assert len(names) >= 25 and "vegas_iterate" in names and "vegas_refine" in names
    raw = C.CDLL(B.LIB_PATH)
    for n in names:
        assert hasattr(raw, n), "libvegas_b200.so does not export %s" % n
        assert n in B.SIGNATURES, "binding.py has no signature for %s" % n
    assert sorted(B.SIGNATURES) == names


def test_host_only_entry_points(B):
    assert B.vegas_version().startswith("vegas_b200")
    assert B.vegas_workspace_bytes(20, 50) > 148 * (4 + 1000) * 8
    assert B.vegas_workspace_bytes(0, 50) == 0 and B.vegas_workspace_bytes(4, 300) == 0
    assert B.lib.vegas_debug_scratch_bytes(4, 100) >= 100 * 4 * 16 + 800
    assert "invalid" in B.vegas_strerror(B.VEGAS_EINVAL) and B.vegas_strerror(0) == "ok"
    # C9 closed forms through the product's own combine
    I, s, c = B.vegas_combine([1.0, 3.0], [0.5, 0.5])
    assert I == 2.0 and s == pytest.approx(0.5 / np.sqrt(2)) and c == pytest.approx(8.0)
    assert B.vegas_combine([1.0, 0.999], [0.0, 1e-3]) == (0.9995, 0.0, 0.0)
    assert B.vegas_combine([9.0, 1.0, 3.0], [1e-3, 0.5, 0.5], n_skip=1)[0] == 2.0
    I, s, c = B.vegas_combine([1.0, 2.0], [1e-200, 2e-200])      # no overflow of 1/sigma^2
    assert I == pytest.approx(1.2) and s == pytest.approx(1e-200 / np.sqrt(1.25))
    with pytest.raises(B.VegasError):
        B.vegas_combine([1.0], [1.0], n_skip=1)
    # an iteration that ended in VEGAS_ENUMERIC (non-finite I or sigma) is not averaged away: ENUMERIC, NaN outputs
    I, s, c = C.c_double(7.0), C.c_double(7.0), C.c_double(7.0)
    for Ik, sk in (([1.0, 2.0], [0.1, float("nan")]), ([1.0, float("inf")], [0.1, 0.1]), ([1.0, 2.0], [0.1, -1.0])):
        Ik, sk = np.array(Ik), np.array(sk)
        f64p = C.POINTER(C.c_double)
        rc = B.lib.vegas_combine(2, 0, Ik.ctypes.data_as(f64p), sk.ctypes.data_as(f64p), C.byref(I), C.byref(s), C.byref(c))
        assert rc == B.VEGAS_ENUMERIC and np.isnan(I.value) and np.isnan(s.value) and np.isnan(c.value)


def test_null_arguments_are_rejected(B):
    assert B.lib.vegas_create(4, 50, None, 0, C.byref(C.c_void_p())) == B.VEGAS_EINVAL
    assert B.lib.vegas_destroy(None) == B.VEGAS_EINVAL
    assert B.lib.vegas_refine(None, None, 1.5, None) == B.VEGAS_EINVAL
    assert B.lib.vegas_launch_count(None) == 0


def test_no_cpu_fallback(B):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(B.VegasError) as e:
        B.VegasGrid(4, 50)
    assert e.value.code == B.VEGAS_ECUDA
    # straight through the C ABI with a fake workspace pointer: the CUDA runtime refuses
    h = C.c_void_p()
    assert B.lib.vegas_create(4, 50, C.c_void_p(256 * 4096), B.vegas_workspace_bytes(4, 50), C.byref(h)) \
        == B.VEGAS_ECUDA


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2002_12921_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "vegas_oracle" not in text, f
