"""The oracle's pins once more against a build of oracle/vegas_oracle.c under -fsanitize=address,undefined
(SURVEY.md section 5).  The oracle is what every parity claim rests on: an out-of-bounds read of a grid row or a
signed overflow in an index would not necessarily change a digit that a pin looks at.  Every sanitizer report is fatal
(-fno-sanitize-recover), so the inner pytest run fails on the first one.  CPU only; runs the Philox / layout pins
and the method pins (sample, accumulate, estimate, refine, combine, integrate) in a child process, because the
sanitizer runtime has to be loaded before the interpreter starts."""
import os
import shutil
import subprocess
import sys

import pytest

from conftest import ROOT


def test_oracle_pins_under_address_and_undefined_behaviour_sanitizers():
    if not shutil.which("gcc"):
        pytest.skip("gcc is not available")
    asan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    if not os.path.isabs(asan) or not os.path.exists(asan):
        pytest.skip("the address sanitizer runtime is not installed")
    env = dict(os.environ, VEGAS_ORACLE_SANITIZE="1", LD_PRELOAD=os.path.realpath(asan),
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=0:halt_on_error=1", UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1")
    files = [os.path.join(ROOT, "tests", f) for f in ("test_oracle_philox.py", "test_oracle_method.py")]
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider"] + files,
                       env=env, cwd=ROOT, capture_output=True, text=True, timeout=1500)
    tail = (r.stdout + r.stderr)[-3000:]
    assert r.returncode == 0, tail
    assert "passed" in r.stdout and "failed" not in r.stdout, tail
    assert "runtime error" not in tail and "AddressSanitizer" not in tail, tail
    assert os.path.exists(os.path.join(ROOT, "oracle", "libvegas_oracle_san.so"))      # the child really loaded that build
