"""Build the CPU oracle (oracle/vegas_oracle.c) into oracle/libvegas_oracle.so with gcc.

TEST INFRASTRUCTURE ONLY -- see the header of vegas_oracle.c.  Called by tests/conftest.py,
__graft_entry__.build() and bench.py's cpu_baseline / --impl reference legs.
-ffp-contract=off: x = X[b] + delta*r is evaluated as written (no FMA contraction), so the
oracle's digits do not depend on the host's instruction set.
"""
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(_HERE, "vegas_oracle.c")
# VEGAS_ORACLE_SANITIZE=1: the same source under -fsanitize=address,undefined as a library of its own;
# every report is fatal.  The process that loads it must have the sanitizer runtime loaded first
# (LD_PRELOAD=$(gcc -print-file-name=libasan.so)); tests/test_oracle_sanitized.py runs the oracle's pins that way.
SANITIZE = os.environ.get("VEGAS_ORACLE_SANITIZE", "") not in ("", "0")
LIB = os.path.join(_HERE, "libvegas_oracle_san.so" if SANITIZE else "libvegas_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= max(os.path.getmtime(SRC), os.path.getmtime(os.path.abspath(__file__)))):
        return LIB
    tmp = LIB + ".tmp%d" % os.getpid()
    flags = ["-O2"] if not SANITIZE else ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=all",
                                          "-fno-omit-frame-pointer"]
    cmd = ["gcc"] + flags + ["-std=c99", "-ffp-contract=off", "-fPIC", "-shared", "-Wall", "-Wextra",
                             "-o", tmp, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
