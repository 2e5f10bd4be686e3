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
LIB = os.path.join(_HERE, "libvegas_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    tmp = LIB + ".tmp%d" % os.getpid()
    cmd = ["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fPIC", "-shared", "-Wall", "-Wextra",
           "-o", tmp, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
