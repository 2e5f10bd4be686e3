"""Build libvegas_b200.so (the C-ABI library of include/vegas.h) in-tree with nvcc for sm_100a.

nvcc cross-compiles without a GPU.  Translation units are compiled in parallel: the generic kernels,
the host driver, and one unit per (integrand, precision) pair of the fast path (vegas_rot_inst.cu with
-DROT_FID / -DROT_FP, 32 dimension instantiations each).  The shared object and the objects under
build/ are git-ignored; the .so travels with the tree to the GPU box.
"""
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
OBJ_DIR = os.path.join(_HERE, "build")
LIB = os.path.join(_HERE, "libvegas_b200.so")
HEADERS = ["vegas_kernels.h", "vegas_device.cuh", "vegas_iterate_rot.cuh", os.path.join("..", "..", "include", "vegas.h")]
# (integrand id, precision) pairs served by the fast path: CONST, GAUSS in both precisions, GENZ and BW_POLY in fp64
ROT_VARIANTS = [(0, 64), (0, 32), (1, 64), (1, 32), (2, 64), (3, 64)]
UNITS = [("vegas_kernels", "vegas_kernels.cu", []), ("vegas_api", "vegas_api.cu", [])] + \
        [("vegas_rot_%d_%d" % (f, p), "vegas_rot_inst.cu", ["-DROT_FID=%d" % f, "-DROT_FP=%d" % p])
         for f, p in ROT_VARIANTS]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden"]


def _newest_source() -> float:
    files = [os.path.join(CSRC, h) for h in HEADERS] + [os.path.join(CSRC, u[1]) for u in UNITS] \
        + [os.path.abspath(__file__)]
    return max(os.path.getmtime(f) for f in files)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= _newest_source():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ_DIR, exist_ok=True)

    def compile_unit(unit):
        name, src, defs = unit
        obj = os.path.join(OBJ_DIR, name + ".o")
        cmd = [nvcc] + NVCC_FLAGS + os.environ.get("VEGAS_NVCC_EXTRA", "").split() + (["-Xptxas", "-v"] if verbose else []) + defs + ["-c", os.path.join(CSRC, src), "-o", obj]
        subprocess.run(cmd, check=True)
        return obj

    with ThreadPoolExecutor(max_workers=min(len(UNITS), os.cpu_count() or 4)) as ex:
        objs = list(ex.map(compile_unit, UNITS))
    tmp = LIB + ".tmp%d" % os.getpid()
    subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "static", "-o", tmp] + objs,
                   check=True)
    os.replace(tmp, LIB)
    return LIB


def build_ubench() -> str:
    """The step-0 pipe microbenchmark (csrc/ubench_pipes.cu), a standalone binary; not part of the library."""
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    out = os.path.join(_HERE, "ubench_pipes.bin")
    subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
                    "-cudart", "static", "-o", out, os.path.join(CSRC, "ubench_pipes.cu")], check=True)
    return out


if __name__ == "__main__":
    import sys
    if "--ubench" in sys.argv:
        print(build_ubench())
    else:
        print(build(force=True, verbose="-v" in sys.argv))
