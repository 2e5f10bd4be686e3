"""B200-native Vegas iteration library (hot path of VegasFlow, arXiv 2002.12921).

    from paper_2002_12921_b200 import binding          # ctypes face of include/vegas.h (needs the built .so)

The product is libvegas_b200.so (csrc/, C ABI in include/vegas.h); `binding` marshals arguments.
Nothing here imports the CPU oracle (oracle/), which is test infrastructure.  The seeded synthetic inputs that tests,
bench.py and smoke() hand to both sides live in the top-level module `workloads`, outside this package.
"""
__all__ = ["binding", "build"]
