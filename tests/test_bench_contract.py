"""Host-side pieces of bench.py that need no GPU: the per-event instruction counts the roofline fraction is computed
from are SURVEY.md 8(d)'s table (line 502 ff.: N_issue per config), the variant rows count their own Philox work, and
both arms (--impl b200 / reference) describe the workload with the same `config` keys and values."""
import importlib.util
import os

import pytest

import workloads as W
from conftest import ROOT


@pytest.fixture(scope="module")
def bench():
    spec = importlib.util.spec_from_file_location("bench_module", os.path.join(ROOT, "bench.py"))
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    return m


def test_instruction_counts_are_the_surveys(bench):
    # SURVEY.md 8(d), column N_issue: cfg1 116, cfg2 206, cfg3 fp64 476 / fp32 462, cfg4 297, cfg5 183
    want = {(1, 64): 116, (2, 64): 206, (3, 64): 476, (3, 32): 462, (4, 64): 297, (5, 64): 183}
    for (cfg, prec), n in want.items():
        assert bench.n_issue(W.config(cfg), prec) == n, (cfg, prec)
    w = W.config(3)
    # u53 draws two words per dimension: ceil(d/2) = 10 blocks of 42 instead of 5; q32 runs the method's stream
    assert bench.philox_blocks(w) == 5 and bench.philox_blocks(w, 1) == 10
    assert bench.n_issue(w, 64, 1) == 476 + 5 * 42 and bench.n_issue(w, 64, 2) == 476
    slots, parts = bench.refined_slots(w, 64, 1)
    assert parts["philox_pairs"] == 200 and slots == pytest.approx(686 + 2.4 * 200)


def test_both_arms_name_the_workload_alike(bench):
    w = W.config(3)
    c = bench.base_config(w)
    assert c == {"workload": "cfg3_gauss_d20", "dim": 20, "n_bins": 50, "integrand": "gauss",
                 "n_events_per_gpu_per_step": 100_000_000, "chunk_events": 10_000_000, "alpha": 1.5, "seed": 3}
    assert bench.base_config(w, 25_000_000)["n_events_per_gpu_per_step"] == 25_000_000      # --scaling strong at 4 GPUs
