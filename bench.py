#!/usr/bin/env python
"""bench.py -- events/s of one Vegas iteration (fused iterate kernel + reduce + finalize + refine) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3] [--precision 64|32]
    python bench.py --impl reference ...      # the CPU oracle on the host cores, same metric/config

A "step" is one pass of the whole hot path over one batch: one Vegas iteration
of the workload's n_events events (in its chunk size) followed by the grid refinement.  Warm-up steps
are the first iterations of the chain, so the timed steps run on an adapted grid (equiprobable bins:
the conflict-heavy state the method spends its time in).  Inputs are seeded and synthetic
(workloads/__init__.py).  One JSON line on stdout (rank 0).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "events/sec per Vegas iteration"
UNIT = "events/s"
SM_COUNT, ISSUE_LANES, FP64_LANES = 148, 128, 64          # per SM per clock (guide + profiles/r01_s7_ubench_pipes.md)
INTEGRAND_DIM_FP = {0: 0, 1: 2, 2: 3, 3: 4}                # SURVEY.md 8(d) counting rule
INTEGRAND_EVENT_FP = {0: {64: 0, 32: 0}, 1: {64: 19, 32: 5}, 2: {64: 8, 32: 8}, 3: {64: 12, 32: 12}}


def philox_blocks(w, variant=0):
    """Philox4x32-10 blocks per event: one per 4 dimensions (C2); the u53 variant (C3') draws two words per dimension."""
    return (w.dim + 1) // 2 if variant == 1 else (w.dim + 3) // 4


def n_issue(w, precision, variant=0):
    """Algorithmic thread-level instructions per event (SURVEY.md 8(d) counting rule).  variant 1 (u53): the
    same rule with ceil(d/2) Philox blocks (its 53-bit split is counted like the 32-bit one: a lower bound); variant 2
    (q32) runs the same instruction stream as the method."""
    d = w.dim
    per_dim_fp = INTEGRAND_DIM_FP[w.integrand_id] * (d - 1 if w.integrand_id == 3 else d)
    return 42 * philox_blocks(w, variant) + d * (4 + 1 + 2 + 3) + per_dim_fp + 3 + 4 + INTEGRAND_EVENT_FP[w.integrand_id][precision]


def n_wide(w):
    """32x32->64 multiplies per event in the SURVEY count: 20 per Philox block plus the split of every dimension."""
    return 20 * ((w.dim + 3) // 4) + w.dim


# Refined machine model from the round-2 microbenchmarks (profiles/r02_ubench_pipes.md; "refine them
# only via the step-0 microbenchmarks"): one Philox round of one block -- 2 IMAD.WIDE.U32 + 2 LOP3 -- costs 8.8 scheduler
# clocks per warp (9.9 measured with the one register move the benchmark loop carries per round), not the 4 its
# instruction count suggests, and instructions added to the rounds cost 1.0 .. 1.9 clocks each ON TOP (DFMA, LOP3, IMAD
# alike): nothing hides under the wide multiplies.  The refined bound charges each of the 20 ceil(d/4) Philox
# multiply+XOR pairs of the SURVEY count 4.4 clocks instead of 2 and every other instruction its one issue slot.
PHILOX_PAIR_CLK = 4.4


def refined_slots(w, precision, variant=0):
    nblk = philox_blocks(w, variant)
    ni = n_issue(w, precision, variant)
    extra = (PHILOX_PAIR_CLK - 2.0) * 20 * nblk
    return ni + extra, {"issue": ni, "philox_pairs": 20 * nblk, "clk_per_pair": PHILOX_PAIR_CLK, "extra_clk": extra}


def ncu_traffic(workload, precision):
    """DRAM bytes per K1 launch from the committed `ncu --set full` summaries (the newest round that captured this
    workload: profiles/r03_traffic.json, else profiles/r02_traffic.json), with its source."""
    for name in ("r03_traffic.json", "r02_traffic.json"):
        try:
            with open(os.path.join(ROOT, "profiles", name)) as fh:
                t = json.load(fh)
            e = t["entries"].get("%s/%d" % (workload, precision))
            if e:
                return e["dram_bytes_per_launch"], {"source": t["source"], "commit": t["commit"], "file": "profiles/" + name,
                                                    "events_per_launch": e["events_per_launch"]}
        except Exception:
            pass
    return None, None


def n_fp(w, precision):
    d = w.dim
    per_dim_fp = INTEGRAND_DIM_FP[w.integrand_id] * (d - 1 if w.integrand_id == 3 else d)
    return 3 * d + per_dim_fp + 4 + INTEGRAND_EVENT_FP[w.integrand_id][precision]


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return json.load(fh)
    except Exception:
        return {}


class ClockSampler:
    """SM clock, power and throttle reasons polled through NVML every 2 ms in a thread (nvidia-smi's 100 ms loop
    cannot witness a 2.5 ms step); windows are cut out of the one sample stream by perf_counter time stamps."""
    PERIOD_S = 0.002

    def __init__(self, gpu_index):
        self.gpu, self.rows, self.stop_flag, self.thread, self.smax = gpu_index, [], False, None, None

    def start(self):
        try:
            import pynvml as N
            N.nvmlInit()
            idx = self.gpu
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            if vis:
                try:
                    idx = int(vis.split(",")[self.gpu])
                except Exception:
                    idx = self.gpu
            h = N.nvmlDeviceGetHandleByIndex(idx)
            self.smax = float(N.nvmlDeviceGetMaxClockInfo(h, N.NVML_CLOCK_SM))
            reasons = {"hw_slowdown": N.nvmlClocksEventReasonHwSlowdown, "hw_thermal_slowdown": N.nvmlClocksEventReasonHwThermalSlowdown,
                       "sw_thermal_slowdown": N.nvmlClocksEventReasonSwThermalSlowdown, "sw_power_cap": N.nvmlClocksEventReasonSwPowerCap}
            get_reasons = getattr(N, "nvmlDeviceGetCurrentClocksEventReasons", None) or N.nvmlDeviceGetCurrentClocksThrottleReasons

            def loop():
                while not self.stop_flag:
                    try:
                        clk = float(N.nvmlDeviceGetClockInfo(h, N.NVML_CLOCK_SM))
                        pw = N.nvmlDeviceGetPowerUsage(h) / 1000.0
                        mask = int(get_reasons(h))
                        self.rows.append((time.perf_counter(), clk, pw, [k for k, b in reasons.items() if mask & b]))
                    except Exception:
                        pass
                    time.sleep(self.PERIOD_S)

            self.thread = threading.Thread(target=loop, daemon=True)
            self.thread.start()
        except Exception:
            self.thread = None

    def window(self, t_begin, t_end, label):
        rows = [r for r in self.rows if t_begin <= r[0] <= t_end]
        sm = [r[1] for r in rows]
        smax = self.smax or (max(sm) if sm else None)
        busy = [c for c in sm if smax and c > 0.5 * smax] or sm
        reasons = sorted({k for r in rows for k in r[3]})
        return {"sm_mhz": statistics.median(busy) if busy else None, "sm_max_mhz": smax, "reasons": reasons,
                "power_w_max": max((r[2] for r in rows), default=None), "samples": len(sm),
                "sampler": "NVML every %g ms" % (1e3 * self.PERIOD_S), "window": label}

    def stop(self):
        self.stop_flag = True
        if self.thread:
            self.thread.join(timeout=1)


def cpu_baseline(w, edges, target_cpu_seconds=16.0):
    """The oracle, as it stands, on the host cores: a bounded sample of the same workload."""
    import oracle as O
    cores = os.cpu_count() or 1
    t0 = time.perf_counter()
    O.iterate(edges, 200_000, w.seed, 0, w.integrand_id, w.params, threads=1)
    rate1 = 200_000 / (time.perf_counter() - t0)
    n = int(min(w.n_events, max(cores * 100_000, rate1 * target_cpu_seconds)))
    t0 = time.perf_counter()
    O.iterate(edges, n, w.seed, 1, w.integrand_id, w.params, threads=cores)
    dt = time.perf_counter() - t0
    return {"value": n / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "%d of %d events of one %s iteration on the adapted grid, %d threads over disjoint "
                      "event ranges (%.1f s wall)" % (n, w.n_events, w.name, cores, dt),
            "per_core": n / dt / cores}


def base_config(w, n_events_per_gpu_per_step=None):
    """The keys both arms (--impl b200 / reference) report under `config`, with the same names and values."""
    import workloads as W
    return {"workload": w.name, "dim": w.dim, "n_bins": w.n_bins, "integrand": W.INTEGRAND_NAMES[w.integrand_id],
            "n_events_per_gpu_per_step": w.n_events if n_events_per_gpu_per_step is None else n_events_per_gpu_per_step,
            "chunk_events": w.chunk_events, "alpha": w.alpha, "seed": w.seed}


def run_reference(args, w, precision):
    """--impl reference: the oracle timed on the host cores; each step = one iteration + refine over a
    bounded sample of the workload's events."""
    import oracle as O
    from oracle import build as obuild
    obuild.build()
    cores = os.cpu_count() or 1
    edges = O.uniform_edges(w.dim, w.n_bins)
    t0 = time.perf_counter()
    O.iterate(edges, 100_000, w.seed, 0, w.integrand_id, w.params, threads=1)
    rate1 = 100_000 / (time.perf_counter() - t0)
    budget = 120.0 / max(1, args.steps + args.warmup)              # wall seconds per step
    n = int(min(w.n_events, max(cores * 50_000, rate1 * cores * 0.6 * budget)))
    k = 0
    for _ in range(args.warmup):
        _, _, H = O.iterate(edges, n, w.seed, k, w.integrand_id, w.params, threads=cores)
        edges, _ = O.refine(edges, H, w.alpha)
        k += 1
    t0 = time.perf_counter()
    for _ in range(args.steps):
        _, _, H = O.iterate(edges, n, w.seed, k, w.integrand_id, w.params, threads=cores)
        edges, _ = O.refine(edges, H, w.alpha)
        k += 1
    dt = time.perf_counter() - t0
    value = n * args.steps / dt
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": base_config(w), "sample_events_per_step": n,
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": "%d events per step (bounded sample of %d), %d threads" % (n, w.n_events, cores)},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="cfg3", help="cfg1..cfg5 (BASELINE.json configs)")
    ap.add_argument("--precision", type=int, default=64, choices=[64, 32])
    ap.add_argument("--n-events", type=int, default=0, help="override events per step per GPU")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="weak: every GPU takes the workload's n_events per step; strong: the workload's n_events are split "
                         "over the GPUs, rank g takes [g n/G, (g+1) n/G) (SURVEY.md 8(e)'s own partition)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="skip the `workloads` array (cfg3 fp32, cfg5, cfg4 at 1e8)")
    ap.add_argument("--alpha", type=float, default=None,
                    help="override the damping exponent (0 = plain MC: the grid stays uniform; SURVEY.md 8(d) asks for "
                         "one timing on the uniform grid)")
    ap.add_argument("--user-integrand", action="store_true",
                    help="run the workload's integrand as a run-time compiled user integrand (VEGAS_F_USER; gauss / genz only)")
    ap.add_argument("--launch", default="", help="blocks,threads,table_copies,hist_copies (0 = auto)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)

    import workloads as W
    w = W.config(int(args.workload.replace("cfg", "")))
    if args.n_events:
        w = w.scaled(args.n_events)
    if args.alpha is not None:
        import dataclasses
        w = dataclasses.replace(w, alpha=args.alpha)
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        if rank == 0:
            run_reference(args, w, args.precision)
        return

    import numpy as np
    import torch
    import torch.distributed as dist
    if local_rank == 0:
        from paper_2002_12921_b200 import build as lib_build
        lib_build.build()                                         # no-op when libvegas_b200.so is up to date
    if world > 1:
        import time as _t
        from paper_2002_12921_b200.build import LIB as _lib_path
        while not os.path.exists(_lib_path):                      # other ranks wait for rank 0's build
            _t.sleep(0.5)
    from paper_2002_12921_b200 import binding as B
    from paper_2002_12921_b200 import distributed as D

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the library has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local_rank)
    sampler.start()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2
    peaks = measured_peaks()
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))

    def measure(w, precision, steps, warmup, label, with_cpu_baseline=False, variant=0):
        """Warm-up (the chain's first iterations adapt the grid), `steps` device-timed steps, the same steps with the
        library's per-launch events (K1 alone), and the same steps end to end through the C ABI with host buffers."""
        g = B.VegasGrid(w.dim, w.n_bins)
        g.set_params(w.integrand_id, w.params)
        if variant:
            g.set_variant(variant)
        if args.launch:
            g.set_launch(*[int(v) for v in args.launch.split(",")])
        fid = w.integrand_id
        if args.user_integrand:
            from paper_2002_12921_b200 import user_integrands as U
            src = {W.GAUSS: U.GAUSS, W.GENZ_PRODUCT_PEAK: U.GENZ_PRODUCT_PEAK}[w.integrand_id]
            g.set_user_integrand(src, w.params)
            fid = B.VEGAS_F_USER
        shape = g.get_launch(fid, precision)
        # weak scaling: n_events per GPU per step; strong: n_events per step in all, split over the ranks
        n_step = w.n_events * world if args.scaling == "weak" else w.n_events

        def step(k):
            if world == 1:
                # one iteration + refinement, ONE launch (vegas_integrate_from, n_iter = 1), one synchronisation
                r = g.integrate(1, n_step, w.seed, w.alpha, fid, precision, chunk_events=w.chunk_events, first_iteration=k)
                return r["I"], r["sigma"]
            # accumulate -> all-reduce -> finalize + refine: one host synchronisation per sharded step
            I, s, _, st = D.iterate_sharded(g, n_step, w.seed, k, fid, precision, w.chunk_events, rank, world, want_hist=False,
                                            alpha=w.alpha)
            return I, s

        k = 0
        for _ in range(warmup):
            step(k)
            k += 1
        # ---- timed region: `steps` steps, device events per step (L2 flushed between steps, outside the brackets)
        g.reset_counters()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        results = []
        barrier()
        t_begin = time.perf_counter()
        for i in range(steps):
            flush.zero_()
            ev[i][0].record()
            results.append(step(k))
            ev[i][1].record()
            k += 1
        barrier()
        t_wall = time.perf_counter() - t_begin
        per_step_ms = [a.elapsed_time(b) for a, b in ev]
        ms = sum(per_step_ms)
        launches = g.launch_count()
        if world > 1:
            t = torch.tensor([ms], dtype=torch.float64, device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms = float(t.item())
        value = n_step * steps / (ms * 1e-3)

        # ---- the dominant kernel alone: the same steps again with the library's per-launch CUDA events switched on
        # (event pairs on the caller's stream around every K1 launch; kept out of the region `value` is taken from)
        k1_steps = min(steps, 50)
        g.set_profiling(True)
        g.reset_counters()
        evk = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(k1_steps)]
        for i in range(k1_steps):
            flush.zero_()
            evk[i][0].record()
            step(k)
            evk[i][1].record()
            k += 1
        barrier()
        k1_ms, k1_launches = g.kernel_time_ms()
        k1_region_ms = sum(a.elapsed_time(b) for a, b in evk)
        g.set_profiling(False)

        # ---- e2e: the same step through the C ABI with HOST buffers (edges in, I/sigma/hist/edges out)
        edges_host = g.get_edges()

        def e2e_step(k, edges_host):
            g.set_edges(edges_host)
            if world > 1:
                I, s, H, st = D.iterate_sharded(g, n_step, w.seed, k, fid, precision, w.chunk_events, rank, world, want_hist=True)
            else:
                I, s, H, st = g.iterate(n_step, w.seed, k, fid, precision, w.chunk_events, want_hist=True)
            g.refine(w.alpha, hist=H)
            return g.get_edges()

        edges_host = e2e_step(k, edges_host)       # untimed: the stand-alone refinement kernel is loaded on its first launch
        k += 1
        barrier()
        t0 = time.perf_counter()
        for i in range(steps):
            edges_host = e2e_step(k, edges_host)
            k += 1
        barrier()
        t_end = time.perf_counter()
        e2e_s = t_end - t0
        # ---- the sharded call sequence on this one rank (begin, accumulate, reduce, [all-reduce: none at world 1],
        # finalize + refine, one synchronisation): what a small iteration costs through the multi-GPU path
        sharded_ms = None
        if world == 1 and w.n_events <= 10_000_000:
            n_sh = min(steps, 50)
            D.iterate_sharded(g, n_step, w.seed, k, fid, precision, w.chunk_events, 0, 1, want_hist=False, alpha=w.alpha)
            barrier()
            t_sh = time.perf_counter()
            for i in range(n_sh):
                D.iterate_sharded(g, n_step, w.seed, k + 1 + i, fid, precision, w.chunk_events, 0, 1, want_hist=False, alpha=w.alpha)
            barrier()
            sharded_ms = 1e3 * (time.perf_counter() - t_sh) / n_sh
            k += 1 + n_sh
        clocks = sampler.window(t_begin, t_end, "%s: timed steps + K1 steps + e2e steps" % label)
        if world > 1:
            t = torch.tensor([e2e_s], dtype=torch.float64, device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            e2e_s = float(t.item())
        nent = w.dim * w.n_bins
        h2d = 8 * w.dim * (w.n_bins + 1) + 8 * nent + 8 * B.VEGAS_MAX_PARAMS   # edges + hist for refine + by-value params
        d2h = 24 + 8 * nent + 8 * w.dim * (w.n_bins + 1) + 4
        out = None
        if rank == 0:
            clk = float(clocks["sm_mhz"] or sm_max)
            ni, nf = n_issue(w, precision, variant), n_fp(w, precision)
            k1_s = (k1_ms * 1e-3) / max(1, k1_launches)
            events_per_launch = (n_step // world) * k1_steps / max(1, k1_launches)   # the fast path runs the chunk loop in the kernel
            k1_rate = events_per_launch / k1_s                         # events/s of the fused kernel alone
            peak_instr = SM_COUNT * ISSUE_LANES * sm_max * 1e6         # thread-instructions/s at max clock
            rs, rs_parts = refined_slots(w, precision, variant)
            traffic, traffic_src = ncu_traffic(w.name, precision)
            roofline = {"bound": "alu", "kernel": ("k_iterate_rot<%s>" % shape["path"]) if shape["path"] == "rotated" else "k_iterate",
                        "achieved": k1_rate * ni / 1e12, "peak": peak_instr / 1e12, "unit": "Tinstr/s",
                        "frac": k1_rate * ni / peak_instr,
                        "frac_at_measured_clock": k1_rate * ni / (SM_COUNT * ISSUE_LANES * clk * 1e6),
                        "peak_source": "148 SMs x 128 issue lanes x sm_max_mhz of MEASURED_PEAKS.json (%s); one instruction per "
                                       "scheduler per clock confirmed by profiles/r02_ubench_pipes.md" % ("measured" if peaks else "fallback 1965 MHz"),
                        "instr_per_event": ni, "fp_instr_per_event": nf,
                        "refined": {"slots_per_event": rs, "parts": rs_parts, "frac": k1_rate * rs / peak_instr,
                                    "why": "a Philox round (2 IMAD.WIDE.U32 + 2 LOP3) costs 8.8 scheduler clocks per warp, and added "
                                           "instructions cost 1.0-1.9 clk each on top of it (profiles/r02_ubench_pipes.md): each of the "
                                           "count's Philox multiply+XOR pairs is charged 4.4 clk instead of 2 issue slots"},
                        "fp_pipe_frac": k1_rate * nf / (SM_COUNT * (FP64_LANES if precision == 64 else ISSUE_LANES) * sm_max * 1e6),
                        "kernel_events_per_s": k1_rate, "kernel_ms_per_launch": k1_s * 1e3, "kernel_launches": int(k1_launches),
                        "kernel_includes": "the whole iteration: event loop + reduce + finalize + refine run in the one launch",
                        "kernel_share_of_step": k1_ms / k1_region_ms if world == 1 else None,
                        "traffic": traffic, "traffic_source": traffic_src,
                        "traffic_note": "algorithmic global bytes per launch = grid read + partial row write per CTA = %d" % (
                            shape["blocks"] * 8 * (w.dim * (w.n_bins + 1) + (4 + w.dim * w.n_bins)))}
            out = {"workload": w.name, "dtype": "f64" if precision == 64 else "f32", "value": value, "ms_per_step": ms / steps,
                   "ms_per_step_median": statistics.median(per_step_ms),     # this rank's steps (median of repeats)
                   "steps": steps, "warmup": warmup,
                   "config": {**base_config(w, n_step // world if args.scaling == "strong" else w.n_events),
                              "integrand_source": "run-time compiled user source (NVRTC)" if args.user_integrand else "built-in",
                              "launch": shape,
                              "l2": "256 MiB memset between timed steps, outside the event brackets (the path reads ~10 KB of global memory per launch)",
                              "grid": ("uniform (alpha = 0)" if w.alpha == 0 else "adapted by the %d warm-up iterations" % warmup)},
                   "clocks": clocks, "wall_s_timed_region": t_wall,
                   "e2e": {"value": n_step * steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
                   "gpu_launches": int(launches), "roofline": roofline, "sharded_call_sequence_ms_per_step": sharded_ms,
                   "last_iteration": {"I": results[-1][0], "sigma": results[-1][1], "closed_form": w.closed_form}}
            if with_cpu_baseline:
                out["cpu_baseline"] = cpu_baseline(w, edges_host)
        g.close()
        return out

    head = measure(w, args.precision, args.steps, args.warmup, "headline", with_cpu_baseline=(world == 1 and not args.no_cpu_baseline))
    # the other workloads SURVEY.md 8(d) gates (>= 1e8 events per iteration): a few steps each, own clock window
    extra = []
    if world == 1 and not args.no_extra and args.workload == "cfg3" and args.precision == 64 and not args.n_events:
        # ... and the two opt-in variants of the sampling map on the headline workload: what the
        # 32-bit draw saves against 53-bit uniforms, what an fp32-rounded grid table costs
        # ... and cfg1 / cfg2 at their OWN sizes (1e5 / 1e7 events per iteration), which SURVEY.md 8(d) lists as reported:
        # launch- and latency-bound, one launch per iteration
        # order: the three other GATED workloads close the array (a reader that keeps the tail of the line keeps them)
        for cfg, prec, n_ev, variant in ((3, 64, 0, 1), (3, 64, 0, 2), (1, 64, 0, 0), (2, 64, 0, 0),
                                         (3, 32, 0, 0), (5, 64, 0, 0), (4, 64, 100_000_000, 0)):
            we = W.config(cfg)
            if n_ev:
                we = we.scaled(n_ev)
            vname = {0: "", 1: "/u53", 2: "/q32"}[variant]
            r = measure(we, prec, max(3, min(args.steps, 10 if cfg > 2 else 100)), max(args.warmup, 4), "%s/%d%s" % (we.name, prec, vname), variant=variant)
            if r:
                extra.append({"workload": r["workload"], "dtype": r["dtype"],
                              "variant": {0: "none", 1: "u53 (53-bit uniforms, two Philox words per draw)",
                                          2: "q32 (grid-table entries rounded to fp32)"}[variant],
                              "n_events": we.n_events, "chunk_events": we.chunk_events,
                              "value": r["value"], "e2e": r["e2e"]["value"], "ms_per_step": r["ms_per_step"], "steps": r["steps"],
                              "sharded_call_sequence_ms_per_step": r["sharded_call_sequence_ms_per_step"],
                              "kernel_ms_per_launch": r["roofline"]["kernel_ms_per_launch"],
                              "kernel_events_per_s": r["roofline"]["kernel_events_per_s"],
                              "roofline_frac": r["roofline"]["frac"], "refined_frac": r["roofline"]["refined"]["frac"],
                              "instr_per_event": r["roofline"]["instr_per_event"], "launch": r["config"]["launch"],
                              "clocks": r["clocks"], "last_iteration": r["last_iteration"]})
    # one timing of the headline workload on the UNIFORM grid (alpha = 0: the grid never adapts) beside
    # the adapted-grid one
    uniform = None
    if world == 1 and not args.no_extra and args.alpha is None and not args.n_events:
        import dataclasses
        uniform = measure(dataclasses.replace(w, alpha=0.0), args.precision, max(3, min(args.steps, 10)), max(args.warmup, 3),
                          "%s/%d uniform grid" % (w.name, args.precision))
    sampler.stop()
    if rank == 0:
        line = {"metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": head["ms_per_step"], "higher_is_better": True, "scaling": args.scaling,
                "vs_baseline": None, "dtype": head["dtype"], "data": "synthetic", "config": head["config"],
                "clocks": head["clocks"], "wall_s_timed_region": head["wall_s_timed_region"], "e2e": head["e2e"],
                "gpu_launches": head["gpu_launches"], "roofline": head["roofline"], "last_iteration": head["last_iteration"]}
        if "cpu_baseline" in head:
            line["cpu_baseline"] = head["cpu_baseline"]
        if extra:
            line["workloads"] = extra
        line["ms_per_step_median"] = head["ms_per_step_median"]
        if uniform:
            line["uniform_grid"] = {"value": uniform["value"], "ms_per_step": uniform["ms_per_step"],
                                    "kernel_ms_per_launch": uniform["roofline"]["kernel_ms_per_launch"],
                                    "roofline_frac": uniform["roofline"]["frac"], "steps": uniform["steps"],
                                    "note": "same workload with alpha = 0 (the grid stays uniform)"}
        # every workload SURVEY.md 8(d) gates (>= 1e8 events per iteration), compact and LAST on the line
        gated = {"%s/%s" % (head["workload"], head["dtype"]): head}
        gated_names = {"cfg3_gauss_d20/f32", "cfg5_bw_poly_d6/f64", "cfg4_genz_pp_d12/f64"}
        rows = {}
        for name, r in gated.items():
            rows[name] = {"n_events": w.n_events, "value": r["value"], "e2e": r["e2e"]["value"], "frac": r["roofline"]["frac"],
                          "kernel_ms": r["roofline"]["kernel_ms_per_launch"], "instr_per_event": r["roofline"]["instr_per_event"],
                          "sm_mhz": r["clocks"]["sm_mhz"], "reasons": r["clocks"]["reasons"]}
        for e in extra:
            name = "%s/%s" % (e["workload"], e["dtype"])
            if e["variant"] == "none" and name in gated_names and e["n_events"] >= 100_000_000:
                rows[name] = {"n_events": e["n_events"], "value": e["value"], "e2e": e["e2e"], "frac": e["roofline_frac"],
                              "kernel_ms": e["kernel_ms_per_launch"], "instr_per_event": e["instr_per_event"],
                              "sm_mhz": e["clocks"]["sm_mhz"], "reasons": e["clocks"]["reasons"]}
        line["gated"] = rows
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
