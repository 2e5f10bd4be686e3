"""Multi-GPU iteration: events are independent and the RNG is addressed by the global
event index (C2), so rank r of R takes a contiguous event range, every rank holds the full grid, and
ONE exchange per iteration -- an all-reduce(sum) of the 4 + dim*n_bins fp64 totals
{S1_hi, S1_lo, S2_hi, S2_lo, H} -- gives every rank the same I, sigma, histogram and therefore the
same refined grid.  The message is <= 26 KB: latency-bound on NVLink 5 / NVSwitch, so it is left to
NCCL (there is no compute tile to overlap it with; the fused kernel has already finished).

One process per GPU (torch.distributed, backend "nccl"); the same functions run on CPU tensors with
"gloo" (tests/test_distributed_cpu.py), which is how the host logic is covered without GPUs.
"""
from __future__ import annotations


def shard_range(n_events: int, rank: int, world: int):
    """Contiguous split of [0, n_events): (first_event, count) of `rank`; counts differ by <= 1."""
    if world < 1 or not (0 <= rank < world) or n_events < 0:
        raise ValueError("bad shard arguments")
    lo = n_events * rank // world
    hi = n_events * (rank + 1) // world
    return lo, hi - lo


def allreduce_totals(totals, group=None, fixed_order: bool = False):
    """Sum the per-rank totals vector in place over the process group (no-op for one process).
    The (hi, lo) pairs of S1 and S2 are summed component-wise: each stays a valid unevaluated sum.

    fixed_order=False: one all-reduce(sum); the association of the fp64 additions is the collective library's
    (NCCL ring/tree, gloo): every rank receives the same bits, so the grids stay in lockstep, and a run is
    reproducible for a fixed world size and algorithm, but not bit-for-bit against another world size.
    fixed_order=True: all-gather of the R vectors (R x <= 26 KB) and a sum in rank order 0, 1, ..., R-1 on every
    rank: bit-reproducible whatever the collective does (SURVEY.md 8(e) "reduced in fixed rank order if bitwise
    reproducibility is wanted")."""
    import torch
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        if fixed_order:
            parts = [torch.empty_like(totals) for _ in range(dist.get_world_size(group))]
            dist.all_gather(parts, totals.contiguous(), group=group)
            acc = parts[0].clone()
            for t in parts[1:]:
                acc += t
            totals.copy_(acc)
        else:
            dist.all_reduce(totals, op=dist.ReduceOp.SUM, group=group)
    return totals


def iterate_sharded(grid, n_events_total: int, seed: int, iteration: int, integrand_id: int, precision: int = 64,
                    chunk_events: int = 0, rank: int = 0, world: int = 1, want_hist: bool = False, group=None,
                    fixed_order: bool = False, alpha=None):
    """One Vegas iteration of n_events_total events spread over `world` ranks; `grid` is this rank's
    binding.VegasGrid.  Returns (I, sigma, hist or None, status), identical on every rank.
    alpha=None: the grid is left as it is (the caller refines, a second host synchronisation).  alpha given: the
    refinement with that damping exponent (alpha < 0: none) follows the estimate in the same call
    (vegas_finish_sharded): accumulate -> all-reduce on the stream -> finalize + refine -> ONE host synchronisation,
    like the single-GPU iteration."""
    first, count = shard_range(n_events_total, rank, world)
    grid.begin_iteration()
    if count:
        grid.accumulate(first, count, seed, iteration, integrand_id, precision, chunk_events)
    grid.reduce()
    if world > 1:
        allreduce_totals(grid.totals_tensor(), group, fixed_order)
    if alpha is not None:
        return grid.finish_sharded(n_events_total, alpha, want_hist=want_hist)
    return grid.finalize(n_events_total, want_hist=want_hist)
