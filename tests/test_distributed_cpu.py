"""Host logic of the multi-GPU iteration (paper_2002_12921_b200/distributed.py) on CPU: world_size-2
gloo processes, each accumulating ITS event range with the oracle (stand-in for the per-rank kernel;
this is a test), one all-reduce of the totals vector, and the result must equal the single-process
iteration."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2002_12921_b200 import distributed as D
import workloads as W


def test_shard_range_partitions_exactly():
    for n in (0, 1, 7, 1000, 10**9 + 7):
        for world in (1, 2, 3, 8):
            parts = [D.shard_range(n, r, world) for r in range(world)]
            assert parts[0][0] == 0 and sum(c for _, c in parts) == n
            for (a, ca), (b, _) in zip(parts[:-1], parts[1:]):
                assert a + ca == b
            assert max(c for _, c in parts) - min(c for _, c in parts) <= 1
    with pytest.raises(ValueError):
        D.shard_range(10, 2, 2)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, n, out_path):
    import oracle as O
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = W.config(1)
    edges = W.adapted_edges(w.dim, w.n_bins, seed=5)
    first, count = D.shard_range(n, rank, world)
    S1, S2, H = O.accumulate(edges, w.seed, 2, first, count, w.integrand_id, w.params)
    ld = np.longdouble
    tot = np.zeros(4 + w.dim * w.n_bins)
    tot[0] = float(S1); tot[1] = float(S1 - ld(tot[0]))
    tot[2] = float(S2); tot[3] = float(S2 - ld(tot[2]))
    tot[4:] = H.astype(np.float64).ravel()
    t = torch.from_numpy(tot)
    D.allreduce_totals(t)
    I, sg = O.estimate(ld(tot[0]) + ld(tot[1]), ld(tot[2]) + ld(tot[3]), n)
    if rank == 0:
        np.save(out_path, np.concatenate([[I, sg], tot[4:]]))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_gloo_iteration_equals_single_process(tmp_path):
    import oracle as O
    n = 40_001
    out = str(tmp_path / "r0.npy")
    mp.spawn(_worker, args=(2, _free_port(), n, out), nprocs=2, join=True)
    got = np.load(out)
    w = W.config(1)
    edges = W.adapted_edges(w.dim, w.n_bins, seed=5)
    I, sg, H = O.iterate(edges, n, w.seed, 2, w.integrand_id, w.params)
    assert got[0] == pytest.approx(I, rel=1e-14) and got[1] == pytest.approx(sg, rel=1e-12)
    np.testing.assert_allclose(got[2:].reshape(H.shape), H, rtol=1e-14)


class _OracleRankGrid:
    """Stands in for binding.VegasGrid on a CPU rank: the same five calls iterate_sharded makes, with the oracle as the
    per-rank kernel and a CPU tensor as the totals vector (this is a test; the product's grid runs the CUDA kernels)."""

    def __init__(self, edges, params):
        import oracle as O
        self.O, self.edges, self.params = O, edges, params
        self.dim, self.n_bins = edges.shape[0], edges.shape[1] - 1
        self.tot = torch.zeros(4 + self.dim * self.n_bins, dtype=torch.float64)
        self.calls = []

    def begin_iteration(self):
        self.tot.zero_()
        self.calls.append("begin")

    def accumulate(self, first, count, seed, iteration, fid, precision, chunk_events):
        S1, S2, H = self.O.accumulate(self.edges, seed, iteration, first, count, fid, self.params)
        ld = np.longdouble
        t = np.zeros(self.tot.numel())
        t[0] = float(S1); t[1] = float(S1 - ld(t[0])); t[2] = float(S2); t[3] = float(S2 - ld(t[2]))
        t[4:] = H.astype(np.float64).ravel()
        self.tot += torch.from_numpy(t)
        self.calls.append(("accumulate", first, count))

    def reduce(self):
        self.calls.append("reduce")

    def totals_tensor(self):
        return self.tot

    def finalize(self, n_total, want_hist=False):
        ld = np.longdouble
        t = self.tot.numpy()
        I, sg = self.O.estimate(ld(t[0]) + ld(t[1]), ld(t[2]) + ld(t[3]), n_total)
        return I, sg, (t[4:].reshape(self.dim, self.n_bins).copy() if want_hist else None), 0

    def finish_sharded(self, n_total, alpha, want_hist=False):
        I, sg, H, st = self.finalize(n_total, want_hist=True)
        if alpha >= 0:
            self.edges, _ = self.O.refine(self.edges, H, alpha)
        self.calls.append(("finish_sharded", alpha))
        return I, sg, (H if want_hist else None), st


def _worker_sharded(rank, world, port, n, fixed_order, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = W.config(1)
    g = _OracleRankGrid(W.adapted_edges(w.dim, w.n_bins, seed=5), w.params)
    I, sg, H, st = D.iterate_sharded(g, n, w.seed, 2, w.integrand_id, 64, 0, rank, world, want_hist=True,
                                     fixed_order=fixed_order)
    assert g.calls[0] == "begin" and g.calls[1] == ("accumulate",) + D.shard_range(n, rank, world) and g.calls[2] == "reduce"
    # the same iteration with the refinement in the same call: same estimate and histogram, grid refined once, on every rank
    e0 = g.edges.copy()
    I2, sg2, H2, _ = D.iterate_sharded(g, n, w.seed, 2, w.integrand_id, 64, 0, rank, world, want_hist=True,
                                       fixed_order=fixed_order, alpha=w.alpha)
    assert (I2, sg2) == (I, sg) and np.array_equal(H2, H) and g.calls[-1] == ("finish_sharded", w.alpha)
    import oracle as O
    assert np.array_equal(g.edges, O.refine(e0, H, w.alpha)[0]) and not np.array_equal(g.edges, e0)
    np.save(os.path.join(out_dir, "r%d.npy" % rank), np.concatenate([[I, sg], H.ravel(), g.edges.ravel()]))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world,fixed_order", [(2, False), (2, True), (3, True)])
def test_iterate_sharded_itself_over_gloo(tmp_path, world, fixed_order):
    """distributed.iterate_sharded, the function bench.py --gpus N calls, at world_size > 1: every rank must end with the
    same bits, equal to the single-process iteration."""
    import oracle as O
    n = 30_001
    mp.spawn(_worker_sharded, args=(world, _free_port(), n, fixed_order, str(tmp_path)), nprocs=world, join=True)
    got = [np.load(str(tmp_path / ("r%d.npy" % r))) for r in range(world)]
    for r in range(1, world):
        assert np.array_equal(got[0], got[r])                      # lockstep: identical bits on every rank
    w = W.config(1)
    I, sg, H = O.iterate(W.adapted_edges(w.dim, w.n_bins, seed=5), n, w.seed, 2, w.integrand_id, w.params)
    assert got[0][0] == pytest.approx(I, rel=1e-14) and got[0][1] == pytest.approx(sg, rel=1e-12)
    np.testing.assert_allclose(got[0][2:2 + H.size].reshape(H.shape), H, rtol=1e-14)
