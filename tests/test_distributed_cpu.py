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
from paper_2002_12921_b200 import workloads as W


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
