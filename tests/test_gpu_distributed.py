"""distributed.iterate_sharded -- the function bench.py --gpus N calls -- with the real kernels at world_size 2:
two processes on the one GPU, each with its own VegasGrid, the gloo backend on CUDA tensors (NCCL refuses two ranks
on one device; the two ranks' kernels are independent launches that never wait on one another, the exchange is the
host-side collective).  Every rank must end with the same I, sigma, H and refined grid, equal to the oracle's
single-process iteration at 1e-10."""
import os
import socket

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import workloads as W


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, cfg, n, n_iter, fixed_order, out_dir):
    import torch
    import torch.distributed as dist
    from paper_2002_12921_b200 import binding as B
    from paper_2002_12921_b200 import distributed as D
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    torch.cuda.set_device(0)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = W.config(cfg)
    g = B.VegasGrid(w.dim, w.n_bins)
    g.set_params(w.integrand_id, w.params)
    out = []
    for k in range(n_iter):
        # odd iterations: estimate and refinement in one call with one synchronisation (vegas_finish_sharded);
        # even ones: vegas_finalize, then vegas_refine -- the same grid either way
        launches = g.launch_count()
        I, s, H, st = D.iterate_sharded(g, n, w.seed, k, w.integrand_id, 64, w.chunk_events and 50_000, rank, world,
                                        want_hist=True, fixed_order=fixed_order, alpha=w.alpha if k % 2 else None)
        assert st == 0
        assert g.totals_tensor().is_cuda
        if k % 2 == 0:
            assert g.refine(w.alpha) == 0
        assert g.launch_count() - launches >= 4          # accumulate, reduce, finalize, refine: all of them ran here
        out.append(np.concatenate([[I, s], H.ravel(), g.get_edges().ravel()]))
    np.save(os.path.join(out_dir, "r%d.npy" % rank), np.stack(out))
    g.close()
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("cfg,fixed_order", [(1, False), (4, True), (5, False)])
def test_iterate_sharded_two_ranks_on_one_gpu(tmp_path, cfg, fixed_order):
    import torch
    import torch.multiprocessing as mp
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    from paper_2002_12921_b200 import build
    build.build()
    import oracle as O
    w = W.config(cfg)
    n, n_iter, world = 200_003, 3, 2
    mp.spawn(_worker, args=(world, _free_port(), cfg, n, n_iter, fixed_order, str(tmp_path)), nprocs=world, join=True)
    got = [np.load(str(tmp_path / ("r%d.npy" % r))) for r in range(world)]
    assert np.array_equal(got[0], got[1])                              # lockstep: identical bits on both ranks
    # teacher-forced against the oracle: iteration k on the grid the ranks sampled from
    nh, ne = w.dim * w.n_bins, w.dim * (w.n_bins + 1)
    edges = O.uniform_edges(w.dim, w.n_bins)
    for k in range(n_iter):
        I, s = got[0][k, 0], got[0][k, 1]
        H = got[0][k, 2:2 + nh].reshape(w.dim, w.n_bins)
        new_edges = got[0][k, 2 + nh:2 + nh + ne].reshape(w.dim, w.n_bins + 1)
        oI, oS, oH = O.iterate(edges, n, w.seed, k, w.integrand_id, w.params, threads=os.cpu_count() or 8)
        assert I == pytest.approx(oI, rel=1e-10) and s == pytest.approx(oS, rel=1e-10)
        np.testing.assert_allclose(H, oH, rtol=1e-10, atol=0)
        want, _ = O.refine(edges, H, w.alpha)                          # the GPU's own histogram: S8 alone
        np.testing.assert_allclose(new_edges, want, rtol=0, atol=1e-10)
        edges = new_edges
