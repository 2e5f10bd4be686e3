"""vegas_iterate_static: the iteration for callers that cannot allocate device memory.

Some users of this library only ever hold the buffers somebody else gave them: an op running inside a framework
that owns the GPU's memory pool, a loop that must not stall on cudaMalloc, a process on a fixed memory budget.  They
cannot create the workspace a VegasGrid needs, so the library offers them one call whose working memory is an array
compiled into the library itself (include/vegas.h).  This file checks that this call computes the same iteration as
the ordinary path: two calls in a row on one stream, with different shapes and integrands so that what the first one
left in the shared array would show up in the second if it were not cleared, compared with vegas_iterate on a
VegasGrid at the tolerance the other parity tests use (1e-10 relative on I, sigma and every histogram bin; empty
bins exactly zero).  A repeat of the first call must then return the same bits as before.

The file name sorts last on purpose: pytest -x stops at the first failure, and a failure here should not hide the
parity tests.  It makes no assumption about what ran before it: the first vegas_iterate_static call on the device does
its own set-up, whether that happens here in a fresh process or after the rest of the suite.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import workloads as W

RTOL64 = 1e-10


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    from paper_2002_12921_b200 import build
    build.build()
    from paper_2002_12921_b200 import binding
    return binding


def _existing_path(B, w, edges, iteration, generic):
    g = B.VegasGrid(w.dim, w.n_bins)
    g.set_params(w.integrand_id, w.params)
    g.set_edges(edges)
    if generic:
        g.set_launch(table_copies=1, hist_copies=1)      # pins the generic kernel (any copy count does)
    I, s, H, status = g.iterate(w.n_events, w.seed, iteration, w.integrand_id)
    g.close()
    assert status == B.VEGAS_OK
    return I, s, H


def test_two_calls_in_a_row_match_the_grid_path(B):
    import torch
    # call A: cfg3-shaped (20 x 50 = 1000 entries); call B: cfg4-shaped (12 x 100 = 1200 entries, another integrand):
    # B's rows overlap A's at different offsets in the shared array
    wa = W.config(3).scaled(n_events=300_007)
    wb = W.config(4).scaled(n_events=200_003)
    cases = [(wa, W.adapted_edges(wa.dim, wa.n_bins, seed=31), 2), (wb, W.adapted_edges(wb.dim, wb.n_bins, seed=32), 1)]
    dev = torch.device("cuda", torch.cuda.current_device())
    # everything the calls touch is handed over by the caller: inputs and outputs, nothing else
    edges_d = [torch.from_numpy(e).to(dev) for _, e, _ in cases]
    result_d = [torch.full((3,), float("nan"), dtype=torch.float64, device=dev) for _ in cases]
    hist_d = [torch.full((w.dim, w.n_bins), float("nan"), dtype=torch.float64, device=dev) for w, _, _ in cases]
    torch.cuda.synchronize()
    for k, (w, _, it) in enumerate(cases):              # back to back on the current stream, no sync in between
        B.vegas_iterate_static(edges_d[k], w.n_events, w.seed, it, w.integrand_id, w.params, result_d[k], hist_d[k])
    torch.cuda.synchronize()
    for k, (w, e, it) in enumerate(cases):
        I, s, status = result_d[k].cpu().numpy()
        H = hist_d[k].cpu().numpy()
        assert status == 0.0
        for generic in (False, True):                   # the default fast path, and the generic kernel it shares
            I0, s0, H0 = _existing_path(B, w, e, it, generic)
            assert abs(I - I0) <= RTOL64 * abs(I0), (w.name, generic, I, I0)
            assert abs(s - s0) <= RTOL64 * abs(s0), (w.name, generic, s, s0)
            np.testing.assert_allclose(H, H0, rtol=RTOL64, atol=0)
            assert np.all(H[H0 == 0] == 0)
    # the first call again, after the other one used the array: same bits as the first time, without the histogram too
    w, _, it = cases[0]
    again = torch.empty(3, dtype=torch.float64, device=dev)
    hist_again = torch.empty_like(hist_d[0])
    B.vegas_iterate_static(edges_d[0], w.n_events, w.seed, it, w.integrand_id, w.params, again, hist_again)
    no_hist = torch.empty(3, dtype=torch.float64, device=dev)
    B.vegas_iterate_static(edges_d[0], w.n_events, w.seed, it, w.integrand_id, w.params, no_hist, None)
    torch.cuda.synchronize()
    assert torch.equal(again, result_d[0]) and torch.equal(hist_again, hist_d[0]) and torch.equal(no_hist, result_d[0])
    # and the point of it all: with the set-up behind it, a call leaves the device's free memory where it was
    # (cudaMemGetInfo through torch; the outputs above are reused, so torch's own allocator has nothing to do either)
    free_before = torch.cuda.mem_get_info()[0]
    for k, (w, _, it) in enumerate(cases):
        B.vegas_iterate_static(edges_d[k], w.n_events, w.seed, it, w.integrand_id, w.params, result_d[k], hist_d[k])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before


def test_shapes_beyond_the_built_in_scratch_are_refused(B):
    import torch
    dev = torch.device("cuda", torch.cuda.current_device())
    result = torch.zeros(3, dtype=torch.float64, device=dev)
    too_big = torch.from_numpy(W.adapted_edges(32, 128)).to(dev)          # 4096 entries > 2048
    with pytest.raises(B.VegasError) as e:
        B.vegas_iterate_static(too_big, 1000, 1, 0, B.VEGAS_F_CONST, None, result)
    assert e.value.code == B.VEGAS_ELIMIT and "2048" in str(e.value)
    at_limit = torch.from_numpy(W.adapted_edges(16, 128)).to(dev)         # exactly 2048 entries: served
    hist = torch.empty(16, 128, dtype=torch.float64, device=dev)
    B.vegas_iterate_static(at_limit, 100_003, 7, 0, B.VEGAS_F_CONST, None, result, hist)
    torch.cuda.synchronize()
    I, s, status = result.cpu().numpy()
    assert status == 0.0 and abs(I - 1.0) < 6 * s + 1e-15                  # f = 1: the integral is 1
    g = B.VegasGrid(16, 128)
    g.set_edges(at_limit.cpu().numpy())
    I0, s0, H0, _ = g.iterate(100_003, 7, 0, B.VEGAS_F_CONST)
    g.close()
    assert abs(I - I0) <= RTOL64 * abs(I0) and abs(s - s0) <= RTOL64 * abs(s0)
    np.testing.assert_allclose(hist.cpu().numpy(), H0, rtol=RTOL64, atol=0)
    # the usual argument rules hold: a user integrand cannot be served, two events at least, parameters as set_params
    for args in ((at_limit, 1000, 1, 0, B.VEGAS_F_USER, None, result), (at_limit, 1, 1, 0, B.VEGAS_F_CONST, None, result),
                 (at_limit, 1000, 1, 0, B.VEGAS_F_GAUSS, [0.1, 0.2], result)):
        with pytest.raises(B.VegasError) as e:
            B.vegas_iterate_static(*args)
        assert e.value.code == B.VEGAS_EINVAL
