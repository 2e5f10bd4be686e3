"""User-supplied integrands compiled at run time (vegas_set_user_integrand) against the
CPU oracle: the same P3/P4/P5 protocol as the built-in integrands, fp64 tolerances of north_star."""
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle as O
from paper_2002_12921_b200 import user_integrands as U
import workloads as W

THREADS = os.cpu_count() or 8
RTOL64 = 1e-10


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    from paper_2002_12921_b200 import build
    build.build()                                   # no-op when libvegas_b200.so is up to date
    from paper_2002_12921_b200 import binding
    return binding


def _hist_ok(h_gpu, h_ref):
    np.testing.assert_allclose(h_gpu, h_ref, rtol=RTOL64, atol=0)
    assert np.all(h_gpu[h_ref == 0] == 0)


CASES = [
    # (user source, oracle id, dim, n_bins, params)
    ("GAUSS", O.GAUSS, 4, 50, lambda d: W.gauss_params(0.1)),
    ("GAUSS", O.GAUSS, 7, 33, lambda d: W.gauss_params(0.2)),                 # last Philox block with 3 dimensions
    ("GENZ_PRODUCT_PEAK", O.GENZ_PRODUCT_PEAK, 12, 100, lambda d: W.genz_params(d, 4)),
    ("GENZ_PRODUCT_PEAK", O.GENZ_PRODUCT_PEAK, 5, 20, lambda d: W.genz_params(d, 11)),   # last block with 1
    ("GENZ_DISCONTINUOUS", O.GENZ_DISCONTINUOUS, 16, 50, lambda d: W.genz_discontinuous_params(d, 9)),
    ("GENZ_DISCONTINUOUS", O.GENZ_DISCONTINUOUS, 2, 8, lambda d: W.genz_discontinuous_params(d, 2)),    # last block with 2
]


@pytest.mark.parametrize("name,oid,dim,nb,pf", CASES)
def test_user_integrand_iterations_on_oracle_grids(B, name, oid, dim, nb, pf):
    """P3/P4 teacher-forced: every iteration of an oracle chain is repeated on the oracle's grid."""
    p = pf(dim)
    n, seed, alpha = 300_007, 21, 1.5
    ch = O.integrate(dim, nb, 3, n, seed, alpha, oid, p, threads=THREADS)
    g = B.VegasGrid(dim, nb)
    g.set_user_integrand(getattr(U, name), p)
    assert g.get_launch(B.VEGAS_F_USER, 64)["path"] == "rotated"
    for k in range(3):
        g.set_edges(ch["edges_trace"][k])
        I, s, H, st = g.iterate(n, seed, k, B.VEGAS_F_USER, 64, chunk_events=100_000 if k == 1 else 0)
        assert st == 0
        assert I == pytest.approx(ch["per_iter"][k, 0], rel=RTOL64)
        assert s == pytest.approx(ch["per_iter"][k, 1], rel=RTOL64)
        _hist_ok(H, ch["hist_trace"][k])
        assert g.refine(alpha) == 0
        nxt = ch["edges_trace"][k + 1] if k + 1 < 3 else ch["edges"]
        np.testing.assert_allclose(g.get_edges(), nxt, rtol=0, atol=1e-10)
    g.close()


def test_user_integrand_equals_builtin_and_closed_form(B):
    """The user-written Gaussian runs in the same fused kernel as the built-in one: same sample, same result to
    rounding; a free-running vegas_integrate lands on the closed form (5 sigma rule, P7)."""
    w = W.config(2).scaled(n_events=2_000_003, n_iter=6)
    g = B.VegasGrid(w.dim, w.n_bins)
    g.set_params(w.integrand_id, w.params)
    g.set_user_integrand(U.GAUSS, w.params)
    Ib, sb, Hb, _ = g.iterate(w.n_events, w.seed, 0, w.integrand_id, 64)
    Iu, su, Hu, _ = g.iterate(w.n_events, w.seed, 0, B.VEGAS_F_USER, 64)
    assert Iu == pytest.approx(Ib, rel=1e-12) and su == pytest.approx(sb, rel=1e-12)
    np.testing.assert_allclose(Hu, Hb, rtol=1e-11)
    r = g.integrate(w.n_iter, w.n_events, w.seed, w.alpha, B.VEGAS_F_USER, 64, n_skip=2)
    assert abs(r["I"] - w.closed_form) < 5 * r["sigma"] and r["sigma"] < 1e-3
    g.close()


def test_user_integrand_parameters_and_errors(B):
    p = W.genz_discontinuous_params(6, 3)
    g = B.VegasGrid(6, 50)
    # not compiled yet
    with pytest.raises(B.VegasError):
        g.iterate(1000, 1, 0, B.VEGAS_F_USER, 64)
    # a source that does not compile: EINVAL with the compiler's message, and no kernel is installed
    with pytest.raises(B.VegasError) as ei:
        g.set_user_integrand(U.BROKEN, p)
    assert ei.value.code == B.VEGAS_EINVAL and "undeclared_symbol" in str(ei.value)
    with pytest.raises(B.VegasError):
        g.iterate(1000, 1, 0, B.VEGAS_F_USER, 64)
    with pytest.raises(B.VegasError):
        g.set_user_integrand(U.GENZ_DISCONTINUOUS, np.zeros(B.VEGAS_USER_MAX_PARAMS + 1))
    g.set_user_integrand(U.GENZ_DISCONTINUOUS, p)
    with pytest.raises(B.VegasError):
        g.iterate(1000, 1, 0, B.VEGAS_F_USER, 16)                 # precision is 64 or 32
    with pytest.raises(B.VegasError):
        g.debug_sample(0, 16, 1, 0, B.VEGAS_F_USER, 64)
    edges = W.adapted_edges(6, 50, seed=6)
    g.set_edges(edges)
    I1, s1, H1, _ = g.iterate(100_003, 5, 0, B.VEGAS_F_USER, 64)
    oI, oS, oH = O.iterate(edges, 100_003, 5, 0, O.GENZ_DISCONTINUOUS, p)
    assert I1 == pytest.approx(oI, rel=RTOL64) and s1 == pytest.approx(oS, rel=RTOL64)
    # new parameters without recompiling
    p2 = W.genz_discontinuous_params(6, 4)
    g.set_params(B.VEGAS_F_USER, p2)
    I2, s2, H2, _ = g.iterate(100_003, 5, 0, B.VEGAS_F_USER, 64)
    oI2, oS2, oH2 = O.iterate(edges, 100_003, 5, 0, O.GENZ_DISCONTINUOUS, p2)
    assert I2 == pytest.approx(oI2, rel=RTOL64) and s2 == pytest.approx(oS2, rel=RTOL64)
    _hist_ok(H2, oH2)
    # a source that does not compile leaves the installed kernel AND its parameters as they were
    with pytest.raises(B.VegasError):
        g.set_user_integrand(U.BROKEN, W.genz_discontinuous_params(6, 9))
    I2b, s2b, _, _ = g.iterate(100_003, 5, 0, B.VEGAS_F_USER, 64)
    assert I2b == I2 and s2b == s2
    # a launch shape wider than the user kernel is built for (12 warps) is clamped, not launched out of bounds
    g.set_launch(0, 512, 0, 0)
    assert g.get_launch(B.VEGAS_F_USER, 64)["threads"] <= 384
    I2c, s2c, _, _ = g.iterate(100_003, 5, 0, B.VEGAS_F_USER, 64)
    assert I2c == pytest.approx(oI2, rel=RTOL64) and s2c == pytest.approx(oS2, rel=RTOL64)
    g.set_launch(0, 0, 0, 0)
    # replacing the integrand replaces the kernel
    g.set_user_integrand(U.GENZ_PRODUCT_PEAK, W.genz_params(6, 8))
    I3, _, _, _ = g.iterate(100_003, 5, 0, B.VEGAS_F_USER, 64)
    oI3, _, _ = O.iterate(edges, 100_003, 5, 0, O.GENZ_PRODUCT_PEAK, W.genz_params(6, 8))
    assert I3 == pytest.approx(oI3, rel=RTOL64)
    g.close()


def test_host_callback_integrand_matches_the_oracle(B):
    """vegas_iterate_callback (second half): f evaluated by a HOST function on batches of points
    sampled on the device; same sample and sums as the oracle's iteration with the same f (fp64 tolerances)."""
    dim, nb, n, seed = 7, 40, 250_003, 31
    p = W.genz_params(dim, 5)
    c, wv = p[:dim], p[dim:]
    edges = W.adapted_edges(dim, nb, seed=3)
    calls = []

    def f_host(x):                                   # numpy restatement of Eq.(3): the "user's C/Fortran function"
        calls.append(x.shape[0])
        assert x.shape[1] == dim and np.all((x > 0) & (x < 1))
        return 1.0 / np.prod(1.0 / (c * c) + (x - wv) ** 2, axis=1)

    g = B.VegasGrid(dim, nb)
    g.set_edges(edges)
    I, s, H, st = g.iterate_callback(f_host, n, seed, 2, batch_events=100_000)
    assert st == 0 and calls == [100_000, 100_000, 50_003]
    oI, oS, oH = O.iterate(edges, n, seed, 2, O.GENZ_PRODUCT_PEAK, p)
    assert I == pytest.approx(oI, rel=RTOL64) and s == pytest.approx(oS, rel=RTOL64)
    _hist_ok(H, oH)
    # the device integrand on the same grid object gives the same iteration
    g.set_params(B.VEGAS_F_GENZ_PRODUCT_PEAK, p)
    Id, sd, Hd, _ = g.iterate(n, seed, 2, B.VEGAS_F_GENZ_PRODUCT_PEAK, 64)
    assert I == pytest.approx(Id, rel=1e-12) and s == pytest.approx(sd, rel=1e-11)
    # refinement from the callback iteration's histogram
    assert g.refine(1.5) == 0
    want, _ = O.refine(edges, oH, 1.5)
    np.testing.assert_allclose(g.get_edges(), want, rtol=0, atol=1e-10)
    # a non-finite f is reported, not hidden
    I2, s2, _, st2 = g.iterate_callback(lambda x: np.full(x.shape[0], np.inf), 1000, seed, 0, batch_events=512)
    assert st2 == B.VEGAS_ENUMERIC
    g.close()


@pytest.mark.parametrize("name,fid,dim,nb,a", [("GAUSS", O.GAUSS, 6, 50, 0.2), ("GAUSS", O.GAUSS, 20, 50, 0.35),
                                                ("GENZ_PRODUCT_PEAK", O.GENZ_PRODUCT_PEAK, 12, 64, None)])
def test_user_integrand_in_fp32(B, name, fid, dim, nb, a):
    """VEGAS_F_USER with precision 32: the fp32 sampling map (C11) around the user's source, against the fp64 oracle at
    north_star's 1e-5 on I, sigma and H (per-dimension max-norm, reading F3); the fp64 run of the same source beside it."""
    p = W.gauss_params(a) if fid == O.GAUSS else W.genz_params(dim, 4)
    edges = W.adapted_edges(dim, nb, seed=dim)
    g = B.VegasGrid(dim, nb)
    g.set_user_integrand(getattr(U, name), p)
    g.set_edges(edges)
    n = 300_007
    oI, oS, oH = O.iterate(edges, n, 21, 3, fid, p, threads=THREADS)
    I, s, H, st = g.iterate(n, 21, 3, B.VEGAS_F_USER, 32)
    assert st == 0
    assert I == pytest.approx(oI, rel=1e-5) and s == pytest.approx(oS, rel=1e-5)
    assert np.all(np.abs(H - oH) <= 1e-5 * oH.max(axis=1, keepdims=True))
    assert np.any(H != oH)                                   # it really is the fp32 map
    I64, s64, H64, _ = g.iterate(n, 21, 3, B.VEGAS_F_USER, 64)
    assert I64 == pytest.approx(oI, rel=RTOL64) and s64 == pytest.approx(oS, rel=RTOL64)
    g.close()


def test_host_callback_overlapped_and_serial_batches_agree(B):
    """The two-slot form (device samples batch k+1 while the host evaluates batch k) and the one-slot serial form see the
    same batches in the same order and give the same sums; many batches, ragged tail, a slow callback."""
    import time
    dim, nb, n, seed = 5, 30, 123_457, 77
    edges = W.adapted_edges(dim, nb, seed=8)
    g = B.VegasGrid(dim, nb)
    g.set_edges(edges)
    seen = {True: [], False: []}

    def make(mode):
        def f_host(x):
            seen[mode].append((x.shape[0], float(x[0, 0]), float(x[-1, -1])))
            if len(seen[mode]) % 3 == 0:
                time.sleep(0.002)                      # the device is ahead of the host here
            return np.exp(-np.sum((x - 0.4) ** 2, axis=1) / 0.09)
        return f_host

    res = {}
    for mode in (True, False):
        res[mode] = g.iterate_callback(make(mode), n, seed, 1, batch_events=10_000, overlap=mode)
        assert res[mode][3] == 0
    assert seen[True] == seen[False] and len(seen[True]) == 13 and seen[True][-1][0] == 3_457
    assert res[True][0] == res[False][0] and res[True][1] == res[False][1]
    np.testing.assert_allclose(res[True][2], res[False][2], rtol=1e-13)     # the batch kernel's adds are unordered
    # against the oracle's sample: same x, f evaluated here, sums in numpy
    _, bins, x, fJ = O.sample(edges, seed, 1, 0, n, O.CONST)
    v = np.exp(-np.sum((x - 0.4) ** 2, axis=1) / 0.09) * fJ
    assert res[True][0] == pytest.approx(v.mean(), rel=1e-12)
    Hb = np.zeros((dim, nb))
    for j in range(dim):
        np.add.at(Hb[j], bins[:, j], v * v)
    np.testing.assert_allclose(res[True][2], Hb, rtol=1e-10)
    g.close()


def test_user_integrand_shape_limits_and_no_parameters(B):
    # a shape whose table plus one histogram copy exceed the 227 KB of shared memory has no fast path: refused
    g = B.VegasGrid(32, 256)
    with pytest.raises(B.VegasError) as ei:
        g.set_user_integrand(U.GAUSS, [0.1])
    assert ei.value.code == B.VEGAS_EINVAL
    g.close()
    # an integrand without parameters: f = prod_j 2 x_j integrates to 1
    src = """
    struct vegas_user_integrand {
        double prod;
        __device__ void begin(int dim, const double* p) { prod = 1.0; }
        __device__ void dim(int j, double x, const double* p) { prod *= 2.0 * x; }
        __device__ double finish(const double* p) { return prod; }
    };"""
    g = B.VegasGrid(3, 16)
    g.set_user_integrand(src)
    r = g.integrate(5, 1_000_000, 7, 1.5, B.VEGAS_F_USER, 64, n_skip=1)
    assert abs(r["I"] - 1.0) < 5 * r["sigma"] and r["sigma"] < 1e-3
    # host callback with a batch larger than the iteration, and the same f: same sample -> same first iteration
    g2 = B.VegasGrid(3, 16)
    I, s, H, st = g2.iterate_callback(lambda x: np.prod(2.0 * x, axis=1), 1_000_000, 7, 0, batch_events=1 << 21)
    g3 = B.VegasGrid(3, 16)
    g3.set_user_integrand(src)
    Iu, su, Hu, _ = g3.iterate(1_000_000, 7, 0, B.VEGAS_F_USER, 64)
    assert I == pytest.approx(Iu, rel=1e-12) and s == pytest.approx(su, rel=1e-11)
    np.testing.assert_allclose(H, Hu, rtol=1e-11)
    g.close(); g2.close(); g3.close()


def test_one_launch_refinement_of_more_dimensions_than_warps_equals_the_stand_alone_kernel(B):
    """The one-launch iteration refines one dimension per warp and, beyond the kernel's warp count, several in turn
    through the same shared scratch (a user kernel has 12 warps: dim 32 makes three rounds; the 24-warp built-in kernels
    two from dim 25 on).  The stand-alone refinement (K3, one CTA per dimension) never reuses scratch: same edges, bit
    for bit."""
    n, seed, alpha = 200_003, 5, 1.5
    for dim, nb, user in ((32, 50, True), (32, 37, True), (28, 50, False), (32, 64, False)):
        edges = []
        for one_launch in (True, False):
            g = B.VegasGrid(dim, nb)
            if user:
                g.set_user_integrand(U.GAUSS, [0.4])
                fid = B.VEGAS_F_USER
            else:
                g.set_params(B.VEGAS_F_GAUSS, [0.4])
                fid = B.VEGAS_F_GAUSS
            assert g.get_launch(fid, 64)["path"] == "rotated"
            g.set_edges(W.adapted_edges(dim, nb, seed=77))
            if one_launch:
                r = g.integrate(1, n, seed, alpha, fid, 64)
                assert r["status"] == 0
            else:
                assert g.iterate(n, seed, 0, fid, 64)[3] == 0
                assert g.refine(alpha) == 0
            edges.append(g.get_edges())
            g.close()
        assert np.array_equal(edges[0], edges[1]), (dim, nb, user, float(np.max(np.abs(edges[0] - edges[1]))))
        assert not np.array_equal(edges[0], W.adapted_edges(dim, nb, seed=77))


def test_observable_buffer_is_zero_before_any_iteration(B):
    g = B.VegasGrid(3, 20)
    g.set_user_integrand(U.GENZ_PRODUCT_PEAK_WITH_OBSERVABLE, W.genz_params(3, 8))
    g.set_observable(0.0, 1.0, 16)
    assert np.all(g.get_observable_hist() == 0.0)
    g.close()


def test_observable_histogram_during_integration(B):
    """PAPER.md:57 ("exporting histograms during integration"): O[k] += f*J for the bin of the user's observable.
    Expected values: numpy histogram of the oracle's per-event x and f*J (O.sample) over the same events."""
    dim, nb, n, seed = 7, 40, 200_003, 12
    p = W.genz_params(dim, 6)
    edges = W.adapted_edges(dim, nb, seed=9)
    g = B.VegasGrid(dim, nb)
    g.set_edges(edges)
    g.set_user_integrand(U.GENZ_PRODUCT_PEAK_WITH_OBSERVABLE, p)
    lo, hi, nobs = 0.2, 0.9, 35
    g.set_observable(lo, hi, nobs)
    I, s, H, st = g.iterate(n, seed, 4, B.VEGAS_F_USER, 64, chunk_events=70_000)
    got = g.get_observable_hist()
    _, _, ox, of = O.sample(edges, seed, 4, 0, n, O.GENZ_PRODUCT_PEAK, p)
    x = ox[:, dim - 1]
    k = np.floor((x - lo) / (hi - lo) * nobs)
    inside = (k >= 0) & (k < nobs)
    want = np.bincount(k[inside].astype(int), weights=of[inside], minlength=nobs)
    np.testing.assert_allclose(got, want, rtol=1e-10)
    assert 0 < want.sum() < of.sum()                           # the window cuts events on both sides
    oI, oS, oH = O.iterate(edges, n, seed, 4, O.GENZ_PRODUCT_PEAK, p)
    assert I == pytest.approx(oI, rel=RTOL64) and s == pytest.approx(oS, rel=RTOL64)
    _hist_ok(H, oH)
    # it is the LAST iteration's histogram; an integrand without observable() leaves it at zero
    g.iterate(1000, seed, 5, B.VEGAS_F_USER, 64)
    assert g.get_observable_hist().sum() < 0.05 * want.sum()
    g.set_user_integrand(U.GENZ_PRODUCT_PEAK, p)
    g.iterate(n, seed, 4, B.VEGAS_F_USER, 64)
    assert np.all(g.get_observable_hist() == 0.0)
    with pytest.raises(B.VegasError):
        g.set_observable(1.0, 1.0, 10)
    with pytest.raises(B.VegasError):
        g.set_observable(0.0, 1.0, 129)
    g.close()
