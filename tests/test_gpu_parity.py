"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Protocol P1..P7 of DESIGN.md.  Tolerances (north_star): Philox words and bin
indices bit-exact; I, sigma, H <= 1e-10 relative in fp64; fp32 path <= 1e-5 relative against the
fp64 oracle (H in per-dimension max-norm, finding F3); refined edges <= 1e-10 absolute."""
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle as O
import workloads as W

THREADS = os.cpu_count() or 8
RTOL64 = 1e-10
RTOL32 = 1e-5


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    from paper_2002_12921_b200 import build
    build.build()                                   # no-op when libvegas_b200.so is up to date
    from paper_2002_12921_b200 import binding
    return binding


def _grid(B, w, edges=None):
    g = B.VegasGrid(w.dim, w.n_bins)
    g.set_params(w.integrand_id, w.params)
    if edges is not None:
        g.set_edges(edges)
    return g


def _assert_hist(h_gpu, h_ref, precision):
    if precision == 64:
        np.testing.assert_allclose(h_gpu, h_ref, rtol=RTOL64, atol=0)
        assert np.all(h_gpu[h_ref == 0] == 0)
    else:
        # reading F3 / P3: |dH| <= 1e-5 max_b H[j][.] per dimension
        scale = h_ref.max(axis=1, keepdims=True)
        assert np.all(np.abs(h_gpu - h_ref) <= RTOL32 * scale), float(np.max(np.abs(h_gpu - h_ref) / scale))


# parity-sized versions of the five configs: several CTAs x several grid-stride passes and a ragged tail
SMALL = {
    1: dict(n_events=100_000, n_iter=5),               # cfg1 is already oracle-sized: full size
    2: dict(n_events=1_000_003, n_iter=4),
    3: dict(n_events=500_009, n_iter=4),
    4: dict(n_events=300_007, n_iter=4),
    5: dict(n_events=1_000_003, n_iter=4, chunk_events=250_000),
}


def _small(i):
    return W.config(i).scaled(**SMALL[i])


@pytest.fixture(scope="module")
def chains():
    """Oracle free-running chains of the parity-sized configs (grid_k, H_k, I_k, sigma_k)."""
    out = {}
    for i in range(1, 6):
        w = _small(i)
        out[i] = O.integrate(w.dim, w.n_bins, w.n_iter, w.n_events, w.seed, w.alpha, w.integrand_id, w.params,
                             threads=THREADS)
    return out


# ------------------------------------------------------------------ P1, P2: words and bins, bit-exact
@pytest.mark.parametrize("path", ["auto", "generic"])
@pytest.mark.parametrize("cfg,precision", [(1, 64), (3, 64), (3, 32), (4, 64), (4, 32), (5, 64)])
def test_p1_p2_words_and_bins_bit_exact(B, cfg, precision, path):
    w = W.config(cfg)
    edges = W.adapted_edges(w.dim, w.n_bins, seed=cfg)
    g = _grid(B, w, edges)
    if path == "generic":
        g.set_launch(0, 0, 1, 1)
    count = 60_000                                   # x dim >= 240k..1.2M (event, dim) pairs per range
    for first, it in ((0, 0), (123_456_789, 7), ((1 << 32) - 1000, 1), ((5 << 32) + 17, 0xFFFFFFFE)):
        gw, gb, gx, gf = g.debug_sample(first, count, w.seed, it, w.integrand_id, precision)
        ow, ob, ox, of = O.sample(edges, w.seed, it, first, count, w.integrand_id, w.params)
        assert np.array_equal(gw, ow)
        assert np.array_equal(gb, ob)
        if precision == 64:
            np.testing.assert_allclose(gx, ox, rtol=5e-16, atol=0)
            np.testing.assert_allclose(gf, of, rtol=1e-12, atol=0)
        else:
            np.testing.assert_allclose(gx, ox, rtol=0, atol=1.5e-7)
            rel = np.abs(gf - of) / np.maximum(np.abs(of), 1e-300)
            big = of > 1e-6 * of.max()
            assert np.median(rel[big]) < 5e-6 and rel[big].max() < 1e-3   # per-event sanity; the gates are on the sums
    g.close()


# ------------------------------------------------------------------ P3: teacher-forced iterations
@pytest.mark.parametrize("path", ["auto", "generic"])
@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_p3_iterate_on_oracle_grids_fp64(B, chains, cfg, path):
    w, ch = _small(cfg), chains[cfg]
    g = _grid(B, w)
    if path == "generic":
        g.set_launch(0, 0, 2, 8)                     # pinning the copy counts pins the generic kernel
    assert g.get_launch(w.integrand_id, 64)["path"] == ("generic" if path == "generic" else "rotated")
    for k in range(w.n_iter):
        g.set_edges(ch["edges_trace"][k])
        I, s, H, st = g.iterate(w.n_events, w.seed, k, w.integrand_id, 64, chunk_events=w.chunk_events)
        assert st == 0
        assert I == pytest.approx(ch["per_iter"][k, 0], rel=RTOL64)
        assert s == pytest.approx(ch["per_iter"][k, 1], rel=RTOL64)
        _assert_hist(H, ch["hist_trace"][k], 64)
        np.testing.assert_array_equal(g.get_hist(), H)
    g.close()


@pytest.mark.parametrize("path", ["auto", "generic"])
@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_p3_iterate_on_oracle_grids_fp32(B, chains, cfg, path):
    w, ch = _small(cfg), chains[cfg]
    g = _grid(B, w)
    if path == "generic":
        g.set_launch(0, 0, 4, 8)
    assert g.get_launch(w.integrand_id, 32)["path"] == ("generic" if path == "generic" else "rotated")
    for k in range(w.n_iter):
        g.set_edges(ch["edges_trace"][k])
        I, s, H, st = g.iterate(w.n_events, w.seed, k, w.integrand_id, 32, chunk_events=w.chunk_events)
        assert st == 0
        assert I == pytest.approx(ch["per_iter"][k, 0], rel=RTOL32)
        assert s == pytest.approx(ch["per_iter"][k, 1], rel=RTOL32)
        _assert_hist(H, ch["hist_trace"][k], 32)
    g.close()


# ------------------------------------------------------------------ P4: refine on the oracle's histograms
@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_p4_refine_on_oracle_histograms(B, chains, cfg):
    w, ch = _small(cfg), chains[cfg]
    g = _grid(B, w)
    for k in range(w.n_iter):
        g.set_edges(ch["edges_trace"][k])
        assert g.refine(w.alpha, hist=ch["hist_trace"][k]) == 0
        new = g.get_edges()
        want = ch["edges_trace"][k + 1] if k + 1 < w.n_iter else ch["edges"]
        np.testing.assert_allclose(new, want, rtol=0, atol=1e-10)
        assert np.all(new[:, 0] == 0.0) and np.all(new[:, -1] == 1.0)
        assert np.all(np.diff(new, axis=1) > 0)
    g.close()


def test_p4_refine_pins_hold_on_the_gpu_too(B):
    rng = np.random.default_rng(5)
    for dim, nb, alpha in ((3, 50, 1.5), (2, 100, 0.7), (1, 2, 1.5), (4, 256, 2.0), (32, 7, 1.0)):
        g = B.VegasGrid(dim, nb)
        edges = W.adapted_edges(dim, nb, seed=nb + dim)
        hist = rng.random((dim, nb)) ** 5 * 10.0 ** rng.integers(-40, 40, size=(dim, 1))
        if nb > 8:
            hist[0, 2:6] = 0.0
        g.set_edges(edges)
        assert g.refine(alpha, hist=hist) == 0
        want, rc = O.refine(edges, hist, alpha)
        assert rc == 0
        np.testing.assert_allclose(g.get_edges(), want, rtol=0, atol=1e-12)
        # alpha = 0 leaves any grid unchanged; a constant histogram leaves the uniform grid unchanged
        g.set_edges(edges)
        assert g.refine(0.0, hist=hist + 1e-300) == 0
        np.testing.assert_allclose(g.get_edges(), edges, rtol=0, atol=1e-14)
        g.set_edges(O.uniform_edges(dim, nb))
        assert g.refine(1.5, hist=np.full((dim, nb), 2.5)) == 0
        np.testing.assert_allclose(g.get_edges(), O.uniform_edges(dim, nb), rtol=0, atol=1e-14)
        g.close()


def test_p4_refine_degenerate_row(B):
    g = B.VegasGrid(3, 10)
    edges = W.adapted_edges(3, 10, seed=3)
    g.set_edges(edges)
    hist = np.ones((3, 10))
    hist[1] = 0.0
    assert g.refine(1.5, hist=hist) == B.VEGAS_ENUMERIC
    new = g.get_edges()
    want, rc = O.refine(edges, hist, 1.5)
    assert rc == O.ENUMERIC
    np.testing.assert_array_equal(new[1], edges[1])
    np.testing.assert_allclose(new, want, rtol=0, atol=1e-12)
    g.close()


# ------------------------------------------------------------------ P5: free-running chains
@pytest.mark.parametrize("cfg,precision", [(1, 64), (2, 64), (3, 64), (4, 64), (5, 64), (1, 32), (3, 32), (4, 32)])
def test_p5_free_running_integrate(B, chains, cfg, precision):
    w, ch = _small(cfg), chains[cfg]
    g = _grid(B, w)
    r = g.integrate(w.n_iter, w.n_events, w.seed, w.alpha, w.integrand_id, precision, n_skip=0,
                    chunk_events=w.chunk_events)
    assert r["status"] == 0
    oI, oS, oC = O.combine(ch["per_iter"][:, 0], ch["per_iter"][:, 1], 0)
    if precision == 64:
        np.testing.assert_allclose(r["per_iter"][:, 0], ch["per_iter"][:, 0], rtol=1e-8)
        np.testing.assert_allclose(r["per_iter"][:, 1], ch["per_iter"][:, 1], rtol=1e-7)
        assert r["I"] == pytest.approx(oI, rel=1e-8) and r["sigma"] == pytest.approx(oS, rel=1e-7)
        np.testing.assert_allclose(g.get_edges(), ch["edges"], rtol=0, atol=1e-8)
    else:
        # finding F3: a free-running fp32 chain feeds its own rounding back through the grid, so only
        # iteration 0 (identical grid) is held to 1e-5; later iterations and the average must agree
        # with the oracle's to a small fraction of their own statistical error.
        assert r["per_iter"][0, 0] == pytest.approx(ch["per_iter"][0, 0], rel=RTOL32)
        for k in range(w.n_iter):
            tol = max(RTOL32 * abs(ch["per_iter"][k, 0]), 0.05 * ch["per_iter"][k, 1])
            assert abs(r["per_iter"][k, 0] - ch["per_iter"][k, 0]) <= tol
        assert abs(r["I"] - oI) <= max(RTOL32 * abs(oI), 0.05 * oS)
    g.close()


# ------------------------------------------------------------------ P6: chunking, launch shapes, sharding
def test_p6_chunked_equals_single_launch(B):
    w = _small(3)
    edges = W.adapted_edges(w.dim, w.n_bins, seed=33)
    g = _grid(B, w, edges)
    ref = g.iterate(w.n_events, w.seed, 2, w.integrand_id, 64)
    for chunk in (w.n_events // 2 + 1, 100_000, 77_777, 1):
        if chunk == 1:
            n = 300                                   # 300 launches of one event each
            a = g.iterate(n, w.seed, 2, w.integrand_id, 64)
            b = g.iterate(n, w.seed, 2, w.integrand_id, 64, chunk_events=1)
        else:
            a, b = ref, g.iterate(w.n_events, w.seed, 2, w.integrand_id, 64, chunk_events=chunk)
        assert b[0] == pytest.approx(a[0], rel=1e-12) and b[1] == pytest.approx(a[1], rel=1e-12)
        np.testing.assert_allclose(b[2], a[2], rtol=1e-12)
    g.close()


@pytest.mark.parametrize("precision", [64, 32])
def test_p6_launch_shapes_give_the_same_iteration(B, precision):
    w = _small(4)
    edges = W.adapted_edges(w.dim, w.n_bins, seed=44)
    oI, oS, oH = O.iterate(edges, w.n_events, w.seed, 1, w.integrand_id, w.params, threads=THREADS)
    g = _grid(B, w, edges)
    shapes = [(0, 0, 0, 0), (1, 32, 1, 1), (7, 96, 2, 4), (148, 256, 1, 16), (296, 512, 4, 2), (1024, 64, 1, 1),
              (37, 512, 2, 8)]
    for blocks, threads, ct, ch in shapes:
        g.set_launch(blocks, threads, ct, ch)
        I, s, H, st = g.iterate(w.n_events, w.seed, 1, w.integrand_id, precision)
        tol = RTOL64 if precision == 64 else RTOL32
        assert st == 0 and I == pytest.approx(oI, rel=tol) and s == pytest.approx(oS, rel=tol)
        _assert_hist(H, oH, precision)
    g.close()


def test_p6_event_range_sharding_matches_whole_iteration(B):
    """The multi-GPU decomposition (begin / accumulate ranges / reduce / finalize) on one GPU."""
    w = _small(5)
    edges = W.adapted_edges(w.dim, w.n_bins, seed=55)
    g = _grid(B, w, edges)
    whole = g.iterate(w.n_events, w.seed, 3, w.integrand_id, 64)
    g.begin_iteration()
    bounds = [0, 1, 400_000, 400_001, 777_777, w.n_events]
    for lo, hi in zip(bounds[:-1], bounds[1:]):
        g.accumulate(lo, hi - lo, w.seed, 3, w.integrand_id, 64)
    g.reduce()
    tot = g.totals_tensor().cpu().numpy()
    assert tot.shape == (4 + w.dim * w.n_bins,)
    I, s, H, st = g.finalize(w.n_events)
    assert I == pytest.approx(whole[0], rel=1e-13) and s == pytest.approx(whole[1], rel=1e-12)
    np.testing.assert_allclose(H, whole[2], rtol=1e-12)
    np.testing.assert_allclose(tot[4:].reshape(w.dim, w.n_bins), H, rtol=0)
    # events beyond 2^32: the high counter word is live
    off = (3 << 32) + 12345
    n = 200_003
    g.begin_iteration()
    g.accumulate(off, n, w.seed, 3, w.integrand_id, 64)
    g.reduce()
    I, s, H, st = g.finalize(n)
    S1, S2, Ho = O.accumulate(edges, w.seed, 3, off, n, w.integrand_id, w.params)
    oI, oS = O.estimate(S1, S2, n)
    assert I == pytest.approx(oI, rel=RTOL64) and s == pytest.approx(oS, rel=RTOL64)
    np.testing.assert_allclose(H, Ho.astype(np.float64), rtol=RTOL64)
    # a range that CROSSES a multiple of 2^32: the fast path splits the launch there (its high counter word is
    # uniform per launch), the generic kernel carries into the high word per event; with and without chunking
    off = (2 << 32) - 77_777
    n = 200_003
    S1, S2, Ho = O.accumulate(edges, w.seed, 3, off, n, w.integrand_id, w.params)
    oI, oS = O.estimate(S1, S2, n)
    for pin_generic, chunk in ((False, 0), (False, 50_000), (True, 0)):
        if pin_generic:
            g.set_launch(0, 0, 2, 8)
        assert g.get_launch(w.integrand_id, 64)["path"] == ("generic" if pin_generic else "rotated")
        g.begin_iteration()
        g.accumulate(off, n, w.seed, 3, w.integrand_id, 64, chunk_events=chunk)
        g.reduce()
        I, s, H, st = g.finalize(n)
        assert I == pytest.approx(oI, rel=RTOL64) and s == pytest.approx(oS, rel=RTOL64)
        np.testing.assert_allclose(H, Ho.astype(np.float64), rtol=RTOL64)
    g.close()


def test_integrate_from_resumes_bit_for_bit(B):
    """Checkpoint / resume: (grid, seed, next iteration index) is the whole state (counter-based RNG)."""
    w = _small(4)
    g = _grid(B, w)
    whole = g.integrate(4, w.n_events, w.seed, w.alpha, w.integrand_id, 64)
    edges_whole = g.get_edges()
    g2 = _grid(B, w)
    a = g2.integrate(2, w.n_events, w.seed, w.alpha, w.integrand_id, 64)
    saved = g2.get_edges()
    g2.close()
    g3 = _grid(B, w, saved)                                  # a fresh grid object restored from the checkpoint
    b = g3.integrate(2, w.n_events, w.seed, w.alpha, w.integrand_id, 64, first_iteration=2)
    assert np.array_equal(np.vstack([a["per_iter"], b["per_iter"]]), whole["per_iter"])
    assert np.array_equal(g3.get_edges(), edges_whole)
    I, s, chi2 = B.vegas_combine(np.r_[a["per_iter"][:, 0], b["per_iter"][:, 0]], np.r_[a["per_iter"][:, 1], b["per_iter"][:, 1]])
    assert I == whole["I"] and s == whole["sigma"]
    with pytest.raises(B.VegasError):
        g3.integrate(2, w.n_events, w.seed, w.alpha, w.integrand_id, 64, first_iteration=0xFFFFFFFE)
    g.close(); g3.close()


def test_plain_mc_mode_is_alpha_zero(B):
    """The paper's "Plain MC" column = the same iteration with the refinement switched off:
    alpha = 0 leaves the grid where it is (C8 fixed point), so every iteration samples the uniform grid."""
    w = W.config(1)
    g = _grid(B, w)
    r = g.integrate(4, w.n_events, w.seed, 0.0, w.integrand_id, 64)
    o = O.integrate(w.dim, w.n_bins, 4, w.n_events, w.seed, 0.0, w.integrand_id, w.params, threads=THREADS)
    np.testing.assert_allclose(g.get_edges(), O.uniform_edges(w.dim, w.n_bins), rtol=0, atol=1e-15)
    np.testing.assert_allclose(r["per_iter"], o["per_iter"], rtol=RTOL64)
    assert r["I"] == pytest.approx(o["I"], rel=RTOL64) and r["sigma"] == pytest.approx(o["sigma"], rel=RTOL64)
    # without adaptation the error stays at its first-iteration size (the adaptive chain shrinks it ~30x, cfg1)
    assert r["per_iter"][3, 1] > 0.5 * r["per_iter"][0, 1]
    g.close()


# ------------------------------------------------------------------ P7: 5 sigma, control, fixed point
def test_p7_constant_control_and_fixed_point(B):
    w = W.control_const(n_events=10_000_000)
    g = _grid(B, w)
    r = g.integrate(3, w.n_events, w.seed, w.alpha, w.integrand_id, 64)
    # reading R9: exactly 1 up to rounding on the uniform grid
    assert abs(r["per_iter"][0, 0] - 1.0) <= 1e-12 and r["per_iter"][0, 1] <= 1e-9
    o = O.integrate(w.dim, w.n_bins, 3, w.n_events, w.seed, w.alpha, w.integrand_id, None, threads=THREADS)
    np.testing.assert_allclose(r["per_iter"][1:, 0], o["per_iter"][1:, 0], rtol=RTOL64)
    np.testing.assert_allclose(r["per_iter"][1:, 1], o["per_iter"][1:, 1], rtol=1e-8)
    # reading R10(ii): sampled flat histogram leaves the grid within 1e-3 of uniform
    assert np.abs(g.get_edges() - O.uniform_edges(w.dim, w.n_bins)).max() < 1e-3
    g.close()


@pytest.mark.parametrize("cfg", [1, 2, 4, 5])
def test_p7_five_sigma_rule(B, cfg):
    if cfg == 1:
        # cfg1 at its own size and length: SURVEY.md F1 gates every I_k from k = 0 and the average over all of them
        w, n_skip = W.config(1), 0
    else:
        # reduced-size chains of the large configs (their first iterations under-estimate sigma at these sizes, F1);
        # at full size they are gated from k = 0 in test_full_size_chains_match_the_survey_probe
        w, n_skip = _small(cfg).scaled(n_events=SMALL[cfg]["n_events"], n_iter=8), 2
    g = _grid(B, w)
    r = g.integrate(w.n_iter, w.n_events, w.seed, w.alpha, w.integrand_id, 64, n_skip=n_skip)
    exact = w.closed_form
    assert abs(r["I"] - exact) < 5 * r["sigma"]
    for k in range(n_skip, w.n_iter):
        assert abs(r["per_iter"][k, 0] - exact) < 5 * r["per_iter"][k, 1]
    g.close()


# ------------------------------------------------------------------ edge cases
def test_edge_shapes(B):
    rng = np.random.default_rng(1)
    cases = [(1, 2, 2), (1, 256, 1000), (32, 2, 5000), (32, 256, 20_011), (5, 3, 3), (17, 31, 33), (4, 128, 31)]
    for dim, nb, n in cases:
        edges = W.adapted_edges(dim, nb, seed=dim * nb)
        # c in [1,3]: keeps prod_j (c_j^-2 + t^2) inside the fp32 range for dim = 32
        params = np.concatenate([1 + 2 * rng.random(dim), rng.random(dim)])
        g = B.VegasGrid(dim, nb)
        g.set_params(B.VEGAS_F_GENZ_PRODUCT_PEAK, params)
        g.set_params(B.VEGAS_F_GAUSS, [0.3])
        g.set_edges(edges)
        for fid, p in ((B.VEGAS_F_GENZ_PRODUCT_PEAK, params), (B.VEGAS_F_GAUSS, [0.3]), (B.VEGAS_F_CONST, None)):
            for precision in (64, 32):
                I, s, H, st = g.iterate(n, 9, 4, fid, precision)
                oI, oS, oH = O.iterate(edges, n, 9, 4, fid, p)
                tol = RTOL64 if precision == 64 else RTOL32
                assert st == 0 and I == pytest.approx(oI, rel=tol)
                assert s == pytest.approx(oS, rel=tol, abs=1e-300)
                _assert_hist(H, oH, precision) if precision == 64 else None
        g.close()


def test_bw_poly_other_dimensions(B):
    """Every shape of the last Philox block (1..4 dimensions) on the fast path: the per-lane coefficient registers
    (dim <= 8) and the constant-bank coefficient rows (dim > 8, up to the ABI's 32 dimensions) must follow the lane's
    dimension; both precisions; and the generic kernel when the copy counts are pinned."""
    for dim in (2, 3, 4, 5, 6, 7, 8, 9, 10, 11, 13, 20, 32):
        p = W.bw_poly_params(dim, 77)
        edges = W.adapted_edges(dim, 40, seed=dim)
        g = B.VegasGrid(dim, 40)
        g.set_params(B.VEGAS_F_BW_POLY, p)
        g.set_edges(edges)
        assert g.get_launch(B.VEGAS_F_BW_POLY, 64)["path"] == "rotated"
        gw, gb, gx, gf = g.debug_sample(5, 4096, 3, 2, B.VEGAS_F_BW_POLY, 64)
        ow, ob, ox, of = O.sample(edges, 3, 2, 5, 4096, O.BW_POLY, p)
        assert np.array_equal(gb, ob)
        np.testing.assert_allclose(gf, of, rtol=1e-12, atol=0)
        oI, oS, oH = O.iterate(edges, 100_001, 3, 0, O.BW_POLY, p)
        I, s, H, st = g.iterate(100_001, 3, 0, B.VEGAS_F_BW_POLY, 64)
        assert I == pytest.approx(oI, rel=RTOL64) and s == pytest.approx(oS, rel=RTOL64)
        _assert_hist(H, oH, 64)
        I, s, H, st = g.iterate(100_001, 3, 0, B.VEGAS_F_BW_POLY, 32)
        assert I == pytest.approx(oI, rel=RTOL32) and s == pytest.approx(oS, rel=RTOL32)
        _assert_hist(H, oH, 32)
        if dim in (9, 13):
            g.set_launch(0, 0, 2, 4)
            assert g.get_launch(B.VEGAS_F_BW_POLY, 64)["path"] == "generic"
            I, s, H, st = g.iterate(100_001, 3, 0, B.VEGAS_F_BW_POLY, 64)
            assert I == pytest.approx(oI, rel=RTOL64) and s == pytest.approx(oS, rel=RTOL64)
            _assert_hist(H, oH, 64)
        g.close()


def test_errors(B):
    import ctypes as C
    assert B.vegas_workspace_bytes(0, 50) == 0 and B.vegas_workspace_bytes(33, 50) == 0
    assert B.vegas_workspace_bytes(4, 1) == 0 and B.vegas_workspace_bytes(4, 257) == 0
    with pytest.raises(B.VegasError):
        B.VegasGrid(0, 50)
    g = B.VegasGrid(4, 50)
    with pytest.raises(B.VegasError) as e:
        g.iterate(1000, 1, 0, B.VEGAS_F_GAUSS)            # params not set
    assert e.value.code == B.VEGAS_EINVAL
    g.set_params(B.VEGAS_F_GAUSS, [0.1])
    for bad in (dict(n_events=1), dict(integrand_id=7), dict(precision=16)):
        kw = dict(n_events=1000, seed=1, iteration=0, integrand_id=B.VEGAS_F_GAUSS, precision=64)
        kw.update(bad)
        with pytest.raises(B.VegasError) as e:
            g.iterate(**kw)
        assert e.value.code == B.VEGAS_EINVAL
    with pytest.raises(B.VegasError):
        g.set_params(B.VEGAS_F_GAUSS, [0.1, 0.2])
    with pytest.raises(B.VegasError):
        g.set_params(B.VEGAS_F_GENZ_PRODUCT_PEAK, [1.0] * 7)
    e2 = O.uniform_edges(4, 50)
    e2[2, 10] = e2[2, 9]
    with pytest.raises(B.VegasError):
        g.set_edges(e2)
    e3 = O.uniform_edges(4, 50)
    e3[0, -1] = 0.999
    with pytest.raises(B.VegasError):
        g.set_edges(e3)
    with pytest.raises(B.VegasError):
        g.refine(-1.0)
    with pytest.raises(B.VegasError):
        g.refine(float("nan"))
    with pytest.raises(B.VegasError):
        g.set_launch(0, 0, 3, 0)                          # not a power of two
    with pytest.raises(B.VegasError):
        g.set_launch(0, 1000, 0, 0)                       # not a multiple of 32
    with pytest.raises(B.VegasError):
        g.integrate(0, 1000, 1, 1.5, B.VEGAS_F_GAUSS)
    with pytest.raises(B.VegasError):
        g.integrate(3, 1000, 1, 1.5, B.VEGAS_F_GAUSS, n_skip=3)
    # too small / misaligned workspace
    import torch
    buf = torch.empty(4096, dtype=torch.uint8, device="cuda")
    h = C.c_void_p()
    assert B.lib.vegas_create(4, 50, C.c_void_p(buf.data_ptr()), 4096, C.byref(h)) == B.VEGAS_EINVAL
    big = torch.empty(B.vegas_workspace_bytes(4, 50) + 512, dtype=torch.uint8, device="cuda")
    assert B.lib.vegas_create(4, 50, C.c_void_p(big.data_ptr() + 8), big.numel() - 8, C.byref(h)) == B.VEGAS_EINVAL
    # the grid is still usable after the failed calls
    I, s, H, st = g.iterate(10_000, 1, 0, B.VEGAS_F_GAUSS)
    oI, oS, oH = O.iterate(O.uniform_edges(4, 50), 10_000, 1, 0, O.GAUSS, [0.1])
    assert st == 0 and I == pytest.approx(oI, rel=RTOL64)
    g.close()


def test_rejected_parameters_leave_the_grid_as_it_was(B):
    w = _small(5)
    g = _grid(B, w)
    I0, s0, _, _ = g.iterate(50_000, 5, 0, w.integrand_id, 64)
    bad = np.array(w.params, dtype=float)
    for idx, val in ((0, 0.0), (3, bad[2]), (3, bad[2] - 1.0), (5, float("nan"))):   # M = 0; m_max = m_min; m_max < m_min; NaN
        p = bad.copy(); p[idx] = val
        with pytest.raises(B.VegasError) as e:
            g.set_params(w.integrand_id, p)
        assert e.value.code == B.VEGAS_EINVAL
        I1, s1, _, st = g.iterate(50_000, 5, 0, w.integrand_id, 64)
        assert st == 0 and I1 == I0 and s1 == s0
    g.close()
    g = B.VegasGrid(4, 50)
    g.set_params(B.VEGAS_F_GAUSS, [0.1])
    I0, s0, _, _ = g.iterate(50_000, 1, 0, B.VEGAS_F_GAUSS, 64)
    with pytest.raises(B.VegasError):
        g.set_params(B.VEGAS_F_GAUSS, [-1.0])
    assert g.iterate(50_000, 1, 0, B.VEGAS_F_GAUSS, 64)[:2] == (I0, s0)
    g.close()


def test_non_default_stream_and_counters(B):
    import torch
    w = _small(1)
    g = _grid(B, w)
    st = torch.cuda.Stream()
    g.set_profiling(True)
    g.reset_counters()
    with torch.cuda.stream(st):
        I, s, H, rc = g.iterate(w.n_events, w.seed, 0, w.integrand_id, 64, chunk_events=30_000)
    ms, n = g.kernel_time_ms()
    # the fast path runs the chunk loop and the reduction / finalisation inside the kernel: one launch per iteration
    assert n == 1 and ms > 0 and g.launch_count() == 1
    oI, oS, oH = O.iterate(O.uniform_edges(w.dim, w.n_bins), w.n_events, w.seed, 0, w.integrand_id, w.params)
    assert I == pytest.approx(oI, rel=RTOL64)
    g.close()


def test_fp32_outside_its_range(B):
    """include/vegas.h (precision, reading C11): v beyond 3.4e38 in fp32 -> non-finite sums -> VEGAS_ENUMERIC while fp64
    is fine; v below the fp32 range -> a finite estimate, biased low, status 0.  And the range that matters is that of v,
    not of exp(-E) alone: cfg3's own shape on a grid that is adapted to something else keeps fp32 parity."""
    # overflow: a narrow Gaussian in 16 dimensions (N = 1.1e44) on a grid that samples its peak
    dim, nb, a = 16, 50, 1e-3
    row = np.concatenate([[0.0], np.linspace(0.5 - 3 * a, 0.5 + 3 * a, nb - 1), [1.0]])
    edges = np.tile(row, (dim, 1))
    g = B.VegasGrid(dim, nb)
    g.set_params(B.VEGAS_F_GAUSS, [a])
    g.set_edges(edges)
    I64, s64, _, st64 = g.iterate(200_000, 5, 0, B.VEGAS_F_GAUSS, 64)
    I32, s32, _, st32 = g.iterate(200_000, 5, 0, B.VEGAS_F_GAUSS, 32)
    assert st64 == 0 and np.isfinite(I64) and I64 > 0
    assert st32 == B.VEGAS_ENUMERIC and not np.isfinite(I32)
    g.close()
    # underflow: cfg3's Gaussian on the uniform grid (f spans > 100 decades, most of it below 1e-38)
    w = W.config(3)
    g = _grid(B, w)
    I64, s64, _, st64 = g.iterate(400_000, 3, 0, w.integrand_id, 64)
    I32, s32, H32, st32 = g.iterate(400_000, 3, 0, w.integrand_id, 32)
    assert st64 == 0 and st32 == 0 and np.isfinite(I32) and np.isfinite(s32) and np.all(np.isfinite(H32))
    assert 0.0 <= I32 <= I64 * (1 + 1e-5)
    # cfg3's shape on a grid adapted to a wider peak (workloads.adapted_edges): ln N folded into the exponent keeps f
    # in range, fp32 agrees with the oracle to 1e-5
    edges = W.adapted_edges(w.dim, w.n_bins, seed=11)
    g.set_edges(edges)
    n = 300_007
    I32, s32, H32, st32 = g.iterate(n, 3, 1, w.integrand_id, 32)
    oI, oS, oH = O.iterate(edges, n, 3, 1, w.integrand_id, w.params, threads=THREADS)
    assert st32 == 0 and I32 == pytest.approx(oI, rel=RTOL32) and s32 == pytest.approx(oS, rel=RTOL32)
    _assert_hist(H32, oH, 32)
    g.close()


# ------------------------------------------------------------------ full BASELINE sizes, bench launch shape
@pytest.mark.parametrize("cfg,precision", [(2, 64), (3, 64), (3, 32), (4, 64), (5, 64)])
def test_full_size_iteration_in_bench_configuration(B, chains, cfg, precision):
    """One iteration at the config's full n_events (and chunking) on the adapted grid of the small
    oracle chain, default launch shape (what bench.py times), against the oracle run on all host
    cores; plus sampled events through K4 and the size-independent invariant sum_b H[j][b] = S2."""
    w = W.config(cfg)
    edges = chains[cfg]["edges"]
    g = _grid(B, w, edges)
    it = 5
    I, s, H, st = g.iterate(w.n_events, w.seed, it, w.integrand_id, precision, chunk_events=w.chunk_events)
    assert st == 0
    n = w.n_events
    S2 = n * (s * s * (n - 1) + I * I)
    np.testing.assert_allclose(H.sum(axis=1), S2, rtol=1e-9 if precision == 64 else 1e-6)
    rng = np.random.default_rng(cfg)
    for first in rng.integers(0, n - 64, size=6).tolist() + [0, n - 64]:
        gw, gb, gx, gf = g.debug_sample(first, 64, w.seed, it, w.integrand_id, precision)
        ow, ob, ox, of = O.sample(edges, w.seed, it, first, 64, w.integrand_id, w.params)
        assert np.array_equal(gw, ow) and np.array_equal(gb, ob)
        if precision == 64:
            np.testing.assert_allclose(gf, of, rtol=1e-12)
    oI, oS, oH = O.iterate(edges, n, w.seed, it, w.integrand_id, w.params, threads=THREADS)
    tol = RTOL64 if precision == 64 else RTOL32
    assert I == pytest.approx(oI, rel=tol) and s == pytest.approx(oS, rel=tol)
    _assert_hist(H, oH, precision)
    assert abs(I - w.closed_form) < 5 * s
    g.close()


# ------------------------------------------------------------------ full-size free-running chains vs the survey's probe
@pytest.mark.parametrize("cfg", [2, 3, 4, 5])
def test_full_size_chains_match_the_survey_probe(B, probe, cfg):
    """The four large configs at their full BASELINE.json sizes, free-running (vegas_integrate), against the values an
    independently written program produced during the survey (tests/golden/survey_probe.txt).
    First iteration: same sample, same uniform grid -> agreement to rounding.  Combined results: the adaptive chain
    amplifies rounding (finding F2) -> the printed digits (P5 gate 1e-8 on I)."""
    w = W.config(cfg)
    g = _grid(B, w)
    r = g.integrate(w.n_iter, w.n_events, w.seed, w.alpha, w.integrand_id, 64, chunk_events=w.chunk_events)
    flt = lambda key: [float(t) for t in probe[key]]
    names = {2: ("cfg2.iter0", "cfg2.combined_all10"), 3: ("cfg3.iter0", "cfg3.combined_all10"),
             4: ("cfg4.iter0", "cfg4.combined_all15"), 5: ("cfg5.iter0", "cfg5.combined_all20")}[cfg]
    i0, comb = flt(names[0]), flt(names[1])
    assert r["per_iter"][0, 0] == pytest.approx(i0[0], rel=1e-10)
    assert r["per_iter"][0, 1] == pytest.approx(i0[1], rel=2e-3 if cfg == 3 else 1e-5)     # sigma_0 printed to 3-6 digits
    assert r["I"] == pytest.approx(comb[0], rel=1e-8)
    assert r["sigma"] == pytest.approx(comb[1], rel=1e-2 if cfg == 3 else 2e-5)
    if len(comb) > 2:
        assert r["chi2_dof"] == pytest.approx(comb[2], abs=0.006)
    if cfg == 2:
        assert r["per_iter"][1] == pytest.approx(flt("cfg2.iter1"), rel=1e-5)
        assert r["per_iter"][1, 0] == pytest.approx(flt("cfg2.iter1")[0], rel=1e-10)
    if cfg == 3:
        i9, from1 = flt("cfg3.iter9"), flt("cfg3.combined_from1")
        assert r["per_iter"][9, 0] == pytest.approx(i9[0], rel=1e-8) and r["per_iter"][9, 1] == pytest.approx(i9[1], rel=1e-4)
        I, s, chi2 = B.vegas_combine(r["per_iter"][:, 0], r["per_iter"][:, 1], n_skip=1)
        assert I == pytest.approx(from1[0], rel=1e-8) and s == pytest.approx(from1[1], rel=2e-3)
        assert chi2 == pytest.approx(from1[2], abs=0.006)
        # finding F1: the first iterations at d = 20 are far off for any correct implementation; from k = 3 on every
        # estimate is within 5 sigma of the closed form
        assert abs(r["per_iter"][0, 0] - w.closed_form) > 1000 * r["per_iter"][0, 1]
        for k in range(3, 10):
            assert abs(r["per_iter"][k, 0] - w.closed_form) < 5 * r["per_iter"][k, 1]
    else:
        # SURVEY.md F1 (value +- error lands on the closed form): n_skip = 0 for cfg2, 4, 5 -- every
        # I_k from the first, un-adapted iteration on, and the average over all of them; the survey's probe saw
        # largest pulls of 2.50, 2.95 and 2.65
        assert abs(r["I"] - w.closed_form) < 5 * r["sigma"]
        pulls = np.abs(r["per_iter"][:, 0] - w.closed_form) / r["per_iter"][:, 1]
        assert np.all(pulls < 5.0), pulls
        assert pulls.max() == pytest.approx({2: 2.50, 4: 2.95, 5: 2.65}[cfg], abs=0.02)
    g.close()


def test_genz_product_peak_at_the_papers_16_dimensions(B):
    """PAPER.md:86 (Table 1, "Genz Eq.(3) 16-d"): the product peak at the paper's dimension count, teacher-forced on
    oracle grids (P3/P4) and free-running against the arctan closed form (5 sigma)."""
    dim, nb, n, seed = 16, 50, 400_003, 16
    p = W.genz_params(dim, seed)
    ch = O.integrate(dim, nb, 3, n, seed, 1.5, O.GENZ_PRODUCT_PEAK, p, threads=THREADS)
    g = B.VegasGrid(dim, nb)
    g.set_params(B.VEGAS_F_GENZ_PRODUCT_PEAK, p)
    for prec, tol in ((64, RTOL64), (32, RTOL32)):
        for k in range(3):
            g.set_edges(ch["edges_trace"][k])
            I, s, H, st = g.iterate(n, seed, k, B.VEGAS_F_GENZ_PRODUCT_PEAK, prec)
            assert st == 0 and I == pytest.approx(ch["per_iter"][k, 0], rel=tol)
            assert s == pytest.approx(ch["per_iter"][k, 1], rel=tol)
            _assert_hist(H, ch["hist_trace"][k], prec)
    g.set_edges(O.uniform_edges(dim, nb))
    r = g.integrate(8, 4_000_000, seed, 1.5, B.VEGAS_F_GENZ_PRODUCT_PEAK, 64, n_skip=3)
    exact = W.closed_form(W.GENZ_PRODUCT_PEAK, dim, p)
    assert abs(r["I"] - exact) < 5 * r["sigma"] and r["sigma"] / exact < 1e-2
    g.close()


def test_more_than_2_to_the_32_events_in_one_iteration(B):
    """5e9 events in one iteration (event indices beyond 2^32, launches split there by the fast path): the constant
    control stays exactly 1, the Gaussian lands on the closed form, and two half-range accumulations equal the whole."""
    n = 5_000_000_000
    w = W.config(1)
    g = _grid(B, w)
    Ic, sc, _, st = g.iterate(n, 1, 0, B.VEGAS_F_CONST, 64, chunk_events=1_000_000_000)
    assert st == 0 and abs(Ic - 1.0) <= 1e-12 and sc <= 1e-9                       # reading R9
    g.set_edges(W.adapted_edges(w.dim, w.n_bins, seed=1))
    I, s, H, st = g.iterate(n, w.seed, 3, w.integrand_id, 64)
    assert st == 0 and abs(I - w.closed_form) < 5 * s and s / I < 1e-4
    g.begin_iteration()
    g.accumulate(0, n // 2, w.seed, 3, w.integrand_id, 64)
    g.accumulate(n // 2, n - n // 2, w.seed, 3, w.integrand_id, 64, chunk_events=700_000_000)
    g.reduce()
    I2, s2, H2, _ = g.finalize(n)
    assert I2 == pytest.approx(I, rel=1e-12) and s2 == pytest.approx(s, rel=1e-10)
    np.testing.assert_allclose(H2, H, rtol=1e-11)
    np.testing.assert_allclose(H.sum(axis=1), np.full(w.dim, H[0].sum()), rtol=1e-11)   # every dimension sums to S2
    g.close()


@pytest.mark.parametrize("path", ["auto", "generic"])
@pytest.mark.parametrize("dim,nb,pseed", [(16, 50, 9), (2, 8, 2), (7, 33, 5), (20, 50, 11)])
def test_genz_discontinuous_built_in(B, dim, nb, pseed, path):
    """PAPER.md:67-70 Eq.(2) as printed (reading R19), at the paper's 16 dimensions and odd shapes, as a
    built-in fast-path integrand (VEGAS_F_GENZ_DISCONTINUOUS; the oracle's id for it is 4): events, teacher-forced
    iterations and refinement against the oracle; fp64 only."""
    fid = B.VEGAS_F_GENZ_DISCONTINUOUS
    p = W.genz_discontinuous_params(dim, pseed)
    n, n_iter = 200_003, 3
    ch = O.integrate(dim, nb, n_iter, n, pseed, 1.5, O.GENZ_DISCONTINUOUS, p, threads=THREADS)
    g = B.VegasGrid(dim, nb)
    g.set_params(fid, p)
    if path == "generic":
        g.set_launch(0, 0, 2, 4)
    assert g.get_launch(fid, 64)["path"] == ("generic" if path == "generic" else "rotated")
    for k in range(n_iter):
        g.set_edges(ch["edges_trace"][k])
        if k == 1:
            gw, gb, gx, gf = g.debug_sample(7, 20_000, pseed, k, fid, 64)
            ow, ob, ox, of = O.sample(ch["edges_trace"][k], pseed, k, 7, 20_000, O.GENZ_DISCONTINUOUS, p)
            assert np.array_equal(gw, ow) and np.array_equal(gb, ob)
            assert np.array_equal(gf == 0, of == 0)                 # the same events fall on the zero side of a cut
            np.testing.assert_allclose(gf, of, rtol=1e-12, atol=0)
        I, s, H, st = g.iterate(n, pseed, k, fid, 64)
        assert st == 0
        assert I == pytest.approx(ch["per_iter"][k, 0], rel=RTOL64)
        assert s == pytest.approx(ch["per_iter"][k, 1], rel=RTOL64)
        _assert_hist(H, ch["hist_trace"][k], 64)
        assert g.refine(1.5) == 0
        want = ch["edges_trace"][k + 1] if k + 1 < n_iter else ch["edges"]
        np.testing.assert_allclose(g.get_edges(), want, rtol=0, atol=1e-10)
    # fp32 is refused (the cuts are decided in fp64); so are non-positive c_j
    with pytest.raises(B.VegasError):
        g.iterate(1000, 1, 0, fid, 32)
    bad = np.array(p, dtype=float)
    bad[0] = -bad[0]
    with pytest.raises(B.VegasError):
        g.set_params(fid, bad)
    g.close()


def test_genz_discontinuous_chain_within_5_sigma_at_16_dimensions(B):
    p = W.genz_discontinuous_params(16, 9)
    g = B.VegasGrid(16, 50)
    g.set_params(B.VEGAS_F_GENZ_DISCONTINUOUS, p)
    r = g.integrate(8, 2_000_000, 9, 1.5, B.VEGAS_F_GENZ_DISCONTINUOUS, 64, n_skip=3)
    exact = W.closed_form(W.GENZ_DISCONTINUOUS, 16, p)
    assert r["status"] == 0 and abs(r["I"] - exact) <= 5 * r["sigma"] and r["sigma"] < 0.01 * exact
    g.close()
