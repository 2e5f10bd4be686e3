"""Pins for the oracle's per-event map, integrands, accumulation, estimate, refine and combine
(readings C4..C9 of DESIGN.md) against what the mathematics fixes -- no GPU."""
import math
from fractions import Fraction

import numpy as np
import pytest

import oracle as O
import workloads as W


def _flt(probe, key):
    return [float(v) for v in probe[key]]


# ---------------------------------------------------------------- C4: grid map and Jacobian
def test_c4_uniform_edges():
    e = O.uniform_edges(3, 50)
    assert e.shape == (3, 51)
    assert np.all(e[:, 0] == 0.0) and np.all(e[:, -1] == 1.0)
    assert e[1, 7] == 7 / 50 and e[2, 49] == 49 / 50


@pytest.mark.parametrize("dim,nb", [(1, 2), (3, 7), (6, 50), (20, 50), (12, 100)])
def test_c4_map_is_exact_rational_affine(dim, nb):
    edges = W.adapted_edges(dim, nb, seed=dim * 1000 + nb)
    words, bins, x, fJ = O.sample(edges, 77, 3, (1 << 33) + 5, 40, O.CONST)
    for q in range(40):
        J = Fraction(1)
        for j in range(dim):
            w = int(words[q, j])
            assert w == O.word(77, 3, (1 << 33) + 5 + q, j)
            b = (w * nb) >> 32
            assert b == bins[q, j]
            r = Fraction(2 * ((w * nb) & 0xFFFFFFFF) + 1, 2**33)
            lo, hi = Fraction(edges[j, b]), Fraction(edges[j, b + 1])
            delta = Fraction(float(hi - lo))              # the fp64-rounded width the method uses
            exact = lo + delta * r
            assert abs(Fraction(x[q, j]) - exact) <= Fraction(np.spacing(x[q, j])) * 1
            assert edges[j, b] < x[q, j] < edges[j, b + 1]
            J *= nb * delta
        assert abs(Fraction(fJ[q]) - J) <= abs(J) * Fraction(dim + 2, 2**52)   # f = 1


def test_c3_c5_worked_example_from_survey_probe(probe):
    w = W.config(1)
    words, bins, x, fJ = O.sample(O.uniform_edges(4, 50), 1, 0, 0, 3, O.GAUSS, w.params)
    assert bins[0].tolist() == [int(v) for v in probe["cfg1.event0.bins"]]
    assert bins[1].tolist() == [int(v) for v in probe["cfg1.event1.bins"]]
    assert bins[2].tolist() == [int(v) for v in probe["cfg1.event2.bins"]]
    lo = [(int(wd) * 50) & 0xFFFFFFFF for wd in words[0]]
    assert lo == [int(v, 16) for v in probe["cfg1.event0.lo"]]
    np.testing.assert_allclose(x[0], _flt(probe, "cfg1.event0.x"), rtol=4e-16)
    np.testing.assert_allclose(x[1, 0], _flt(probe, "cfg1.event1.x0")[0], rtol=4e-16)
    J0 = _flt(probe, "cfg1.event0.J")[0]
    f = [_flt(probe, "cfg1.event%d.f" % i)[0] for i in range(3)]
    # f is e^-(~29..37): a 1-ulp change of x moves it by ~1e-14 relative
    np.testing.assert_allclose(fJ[0], f[0] * J0, rtol=2e-13)
    np.testing.assert_allclose(fJ[1:], f[1:], rtol=2e-13)


# ---------------------------------------------------------------- C5: integrands
def test_c5_gauss_normalisation_closed_form(probe):
    # (a sqrt(pi))^-d with a = 0.1 is 10^d / pi^(d/2)
    for d, want in zip((4, 8, 20), _flt(probe, "gauss.norm.d4d8d20")):
        got = O.f(O.GAUSS, np.full(d, 0.5), [0.1])
        assert got == pytest.approx(10.0**d / math.pi ** (d / 2), rel=1e-14)
        assert got == pytest.approx(want, rel=1e-14)
    # one e-fold: moving one coordinate by a divides f by e
    x = np.full(4, 0.5)
    x[2] += 0.1
    assert O.f(O.GAUSS, x, [0.1]) == pytest.approx(O.f(O.GAUSS, np.full(4, 0.5), [0.1]) / math.e,
                                                   rel=1e-13)


def _gl_nodes(breaks, n):
    xs, ws = [], []
    g, w = np.polynomial.legendre.leggauss(n)
    for a, b in zip(breaks[:-1], breaks[1:]):
        xs.append(0.5 * (b - a) * g + 0.5 * (a + b))
        ws.append(0.5 * (b - a) * w)
    return np.concatenate(xs), np.concatenate(ws)


def _tensor_quadrature(integrand_id, params, nodes):
    """Integral of oracle.f over [0,1]^d by a tensor Gauss-Legendre rule; nodes = [(x, w)] * d."""
    d = len(nodes)
    total = 0.0
    idx = np.zeros(d, dtype=int)
    sizes = [len(n[0]) for n in nodes]
    x = np.zeros(d)
    for flat in range(int(np.prod(sizes))):
        rem = flat
        wgt = 1.0
        for j in range(d):
            idx[j] = rem % sizes[j]
            rem //= sizes[j]
            x[j] = nodes[j][0][idx[j]]
            wgt *= nodes[j][1][idx[j]]
        total += wgt * O.f(integrand_id, x, params)
    return total


def test_c5_gauss_integral_matches_erf_closed_form(probe):
    nd = _gl_nodes(np.linspace(0, 1, 11), 12)
    for d in (1, 2):
        got = _tensor_quadrature(O.GAUSS, [0.1], [nd] * d)
        assert got == pytest.approx(math.erf(5.0) ** d, rel=1e-12)
        assert got == pytest.approx(W.closed_form(W.GAUSS, d, [0.1]), rel=1e-12)
    for d, want in zip((4, 8, 20), _flt(probe, "gauss.closed.d4d8d20")):
        assert W.closed_form(W.GAUSS, d, [0.1]) == pytest.approx(want, rel=1e-15)
    # a different width, so that a hard-wired a = 0.1 would fail
    got = _tensor_quadrature(O.GAUSS, [0.3], [_gl_nodes(np.linspace(0, 1, 6), 12)] * 2)
    assert got == pytest.approx(math.erf(1 / 0.6) ** 2, rel=1e-12)


def test_c5_genz_product_peak_integral_matches_atan_closed_form(probe):
    w4 = W.config(4)
    c, w = w4.params[:12], w4.params[12:]
    assert w4.closed_form == pytest.approx(_flt(probe, "cfg4.closed_form")[0], rel=1e-14)
    assert [c[0], c[1], w[0]] == pytest.approx(_flt(probe, "cfg4.c0c1w0"), rel=1e-15)
    assert np.all((c > 5) & (c < 15)) and np.all((w > 0) & (w < 1))
    # 2-d slice with dims (0, 1) and then (5, 9): asymmetric peaks, distinct c's
    for dims in ((0, 1), (5, 9)):
        p = np.concatenate([c[list(dims)], w[list(dims)]])
        nodes = []
        for j in dims:
            br = sorted({0.0, 1.0, *np.clip(w[j] + np.array([-0.3, -0.1, -0.03, 0, 0.03, 0.1, 0.3]),
                                            0, 1)})
            nodes.append(_gl_nodes(np.array(br), 24))
        got = _tensor_quadrature(O.GENZ_PRODUCT_PEAK, p, nodes)
        assert got == pytest.approx(W.closed_form(W.GENZ_PRODUCT_PEAK, 2, p), rel=1e-11)
    # point value at the peak: prod c_j^2
    assert O.f(O.GENZ_PRODUCT_PEAK, w, w4.params) == pytest.approx(np.prod(c * c), rel=1e-13)


def test_c5_bw_poly_integral_matches_closed_form(probe):
    w5 = W.config(5)
    assert w5.closed_form == pytest.approx(_flt(probe, "cfg5.closed_form")[0], rel=1e-14)
    assert w5.params[4:6].tolist() == pytest.approx(_flt(probe, "cfg5.a10a11"), rel=1e-15)
    # 3-d version (x0 = mass dimension, two polynomial dimensions with distinct coefficients)
    p = np.concatenate([w5.params[:4], w5.params[4 + 5:4 + 15]])
    M, G, m_min, m_max = p[:4]
    peak = (M * M - m_min**2) / (m_max**2 - m_min**2)
    br = sorted({0.0, 1.0, *np.clip(peak + np.array([-0.1, -0.03, -0.01, -0.003, 0, 0.003, 0.01,
                                                      0.03, 0.1]), 0, 1)})
    nodes = [_gl_nodes(np.array(br), 24), _gl_nodes(np.array([0.0, 1.0]), 6),
             _gl_nodes(np.array([0.0, 1.0]), 6)]
    got = _tensor_quadrature(O.BW_POLY, p, nodes)
    assert got == pytest.approx(W.closed_form(W.BW_POLY, 3, p), rel=1e-11)
    # peak value of the Breit-Wigner factor is 1: f(peak, 0, 0) = a_10 + a_20
    assert O.f(O.BW_POLY, [peak, 0.0, 0.0], p) == pytest.approx(p[4] + p[9], rel=1e-12)
    # f(x0, 1, 1) = bw * sum of all coefficients
    bw = O.f(O.BW_POLY, [0.3, 0.0, 0.0], p) / (p[4] + p[9])
    assert O.f(O.BW_POLY, [0.3, 1.0, 1.0], p) == pytest.approx(bw * p[4:].sum(), rel=1e-12)


def test_c5_genz_discontinuous_as_printed_matches_closed_form():
    """PAPER.md:69 Eq.(2) as printed (reading R19), N = 1: zero where ANY x_j <= a_j, exp(sum c_j x_j) elsewhere.
    Pinned by quadrature with a break at the discontinuity, by point values on both sides of it, and by a chain."""
    p = W.genz_discontinuous_params(2, 9)
    c, a = p[:2], p[2:]
    nodes = [_gl_nodes(np.array([0.0, a[j], 1.0]), 16) for j in range(2)]
    got = _tensor_quadrature(O.GENZ_DISCONTINUOUS, p, nodes)
    want = np.prod([(math.exp(cj) - math.exp(cj * aj)) / cj for cj, aj in zip(c, a)])
    assert got == pytest.approx(want, rel=1e-12)
    assert W.closed_form(W.GENZ_DISCONTINUOUS, 2, p) == pytest.approx(want, rel=1e-14)
    # the zero region is x_j <= a_j (not >=), and one coordinate inside it is enough
    assert O.f(O.GENZ_DISCONTINUOUS, [a[0] * 0.5, 0.9], p) == 0.0
    assert O.f(O.GENZ_DISCONTINUOUS, [0.9, a[1]], p) == 0.0                       # boundary belongs to the zero side
    assert O.f(O.GENZ_DISCONTINUOUS, [0.9, 0.8], p) == pytest.approx(math.exp(c[0] * 0.9 + c[1] * 0.8), rel=1e-15)
    # the paper's 16-d case as a chain: within 5 sigma of the closed form once adapted
    p16 = W.genz_discontinuous_params(16, 9)
    r = O.integrate(16, 50, 6, 200_000, 9, 1.5, O.GENZ_DISCONTINUOUS, p16, n_skip=2, threads=8)
    exact = W.closed_form(W.GENZ_DISCONTINUOUS, 16, p16)
    assert abs(r["I"] - exact) < 5 * r["sigma"] and r["sigma"] / exact < 2e-2


def test_c5_const():
    assert O.f(O.CONST, [0.1, 0.9], None) == 1.0
    assert O.n_params(O.GENZ_PRODUCT_PEAK, 12) == 24 and O.n_params(O.BW_POLY, 6) == 29
    assert O.n_params(O.GAUSS, 20) == 1 and O.n_params(9, 3) < 0


# ---------------------------------------------------------------- C6, C7: accumulate, estimate
@pytest.mark.parametrize("dim,nb,n", [(1, 2, 4), (2, 3, 16), (4, 50, 3001), (12, 100, 1500)])
def test_c6_c7_brute_force_reaccumulation(dim, nb, n):
    edges = W.adapted_edges(dim, nb, seed=n)
    ident = O.GENZ_PRODUCT_PEAK if dim == 12 else O.GAUSS
    params = W.config(4).params if dim == 12 else [0.25]
    I, sg, H = O.iterate(edges, n, 99, 2, ident, params)
    _, bins, _, fJ = O.sample(edges, 99, 2, 0, n, ident, params)
    v = [Fraction(float(t)) for t in fJ]
    S1 = sum(v)
    S2 = sum(Fraction(float(t * t)) for t in fJ)            # v*v rounded to fp64, as the method does
    mean = S1 / n
    var = (S2 / n - mean * mean) / (n - 1)
    assert I == pytest.approx(float(mean), rel=1e-15)
    assert sg == pytest.approx(math.sqrt(float(var)), rel=1e-13)
    Hn = np.zeros((dim, nb))
    for j in range(dim):
        np.add.at(Hn[j], bins[:, j], fJ * fJ)
    np.testing.assert_allclose(H, Hn, rtol=1e-13, atol=0)
    assert np.all(H[Hn == 0] == 0)
    for j in range(dim):                                     # every event lands once per dimension
        assert H[j].sum() == pytest.approx(float(S2), rel=1e-13)


def test_c6_event_ranges_add_up():
    edges = W.adapted_edges(5, 20, seed=4)
    a = O.iterate(edges, 50_000, 8, 1, O.GAUSS, [0.2], threads=1)
    b = O.iterate(edges, 50_000, 8, 1, O.GAUSS, [0.2], threads=5)
    assert a[0] == pytest.approx(b[0], rel=1e-15) and a[1] == pytest.approx(b[1], rel=1e-13)
    np.testing.assert_allclose(a[2], b[2], rtol=1e-15)
    S1a, _, _ = O.accumulate(edges, 8, 1, 0, 1000, O.GAUSS, [0.2])
    S1b, _, _ = O.accumulate(edges, 8, 1, 1000, 500, O.GAUSS, [0.2])
    S1c, _, _ = O.accumulate(edges, 8, 1, 0, 1500, O.GAUSS, [0.2])
    assert float(abs(S1a + S1b - S1c)) <= 1e-17 * float(S1c)


def test_c7_estimator_on_constant_integrand_with_known_variance():
    # f = 1 on a non-uniform grid: E[v] = 1 exactly; E[v^2] = prod_j sum_b (nb Delta_b)^2 / nb
    dim, nb, n = 3, 8, 200_000
    edges = W.adapted_edges(dim, nb, seed=11, strength=1.0)
    widths = np.diff(edges, axis=1)
    second = np.prod(((nb * widths) ** 2).sum(axis=1) / nb)
    sigma_pred = math.sqrt((second - 1.0) / n)
    I, sg, H = O.iterate(edges, n, 5, 0, O.CONST)
    assert abs(I - 1.0) < 5 * sigma_pred
    assert sg == pytest.approx(sigma_pred, rel=0.02)
    # bin b of dimension j is hit with probability 1/nb and carries E[v^2 | b]
    for j in range(dim):
        pred = n * ((nb * widths[j]) ** 2 / nb) * second / (((nb * widths[j]) ** 2).sum() / nb)
        np.testing.assert_allclose(H[j], pred, rtol=0.05)


def test_c7_uniform_grid_constant_is_one():
    I, sg, H = O.iterate(O.uniform_edges(8, 50), 100_000, 2, 0, O.CONST)
    assert abs(I - 1.0) <= 1e-12 and sg <= 1e-9
    np.testing.assert_allclose(H.sum(axis=1), 100_000, rtol=1e-12)


def test_c7_pulls_are_unit_normal():
    # 40 independent seeds of one iteration: (I - exact)/sigma must look like N(0,1)
    edges = O.uniform_edges(2, 50)
    exact = W.closed_form(W.GAUSS, 2, [0.1])
    pulls = []
    for seed in range(100, 140):
        I, sg, _ = O.iterate(edges, 20_000, seed, 0, O.GAUSS, [0.1])
        pulls.append((I - exact) / sg)
    pulls = np.array(pulls)
    assert np.abs(pulls).max() < 5
    assert 0.7 < pulls.std() < 1.35 and abs(pulls.mean()) < 0.6


def test_invalid_arguments():
    e = O.uniform_edges(2, 4)
    with pytest.raises(O.OracleError):
        O.iterate(e, 1, 1, 0, O.CONST)
    bad = e.copy()
    bad[1, 2] = bad[1, 1]
    with pytest.raises(O.OracleError):
        O.accumulate(bad, 1, 0, 0, 10, O.CONST)
    with pytest.raises(O.OracleError):
        O.refine(e, np.ones((2, 4)), -1.0)


# ---------------------------------------------------------------- C8: refine
def _refine_by_interp(edges, hist, alpha):
    """Independent restatement through library routines: the new edges are where the
    piecewise-linear cumulative of the compressed weights crosses k/nb of its total."""
    out = np.empty_like(edges)
    for j, (X, h) in enumerate(zip(edges, hist)):
        nb = len(h)
        s = np.convolve(h, [1, 1, 1], mode="same") / 3.0
        s[0] = (h[0] + h[1]) / 2.0
        s[-1] = (h[-2] + h[-1]) / 2.0
        p = s / s.sum()
        with np.errstate(divide="ignore", invalid="ignore"):
            m = np.where(p > 0, ((1 - p) / np.log(1 / p)) ** alpha, 0.0)
        m = np.where(p >= 1, 1.0, m)
        cum = np.concatenate([[0.0], np.cumsum(m)])
        out[j] = np.interp(np.arange(nb + 1) * (cum[-1] / nb), cum, X)
        out[j, 0], out[j, -1] = 0.0, 1.0
    return out


def test_c8_fixed_points():
    rng = np.random.default_rng(8)
    for dim, nb in ((3, 50), (2, 100), (1, 7)):
        edges = W.adapted_edges(dim, nb, seed=nb)
        # (i) constant histogram on a uniform grid, and on any grid m is constant so the
        # new edges cut the old piecewise-linear map at equal shares: uniform grid unchanged
        u = O.uniform_edges(dim, nb)
        out, rc = O.refine(u, np.full((dim, nb), 3.7), 1.5)
        assert rc == 0
        np.testing.assert_allclose(out, u, rtol=0, atol=1e-14)
        # (ii) alpha = 0: every m_i = 1, grid unchanged whatever the (positive) histogram
        out, rc = O.refine(edges, rng.random((dim, nb)) + 0.01, 0.0)
        assert rc == 0
        np.testing.assert_allclose(out, edges, rtol=0, atol=1e-14)
    # (iii) nb = 2: smoothing equalises the two bins
    e2 = np.array([[0.0, 0.3, 1.0]])
    out, rc = O.refine(e2, np.array([[5.0, 1.0]]), 1.5)
    np.testing.assert_allclose(out, e2, atol=1e-15)


def test_c8_worked_examples(probe):
    u3 = O.uniform_edges(1, 3)
    out, rc = O.refine(u3, np.array([[1.0, 0.0, 0.0]]), 1.5)
    assert rc == 0
    # by hand: s = (1/2, 1/3, 0), p = (0.6, 0.4, 0), m_i = ((1-p)/ln(1/p))^1.5
    m = [((1 - p) / math.log(1 / p)) ** 1.5 for p in (0.6, 0.4)] + [0.0]
    assert m == pytest.approx(_flt(probe, "refine.nb3.H100.m"), rel=1e-14)
    delta = sum(m) / 3
    want = [0.0, (delta / m[0]) / 3, (1 + (2 * delta - m[0]) / m[1]) / 3, 1.0]
    np.testing.assert_allclose(out[0], want, rtol=1e-14)
    np.testing.assert_allclose(out[0], _flt(probe, "refine.nb3.H100.edges"), rtol=1e-14)
    out, rc = O.refine(O.uniform_edges(1, 4), np.array([[1.0, 2.0, 3.0, 4.0]]), 1.5)
    np.testing.assert_allclose(out[0], _flt(probe, "refine.nb4.H1234.edges"), rtol=1e-14)


@pytest.mark.parametrize("alpha", [0.5, 1.0, 1.5, 2.5])
def test_c8_against_interp_restatement(alpha):
    rng = np.random.default_rng(int(alpha * 10))
    for dim, nb in ((4, 50), (3, 100), (2, 5)):
        edges = W.adapted_edges(dim, nb, seed=nb + 1)
        hist = rng.random((dim, nb)) ** 6 * 10.0 ** rng.integers(-30, 30, size=(dim, 1))
        hist[0, nb // 2:nb // 2 + 3] = 0.0                  # empty bins
        if nb > 6:
            hist[1, :6] = 0.0
        out, rc = O.refine(edges, hist, alpha)
        assert rc == 0
        np.testing.assert_allclose(out, _refine_by_interp(edges, hist, alpha), rtol=0, atol=1e-13)
        assert np.all(out[:, 0] == 0.0) and np.all(out[:, -1] == 1.0)
        assert np.all(np.diff(out, axis=1) > 0)


def test_c8_degenerate_rows_are_left_unchanged():
    edges = W.adapted_edges(3, 10, seed=3)
    hist = np.ones((3, 10))
    hist[1] = 0.0
    out, rc = O.refine(edges, hist, 1.5)
    assert rc == O.ENUMERIC
    np.testing.assert_array_equal(out[1], edges[1])
    assert not np.array_equal(out[0], edges[0])
    hist[1] = np.nan
    out, rc = O.refine(edges, hist, 1.5)
    assert rc == O.ENUMERIC
    np.testing.assert_array_equal(out[1], edges[1])
    # one bin holds everything: p = (2/3.., ) stays finite, edges stay monotone
    hist = np.zeros((3, 10))
    hist[:, 4] = 1.0
    out, rc = O.refine(edges, hist, 1.5)
    assert rc == 0 and np.all(np.diff(out, axis=1) > 0)


def test_c8_concentrates_bins_where_the_histogram_is_large():
    nb = 50
    h = np.exp(-((np.arange(nb) + 0.5) / nb - 0.5) ** 2 / 0.005)[None, :]
    out, _ = O.refine(O.uniform_edges(1, nb), h, 1.5)
    w = np.diff(out[0])
    assert w[nb // 2] < 0.5 / nb and w[0] > 2.0 / nb


# ---------------------------------------------------------------- C9: combine
def test_c9_closed_forms():
    I, s, c = O.combine([1.0, 3.0], [0.5, 0.5])
    assert I == 2.0 and s == pytest.approx(0.5 / math.sqrt(2)) and c == pytest.approx(8.0 / 1)
    I, s, c = O.combine([2.5, 2.5, 2.5], [0.1, 0.2, 0.3])
    assert I == 2.5 and c == 0.0 and s == pytest.approx((100 + 25 + 100 / 9) ** -0.5)
    # weights 1/sigma^2: (1*1 + 4*0.25... ) by hand
    I, s, c = O.combine([1.0, 2.0], [1.0, 2.0])
    assert I == pytest.approx((1.0 + 2.0 / 4) / (1 + 0.25))
    assert s == pytest.approx(1 / math.sqrt(1.25))
    assert c == pytest.approx((1.0 - 1.2) ** 2 + (2.0 - 1.2) ** 2 / 4)
    # n_skip drops the early iterations
    assert O.combine([9.0, 1.0, 3.0], [1e-3, 0.5, 0.5], n_skip=1)[0] == 2.0
    # sigma_k = 0 rule: plain mean, sigma = 0
    assert O.combine([1.0, 0.999], [0.0, 1e-3]) == (0.9995, 0.0, 0.0)
    assert O.combine([4.0], [0.3]) == (4.0, 0.3, 0.0)
    with pytest.raises(O.OracleError):
        O.combine([1.0], [1.0], n_skip=1)


# ---------------------------------------------------------------- whole chains
def test_chain_cfg1_matches_survey_probe_and_closed_form(probe):
    w = W.config(1)
    r = O.integrate(w.dim, w.n_bins, w.n_iter, w.n_events, w.seed, w.alpha, w.integrand_id, w.params)
    per = np.array(_flt(probe, "cfg1.per_iter")).reshape(5, 2)
    np.testing.assert_allclose(r["per_iter"][:, 0], per[:, 0], rtol=1e-11)
    np.testing.assert_allclose(r["per_iter"][:, 1], per[:, 1], rtol=2e-5)     # printed to 6 digits
    comb = _flt(probe, "cfg1.combined")
    assert r["I"] == pytest.approx(comb[0], rel=1e-11)
    assert r["sigma"] == pytest.approx(comb[1], rel=2e-6)
    assert r["chi2_dof"] == pytest.approx(comb[2], abs=1e-3)
    np.testing.assert_allclose(r["hist_trace"][0][0][:3], _flt(probe, "cfg1.H0.dim0.bins012"),
                               rtol=1e-11)
    np.testing.assert_allclose(r["edges_trace"][1][0][1:4], _flt(probe, "cfg1.edges1.dim0.e123"),
                               rtol=1e-11)
    # 5-sigma rule against the erf closed form (north_star), every iteration and the average
    exact = w.closed_form
    assert np.all(np.abs(r["per_iter"][:, 0] - exact) < 5 * r["per_iter"][:, 1])
    assert abs(r["I"] - exact) < 5 * r["sigma"]
    # adaptation must shrink the error by more than an order of magnitude
    assert r["per_iter"][-1, 1] < r["per_iter"][0, 1] / 10
    # the threaded driver gives the same chain
    r2 = O.integrate(w.dim, w.n_bins, w.n_iter, w.n_events, w.seed, w.alpha, w.integrand_id,
                     w.params, threads=4)
    np.testing.assert_allclose(r2["per_iter"], r["per_iter"], rtol=1e-12)
    np.testing.assert_allclose(r2["edges"], r["edges"], rtol=0, atol=1e-12)


def test_chain_cfg2_first_iterations_match_survey_probe(probe):
    w = W.config(2)
    r = O.integrate(w.dim, w.n_bins, 2, w.n_events, w.seed, w.alpha, w.integrand_id, w.params,
                    threads=8)
    for k in (0, 1):
        want = _flt(probe, "cfg2.iter%d" % k)
        assert r["per_iter"][k, 0] == pytest.approx(want[0], rel=1e-11)
        assert r["per_iter"][k, 1] == pytest.approx(want[1], rel=2e-6)
    assert abs(r["per_iter"][1, 0] - w.closed_form) < 5 * r["per_iter"][1, 1]


def test_chain_constant_control_and_fixed_point(probe):
    w = W.control_const(n_events=10_000_000)
    r = O.integrate(w.dim, w.n_bins, 2, w.n_events, w.seed, w.alpha, w.integrand_id, None, threads=8)
    assert abs(r["per_iter"][0, 0] - 1.0) <= 1e-12 and r["per_iter"][0, 1] <= 1e-9     # reading R9
    want = _flt(probe, "cfg2.control.iter1")
    assert r["per_iter"][1, 0] == pytest.approx(want[0], rel=1e-12)
    assert r["per_iter"][1, 1] == pytest.approx(want[1], rel=2e-5)
    # reading R10(ii): a sampled flat histogram moves the edges by a few 1e-5 only
    assert np.abs(r["edges_trace"][1] - O.uniform_edges(w.dim, w.n_bins)).max() < 1e-3
    assert abs(r["edges_trace"][1][0][1] - 0.0199925) < 2e-7
    assert abs(r["edges_trace"][1][0][5] - 0.0999710) < 2e-7


def test_chain_small_genz_and_bw_within_5_sigma():
    for w, n in ((W.config(4), 200_000), (W.config(5), 200_000)):
        r = O.integrate(w.dim, w.n_bins, 6, n, w.seed, w.alpha, w.integrand_id, w.params,
                        n_skip=2, threads=8)
        exact = w.closed_form
        assert abs(r["I"] - exact) < 5 * r["sigma"]
        assert r["sigma"] / exact < 2e-2
        for k in range(2, 6):
            assert abs(r["per_iter"][k, 0] - exact) < 5 * r["per_iter"][k, 1]
