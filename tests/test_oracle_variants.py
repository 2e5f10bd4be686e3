"""Pins for the oracle's sampling-map variants (readings C3' and C4' of DESIGN.md section 2)
against what the mathematics fixes -- no GPU.

  C3' (O.V_U53): 53-bit uniforms from two Philox words per draw, counter (j>>1, iteration, e lo, e hi).
  C4' (O.V_Q32): the per-bin pair (X_b, Delta_b) of the map rounded to fp32; master grid and refinement in fp64.
"""
import math
from fractions import Fraction

import numpy as np
import pytest

import oracle as O
import workloads as W


# ---------------------------------------------------------------- C3': two-word layout and the 53-bit split
def test_c3p_layout_against_independent_python_integers():
    # workloads._draw_block is a Python-integer Philox written for the parameter draws; neither the oracle nor the
    # kernels call it.  A dropped shift, swapped words or the C2 counter (j>>2) in place of (j>>1) fails here.
    for seed, it, ev in [(1, 0, 0), (0xDEADBEEF12345678, 7, (1 << 32) + 3), (3, 0xFFFFFFFE, (1 << 40) - 1)]:
        key = (seed & 0xFFFFFFFF, seed >> 32)
        for j in range(9):
            out = W._draw_block((j >> 1, it, ev & 0xFFFFFFFF, ev >> 32), key)
            hi, lo = out[2 * (j & 1)], out[2 * (j & 1) + 1]
            assert O.word53(seed, it, ev, j) == (hi << 21) | (lo >> 11)
            assert O.word53(seed, it, ev, j) < 1 << 53


def test_c3p_two_dimensions_share_one_block_and_differ_from_c2():
    # dimensions 0 and 1 come from the same block (words 0,1 and 2,3); dimension 2 from the next counter
    U = [O.word53(5, 1, 9, j) for j in range(4)]
    blk0 = [int(v) for v in O.philox4x32_10([0, 1, 9, 0], [5, 0])]
    blk1 = [int(v) for v in O.philox4x32_10([1, 1, 9, 0], [5, 0])]
    assert U[0] >> 21 == blk0[0] and U[1] >> 21 == blk0[2] and U[2] >> 21 == blk1[0] and U[3] >> 21 == blk1[2]
    assert U[0] & ((1 << 21) - 1) == blk0[1] >> 11


@pytest.mark.parametrize("nb", [2, 3, 50, 100, 255, 256])
def test_c3p_split_is_exact_rational(nb):
    rng = np.random.default_rng(nb)
    Us = [0, 1, (1 << 53) - 1, (1 << 52), (1 << 53) // nb, (1 << 53) // nb + 1] + [int(v) for v in rng.integers(0, 1 << 53, 300)]
    # first and last U of a few bins
    for b in (0, 1, nb // 2, nb - 1):
        first = -((-b * (1 << 53)) // nb)          # ceil(b 2^53 / nb)
        Us += [first, max(first - 1, 0)]
    for U in Us:
        b, r = O.split53(U, nb)
        P = U * nb
        assert b == P >> 53 and 0 <= b < nb
        assert Fraction(r) == Fraction(P & ((1 << 53) - 1), 1 << 53)      # exact, no rounding
        assert 0.0 <= r < 1.0
        # (b + r)/nb is U 2^-53 exactly: the bin and offset reassemble the 53-bit uniform
        assert (b + Fraction(r)) / nb == Fraction(U, 1 << 53)


def test_c3p_uniformity_of_bins_and_offsets():
    edges = O.uniform_edges(3, 50)
    _, bins, x, _ = O.sample(edges, 11, 0, 0, 60000, O.CONST, variant=O.V_U53)
    cnt = np.bincount(bins[:, 1], minlength=50)
    assert abs(cnt - 1200).max() < 6 * math.sqrt(1200)
    assert abs(x.mean() - 0.5) < 5 * math.sqrt(1 / 12 / x.size)
    # the C2/C3 stream of the same seed is a different sample
    _, bins32, _, _ = O.sample(edges, 11, 0, 0, 100, O.CONST)
    assert not np.array_equal(bins32, bins[:100])


# ---------------------------------------------------------------- C4': fp32-rounded table entries
def test_c4p_q32_is_round_to_nearest_fp32():
    for v in [0.0, 1.0, 0.1, 1 / 3, 0.5 + 2.0**-25, 0.5 + 2.0**-24, 0.5 + 3 * 2.0**-25, 1e-30, 0.7499999701976776]:
        assert O.q32(v) == float(np.float32(v))
    assert O.q32(0.5 + 2.0**-25) == 0.5                      # tie to even
    assert O.q32(0.5 + 3 * 2.0**-25) == 0.5 + 2.0**-23        # tie to even, upwards


@pytest.mark.parametrize("variant", [O.V_Q32, O.V_Q32 | O.V_U53])
@pytest.mark.parametrize("dim,nb", [(1, 2), (3, 7), (6, 50), (20, 50), (12, 100)])
def test_c4p_map_is_the_exact_rational_map_of_the_rounded_entries(dim, nb, variant):
    edges = W.adapted_edges(dim, nb, seed=dim * 1000 + nb)
    first = (1 << 33) + 5
    words, bins, x, fJ = O.sample(edges, 77, 3, first, 40, O.CONST, variant=variant)
    _, _, x_plain, fJ_plain = O.sample(edges, 77, 3, first, 40, O.CONST, variant=variant & O.V_U53)
    for q in range(40):
        J = Fraction(1)
        for j in range(dim):
            if variant & O.V_U53:
                U = O.word53(77, 3, first + q, j)
                b = (U * nb) >> 53
                r = Fraction((U * nb) & ((1 << 53) - 1), 1 << 53)
            else:
                w = O.word(77, 3, first + q, j)
                b = (w * nb) >> 32
                r = Fraction(2 * ((w * nb) & 0xFFFFFFFF) + 1, 2**33)
            assert b == bins[q, j]
            x0 = Fraction(float(np.float32(edges[j, b])))
            delta = Fraction(float(np.float32(edges[j, b + 1] - edges[j, b])))      # width in fp64, then rounded
            exact = x0 + delta * r
            assert abs(Fraction(x[q, j]) - exact) <= Fraction(np.spacing(x[q, j]))   # one product, one sum
            J *= nb * delta
        assert abs(Fraction(fJ[q]) - J) <= abs(J) * Fraction(dim + 2, 2**52)         # f = 1
    # the rounded map stays within fp32 rounding of the plain one: |dx| <= 2^-24 (|X_b| + Delta), |dJ/J| <= d 2^-24
    assert np.all(np.abs(x - x_plain) <= 2.0**-24 * 1.0000001)
    assert np.all(np.abs(fJ / fJ_plain - 1) <= dim * 2.0**-24 * 1.01)
    assert np.any(x != x_plain)


def test_c4p_exactly_representable_grid_is_unchanged():
    # a uniform grid with a power-of-two bin count is exact in fp32: the variant must reproduce the plain map bit for bit
    edges = O.uniform_edges(4, 64)
    a = O.sample(edges, 9, 2, 0, 500, O.GAUSS, [0.3])
    b = O.sample(edges, 9, 2, 0, 500, O.GAUSS, [0.3], variant=O.V_Q32)
    for u, v in zip(a, b):
        assert np.array_equal(u, v)


# ---------------------------------------------------------------- C6/C7 with the variants, chains
@pytest.mark.parametrize("variant", [O.V_U53, O.V_Q32, O.V_U53 | O.V_Q32])
def test_variants_brute_force_reaccumulation(variant):
    w = W.config(4)
    dim, nb, n = 5, 20, 4000
    params = np.concatenate([w.params[:dim], w.params[w.dim:w.dim + dim]])
    edges = W.adapted_edges(dim, nb, seed=42)
    _, bins, x, fJ = O.sample(edges, 4, 1, 0, n, O.GENZ_PRODUCT_PEAK, params, variant=variant)
    I, sg, H = O.iterate(edges, n, 4, 1, O.GENZ_PRODUCT_PEAK, params, variant=variant)
    v = fJ.astype(np.longdouble)
    S1, S2 = v.sum(), (v * v).sum()
    mean = S1 / n
    assert abs(I - float(mean)) <= 1e-15 * abs(I)
    assert abs(sg - float(np.sqrt((S2 / n - mean * mean) / (n - 1)))) <= 1e-12 * sg
    Hb = np.zeros((dim, nb), dtype=np.longdouble)
    for j in range(dim):
        np.add.at(Hb[j], bins[:, j], v * v)
    np.testing.assert_allclose(H, Hb.astype(np.float64), rtol=1e-14)
    for j in range(dim):
        assert abs(H[j].sum() - float(S2)) <= 1e-13 * float(S2)
    # threads only split the event range
    I2, sg2, H2 = O.iterate(edges, n, 4, 1, O.GENZ_PRODUCT_PEAK, params, threads=3, variant=variant)
    assert abs(I2 - I) <= 1e-15 * abs(I) and np.allclose(H2, H, rtol=1e-14, atol=0)


@pytest.mark.parametrize("variant", [O.V_U53, O.V_Q32, O.V_U53 | O.V_Q32])
def test_variant_chains_within_5_sigma_of_the_closed_form(variant):
    w = W.config(1)
    res = O.integrate(w.dim, w.n_bins, 5, 50000, w.seed, w.alpha, w.integrand_id, w.params, variant=variant)
    assert res["status"] == O.OK
    assert abs(res["I"] - w.closed_form) <= 5 * res["sigma"]
    for Ik, sk in res["per_iter"][1:]:
        assert abs(Ik - w.closed_form) <= 5 * sk
    # f = 1 on the uniform grid: exactly 1 up to rounding for the 53-bit draw; within d 2^-24 for the rounded table
    I, sg, _ = O.iterate(O.uniform_edges(4, 50), 20000, 1, 0, O.CONST, variant=variant)
    assert abs(I - 1.0) <= (1e-12 if variant == O.V_U53 else 4 * 2.0**-24)


def test_variant_zero_is_the_method_and_bad_masks_are_rejected():
    edges = W.adapted_edges(3, 10, seed=1)
    a = O.iterate(edges, 3000, 2, 0, O.GAUSS, [0.2])
    b = O.iterate(edges, 3000, 2, 0, O.GAUSS, [0.2], variant=0)
    assert a[0] == b[0] and a[1] == b[1] and np.array_equal(a[2], b[2])
    with pytest.raises(O.OracleError):
        O.sample(edges, 1, 0, 0, 4, O.CONST, variant=4)
