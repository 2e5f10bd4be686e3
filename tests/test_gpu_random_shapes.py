"""Seeded sweep over random shapes: dimension 1..32, n_bins 2..256, every built-in integrand, both precisions, both
kernels, ragged event counts, chunking and event offsets -- one teacher-forced iteration each against the oracle (P3),
plus the refinement (P4).  Catches what the five configs cannot: odd last-block shapes, tiny grids, shapes that fall
back to the generic kernel because their shared memory does not fit."""
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle as O
import workloads as W

THREADS = os.cpu_count() or 8


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    from paper_2002_12921_b200 import build
    build.build()
    from paper_2002_12921_b200 import binding
    return binding


def _case(rng):
    fid = int(rng.integers(0, 4))
    dim = int(rng.integers(2 if fid == 3 else 1, 33))
    nb = int(rng.choice([2, 3, 7, 16, 33, 50, 64, 100, 128, 200, 256]))
    if fid == 0:
        p = None
    elif fid == 1:
        p = W.gauss_params(float(rng.uniform(0.08, 0.6)))
    elif fid == 2:
        p = W.genz_params(dim, int(rng.integers(1, 1000)))
    else:
        p = W.bw_poly_params(dim, int(rng.integers(1, 1000)))
    precision = int(rng.choice([64, 64, 32]))
    return dict(fid=fid, dim=dim, nb=nb, params=p, precision=precision,
                n=int(rng.integers(20_000, 120_000)), seed=int(rng.integers(1, 2**40)),
                iteration=int(rng.integers(0, 2**31)), first=int(rng.choice([0, 0, 12345, (1 << 32) - 30_000, 7 << 33])),
                chunk=int(rng.choice([0, 0, 17_000, 50_001])), threads=int(rng.choice([0, 0, 0, 128, 256, 352])),
                generic=bool(rng.random() < 0.25), grid_seed=int(rng.integers(1, 1000)))


def _r23_bound(fid, params, edges):
    """Reading R23: the fp32 table entry of the Breit-Wigner variable u_0 = scale_0 (x_0 - shift_0), scale_0 =
    (m_max^2 - m_min^2)/(M Gamma), shift_0 = (M^2 - m_min^2)/(m_max^2 - m_min^2), carries an absolute error of up to
    2^-24 scale_0 (|X_b - shift_0| + 2 Delta_b); in the bin that holds the resonance (|u_0| ~ 1) that is a relative
    error of the same size on f (and on I, sigma), twice that on H.  0 for the other integrands."""
    if fid != 3:
        return 0.0
    M, G, m_min, m_max = params[:4]
    ds = m_max * m_max - m_min * m_min
    scale0, shift0 = ds / (M * G), (M * M - m_min * m_min) / ds
    X = edges[0]
    b = int(np.searchsorted(X, shift0, side="right")) - 1
    return 2.0 ** -24 * scale0 * (max(abs(X[b] - shift0), abs(X[b + 1] - shift0)) + 2 * (X[b + 1] - X[b]))


N_CASES = int(os.environ.get("VEGAS_SWEEP_CASES", "48"))       # a longer sweep: VEGAS_SWEEP_CASES=400 pytest ...


@pytest.mark.parametrize("case_id", range(N_CASES))
def test_random_shape_iteration_and_refinement(B, case_id):
    c = _case(np.random.default_rng(1000 + case_id))
    dim, nb, fid, prec = c["dim"], c["nb"], c["fid"], c["precision"]
    edges = W.adapted_edges(dim, nb, seed=c["grid_seed"])
    g = B.VegasGrid(dim, nb)
    if fid != 0:
        g.set_params(fid, c["params"])
    g.set_edges(edges)
    if c["generic"]:
        try:
            g.set_launch(0, 0, 2, 4)
        except B.VegasError:                              # these copy counts do not fit next to a large grid
            g.set_launch(0, 0, 1, 1)
    elif c["threads"]:
        g.set_launch(0, c["threads"], 0, 0)
    path = g.get_launch(fid, prec)["path"]
    assert path in ("rotated", "generic") and (path == "generic" or not c["generic"])
    g.begin_iteration()
    g.accumulate(c["first"], c["n"], c["seed"], c["iteration"], fid, prec, chunk_events=c["chunk"])
    g.reduce()
    I, s, H, st = g.finalize(c["n"])
    S1, S2, Ho = O.accumulate(edges, c["seed"], c["iteration"], c["first"], c["n"], fid, c["params"])
    oI, oS = O.estimate(S1, S2, c["n"])
    Ho = Ho.astype(np.float64)
    info = "case %r path %s" % ({k: v for k, v in c.items() if k != "params"}, path)
    if prec == 64:
        assert st == 0 and I == pytest.approx(oI, rel=1e-10), info
        assert s == pytest.approx(oS, rel=1e-10, abs=1e-300), info
        np.testing.assert_allclose(H, Ho, rtol=1e-10, atol=0, err_msg=info)
    else:
        # fp32 per-event arithmetic against the fp64 oracle: 1e-5 on I, sigma and H (north_star; H in the
        # per-dimension max-norm, reading F3) -- except where reading R23 derives a wider bound:
        # BW_POLY on a grid whose bin AT the resonance is wider than ~0.1
        tol = max(1e-5, _r23_bound(fid, c["params"], edges))
        assert st == 0 and I == pytest.approx(oI, rel=tol), info
        assert s == pytest.approx(oS, rel=tol, abs=1e-300), info
        assert np.all(np.abs(H - Ho) <= max(1e-5, 2 * _r23_bound(fid, c["params"], edges)) * Ho.max(axis=1, keepdims=True)), \
            (info, float(np.max(np.abs(H - Ho) / Ho.max(axis=1, keepdims=True))))
    # refinement of the oracle's histogram on the GPU vs the oracle's own (skip all-zero rows: ENUMERIC on both sides)
    want, ost = O.refine(edges, Ho, 1.5)
    rc = g.refine(1.5, hist=Ho)
    assert (rc != 0) == (ost != 0), info
    np.testing.assert_allclose(g.get_edges(), want, rtol=0, atol=1e-10, err_msg=info)
    g.close()
