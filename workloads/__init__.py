"""Seeded synthetic workloads: the five BASELINE.json configs and their parameter draws.

This module is the ONLY thing the CUDA path's tests/bench and the CPU oracle's tests have in
common.  It holds inputs, not the method: sizes, seeds, integrand ids, the integrand parameter
arrays and the analytic value of each integral.  It lives outside the product package and imports neither the CUDA binding nor
``oracle``.  Parameters are handed to both implementations as plain fp64 arrays.

Parameter draws (reading C10 of DESIGN.md; BASELINE.json:configs[3] "c_i drawn uniform in
[5,15] and w_i uniform in [0,1] from seed=4", configs[4] "coefficients uniform in [0,1] from
seed=5"): u_q = (word_q + 0.5) * 2^-32 where word_q is output word q&3 of the Philox4x32-10
block with counter (q>>2, 0xFFFFFFFF, 0, 0) and key (seed lo, seed hi).  The generator below is
a third, self-contained restatement in Python integers used for nothing but these draws;
neither the oracle nor the kernels call it.

The workloads stand in for the paper's own benchmark integrands, whose parameters are not
printed: cfg1-3 <-> SymGauss rows (Eq.(1)), cfg4 <->
Genz product peak (Eq.(3)), cfg5 <-> the single-top LO computation
(PAPER.md:134-138), which cannot be built here.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

CONST, GAUSS, GENZ_PRODUCT_PEAK, BW_POLY, GENZ_DISCONTINUOUS = 0, 1, 2, 3, 4
INTEGRAND_NAMES = {CONST: "const", GAUSS: "gauss", GENZ_PRODUCT_PEAK: "genz_product_peak",
                   BW_POLY: "bw_poly", GENZ_DISCONTINUOUS: "genz_discontinuous"}

_M0, _M1 = 0xD2511F53, 0xCD9E8D57
_W0, _W1 = 0x9E3779B9, 0xBB67AE85
_MASK = 0xFFFFFFFF


def _draw_block(counter, key):
    c0, c1, c2, c3 = counter
    k0, k1 = key
    for rnd in range(10):
        if rnd:
            k0 = (k0 + _W0) & _MASK
            k1 = (k1 + _W1) & _MASK
        p0, p1 = _M0 * c0, _M1 * c2
        c0, c1, c2, c3 = ((p1 >> 32) ^ c1 ^ k0) & _MASK, p1 & _MASK, \
                         ((p0 >> 32) ^ c3 ^ k1) & _MASK, p0 & _MASK
    return c0, c1, c2, c3


def parameter_uniforms(seed: int, count: int) -> np.ndarray:
    """C10: count uniforms in (0,1) reserved for parameter generation (iteration 0xFFFFFFFF)."""
    key = (seed & _MASK, (seed >> 32) & _MASK)
    out = np.empty(count, dtype=np.float64)
    for q in range(count):
        w = _draw_block((q >> 2, 0xFFFFFFFF, 0, 0), key)[q & 3]
        out[q] = (w + 0.5) / 4294967296.0
    return out


@dataclass
class Workload:
    name: str
    dim: int
    n_bins: int
    n_iter: int
    n_events: int
    chunk_events: int          # 0 = one launch per iteration
    seed: int
    integrand_id: int
    params: np.ndarray
    alpha: float = 1.5
    n_skip: int = 0            # iterations excluded from the 5-sigma-gated average (finding F1)
    precisions: tuple = (64,)
    note: str = ""
    extra: dict = field(default_factory=dict)

    @property
    def closed_form(self) -> float:
        return closed_form(self.integrand_id, self.dim, self.params)

    def scaled(self, n_events: int, n_iter: int | None = None, chunk_events: int | None = None):
        """Same workload at a smaller size (for oracle-speed parity cases)."""
        return Workload(self.name, self.dim, self.n_bins, self.n_iter if n_iter is None else n_iter,
                        int(n_events), self.chunk_events if chunk_events is None else chunk_events,
                        self.seed, self.integrand_id, self.params, self.alpha, self.n_skip,
                        self.precisions, self.note, dict(self.extra))


def closed_form(integrand_id: int, dim: int, params) -> float:
    """Analytic integral over [0,1]^dim of the built-in integrands (erf / atan closed forms)."""
    p = np.asarray(params, dtype=np.float64)
    if integrand_id == CONST:
        return 1.0
    if integrand_id == GAUSS:
        return math.erf(1.0 / (2.0 * p[0])) ** dim
    if integrand_id == GENZ_PRODUCT_PEAK:
        c, w = p[:dim], p[dim:2 * dim]
        val = 1.0
        for cj, wj in zip(c, w):
            val *= cj * (math.atan(cj * (1.0 - wj)) + math.atan(cj * wj))
        return val
    if integrand_id == BW_POLY:
        M, G, m_min, m_max = p[:4]
        a = p[4:].reshape(dim - 1, 5)
        s_min, s_max = m_min * m_min, m_max * m_max
        bw = (M * G / (s_max - s_min)) * (math.atan((s_max - M * M) / (M * G))
                                          - math.atan((s_min - M * M) / (M * G)))
        poly = sum(a[i, k] / (k + 1.0) for i in range(dim - 1) for k in range(5))
        return bw * poly
    if integrand_id == GENZ_DISCONTINUOUS:        # PAPER.md:69 Eq.(2) as printed, N = 1: zero where any x_j <= a_j
        c, a = p[:dim], p[dim:2 * dim]
        val = 1.0
        for cj, aj in zip(c, a):
            val *= (math.exp(cj) - math.exp(cj * aj)) / cj
        return val
    raise ValueError("unknown integrand id %r" % integrand_id)


def genz_discontinuous_params(dim: int, seed: int) -> np.ndarray:
    """c_j = 0.5 + u_j, a_j = 0.3 u_{dim+j} (C10 draws): the zero region removes 1 - prod(1 - a_j) of the volume."""
    u = parameter_uniforms(seed, 2 * dim)
    return np.concatenate([0.5 + u[:dim], 0.3 * u[dim:2 * dim]])


def gauss_params(a: float = 0.1) -> np.ndarray:
    return np.array([a], dtype=np.float64)


def genz_params(dim: int, seed: int) -> np.ndarray:
    u = parameter_uniforms(seed, 2 * dim)
    return np.concatenate([5.0 + 10.0 * u[:dim], u[dim:2 * dim]])


def bw_poly_params(dim: int, seed: int, M=80.4, Gamma=2.1, m_min=10.0, m_max=200.0) -> np.ndarray:
    u = parameter_uniforms(seed, 5 * (dim - 1))
    return np.concatenate([[M, Gamma, m_min, m_max], u])


def config(i: int) -> Workload:
    """BASELINE.json:configs[i-1] (1-based, as SURVEY.md numbers them cfg1..cfg5)."""
    if i == 1:
        return Workload("cfg1_gauss_d4", 4, 50, 5, 100_000, 0, 1, GAUSS, gauss_params())
    if i == 2:
        return Workload("cfg2_gauss_d8", 8, 50, 10, 10_000_000, 0, 2, GAUSS, gauss_params())
    if i == 3:
        return Workload("cfg3_gauss_d20", 20, 50, 10, 100_000_000, 10_000_000, 3, GAUSS,
                        gauss_params(), n_skip=3, precisions=(64, 32),
                        note="5-sigma gate from iteration 3 on (finding F1)")
    if i == 4:
        return Workload("cfg4_genz_pp_d12", 12, 100, 15, 50_000_000, 0, 4, GENZ_PRODUCT_PEAK,
                        genz_params(12, 4))
    if i == 5:
        return Workload("cfg5_bw_poly_d6", 6, 50, 20, 1_000_000_000, 25_000_000, 5, BW_POLY,
                        bw_poly_params(6, 5))
    raise ValueError("configs are numbered 1..5")


def control_const(dim: int = 8, n_bins: int = 50, n_events: int = 10_000_000, seed: int = 2):
    """cfg2's constant f=1 control run."""
    return Workload("cfg2_control_const", dim, n_bins, 10, n_events, 0, seed, CONST,
                    np.zeros(0))


def adapted_edges(dim: int, n_bins: int, seed: int = 12345, strength: float = 3.0) -> np.ndarray:
    """A synthetic non-uniform grid with strictly increasing edges, 0 and 1 at the ends, bins
    narrower towards x = 1/2 (what a peaked integrand produces).  Used for injected-grid
    parity cases that do not need an oracle chain first.  numpy PCG64 stream, fixed seed."""
    rng = np.random.default_rng(seed)
    edges = np.empty((dim, n_bins + 1))
    centres = (np.arange(n_bins) + 0.5) / n_bins
    for j in range(dim):
        w = 1.0 / (1.0 + strength * np.exp(-((centres - 0.5) / 0.15) ** 2)) \
            * (0.5 + rng.random(n_bins))
        c = np.concatenate([[0.0], np.cumsum(w)])
        e = c / c[-1]
        e[0], e[-1] = 0.0, 1.0
        edges[j] = e
    return edges
