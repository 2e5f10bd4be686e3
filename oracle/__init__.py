"""Python face of the CPU oracle (oracle/vegas_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / ``--impl reference`` legs
may import this package; the product (paper_2002_12921_b200) never does and shares no code
with it.  Everything numerical happens in the C file; this module only marshals numpy arrays
through ctypes and, for ``iterate(..., threads=P)``, runs the single-threaded C routine on P
disjoint event ranges (the RNG is counter-based, C2, so the union is the same sample set) and
adds the long-double partial sums in range order.

Readings C1..C9 are those of SURVEY.md section 8(c), restated in DESIGN.md.
"""
from __future__ import annotations

import ctypes as C
from concurrent.futures import ThreadPoolExecutor

import numpy as np

from .build import build as _build

CONST, GAUSS, GENZ_PRODUCT_PEAK, BW_POLY, GENZ_DISCONTINUOUS = 0, 1, 2, 3, 4
# variants of the sampling map (readings C3', C4'); a bit mask
V_U53, V_Q32 = 1, 2
OK, EINVAL, ENUMERIC = 0, -1, -3

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build())
        u32p, i32p, f64p = (C.POINTER(C.c_uint32), C.POINTER(C.c_int32), C.POINTER(C.c_double))
        L.oracle_philox4x32_10.argtypes = [u32p, u32p, u32p]
        L.oracle_philox4x32_10.restype = None
        L.oracle_word.argtypes = [C.c_uint64, C.c_uint32, C.c_uint64, C.c_int]
        L.oracle_word.restype = C.c_uint32
        L.oracle_split.argtypes = [C.c_uint32, C.c_int, i32p, f64p]
        L.oracle_split.restype = None
        L.oracle_n_params.argtypes = [C.c_int, C.c_int]
        L.oracle_n_params.restype = C.c_int
        L.oracle_f.argtypes = [C.c_int, C.c_int, f64p, f64p]
        L.oracle_f.restype = C.c_double
        L.oracle_word53.argtypes = [C.c_uint64, C.c_uint32, C.c_uint64, C.c_int]
        L.oracle_word53.restype = C.c_uint64
        L.oracle_split53.argtypes = [C.c_uint64, C.c_int, i32p, f64p]
        L.oracle_split53.restype = None
        L.oracle_q32.argtypes = [C.c_double]
        L.oracle_q32.restype = C.c_double
        L.oracle_sample_v.argtypes = [C.c_int, C.c_int, C.c_int, f64p, C.c_uint64, C.c_uint32, C.c_uint64,
                                      C.c_uint64, C.c_int, f64p, u32p, i32p, f64p, f64p]
        L.oracle_sample_v.restype = C.c_int
        L.oracle_accumulate_v.argtypes = [C.c_int, C.c_int, C.c_int, f64p, C.c_uint64, C.c_uint32,
                                          C.c_uint64, C.c_uint64, C.c_int, f64p, f64p, f64p, f64p]
        L.oracle_accumulate_v.restype = C.c_int
        L.oracle_estimate.argtypes = [f64p, C.c_uint64, f64p, f64p]
        L.oracle_estimate.restype = C.c_int
        L.oracle_iterate.argtypes = [C.c_int, C.c_int, f64p, C.c_uint64, C.c_uint64, C.c_uint32,
                                     C.c_int, f64p, f64p, f64p, f64p]
        L.oracle_iterate.restype = C.c_int
        L.oracle_refine.argtypes = [C.c_int, C.c_int, f64p, f64p, C.c_double, f64p]
        L.oracle_refine.restype = C.c_int
        L.oracle_combine.argtypes = [C.c_int, C.c_int, f64p, f64p, f64p, f64p, f64p]
        L.oracle_combine.restype = C.c_int
        L.oracle_uniform_edges.argtypes = [C.c_int, C.c_int, f64p]
        L.oracle_uniform_edges.restype = None
        L.oracle_integrate_v.argtypes = [C.c_int, C.c_int, C.c_int, f64p, C.c_int, C.c_int, C.c_uint64,
                                         C.c_uint64, C.c_double, C.c_int, f64p, f64p, f64p, f64p,
                                         f64p, f64p, f64p]
        L.oracle_integrate_v.restype = C.c_int
        _lib = L
    return _lib


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a, ctype=C.c_double):
    return a.ctypes.data_as(C.POINTER(ctype)) if a is not None else None


def _params(params):
    p = _f64(np.atleast_1d(np.asarray(params if params is not None else [], dtype=np.float64)))
    if p.size == 0:
        p = np.zeros(1)
    return p


class OracleError(RuntimeError):
    def __init__(self, code):
        super().__init__("oracle error %d" % code)
        self.code = code


def philox4x32_10(ctr, key):
    """C1: one Philox4x32-10 block; ctr 4 x u32, key 2 x u32 -> 4 x u32."""
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().oracle_philox4x32_10(_p(c, C.c_uint32), _p(k, C.c_uint32), _p(out, C.c_uint32))
    return out


def word(seed, iteration, event, j):
    """C2: the 32-bit word of (seed, iteration, event, dimension j)."""
    return int(lib().oracle_word(int(seed), int(iteration), int(event), int(j)))


def split(w, n_bins):
    """C3: word -> (bin, r)."""
    b, r = C.c_int32(), C.c_double()
    lib().oracle_split(int(w), int(n_bins), C.byref(b), C.byref(r))
    return b.value, r.value


def word53(seed, iteration, event, j):
    """C3': the 53-bit integer U of (seed, iteration, event, dimension j), two Philox words per draw."""
    return int(lib().oracle_word53(int(seed), int(iteration), int(event), int(j)))


def split53(U, n_bins):
    """C3': U -> (bin, r) with r in [0,1)."""
    b, r = C.c_int32(), C.c_double()
    lib().oracle_split53(int(U), int(n_bins), C.byref(b), C.byref(r))
    return b.value, r.value


def q32(v):
    """C4': a table entry rounded to fp32 and widened back."""
    return float(lib().oracle_q32(float(v)))


def n_params(integrand_id, dim):
    return int(lib().oracle_n_params(integrand_id, dim))


def f(integrand_id, x, params=None):
    """C5: integrand value at one point x (length-d array)."""
    x = _f64(x)
    p = _params(params)
    return float(lib().oracle_f(integrand_id, x.size, _p(x), _p(p)))


def uniform_edges(dim, n_bins):
    """C4: uniform start grid, X[j][i] = i / n_bins; shape [dim, n_bins+1]."""
    e = np.zeros((dim, n_bins + 1))
    lib().oracle_uniform_edges(dim, n_bins, _p(e))
    return e


def sample(edges, seed, iteration, first_event, count, integrand_id, params=None, variant=0):
    """C2..C5 for events [first_event, first_event+count): (words, bins, x, fJ).
    With V_U53 the words column holds the top 32 bits of each 53-bit U."""
    edges = _f64(edges)
    dim, nb = edges.shape[0], edges.shape[1] - 1
    p = _params(params)
    words = np.zeros((count, dim), dtype=np.uint32)
    bins = np.zeros((count, dim), dtype=np.int32)
    x = np.zeros((count, dim))
    fJ = np.zeros(count)
    rc = lib().oracle_sample_v(int(variant), dim, nb, _p(edges), int(seed), int(iteration), int(first_event),
                               int(count), integrand_id, _p(p), _p(words, C.c_uint32),
                               _p(bins, C.c_int32), _p(x), _p(fJ))
    if rc:
        raise OracleError(rc)
    return words, bins, x, fJ


def accumulate(edges, seed, iteration, first_event, count, integrand_id, params=None, variant=0):
    """C6 on one event range: (S1, S2, H) as np.longdouble scalars / array [dim, n_bins]."""
    edges = _f64(edges)
    dim, nb = edges.shape[0], edges.shape[1] - 1
    p = _params(params)
    sums = np.zeros(4)
    hi = np.zeros((dim, nb))
    lo = np.zeros((dim, nb))
    rc = lib().oracle_accumulate_v(int(variant), dim, nb, _p(edges), int(seed), int(iteration), int(first_event),
                                   int(count), integrand_id, _p(p), _p(sums), _p(hi), _p(lo))
    if rc:
        raise OracleError(rc)
    ld = np.longdouble
    return (ld(sums[0]) + ld(sums[1]), ld(sums[2]) + ld(sums[3]),
            hi.astype(ld) + lo.astype(ld))


def estimate(S1, S2, n_events):
    """C7: (I, sigma) from long-double sums."""
    ld = np.longdouble
    s = np.zeros(4)
    s[0] = float(S1); s[1] = float(ld(S1) - ld(s[0]))
    s[2] = float(S2); s[3] = float(ld(S2) - ld(s[2]))
    I, sg = C.c_double(), C.c_double()
    rc = lib().oracle_estimate(_p(s), int(n_events), C.byref(I), C.byref(sg))
    if rc:
        raise OracleError(rc)
    return I.value, sg.value


def iterate(edges, n_events, seed, iteration, integrand_id, params=None, threads=1, variant=0):
    """One Vegas iteration (C2..C7) on the given grid: (I, sigma, H[dim, n_bins] fp64).

    threads > 1 runs the single-threaded C routine on disjoint event ranges concurrently
    (ctypes drops the GIL) and adds the long-double partial sums in range order."""
    n_events = int(n_events)
    if n_events < 2:
        raise OracleError(EINVAL)
    threads = max(1, min(int(threads), n_events // 1024 or 1))
    bounds = [n_events * t // threads for t in range(threads + 1)]
    jobs = [(bounds[t], bounds[t + 1] - bounds[t]) for t in range(threads)]

    def run(job):
        return accumulate(edges, seed, iteration, job[0], job[1], integrand_id, params, variant)

    if threads == 1:
        parts = [run(jobs[0])]
    else:
        with ThreadPoolExecutor(max_workers=threads) as ex:
            parts = list(ex.map(run, jobs))
    S1 = np.longdouble(0)
    S2 = np.longdouble(0)
    H = np.zeros_like(parts[0][2])
    for a, b, h in parts:
        S1 = S1 + a
        S2 = S2 + b
        H = H + h
    I, sg = estimate(S1, S2, n_events)
    return I, sg, H.astype(np.float64)


def refine(edges, hist, alpha):
    """C8: new edges [dim, n_bins+1] from a histogram; returns (new_edges, status)."""
    edges = _f64(edges)
    hist = _f64(hist)
    dim, nb = edges.shape[0], edges.shape[1] - 1
    out = np.zeros_like(edges)
    rc = lib().oracle_refine(dim, nb, _p(edges), _p(hist), float(alpha), _p(out))
    if rc == EINVAL:
        raise OracleError(rc)
    return out, rc


def combine(I_k, sigma_k, n_skip=0):
    """C9: inverse-variance combination -> (I, sigma, chi2_dof)."""
    I_k = _f64(I_k)
    sigma_k = _f64(sigma_k)
    I, s, c = C.c_double(), C.c_double(), C.c_double()
    rc = lib().oracle_combine(I_k.size, int(n_skip), _p(I_k), _p(sigma_k), C.byref(I),
                              C.byref(s), C.byref(c))
    if rc:
        raise OracleError(rc)
    return I.value, s.value, c.value


def integrate(dim, n_bins, n_iter, n_events, seed, alpha, integrand_id, params=None, n_skip=0,
              edges=None, threads=1, variant=0):
    """Whole chain (C2..C9).  Returns a dict with I, sigma, chi2_dof, per_iter [n_iter,2],
    edges_trace [n_iter, dim, n_bins+1] (grid each iteration sampled from), hist_trace
    [n_iter, dim, n_bins], edges (final grid), status.  threads > 1 uses iterate(threads=...)
    per iteration (same arithmetic per event; partial sums added in range order)."""
    edges = uniform_edges(dim, n_bins) if edges is None else _f64(edges).copy()
    p = _params(params)
    per_iter = np.zeros((n_iter, 2))
    et = np.zeros((n_iter, dim, n_bins + 1))
    ht = np.zeros((n_iter, dim, n_bins))
    status = OK
    if threads == 1:
        I, s, c = C.c_double(), C.c_double(), C.c_double()
        status = lib().oracle_integrate_v(int(variant), dim, n_bins, _p(edges), n_iter, n_skip, int(n_events),
                                          int(seed), float(alpha), integrand_id, _p(p),
                                          C.byref(I), C.byref(s), C.byref(c), _p(per_iter),
                                          _p(et), _p(ht))
        if status == EINVAL:
            raise OracleError(status)
        res = (I.value, s.value, c.value)
    else:
        for k in range(n_iter):
            et[k] = edges
            Ik, sk, H = iterate(edges, n_events, seed, k, integrand_id, params, threads, variant)
            ht[k] = H
            per_iter[k] = (Ik, sk)
            if alpha >= 0:
                edges, rc = refine(edges, H, alpha)
                if rc:
                    status = rc
        res = combine(per_iter[:, 0], per_iter[:, 1], n_skip)
    return dict(I=res[0], sigma=res[1], chi2_dof=res[2], per_iter=per_iter, edges_trace=et,
                hist_trace=ht, edges=edges, status=status)
