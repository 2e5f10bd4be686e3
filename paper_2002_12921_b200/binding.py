"""ctypes binding of libvegas_b200.so: the entry points of include/vegas.h under the same names.

Argument marshalling only -- every step of the hot path runs in the library's CUDA kernels.
PyTorch is used for device memory (the workspace) and streams, nothing else.  There is no CPU
fallback: if the shared library is missing this module raises at import, and without a CUDA
device the compute calls return VEGAS_ECUDA (raised as VegasError).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libvegas_b200.so")

VEGAS_OK, VEGAS_EINVAL, VEGAS_ECUDA, VEGAS_ENUMERIC, VEGAS_ELIMIT = 0, -1, -2, -3, -4
VEGAS_STATIC_MAX_ENTRIES = 2048
VEGAS_F_CONST, VEGAS_F_GAUSS, VEGAS_F_GENZ_PRODUCT_PEAK, VEGAS_F_BW_POLY, VEGAS_F_USER = 0, 1, 2, 3, 4
VEGAS_F_GENZ_DISCONTINUOUS = 5
VEGAS_USER_MAX_PARAMS = 64
VEGAS_FP64, VEGAS_FP32 = 64, 32
VEGAS_VARIANT_NONE, VEGAS_VARIANT_U53, VEGAS_VARIANT_Q32 = 0, 1, 2
VEGAS_MAX_DIM, VEGAS_MAX_BINS, VEGAS_MAX_PARAMS = 32, 256, 160

if not os.path.exists(LIB_PATH):
    raise ImportError(
        "libvegas_b200.so is not built (%s). Run `python -m paper_2002_12921_b200.build` or "
        "`python -c 'import __graft_entry__ as g; g.build()'`; there is no CPU fallback." % LIB_PATH)

lib = C.CDLL(LIB_PATH)

_f64p, _u32p, _i32p = C.POINTER(C.c_double), C.POINTER(C.c_uint32), C.POINTER(C.c_int32)
_vp, _u64 = C.c_void_p, C.c_uint64

# name -> (restype, argtypes); one entry per declaration in include/vegas.h
SIGNATURES = {
    "vegas_workspace_bytes": (C.c_size_t, [C.c_int, C.c_int]),
    "vegas_create": (C.c_int, [C.c_int, C.c_int, _vp, C.c_size_t, C.POINTER(_vp)]),
    "vegas_destroy": (C.c_int, [_vp]),
    "vegas_set_params": (C.c_int, [_vp, C.c_int, _f64p, C.c_int]),
    "vegas_set_user_integrand": (C.c_int, [_vp, C.c_char_p, _f64p, C.c_int, C.c_char_p, C.c_size_t]),
    "vegas_set_observable": (C.c_int, [_vp, C.c_double, C.c_double, C.c_int]),
    "vegas_get_observable_hist": (C.c_int, [_vp, _f64p, _vp]),
    "vegas_callback_scratch_bytes": (C.c_size_t, [C.c_int, C.c_uint32]),
    "vegas_iterate_callback": (C.c_int, [_vp, _u64, C.c_uint32, _u64, C.c_uint32, _vp, _vp, _vp, C.c_size_t, _vp,
                                         _f64p, _f64p, _f64p]),
    "vegas_set_edges": (C.c_int, [_vp, _f64p, _vp]),
    "vegas_get_edges": (C.c_int, [_vp, _f64p, _vp]),
    "vegas_get_hist": (C.c_int, [_vp, _f64p, _vp]),
    "vegas_iterate": (C.c_int, [_vp, _u64, _u64, _u64, C.c_uint32, C.c_int, C.c_int, _vp, _f64p, _f64p, _f64p]),
    "vegas_iterate_static": (C.c_int, [_vp, C.c_int, C.c_int, _u64, _u64, C.c_uint32, C.c_int, _f64p, C.c_int, C.c_int,
                                       _vp, _vp, _vp]),
    "vegas_begin_iteration": (C.c_int, [_vp, _vp]),
    "vegas_accumulate": (C.c_int, [_vp, _u64, _u64, _u64, _u64, C.c_uint32, C.c_int, C.c_int, _vp]),
    "vegas_reduce": (C.c_int, [_vp, _vp]),
    "vegas_finalize": (C.c_int, [_vp, _u64, _vp, _f64p, _f64p, _f64p]),
    "vegas_finish_sharded": (C.c_int, [_vp, _u64, C.c_double, _vp, _f64p, _f64p, _f64p]),
    "vegas_totals_device": (_vp, [_vp]),
    "vegas_totals_count": (C.c_size_t, [_vp]),
    "vegas_refine": (C.c_int, [_vp, _f64p, C.c_double, _vp]),
    "vegas_integrate": (C.c_int, [_vp, C.c_int, C.c_int, _u64, _u64, _u64, C.c_double, C.c_int, C.c_int, _vp,
                                  _f64p, _f64p, _f64p, _f64p]),
    "vegas_integrate_from": (C.c_int, [_vp, C.c_uint32, C.c_int, C.c_int, _u64, _u64, _u64, C.c_double, C.c_int, C.c_int,
                                       _vp, _f64p, _f64p, _f64p, _f64p]),
    "vegas_combine": (C.c_int, [C.c_int, C.c_int, _f64p, _f64p, _f64p, _f64p, _f64p]),
    "vegas_debug_scratch_bytes": (C.c_size_t, [C.c_int, C.c_uint32]),
    "vegas_debug_sample": (C.c_int, [_vp, _u64, C.c_uint32, _u64, C.c_uint32, C.c_int, C.c_int, _vp, _vp,
                                     _u32p, _i32p, _f64p, _f64p]),
    "vegas_set_launch": (C.c_int, [_vp, C.c_int, C.c_int, C.c_int, C.c_int]),
    "vegas_get_launch": (C.c_int, [_vp, C.c_int, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int),
                                   C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_size_t)]),
    "vegas_set_variant": (C.c_int, [_vp, C.c_int]),
    "vegas_get_variant": (C.c_int, [_vp]),
    "vegas_set_profiling": (C.c_int, [_vp, C.c_int]),
    "vegas_kernel_time_ms": (C.c_int, [_vp, _f64p, C.POINTER(_u64)]),
    "vegas_launch_count": (_u64, [_vp]),
    "vegas_reset_counters": (C.c_int, [_vp]),
    "vegas_strerror": (C.c_char_p, [C.c_int]),
    "vegas_last_cuda_error": (C.c_char_p, [_vp]),
    "vegas_version": (C.c_char_p, []),
}
for _name, (_res, _args) in SIGNATURES.items():
    _fn = getattr(lib, _name)          # AttributeError here = the library does not export it
    _fn.restype = _res
    _fn.argtypes = _args


HOST_INTEGRAND = C.CFUNCTYPE(None, _f64p, _u64, C.c_int, _f64p, _vp)


class VegasError(RuntimeError):
    def __init__(self, code, detail=""):
        msg = lib.vegas_strerror(code).decode()
        super().__init__("vegas error %d: %s%s" % (code, msg, (" [%s]" % detail) if detail else ""))
        self.code = code


def _ptr(a, ctype=C.c_double):
    return a.ctypes.data_as(C.POINTER(ctype)) if a is not None else None


def _stream(stream):
    if stream is None:
        import torch
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    if hasattr(stream, "cuda_stream"):
        return C.c_void_p(stream.cuda_stream)
    return C.c_void_p(int(stream))


def vegas_workspace_bytes(dim, n_bins):
    return int(lib.vegas_workspace_bytes(dim, n_bins))


def vegas_version():
    return lib.vegas_version().decode()


def vegas_strerror(code):
    return lib.vegas_strerror(code).decode()


def vegas_combine(I_k, sigma_k, n_skip=0):
    I_k = np.ascontiguousarray(I_k, dtype=np.float64)
    sigma_k = np.ascontiguousarray(sigma_k, dtype=np.float64)
    I, s, c = C.c_double(), C.c_double(), C.c_double()
    rc = lib.vegas_combine(I_k.size, n_skip, _ptr(I_k), _ptr(sigma_k), C.byref(I), C.byref(s), C.byref(c))
    if rc:
        raise VegasError(rc)
    return I.value, s.value, c.value


def vegas_iterate_static(edges, n_events, seed, iteration, integrand_id, params, result, hist=None,
                         precision=VEGAS_FP64, stream=None):
    """One iteration without a grid handle and without any device workspace (include/vegas.h: vegas_iterate_static).

    For code that only holds the buffers it was given -- an op inside a framework that owns the GPU memory pool, a
    latency-bound loop, a process on a fixed memory budget -- and so cannot allocate the workspace a VegasGrid needs.
    edges [dim, n_bins+1], result [>=3] and hist [dim, n_bins] (optional) are CUDA float64 torch tensors owned by the
    caller, contiguous, on the current device; params is a host array as for set_params.  Only enqueues work on the
    stream: result = {I, sigma, status} and hist are valid once the stream gets there (torch.cuda.synchronize() or
    an event).  Shapes with dim * n_bins > VEGAS_STATIC_MAX_ENTRIES raise VegasError(VEGAS_ELIMIT).  All calls on a
    GPU share one built-in scratch array: issue them on one stream, or order them with events."""
    import torch
    for t, what in ((edges, "edges"), (result, "result"), (hist, "hist")):
        if t is None and what == "hist":
            continue
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
            raise VegasError(VEGAS_EINVAL, "%s must be a contiguous CUDA float64 tensor" % what)
    dim, n_bins = int(edges.shape[0]), int(edges.shape[1]) - 1
    if result.numel() < 3 or (hist is not None and tuple(hist.shape) != (dim, n_bins)):
        raise VegasError(VEGAS_EINVAL, "result needs 3 elements, hist the shape [dim, n_bins]")
    p = np.ascontiguousarray(np.atleast_1d(np.asarray(params if params is not None else [], dtype=np.float64)))
    rc = lib.vegas_iterate_static(_vp(edges.data_ptr()), dim, n_bins, int(n_events), int(seed), int(iteration),
                                  integrand_id, _ptr(p) if p.size else None, p.size, precision, _stream(stream),
                                  _vp(result.data_ptr()), _vp(hist.data_ptr()) if hist is not None else None)
    if rc:
        raise VegasError(rc)


class VegasGrid:
    """A vegas_grid handle plus the torch-allocated device workspace it lives in.

    Methods mirror the C entry points (vegas_<method>); ENUMERIC is returned as a status, other
    errors raise VegasError."""

    def __init__(self, dim, n_bins, device=None):
        import torch
        if not torch.cuda.is_available():
            raise VegasError(VEGAS_ECUDA, "no CUDA device; this library has no CPU fallback")
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        nbytes = vegas_workspace_bytes(dim, n_bins)
        if nbytes == 0:
            raise VegasError(VEGAS_EINVAL, "dim=%r n_bins=%r" % (dim, n_bins))
        self.dim, self.n_bins = dim, n_bins
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = self.workspace.data_ptr()
            aligned = (base + 255) // 256 * 256
            handle = C.c_void_p()
            rc = lib.vegas_create(dim, n_bins, C.c_void_p(aligned), nbytes, C.byref(handle))
        if rc:
            raise VegasError(rc)
        self._h = handle
        self._debug_scratch = None

    # -- lifetime
    def close(self):
        if getattr(self, "_h", None):
            lib.vegas_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc, allow_numeric=False):
        if rc == VEGAS_OK or (allow_numeric and rc == VEGAS_ENUMERIC):
            return rc
        raise VegasError(rc, lib.vegas_last_cuda_error(self._h).decode() if rc == VEGAS_ECUDA else "")

    # -- state
    def set_params(self, integrand_id, params):
        p = np.ascontiguousarray(np.atleast_1d(np.asarray(params if params is not None else [], dtype=np.float64)))
        self._check(lib.vegas_set_params(self._h, integrand_id, _ptr(p) if p.size else None, p.size))

    def set_user_integrand(self, cuda_source, params=None):
        """Compile `cuda_source` (struct vegas_user_integrand, see include/vegas.h) into the fused kernel for this
        grid; use integrand_id VEGAS_F_USER afterwards.  Returns the compiler log; raises VegasError (with the log
        as detail) when the source does not compile."""
        p = np.ascontiguousarray(np.atleast_1d(np.asarray(params if params is not None else [], dtype=np.float64)))
        log = C.create_string_buffer(1 << 16)
        rc = lib.vegas_set_user_integrand(self._h, cuda_source.encode(), _ptr(p) if p.size else None, p.size,
                                          log, len(log))
        text = log.value.decode(errors="replace")
        if rc != VEGAS_OK:
            raise VegasError(rc, text or lib.vegas_last_cuda_error(self._h).decode())
        return text

    def set_observable(self, lo, hi, n_obs_bins):
        self._check(lib.vegas_set_observable(self._h, float(lo), float(hi), int(n_obs_bins)))
        self._n_obs = int(n_obs_bins)

    def get_observable_hist(self, stream=None):
        out = np.zeros(self._n_obs)
        self._check(lib.vegas_get_observable_hist(self._h, _ptr(out), _stream(stream)))
        return out

    def set_edges(self, edges, stream=None):
        e = np.ascontiguousarray(edges, dtype=np.float64)
        if e.shape != (self.dim, self.n_bins + 1):
            raise VegasError(VEGAS_EINVAL, "edges shape %r" % (e.shape,))
        self._check(lib.vegas_set_edges(self._h, _ptr(e), _stream(stream)))

    def get_edges(self, stream=None):
        e = np.empty((self.dim, self.n_bins + 1))
        self._check(lib.vegas_get_edges(self._h, _ptr(e), _stream(stream)))
        return e

    def get_hist(self, stream=None):
        h = np.empty((self.dim, self.n_bins))
        self._check(lib.vegas_get_hist(self._h, _ptr(h), _stream(stream)))
        return h

    # -- the hot path
    def iterate(self, n_events, seed, iteration, integrand_id, precision=VEGAS_FP64, chunk_events=0,
                want_hist=True, stream=None):
        """-> (I, sigma, hist or None, status)"""
        I, s = C.c_double(), C.c_double()
        h = np.empty((self.dim, self.n_bins)) if want_hist else None
        rc = lib.vegas_iterate(self._h, int(n_events), int(chunk_events), int(seed), int(iteration), integrand_id,
                               precision, _stream(stream), C.byref(I), C.byref(s), _ptr(h))
        return I.value, s.value, h, self._check(rc, allow_numeric=True)

    def iterate_callback(self, fn, n_events, seed, iteration, batch_events=1 << 18, want_hist=True, stream=None,
                         overlap=True):
        """One iteration with a HOST integrand: fn(x) takes a float64 array [n, dim] and returns n values.
        overlap: scratch for two batches (the device samples batch k+1 while fn evaluates batch k); False hands the
        library half of it, which processes the batches strictly one after the other.
        -> (I, sigma, hist or None, status)"""
        import torch
        n_batch = int(min(batch_events, n_events))
        nbytes = lib.vegas_callback_scratch_bytes(self.dim, n_batch) // (1 if overlap else 2)
        scratch = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        ptr = (scratch.data_ptr() + 255) // 256 * 256
        dim = self.dim

        @HOST_INTEGRAND
        def _cb(x, n, d, f, user):
            xs = np.ctypeslib.as_array(x, shape=(n, d))
            out = np.ctypeslib.as_array(f, shape=(n,))
            out[:] = np.asarray(fn(xs), dtype=np.float64)

        I, s = C.c_double(), C.c_double()
        H = np.zeros((self.dim, self.n_bins)) if want_hist else None
        rc = lib.vegas_iterate_callback(self._h, int(n_events), n_batch, int(seed), int(iteration),
                                        C.cast(_cb, _vp), None, _vp(ptr), nbytes, _stream(stream),
                                        C.byref(I), C.byref(s), _ptr(H) if want_hist else None)
        self._check(rc, allow_numeric=True)
        return I.value, s.value, H, rc

    def begin_iteration(self, stream=None):
        self._check(lib.vegas_begin_iteration(self._h, _stream(stream)))

    def accumulate(self, first_event, count, seed, iteration, integrand_id, precision=VEGAS_FP64, chunk_events=0,
                   stream=None):
        self._check(lib.vegas_accumulate(self._h, int(first_event), int(count), int(chunk_events), int(seed),
                                         int(iteration), integrand_id, precision, _stream(stream)))

    def reduce(self, stream=None):
        self._check(lib.vegas_reduce(self._h, _stream(stream)))

    def finalize(self, n_events_total, want_hist=True, stream=None):
        I, s = C.c_double(), C.c_double()
        h = np.empty((self.dim, self.n_bins)) if want_hist else None
        rc = lib.vegas_finalize(self._h, int(n_events_total), _stream(stream), C.byref(I), C.byref(s), _ptr(h))
        return I.value, s.value, h, self._check(rc, allow_numeric=True)

    def finish_sharded(self, n_events_total, alpha, want_hist=True, stream=None):
        """finalize + refine (alpha >= 0) after the ranks' all-reduce, one synchronisation -> (I, sigma, hist or None, status)"""
        I, s = C.c_double(), C.c_double()
        h = np.empty((self.dim, self.n_bins)) if want_hist else None
        rc = lib.vegas_finish_sharded(self._h, int(n_events_total), float(alpha), _stream(stream), C.byref(I), C.byref(s), _ptr(h))
        return I.value, s.value, h, self._check(rc, allow_numeric=True)

    def totals_tensor(self):
        """The reduced totals {S1_hi, S1_lo, S2_hi, S2_lo, H[dim][n_bins]} as a torch fp64 view of the
        workspace (for the one all-reduce of a multi-GPU iteration)."""
        import torch
        n = int(lib.vegas_totals_count(self._h))
        addr = int(lib.vegas_totals_device(self._h))
        off = addr - self.workspace.data_ptr()
        return self.workspace[off:off + 8 * n].view(torch.float64)

    def refine(self, alpha, hist=None, stream=None):
        """-> status (VEGAS_OK or VEGAS_ENUMERIC)"""
        h = None if hist is None else np.ascontiguousarray(hist, dtype=np.float64)
        if h is not None and h.shape != (self.dim, self.n_bins):
            raise VegasError(VEGAS_EINVAL, "hist shape %r" % (h.shape,))
        return self._check(lib.vegas_refine(self._h, _ptr(h), float(alpha), _stream(stream)), allow_numeric=True)

    def integrate(self, n_iter, n_events, seed, alpha, integrand_id, precision=VEGAS_FP64, n_skip=0,
                  chunk_events=0, stream=None, first_iteration=0):
        """-> dict(I, sigma, chi2_dof, per_iter [n_iter,2], status); first_iteration > 0 continues a run"""
        I, s, c = C.c_double(), C.c_double(), C.c_double()
        per = np.zeros((max(int(n_iter), 1), 2))
        rc = lib.vegas_integrate_from(self._h, int(first_iteration), int(n_iter), int(n_skip), int(n_events),
                                      int(chunk_events), int(seed), float(alpha), integrand_id, precision,
                                      _stream(stream), C.byref(I), C.byref(s), C.byref(c), _ptr(per))
        self._check(rc, allow_numeric=True)
        return dict(I=I.value, sigma=s.value, chi2_dof=c.value, per_iter=per, status=rc)

    def debug_sample(self, first_event, count, seed, iteration, integrand_id, precision=VEGAS_FP64, stream=None):
        """-> (words [count,dim] u32, bins [count,dim] i32, x [count,dim] f64, fJ [count] f64)"""
        import torch
        need = int(lib.vegas_debug_scratch_bytes(self.dim, int(count))) + 256
        if self._debug_scratch is None or self._debug_scratch.numel() < need:
            self._debug_scratch = torch.empty(need, dtype=torch.uint8, device=self.device)
        ptr = (self._debug_scratch.data_ptr() + 255) // 256 * 256
        words = np.empty((count, self.dim), dtype=np.uint32)
        bins = np.empty((count, self.dim), dtype=np.int32)
        x = np.empty((count, self.dim))
        fJ = np.empty(count)
        self._check(lib.vegas_debug_sample(self._h, int(first_event), int(count), int(seed), int(iteration),
                                           integrand_id, precision, C.c_void_p(ptr), _stream(stream),
                                           _ptr(words, C.c_uint32), _ptr(bins, C.c_int32), _ptr(x), _ptr(fJ)))
        return words, bins, x, fJ

    # -- launch shape and instrumentation
    def set_launch(self, blocks=0, threads=0, table_copies=0, hist_copies=0):
        self._check(lib.vegas_set_launch(self._h, blocks, threads, table_copies, hist_copies))

    def get_launch(self, integrand_id=VEGAS_F_CONST, precision=VEGAS_FP64):
        pa, b, t, ct, ch, sh = C.c_int(), C.c_int(), C.c_int(), C.c_int(), C.c_int(), C.c_size_t()
        self._check(lib.vegas_get_launch(self._h, integrand_id, precision, C.byref(pa), C.byref(b), C.byref(t),
                                         C.byref(ct), C.byref(ch), C.byref(sh)))
        return dict(path="rotated" if pa.value else "generic", blocks=b.value, threads=t.value,
                    table_copies=ct.value, hist_copies=ch.value, shared_bytes=sh.value)

    def set_variant(self, variant):
        """VEGAS_VARIANT_NONE / _U53 (53-bit uniforms) / _Q32 (fp32-rounded table entries); fp64 fast path only."""
        self._check(lib.vegas_set_variant(self._h, int(variant)))

    def get_variant(self):
        return int(lib.vegas_get_variant(self._h))

    def set_profiling(self, on=True):
        self._check(lib.vegas_set_profiling(self._h, int(bool(on))))

    def kernel_time_ms(self):
        ms, n = C.c_double(), C.c_uint64()
        self._check(lib.vegas_kernel_time_ms(self._h, C.byref(ms), C.byref(n)))
        return ms.value, n.value

    def launch_count(self):
        return int(lib.vegas_launch_count(self._h))

    def reset_counters(self):
        self._check(lib.vegas_reset_counters(self._h))
