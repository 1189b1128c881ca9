"""Thin ctypes binding of libpn_b200.so (C ABI in include/pn.h).  Argument marshalling only: every
step of the path runs in the CUDA kernels.  torch is used for device memory and streams.

There is NO CPU fallback: if the shared library is missing or no CUDA device is present, the calls
raise.  This module never imports oracle/.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpn_b200.so")

PN_FP64, PN_FP32, PN_MIXED = 0, 1, 2
PN_OK, PN_EINVAL, PN_ECUDA, PN_ENOTCONVERGED, PN_ENONFINITE, PN_ETOOLARGE = 0, 1, 2, 3, 4, 5
PN_STATIC_MAX_GROUPS, PN_STATIC_SCRATCH_BYTES = 1024, 344064
FAIL_MAXSTEPS, FAIL_HUNDERFLOW, FAIL_NONFINITE, FAIL_LANDING, FAIL_BADINPUT = -1, -2, -3, -4, -5

EXPORTS = ["pn_integrate", "pn_integrate_ex", "pn_histogram", "pn_histogram_ex", "pn_statistics", "pn_statistics_static", "pn_merge_statistics", "pn_generate", "pn_run_ensembles", "pn_selfcheck", "pn_stream_status", "pn_stream_release",
           "pn_measure_fma_peak", "pn_measure_fma_operands", "pn_last_counters", "pn_last_redo_count", "pn_last_kernel_ms", "pn_launch_count", "pn_strerror",
           "pn_last_cuda_error", "pn_shutdown", "pn_version"]


class PnOptions(C.Structure):
    _fields_ = [("size", C.c_int), ("fixed_steps", C.c_int), ("h0", C.c_double), ("max_steps", C.c_int),
                ("term_mask", C.c_uint), ("tau_land", C.c_double), ("layout", C.c_int), ("host_buffers", C.c_int),
                ("async_", C.c_int), ("input_order", C.c_int), ("out_time", C.c_void_p), ("out_rejected", C.c_void_p),
                ("stream", C.c_void_p), ("block_threads", C.c_int), ("grid_blocks", C.c_int), ("variant", C.c_int),
                ("hist_bins", C.c_int), ("hist_counts", C.c_void_p), ("hist_skipped", C.c_void_p)]


class PnStatsOut(C.Structure):
    _fields_ = [("size", C.c_int), ("pearson_r", C.c_void_p), ("moments", C.c_void_p), ("n_skipped", C.c_void_p),
                ("hist1", C.c_void_p), ("hist2", C.c_void_p), ("hist2_max", C.c_void_p), ("hist2_norm", C.c_void_p)]


class PnEnsemble(C.Structure):
    _fields_ = [("size", C.c_int), ("key", C.c_ulonglong * 2), ("omega0", C.c_double), ("q_lo", C.c_double),
                ("q_hi", C.c_double), ("m1_fixed", C.c_double), ("chi1_lo", C.c_double), ("chi1_hi", C.c_double),
                ("chi2_lo", C.c_double), ("chi2_hi", C.c_double), ("s1_tilt_deg", C.c_double)]


def make_ensemble(key, omega0, q=(1.0, 1.0), chi1=(1.0, 1.0), chi2=(1.0, 1.0), m1_fixed=None, s1_tilt_deg=None) -> PnEnsemble:
    e = PnEnsemble()
    e.size = C.sizeof(PnEnsemble)
    e.key[0], e.key[1] = int(key[0]), int(key[1])
    e.omega0, e.q_lo, e.q_hi = float(omega0), float(q[0]), float(q[1])
    e.m1_fixed = float(m1_fixed) if m1_fixed is not None else 0.0
    e.chi1_lo, e.chi1_hi, e.chi2_lo, e.chi2_hi = float(chi1[0]), float(chi1[1]), float(chi2[0]), float(chi2[1])
    e.s1_tilt_deg = float(s1_tilt_deg) if s1_tilt_deg is not None else -1.0
    return e


class PnCheckOut(C.Structure):
    _fields_ = [("size", C.c_int), ("n_checked", C.c_longlong), ("n_failed_ref", C.c_longlong), ("max_dot_dev", C.c_double * 3),
                ("worst_index", C.c_longlong * 3), ("max_time_rel_dev", C.c_double), ("ms_reference", C.c_float)]


class PnError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(msg)
        self.status = status


_lib = None


def load():
    """Loads the library; raises (loudly) if it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_0908_3889_b200.build` "
                              "(there is no CPU fallback)")
        lib = C.CDLL(LIB_PATH)
        vp, d, ll, i = C.c_void_p, C.c_double, C.c_longlong, C.c_int
        lib.pn_integrate.argtypes = [vp, vp, ll, d, d, d, d, i, vp, vp]
        lib.pn_integrate_ex.argtypes = [vp, vp, ll, d, d, d, d, i, vp, vp, C.POINTER(PnOptions)]
        lib.pn_histogram.argtypes = [vp, ll, i, vp, vp]
        lib.pn_histogram_ex.argtypes = [vp, ll, i, vp, vp, C.POINTER(PnOptions)]
        lib.pn_statistics.argtypes = [vp, vp, vp, ll, ll, i, i, C.POINTER(PnStatsOut), C.POINTER(PnOptions)]
        lib.pn_statistics_static.argtypes = [vp, vp, vp, ll, ll, i, i, C.POINTER(PnStatsOut), vp, i]
        lib.pn_merge_statistics.argtypes = [vp, i, i, vp, vp, C.POINTER(PnOptions)]
        lib.pn_generate.argtypes = [C.POINTER(PnEnsemble), i, ll, ll, ll, vp, vp, C.POINTER(PnOptions)]
        lib.pn_run_ensembles.argtypes = [C.POINTER(PnEnsemble), i, ll, ll, ll, d, d, d, i, i, i, C.POINTER(PnStatsOut), C.POINTER(PnOptions)]
        lib.pn_selfcheck.argtypes = [vp, vp, vp, vp, ll, d, d, C.POINTER(C.c_ulonglong), d, d, C.POINTER(PnCheckOut), vp, ll,
                                     C.POINTER(PnOptions)]
        lib.pn_stream_status.argtypes = [vp]
        lib.pn_stream_release.argtypes = [vp]
        lib.pn_measure_fma_peak.argtypes = [i, d, C.POINTER(d), C.POINTER(d)]
        lib.pn_measure_fma_operands.argtypes = [i, i, C.POINTER(d)]
        lib.pn_last_counters.argtypes = [C.POINTER(C.c_ulonglong)] * 4
        lib.pn_last_kernel_ms.argtypes = [C.POINTER(C.c_float)]
        lib.pn_launch_count.restype = C.c_ulonglong
        lib.pn_last_redo_count.restype = C.c_ulonglong
        lib.pn_strerror.argtypes = [i]
        lib.pn_strerror.restype = C.c_char_p
        lib.pn_last_cuda_error.restype = C.c_char_p
        _lib = lib
    return _lib


def _check(st, allow=()):
    if st != PN_OK and st not in allow:
        lib = load()
        msg = lib.pn_strerror(st).decode()
        if st == PN_ECUDA:
            msg += ": " + lib.pn_last_cuda_error().decode()
        raise PnError(st, f"pn status {st}: {msg}")
    return st


def _ptr(a):
    """Address of a torch tensor (device or host) or a numpy array; None -> NULL."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        return a.ctypes.data
    return a.data_ptr()


def _is_host(a) -> bool:
    return isinstance(a, np.ndarray) or (hasattr(a, "is_cuda") and not a.is_cuda)


_DTYPES = {"f64": ("float64",), "i32": ("int32",), "i64": ("int64", "uint64")}


def _require(name, a, dtype, shape=None, host=None, at_least=False):
    """The C ABI takes raw pointers: a wrong dtype, a non-contiguous view, a short array or a tensor on another device
    would be read or written out of bounds by the kernels.  Checked here, before the call (None passes).
    at_least: an output that only has to be large enough (element count), whatever its shape."""
    if a is None:
        return
    dt = str(a.dtype).replace("torch.", "")
    if dt not in _DTYPES[dtype]:
        raise ValueError(f"{name}: dtype {dt}, expected {_DTYPES[dtype][0]}")
    contiguous = a.flags["C_CONTIGUOUS"] if isinstance(a, np.ndarray) else a.is_contiguous()
    if not contiguous:
        raise ValueError(f"{name}: array is not contiguous")
    if shape is not None and at_least:
        need = int(np.prod([int(w) for w in shape])) if len(shape) else 1
        have = int(np.prod([int(x) for x in a.shape])) if len(a.shape) else 1
        if have < need:
            raise ValueError(f"{name}: {have} elements, the call writes {need}")
    elif shape is not None:
        got = tuple(int(x) for x in a.shape)
        if len(got) != len(shape) or any(w is not None and g != w for g, w in zip(got, shape)):
            raise ValueError(f"{name}: shape {got}, expected {tuple('*' if w is None else w for w in shape)}")
    if host is not None and _is_host(a) != host:
        raise ValueError(f"{name}: all arrays of one call must live on the same side (host or device)")
    if not _is_host(a):
        import torch

        if a.device.index != torch.cuda.current_device():
            raise ValueError(f"{name}: tensor is on cuda:{a.device.index}, the current device is cuda:{torch.cuda.current_device()}")


def make_options(*, fixed_steps=0, h0=0.0, max_steps=0, term_mask=0, tau_land=0.0, layout=0, host_buffers=False,
                 async_=False, input_order=False, out_time=None, out_rejected=None, stream=None, block_threads=0,
                 grid_blocks=0, variant=0, hist_bins=0, hist_counts=None, hist_skipped=None) -> PnOptions:
    o = PnOptions()
    o.size = C.sizeof(PnOptions)
    o.fixed_steps, o.h0, o.max_steps, o.term_mask, o.tau_land = int(fixed_steps), float(h0), int(max_steps), int(term_mask), float(tau_land)
    o.layout, o.host_buffers, o.async_, o.input_order = int(layout), int(bool(host_buffers)), int(bool(async_)), int(bool(input_order))
    o.out_time, o.out_rejected = _ptr(out_time), _ptr(out_rejected)
    o.stream = None if stream is None else int(getattr(stream, "cuda_stream", stream))
    o.block_threads, o.grid_blocks, o.variant = int(block_threads), int(grid_blocks), int(variant)
    o.hist_bins, o.hist_counts, o.hist_skipped = int(hist_bins), _ptr(hist_counts), _ptr(hist_skipped)
    return o


def pn_integrate(init_states, masses, omega0, omegaf, rtol, atol, precision, out_final, out_steps, *,
                 allow_failures=False, **opts):
    """pn_integrate_ex of include/pn.h.  Arrays are torch CUDA tensors (float64 / int32, contiguous), or
    numpy / CPU tensors when every array is on the host (host_buffers is then set automatically).
    Returns the pn_status (raises PnError unless it is PN_OK, or a per-system failure with allow_failures)."""
    lib = load()
    n = int(out_steps.shape[0])
    host = _is_host(init_states)
    soa = opts.get("layout", 0) == 1
    _require("init_states", init_states, "f64", (10, n) if soa else (n, 10), host)
    _require("masses", masses, "f64", (2, n) if soa else (n, 2), host)
    _require("out_final", out_final, "f64", (10, n) if soa else (n, 10), host)
    _require("out_steps", out_steps, "i32", (n,), host)
    _require("out_time", opts.get("out_time"), "f64", (n,), host)
    _require("out_rejected", opts.get("out_rejected"), "i32", (n,), host)
    _require("hist_counts", opts.get("hist_counts"), "i64", (3, max(int(opts.get("hist_bins", 0)), 0)), host, at_least=True)
    _require("hist_skipped", opts.get("hist_skipped"), "i64", (3,), host, at_least=True)
    if host:
        opts["host_buffers"] = True
    o = make_options(**opts)
    st = lib.pn_integrate_ex(_ptr(init_states), _ptr(masses), n, float(omega0), float(omegaf), float(rtol),
                             float(atol), int(precision), _ptr(out_final), _ptr(out_steps), C.byref(o))
    return _check(st, allow=(PN_ENOTCONVERGED, PN_ENONFINITE, PN_EINVAL) if allow_failures else ())


def pn_histogram(final_states, bins, counts, n_skipped=None, *, n=None, **opts):
    """pn_histogram_ex of include/pn.h: counts[3, bins] uint64 (torch int64 storage is accepted)."""
    lib = load()
    soa = opts.get("layout", 0) == 1
    if n is None:
        n = int(final_states.shape[1] if soa else final_states.shape[0])
    host = _is_host(final_states)
    _require("final_states", final_states, "f64", (10, None) if soa else (None, 10), host)
    if int(final_states.shape[1 if soa else 0]) < n:
        raise ValueError("final_states holds fewer than n systems")
    _require("counts", counts, "i64", (3, max(int(bins), 0)), host, at_least=True)
    _require("n_skipped", n_skipped, "i64", (3,), host, at_least=True)
    if host:
        opts["host_buffers"] = True
    o = make_options(**opts)
    return _check(lib.pn_histogram_ex(_ptr(final_states), int(n), int(bins), _ptr(counts), _ptr(n_skipped), C.byref(o)))


def pn_statistics(init_states, final_states, steps=None, *, group_size=0, bins1=0, bins2=0, pearson_r=None,
                  moments=None, n_skipped=None, hist1=None, hist2=None, hist2_max=None, hist2_norm=None, **opts):
    """pn_statistics of include/pn.h.  Output arrays are caller-allocated (torch CUDA tensors, or numpy when
    the inputs are on the host); any of them may be None.  init_states may be None (final-only mode)."""
    lib = load()
    n = int(final_states.shape[0])
    host = _is_host(final_states)
    gs = int(group_size) if int(group_size) > 0 else max(n, 1)
    G = n // gs if n else 0
    _require("final_states", final_states, "f64", (n, 10), host)
    _require("init_states", init_states, "f64", (n, 10), host)
    _require("steps", steps, "i32", (n,), host)
    _require("pearson_r", pearson_r, "f64", (G, 3), host, at_least=True)
    _require("moments", moments, "f64", (G, 3, 6), host, at_least=True)
    _require("n_skipped", n_skipped, "i64", (G, 3), host, at_least=True)
    _require("hist1", hist1, "i64", (G, 3, int(bins1)), host, at_least=True)
    _require("hist2", hist2, "i64", (G, 3, int(bins2), int(bins2)), host, at_least=True)
    _require("hist2_max", hist2_max, "i64", (G, 3), host, at_least=True)
    _require("hist2_norm", hist2_norm, "f64", (G, 3, int(bins2), int(bins2)), host, at_least=True)
    if host:
        opts["host_buffers"] = True
    o = make_options(**opts)
    out = PnStatsOut()
    out.size = C.sizeof(PnStatsOut)
    out.pearson_r, out.moments, out.n_skipped = _ptr(pearson_r), _ptr(moments), _ptr(n_skipped)
    out.hist1, out.hist2, out.hist2_max, out.hist2_norm = _ptr(hist1), _ptr(hist2), _ptr(hist2_max), _ptr(hist2_norm)
    return _check(lib.pn_statistics(_ptr(init_states), _ptr(final_states), _ptr(steps), n, int(group_size), int(bins1),
                                    int(bins2), C.byref(out), C.byref(o)))


def pn_statistics_static(init_states, final_states, steps=None, *, group_size=0, bins1=0, bins2=0, pearson_r=None,
                         moments=None, n_skipped=None, hist1=None, hist2=None, hist2_max=None, hist2_norm=None,
                         stream=None, async_=False):
    """pn_statistics_static of include/pn.h: the statistics of pn_statistics for a caller that must not allocate device
    memory while it runs (all of HBM already sits in a framework's caching allocator, other streams would be stalled by
    cudaMalloc's device-wide synchronisation, or the process has a fixed memory budget).  The kernels' scratch is a
    fixed 336 KB array inside the library; at most PN_STATIC_MAX_GROUPS ensembles per call (PnError with status
    PN_ETOOLARGE beyond).  Torch CUDA tensors only: inputs and outputs stay the caller's.  Calls share the array, so
    calls that could overlap on the GPU (unordered streams) must not be issued; make the first call on a device outside
    stream capture (it looks the array's address up)."""
    lib = load()
    n = int(final_states.shape[0])
    gs = int(group_size) if int(group_size) > 0 else max(n, 1)
    G = n // gs if n else 0
    for name, a in (("final_states", final_states), ("init_states", init_states), ("steps", steps)):
        if a is not None and _is_host(a):
            raise ValueError(f"{name}: pn_statistics_static takes device tensors only (staging host arrays would need an allocation)")
    _require("final_states", final_states, "f64", (n, 10), False)
    _require("init_states", init_states, "f64", (n, 10), False)
    _require("steps", steps, "i32", (n,), False)
    _require("pearson_r", pearson_r, "f64", (G, 3), False, at_least=True)
    _require("moments", moments, "f64", (G, 3, 6), False, at_least=True)
    _require("n_skipped", n_skipped, "i64", (G, 3), False, at_least=True)
    _require("hist1", hist1, "i64", (G, 3, int(bins1)), False, at_least=True)
    _require("hist2", hist2, "i64", (G, 3, int(bins2), int(bins2)), False, at_least=True)
    _require("hist2_max", hist2_max, "i64", (G, 3), False, at_least=True)
    _require("hist2_norm", hist2_norm, "f64", (G, 3, int(bins2), int(bins2)), False, at_least=True)
    out = PnStatsOut()
    out.size = C.sizeof(PnStatsOut)
    out.pearson_r, out.moments, out.n_skipped = _ptr(pearson_r), _ptr(moments), _ptr(n_skipped)
    out.hist1, out.hist2, out.hist2_max, out.hist2_norm = _ptr(hist1), _ptr(hist2), _ptr(hist2_max), _ptr(hist2_norm)
    s = None if stream is None else int(getattr(stream, "cuda_stream", stream))
    return _check(lib.pn_statistics_static(_ptr(init_states), _ptr(final_states), _ptr(steps), n, int(group_size), int(bins1),
                                           int(bins2), C.byref(out), s, int(bool(async_))))


def pn_merge_statistics(parts, moments=None, pearson_r=None, **opts):
    """pn_merge_statistics of include/pn.h: parts [R, G, 3, 6] (torch CUDA float64) -> moments [G, 3, 6], pearson_r [G, 3]."""
    lib = load()
    _require("parts", parts, "f64", (None, None, 3, 6), False)
    _require("moments", moments, "f64", (int(parts.shape[1]), 3, 6), False, at_least=True)
    _require("pearson_r", pearson_r, "f64", (int(parts.shape[1]), 3), False, at_least=True)
    o = make_options(**opts)
    return _check(lib.pn_merge_statistics(_ptr(parts), int(parts.shape[0]), int(parts.shape[1]), _ptr(moments), _ptr(pearson_r),
                                          C.byref(o)))


def pn_generate(ensembles, n_total, init_states, masses, *, first=0, count=None, **opts):
    """pn_generate of include/pn.h.  `ensembles`: one PnEnsemble (make_ensemble) or a list of them; output arrays
    [len(ensembles)*count, 10] and [.., 2] float64 (torch CUDA tensors, or numpy for host buffers)."""
    lib = load()
    ens = ensembles if isinstance(ensembles, (list, tuple)) else [ensembles]
    arr = (PnEnsemble * len(ens))(*ens)
    count = int(n_total) - int(first) if count is None else int(count)
    host = _is_host(init_states)
    _require("init_states", init_states, "f64", (len(ens) * max(count, 0), 10), host, at_least=True)
    _require("masses", masses, "f64", (len(ens) * max(count, 0), 2), host, at_least=True)
    if host:
        opts["host_buffers"] = True
    o = make_options(**opts)
    return _check(lib.pn_generate(arr, len(ens), int(n_total), int(first), count, _ptr(init_states), _ptr(masses), C.byref(o)))


def pn_run_ensembles(ensembles, n_total, omegaf, rtol, atol, *, first=0, count=None, precision=PN_FP64, bins1=0, bins2=0,
                     pearson_r=None, moments=None, n_skipped=None, hist1=None, hist2=None, hist2_max=None, hist2_norm=None,
                     allow_failures=False, **opts):
    """pn_run_ensembles of include/pn.h: seed in, statistics out (no state arrays).  `ensembles`: one PnEnsemble or a list;
    outputs as in pn_statistics with one group per ensemble (torch CUDA tensors, or numpy for host buffers)."""
    lib = load()
    ens = ensembles if isinstance(ensembles, (list, tuple)) else [ensembles]
    arr = (PnEnsemble * len(ens))(*ens)
    count = int(n_total) - int(first) if count is None else int(count)
    G = len(ens)
    outs = [a for a in (pearson_r, moments, n_skipped, hist1, hist2, hist2_max, hist2_norm) if a is not None]
    host = _is_host(outs[0]) if outs else False
    _require("pearson_r", pearson_r, "f64", (G, 3), host, at_least=True)
    _require("moments", moments, "f64", (G, 3, 6), host, at_least=True)
    _require("n_skipped", n_skipped, "i64", (G, 3), host, at_least=True)
    _require("hist1", hist1, "i64", (G, 3, max(int(bins1), 0)), host, at_least=True)
    _require("hist2", hist2, "i64", (G, 3, max(int(bins2), 0), max(int(bins2), 0)), host, at_least=True)
    _require("hist2_max", hist2_max, "i64", (G, 3), host, at_least=True)
    _require("hist2_norm", hist2_norm, "f64", (G, 3, max(int(bins2), 0), max(int(bins2), 0)), host, at_least=True)
    if host:
        opts["host_buffers"] = True
    o = make_options(**opts)
    out = PnStatsOut()
    out.size = C.sizeof(PnStatsOut)
    out.pearson_r, out.moments, out.n_skipped = _ptr(pearson_r), _ptr(moments), _ptr(n_skipped)
    out.hist1, out.hist2, out.hist2_max, out.hist2_norm = _ptr(hist1), _ptr(hist2), _ptr(hist2_max), _ptr(hist2_norm)
    st = lib.pn_run_ensembles(arr, len(ens), int(n_total), int(first), count, float(omegaf), float(rtol), float(atol), int(precision),
                              int(bins1), int(bins2), C.byref(out), C.byref(o))
    return _check(st, allow=(PN_ENOTCONVERGED, PN_ENONFINITE) if allow_failures else ())


def pn_selfcheck(init_states, masses, final_states, omegaf, *, fraction=0.01, key=(0, 0), times=None, rtol_ref=0.0,
                 atol_ref=0.0, checked_indices=None, allow_failures=False, **opts):
    """pn_selfcheck of include/pn.h (the paper's 1 % double-precision cross-check).  Returns a dict."""
    lib = load()
    n = int(final_states.shape[0])
    host = _is_host(final_states)
    _require("init_states", init_states, "f64", (n, 10), host)
    _require("masses", masses, "f64", (n, 2), host)
    _require("final_states", final_states, "f64", (n, 10), host)
    _require("times", times, "f64", (n,), host)
    _require("checked_indices", checked_indices, "i64", (None,), host)
    if host:
        opts["host_buffers"] = True
    o = make_options(**opts)
    out = PnCheckOut()
    out.size = C.sizeof(PnCheckOut)
    k = (C.c_ulonglong * 2)(int(key[0]), int(key[1]))
    cap = 0 if checked_indices is None else int(checked_indices.shape[0])
    st = lib.pn_selfcheck(_ptr(init_states), _ptr(masses), _ptr(final_states), _ptr(times), n, float(omegaf), float(fraction), k,
                          float(rtol_ref), float(atol_ref), C.byref(out), _ptr(checked_indices), cap, C.byref(o))
    _check(st, allow=(PN_ENOTCONVERGED, PN_ENONFINITE, PN_EINVAL) if allow_failures else ())
    return dict(status=st, n_checked=int(out.n_checked), n_failed_ref=int(out.n_failed_ref), max_dot_dev=list(out.max_dot_dev),
                worst_index=list(out.worst_index), max_time_rel_dev=float(out.max_time_rel_dev), ms_reference=float(out.ms_reference))


def pn_stream_status(stream=None):
    return load().pn_stream_status(None if stream is None else int(getattr(stream, "cuda_stream", stream)))


def pn_stream_release(stream=None):
    """pn_stream_release of include/pn.h: frees the library's scratch context of `stream` (call before destroying it)."""
    return _check(load().pn_stream_release(None if stream is None else int(getattr(stream, "cuda_stream", stream))))


def pn_measure_fma_peak(precision=PN_FP64, seconds=0.25):
    t, mhz = C.c_double(0), C.c_double(0)
    _check(load().pn_measure_fma_peak(int(precision), float(seconds), C.byref(t), C.byref(mhz)))
    return t.value, mhz.value


def pn_measure_fma_operands(precision=PN_FP64, n_register_sources=3):
    c = C.c_double(0)
    _check(load().pn_measure_fma_operands(int(precision), int(n_register_sources), C.byref(c)))
    return c.value


def pn_last_counters():
    v = [C.c_ulonglong(0) for _ in range(4)]
    load().pn_last_counters(*[C.byref(x) for x in v])
    return dict(trial_steps=v[0].value, rejected=v[1].value, landing_trials=v[2].value, failed=v[3].value,
                redo=int(load().pn_last_redo_count()))


def pn_last_kernel_ms():
    ms = (C.c_float * 4)()
    load().pn_last_kernel_ms(ms)
    return dict(stage_in=ms[0], integrate=ms[1], stage_out=ms[2], histogram=ms[3])


def pn_launch_count() -> int:
    return int(load().pn_launch_count())


def pn_shutdown():
    return load().pn_shutdown()


def pn_version() -> int:
    return int(load().pn_version())
