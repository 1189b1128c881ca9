"""ctypes front end of the CPU oracle (oracle/pn_oracle.c).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It imports nothing from paper_0908_3889_b200 and the product imports nothing from here.

The arithmetic lives in pn_oracle.c (Eqs. (1)-(4) of arXiv:0908.3889; Dormand-Prince
stepper); this file only builds the shared library with gcc and marshals numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pn_oracle.c")
_LIB = os.path.join(_HERE, "libpn_oracle.so")
_OPCOUNT = os.path.join(_HERE, "pn_oracle_opcount")

FAIL_MAXSTEPS, FAIL_HUNDERFLOW, FAIL_NONFINITE, FAIL_LANDING, FAIL_BADINPUT = -1, -2, -3, -4, -5
MASK_ALL = 0x100FF
MASK_SPIN = 1 << 16


def build(force: bool = False) -> str:
    """Compile libpn_oracle.so next to the source (gcc, -O2, no FMA contraction, OpenMP over systems)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", _SRC, "-o", _LIB, "-lm"]
        )
    return _LIB


def op_counts() -> dict:
    """Build and run the op-counting variant (same source compiled as C++ with a counting scalar)."""
    import json

    if not os.path.exists(_OPCOUNT) or os.path.getmtime(_OPCOUNT) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-x", "c++", "-O1", "-DPN_COUNT_OPS", _SRC, "-o", _OPCOUNT])
    return json.loads(subprocess.check_output([_OPCOUNT]).decode())


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        dp, ip, llp, ullp = (C.POINTER(C.c_double), C.POINTER(C.c_int), C.POINTER(C.c_longlong),
                             C.POINTER(C.c_ulonglong))
        lib.pn_oracle_rhs.argtypes = [dp, dp, C.c_longlong, C.c_uint, dp]
        lib.pn_oracle_rhs.restype = None
        lib.pn_oracle_tableau.argtypes = [llp] * 6
        lib.pn_oracle_tableau.restype = None
        lib.pn_oracle_integrate.argtypes = [dp, dp, C.c_longlong, C.c_double, C.c_double, C.c_double, C.c_int,
                                            C.c_double, C.c_int, C.c_uint, C.c_double, dp, ip, dp, ip, C.c_int]
        lib.pn_oracle_integrate.restype = C.c_longlong
        lib.pn_oracle_histogram.argtypes = [dp, C.c_longlong, C.c_int, ullp, ullp, dp]
        lib.pn_oracle_histogram.restype = None
        lib.pn_oracle_num_threads.restype = C.c_int
        _lib = lib
    return _lib


def _d(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def num_threads() -> int:
    return int(_load().pn_oracle_num_threads())


def rhs(y, masses, term_mask: int = 0) -> np.ndarray:
    """f(y) of Eqs. (1)-(4) for states y[n,10] and masses[n,2]."""
    y = np.ascontiguousarray(np.atleast_2d(y), dtype=np.float64)
    masses = np.ascontiguousarray(np.atleast_2d(masses), dtype=np.float64)
    assert y.shape[1] == 10 and masses.shape == (y.shape[0], 2)
    f = np.empty_like(y)
    _load().pn_oracle_rhs(_d(y), _d(masses), y.shape[0], term_mask, _d(f))
    return f


def tableau():
    """Dormand-Prince coefficients as exact fractions: (a[7][6], c[7], bhat[7]); b = a[6]."""
    from fractions import Fraction

    arrs = [np.zeros(n, dtype=np.int64) for n in (42, 42, 7, 7, 7, 7)]
    _load().pn_oracle_tableau(*[a.ctypes.data_as(C.POINTER(C.c_longlong)) for a in arrs])
    an, ad, cn, cd, bn, bd = arrs
    a = [[Fraction(int(an[6 * s + j]), int(ad[6 * s + j])) for j in range(6)] for s in range(7)]
    c = [Fraction(int(cn[s]), int(cd[s])) for s in range(7)]
    bh = [Fraction(int(bn[s]), int(bd[s])) for s in range(7)]
    return a, c, bh


def integrate(init_states, masses, omegaf, rtol, atol, *, fixed_steps=0, h0=0.0, max_steps=0, term_mask=0,
              tau_land=0.0, n_threads=0):
    """Adaptive (or fixed-step) DP5(4) integration of n systems.

    Returns dict(final[n,10], steps[n], time[n], rejected[n], n_failed).
    """
    y0 = np.ascontiguousarray(np.atleast_2d(init_states), dtype=np.float64)
    ms = np.ascontiguousarray(np.atleast_2d(masses), dtype=np.float64)
    n = y0.shape[0]
    assert y0.shape == (n, 10) and ms.shape == (n, 2)
    final = np.empty((n, 10))
    steps = np.empty(n, dtype=np.int32)
    time = np.empty(n)
    rej = np.empty(n, dtype=np.int32)
    ip = C.POINTER(C.c_int)
    nf = _load().pn_oracle_integrate(_d(y0), _d(ms), n, float(omegaf), float(rtol), float(atol), int(fixed_steps),
                                     float(h0), int(max_steps), int(term_mask), float(tau_land), _d(final),
                                     steps.ctypes.data_as(ip), _d(time), rej.ctypes.data_as(ip), int(n_threads))
    return dict(final=final, steps=steps, time=time, rejected=rej, n_failed=int(nf))


def histogram(final_states, bins: int):
    """3 x bins counts of S1^.S2^, S1^.L^, S2^.L^ plus skipped[3] and the dots[n,3] themselves."""
    y = np.ascontiguousarray(np.atleast_2d(final_states), dtype=np.float64)
    n = y.shape[0]
    counts = np.zeros((3, bins), dtype=np.uint64)
    skipped = np.zeros(3, dtype=np.uint64)
    dots = np.empty((n, 3))
    up = C.POINTER(C.c_ulonglong)
    _load().pn_oracle_histogram(_d(y), n, int(bins), counts.ctypes.data_as(up), skipped.ctypes.data_as(up), _d(dots))
    return counts, skipped, dots
