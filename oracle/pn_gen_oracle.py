"""ctypes front end of the generator oracle (oracle/pn_gen_oracle.c).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
module.  It imports nothing from paper_0908_3889_b200 and the product imports nothing from here.
The arithmetic (Philox4x64-10, the variate layout, the sphere sampling)
lives in pn_gen_oracle.c; this file only builds it with gcc and marshals numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pn_gen_oracle.c")
_LIB = os.path.join(_HERE, "libpn_gen_oracle.so")


class Spec(C.Structure):
    _fields_ = [("key", C.c_uint64 * 2), ("omega0", C.c_double), ("q_lo", C.c_double), ("q_hi", C.c_double),
                ("m1_fixed", C.c_double), ("chi1_lo", C.c_double), ("chi1_hi", C.c_double), ("chi2_lo", C.c_double),
                ("chi2_hi", C.c_double), ("s1_tilt_deg", C.c_double)]


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-shared", "-fPIC", _SRC, "-o", _LIB, "-lm"])
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        u64p = C.POINTER(C.c_uint64)
        lib.pn_gen_oracle_philox4x64_10.argtypes = [u64p, u64p, u64p]
        lib.pn_gen_oracle_philox4x64_10.restype = None
        lib.pn_gen_oracle_raw_block.argtypes = [u64p, C.c_uint64, C.c_longlong, u64p]
        lib.pn_gen_oracle_raw_block.restype = None
        lib.pn_gen_oracle_uniform.argtypes = [u64p, C.c_uint64]
        lib.pn_gen_oracle_uniform.restype = C.c_double
        lib.pn_gen_oracle_generate.argtypes = [C.POINTER(Spec), C.c_longlong, C.c_longlong, C.c_longlong,
                                               C.POINTER(C.c_double), C.POINTER(C.c_double)]
        lib.pn_gen_oracle_generate.restype = None
        _lib = lib
    return _lib


def _u64(a):
    a = np.ascontiguousarray(a, dtype=np.uint64)
    return a, a.ctypes.data_as(C.POINTER(C.c_uint64))


def philox4x64_10(counter, key) -> np.ndarray:
    c, cp = _u64(counter)
    k, kp = _u64(key)
    out = np.zeros(4, dtype=np.uint64)
    _load().pn_gen_oracle_philox4x64_10(cp, kp, out.ctypes.data_as(C.POINTER(C.c_uint64)))
    return out


def raw(key, first: int, n: int) -> np.ndarray:
    k, kp = _u64(key)
    out = np.zeros(n, dtype=np.uint64)
    _load().pn_gen_oracle_raw_block(kp, int(first), int(n), out.ctypes.data_as(C.POINTER(C.c_uint64)))
    return out


def make_spec(key, omega0, q=(1.0, 1.0), chi1=(1.0, 1.0), chi2=(1.0, 1.0), m1_fixed=None, s1_tilt_deg=None) -> Spec:
    s = Spec()
    s.key[0], s.key[1] = int(key[0]), int(key[1])
    s.omega0 = float(omega0)
    s.q_lo, s.q_hi = float(q[0]), float(q[1])
    s.m1_fixed = float(m1_fixed) if m1_fixed is not None else 0.0
    s.chi1_lo, s.chi1_hi = float(chi1[0]), float(chi1[1])
    s.chi2_lo, s.chi2_hi = float(chi2[0]), float(chi2[1])
    s.s1_tilt_deg = float(s1_tilt_deg) if s1_tilt_deg is not None else -1.0
    return s


def generate(spec: Spec, n_total: int, first: int = 0, count: int | None = None):
    """(init_states[count,10], masses[count,2]) of systems first..first+count-1 of an n_total ensemble."""
    count = n_total - first if count is None else count
    y0 = np.empty((count, 10))
    m = np.empty((count, 2))
    dp = C.POINTER(C.c_double)
    _load().pn_gen_oracle_generate(C.byref(spec), int(n_total), int(first), int(count), y0.ctypes.data_as(dp),
                                   m.ctypes.data_as(dp))
    return y0, m
