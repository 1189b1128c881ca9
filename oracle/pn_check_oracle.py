"""CPU oracle of the built-in cross-check.  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this module.
It imports nothing from paper_0908_3889_b200 and shares no code with the CUDA path.

The paper validates its single-precision GPU runs by evolving "a random ~1 % subset" of the batch in double
precision and comparing the final states.  Written out step by step:

  1. selection: system i is in the subset iff u_i < fraction, where u_i is element i of the uniform stream of
     key `key` (Philox4x64-10 in numpy's layout, oracle/pn_gen_oracle.c: u_i = (raw[i] >> 11) 2^-53);
  2. reference: the selected systems are integrated by the FP64 oracle (oracle/pn_oracle.c) from their initial
     states to omega_f at (rtol_ref, atol_ref);
  3. comparison: for each of the three unit dot products (oracle/pn_stats_oracle.unit_dots) the largest
     |d(checked final state) - d(reference final state)| over the subset and the (lowest) index where it occurs;
     and the largest relative deviation of the final time, if times are given.  Systems whose reference
     integration failed are counted in n_failed_ref and left out; a dot product undefined on either side is left out.

Pins (tests/test_oracle_check.py): the selection mask against numpy.random.Generator(Philox).random(N) < fraction,
its size against the binomial law, identical states -> zero deviation, a planted perturbation is found at the right
index with the right size.  Parity unpinned: none (steps 2 and 3 reuse pinned oracles).
"""
from __future__ import annotations

import numpy as np

from . import pn_gen_oracle, pn_oracle, pn_stats_oracle


def selection(n: int, fraction: float, key) -> np.ndarray:
    """Sorted indices i in [0, n) with u_i < fraction."""
    raw = pn_gen_oracle.raw(key, 0, n)
    u = (raw >> np.uint64(11)).astype(np.float64) * 2.0**-53
    return np.nonzero(u < float(fraction))[0]


def selfcheck(init_states, masses, final_states, times, omegaf, fraction, key, rtol_ref=1e-10, atol_ref=1e-12) -> dict:
    y0 = np.asarray(init_states, dtype=np.float64)
    idx = selection(y0.shape[0], fraction, key)
    out = dict(indices=idx, n_checked=int(idx.size), n_failed_ref=0, max_dot_dev=np.zeros(3),
               worst_index=np.full(3, -1, dtype=np.int64), max_time_rel_dev=0.0)
    if idx.size == 0:
        return out
    ref = pn_oracle.integrate(y0[idx], np.asarray(masses, dtype=np.float64)[idx], omegaf, rtol_ref, atol_ref)
    ok = ref["steps"] > 0
    out["n_failed_ref"] = int(np.count_nonzero(~ok))
    d_ref = pn_stats_oracle.unit_dots(ref["final"])
    d_chk = pn_stats_oracle.unit_dots(np.asarray(final_states, dtype=np.float64)[idx])
    for k in range(3):
        dev = np.abs(d_chk[:, k] - d_ref[:, k])
        dev[~ok | ~np.isfinite(dev)] = -1.0
        if dev.max() >= 0.0:
            j = int(np.argmax(dev))                 # first (lowest index) maximum
            out["max_dot_dev"][k] = dev[j]
            out["worst_index"][k] = idx[j]
    if times is not None:
        t = np.asarray(times, dtype=np.float64)[idx]
        rel = np.abs(t / ref["time"] - 1.0)
        rel[~ok | ~np.isfinite(rel)] = 0.0
        out["max_time_rel_dev"] = float(rel.max())
    out["ref_final"] = ref["final"]
    return out
