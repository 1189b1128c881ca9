"""paper_0908_3889_b200 -- batched post-Newtonian inspiral integration on one B200 (sm_100a).

The product is libpn_b200.so (hand-written CUDA behind the C ABI of include/pn.h); this package holds
its sources (csrc/), the build step (build.py), the ctypes binding (binding.py) and the seeded
workload generators (workloads.py).  There is no CPU fallback.
"""
from .binding import (PN_ETOOLARGE, PN_FP32, PN_FP64, PN_MIXED, PN_STATIC_MAX_GROUPS, PnError, make_ensemble, pn_generate, pn_histogram, pn_integrate, pn_last_counters,  # noqa: F401
                      pn_last_kernel_ms, pn_launch_count, pn_measure_fma_operands, pn_measure_fma_peak, pn_merge_statistics, pn_run_ensembles, pn_selfcheck, pn_shutdown, pn_statistics, pn_statistics_static, pn_stream_release, pn_stream_status,
                      pn_version)
from .pipeline import run_ensembles  # noqa: E402,F401
