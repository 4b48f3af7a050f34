"""paper_1802_05065_b200 -- B200-native first-passage-time Monte Carlo (arXiv:1802.05065 hot path).

The product is the C-ABI shared library ``libfpt_b200.so`` (``include/fpt.h``, sources under ``csrc/``); this package is
the thin ctypes binding (argument marshalling only) plus the five benchmark workloads as plain data.  There is no CPU
fallback: importing works without the library, but the first call raises if it has not been built.
"""
from .binding import (FptError, FptHist, FptLaunchOpts, FptParams, FptStats, alloc_stats, dbg_normals_f32, dbg_set_helper_seq0, dbg_set_slice_quantum, dbg_normals_f64, dbg_philox, dbg_selfcheck, dbg_sincos_f32,  # noqa: F401
                      dbg_sincos_f64, dbg_trace, dbg_unary_f32, dbg_unary_f64, fp32_peak, fp64_peak, histogram, last_stats, launch_opts,
                      lib, make_params, read_stats, set_launch, set_schedule, set_specialise, set_tail_helper, simulate, simulate_ex, simulate_hist, simulate_host, simulate_noalloc, simulate_sweep, version)
from . import analysis, sharding, units  # noqa: F401
from .workloads import CONFIGS, workload  # noqa: F401
