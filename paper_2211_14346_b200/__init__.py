"""paper_2211_14346_b200 — B200-native ttH selection + kinematic reconstruction (arXiv 2211.14346, §4).

Thin Python binding over the C ABI of ``libhepf.so`` (``include/hepf.h``): argument marshalling only — every
step of the path runs in the hand-written sm_100a kernels under ``csrc/``.  PyTorch supplies device memory and
streams.  There is no CPU fallback: importing works anywhere, calling needs the built library and a CUDA device.
"""
from .binding import (BEST_DTYPE, CHI2_DTYPE, CHI2_DILEP_DTYPE, DeviceEvents, HepfError, chi2_dilep, chi2_semilep, chi2_single_top, default_params, fp64_peak_probe, histogram, last_error, launch_count,
                      lib_path, load, make_cuts, philox_normal, reconstruct_tth, reconstruct_tth_n, select, select_record, tth_host, tth_system, histogram_values, cut_stats, plan_chain, select_planned, select_static, SELECT_STATIC_MAX_EVENTS)

__all__ = ["BEST_DTYPE", "CHI2_DTYPE", "CHI2_DILEP_DTYPE", "chi2_dilep", "chi2_semilep", "chi2_single_top", "DeviceEvents", "HepfError", "default_params", "fp64_peak_probe", "histogram", "last_error",
           "launch_count", "lib_path", "load", "make_cuts", "philox_normal", "reconstruct_tth", "reconstruct_tth_n", "select", "select_record", "tth_host", "tth_system", "histogram_values", "cut_stats", "plan_chain", "select_planned", "select_static", "SELECT_STATIC_MAX_EVENTS"]
