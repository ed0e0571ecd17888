"""paper_2001_03389_b200 -- B200-native sigma-cut RFI cleaning (librfim) and its Python binding.

The product is the C-ABI library `librfim.so` (include/rfim.h) built from csrc/; `binding` marshals
arguments to it.  `synth` is the seeded input generator used by tests and bench.  Nothing here
imports the CPU oracle, and nothing falls back to the CPU.
"""
from .binding import (MEAN, MEDIAN, OP_FREQ, OP_HOST, OP_TIME, OP_TIME_FREQ, VARIANT_AUTO, VARIANT_FD_QBIN, VARIANT_FD_QUAD, VARIANT_FD_STREAM,  # noqa: F401
                      VARIANT_FD_STRIP, VARIANT_FD_STRIP_BULK, VARIANT_FD_STRIP_CLUSTER, VARIANT_GENERIC,
                      VARIANT_STAGED, VARIANT_STAGED_1W, VARIANT_STAGED_2W, RfimError, RfimOpts,
                      rfim_freq_sigma_cut, rfim_freq_sigma_cut_noalloc, rfim_launch_count, rfim_last_variant, rfim_sigma_cut_host,
                      rfim_time_freq_sigma_cut, rfim_time_sigma_cut, rfim_version, rfim_workspace_bytes)
