"""paper_2504_02034_b200 -- thin Python binding of libchim (include/chim.h).

Argument marshalling only: every step of the hot path runs in the CUDA kernels of libchim.so.  PyTorch is
used for device memory and streams.  There is no CPU fallback: if libchim.so has not been built
(`python -m paper_2504_02034_b200.build` or `__graft_entry__.build()`), loading fails loudly.
"""
from .binding import (CHIM_BW_FIXED, CHIM_BW_SCOTT, CHIM_FLAG_BW_DEGENERATE, CHIM_FLAG_DL_NONMONOTONE,
                      CHIM_FLAG_EVENT_ZERO, CHIM_FLAG_LAMBDA_DOMAIN, CHIM_FLAG_NEFF_LOW, CHIM_FLAG_TABLE_RANGE,
                      CHIM_FLAG_XI_ZERO, CHIM_KDE_AUTO, CHIM_KDE_DIRECT, CHIM_KDE_POWER, CHIM_KDE_NONE, CHIM_KERNEL_GAUSS, CHIM_KERNEL_EPANECHNIKOV, CHIM_MEM_DEVICE, CHIM_MEM_HOST, CHIM_ON_GRID, CHIM_ON_SAMPLES, ChimConfig,
                      ChimAluPeaks, ChimError, ChimKernelTimes, ChimStats, Context, chim_create, chim_default_config, chim_destroy,
                      chim_get_stats, chim_init_events, chim_set_event_groups, chim_build_pcat, chim_build_pcat_static, CHIM_PCAT_STATIC_MAX_GALAXIES, chim_build_pgal, chim_loglike_grad_batch, chim_init_injections, chim_last_error,
                      chim_loglike_batch, chim_loglike_batch_host, chim_measure_alu_peaks, chim_version, lib, lib_path)
from .sharding import gather_lambda_results, shard_lambda

__all__ = [n for n in dir() if not n.startswith("_")]
