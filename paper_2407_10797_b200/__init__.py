"""B200-native batched semi-coherent F-statistic (arXiv 2407.10797) -- Python binding of the C ABI.

The functions here carry the names of include/fstat.h and only marshal arguments: every step of the
path (a0 table fold, a1 prologue, a2-a5 fused template + inner products, a6 epilogue) runs in the
sm_100a kernels of ``libfstat_b200.so``.  PyTorch appears only as the owner of device memory and
streams.  There is no CPU fallback: importing works without a GPU (so that symbols can be checked),
but every compute call returns FSTAT_ECUDA -> ``FstatError`` when no sm_100 device exists, and a
missing shared object raises at import of the first call.

This package never imports ``oracle`` (the CPU oracle is test infrastructure) and vice versa.
"""
from __future__ import annotations

from .binding import (  # noqa: F401
    FstatError, Options, Plan, STATUS, TDI_CHANNELS,
    fstat_default_options, fstat_plan_create, fstat_plan_set_partitions, fstat_eval_batch,
    fstat_eval_batch_noalloc, fstat_noalloc_scratch_bytes,
    fstat_eval_batch_host, fstat_eval_batch_bands, fstat_eval_batch_bands_host, fstat_eval_amplitudes_bands, fstat_eval_batch_channels, fstat_eval_amplitudes, fstat_eval_template, fstat_plan_destroy, fstat_plan_n_bins,
    fstat_plan_n_part, fstat_plan_device, fstat_plan_n_ctas, fstat_plan_launch_count, fstat_plan_table_bytes, fstat_plan_band_stats,
    fstat_plan_main_kernel_ms, fstat_plan_level_bins, fstat_edges_equal_bins, fstat_probe_pipe_peak,
    fstat_status_str, fstat_last_error, library_path, load_library, EXPORTED_SYMBOLS,
    Pso, PsoOptions, fstat_pso_default_options, fstat_pso_create, fstat_pso_iterate, fstat_pso_best,
    fstat_pso_state, fstat_pso_iterations_done, fstat_pso_destroy,
)
