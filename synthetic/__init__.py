"""Seeded synthetic inputs shared by the oracle-side tests and the CUDA-side tests/bench.

This package holds NONE of the method's arithmetic (no waveform, no response, no inner
product, no F-statistic): only the frequency grids, the analytic noise PSD used to colour
the noise, the seeded Gaussian noise, the particle draws and the partition edges of
BASELINE.json's five configs (recipe: DESIGN.md "Synthetic inputs").
The injection template is supplied by the caller as an array, so that the oracle-side
callers use the oracle's template and the CUDA-side bench uses the library's own.
"""
from .lisa_data import (  # noqa: F401
    YEAR_S, C_SI, ARM_LENGTH_M, CONFIGS, BANDS_SMALL, Config, Dataset,
    frequency_grid, psd_tdi_x, psd_tdi, coloured_noise, equal_bin_edges, injection_params,
    injection_amplitudes, draw_particles, paper_range_particles, make_dataset, config_by_name,
)
