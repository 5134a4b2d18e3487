"""B200-native GPUMCD hot path (arxiv 1101.1245): coupled photon-electron Monte Carlo dose.

``binding`` mirrors the C ABI of include/gpumcd.h; ``inputs`` generates the seeded synthetic
workloads (tables, phantoms, spectra); ``evaluation`` holds the dose-comparison metrics of the
paper (gamma index, Eq. 14-15; uncertainty, Eq. 12-13).
"""
from .binding import (GPUMCD_ERR_BANK_OVERFLOW, GPUMCD_ERR_CUDA, GPUMCD_ERR_INVALID_ARG, GPUMCD_ERR_NO_SOURCE,  # noqa: F401
                      GPUMCD_ERR_OOM, GPUMCD_ERR_TABLE_RANGE, GPUMCD_OK, GPUMCD_STATIC_MAX_VOXELS, Context, GpumcdError, gpumcd_create, gpumcd_create_host, gpumcd_default_options,  # noqa: F401
                      gpumcd_destroy, gpumcd_get_counters, gpumcd_get_energy_tally, gpumcd_last_error,
                      gpumcd_get_profile, gpumcd_probe_tally, gpumcd_selftest_philox, gpumcd_release_l2, gpumcd_run, gpumcd_run_host, gpumcd_run_trace, gpumcd_run_uncertainty, gpumcd_run_uncertainty_static,
                      gpumcd_set_history_offset, gpumcd_set_phantom, gpumcd_set_phantom_host, gpumcd_set_profiling,
                      gpumcd_set_source, load_library)
