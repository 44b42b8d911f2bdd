"""Seeded synthetic inputs for the realfast search hot path.

This package serves BOTH the CPU oracle (``oracle/``) and the CUDA path
(``paper_1802_03084_b200``) with identical input bytes.  It holds no part of
the search method (no delay table used for searching, no gridding, no FFT, no
statistics): only the observation geometry, the noise, and the mock-transient
signal model ("mock transient sources ... inserted after
calibration").  Neither the oracle nor the CUDA path is imported here.
"""
from .configs import CONFIGS, Config, get_config  # noqa: F401
from .generate import (  # noqa: F401
    Transient,
    antenna_enu,
    baseline_uvw_m,
    channel_freqs_hz,
    chan_weights,
    default_cell_rad,
    dm_list,
    make_segment,
    noise_rows,
    transients,
)
