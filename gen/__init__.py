"""Seeded synthetic inputs for the single-pulse-detection path.

This package serves BOTH the oracle-side tests and the CUDA-side tests/bench.  It holds
none of the method's arithmetic (no statistics, no boxcars, no SNR, no thresholding):
only noise, baselines and injected pulses of known position / width / amplitude.
"""
from .synth import (  # noqa: F401
    SEED0,
    Config,
    Pulse,
    CONFIGS,
    get_config,
    custom_config,
    pulse_table,
    pulse_rows,
    make_rows,
    make_array,
)
