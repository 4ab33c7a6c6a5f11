"""Seeded synthetic inputs shaped like SIE embedding clusters (BASELINE.json configs 0-4).

This package holds ONLY input generation. It contains none of the method's arithmetic
(no transform, no pair integrals, no amplitudes, no G, no trace) and is the one module
shared by `oracle/` (test infrastructure) and `paper_2412_18553_b200/` (the CUDA product).
"""
from .gen import (  # noqa: F401
    ClusterSpec,
    ClusterInputs,
    config_specs,
    make_cluster,
    npair,
    occupied_subset,
    virtual_subset,
)
