"""Seeded synthetic inputs for the CAS hot path (shared by oracle tests, GPU tests and bench.py).

This module holds NO arithmetic of the method (no attention, no Adam, no rotation policy): it only
draws random numbers with the shapes/distributions of BASELINE.json's five configs and rounds them
once to the config's storage dtype.  Both the oracle (``oracle/``) and the CUDA path
(``paper_2606_04557_b200``) consume exactly these arrays; neither imports the other.
"""
from .configs import CONFIGS, CasConfig, get_config  # noqa: F401
from .generate import (  # noqa: F401
    BASE_SEED,
    Workload,
    make_workload,
    round_to_dtype,
)
