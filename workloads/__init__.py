"""Seeded synthetic inputs shared by the oracle tests and the CUDA path.

This package holds NONE of the method's arithmetic (no conductances, no matrix,
no solver): it only turns a config id + seed into plain arrays (cell fields and
power maps) that are handed identically to `oracle/` and to the C-ABI library.
"""
from .generators import (  # noqa: F401
    Workload, make_workload, power_for_step, splitmix64, uniform01, normal01,
    CONFIG_NAMES, SEEDS,
)
