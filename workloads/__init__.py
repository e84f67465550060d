"""Seeded synthetic workloads (BASELINE.json `configs`) shared by the oracle tests,
the GPU parity tests, ``bench.py`` and ``smoke()``.

This package holds the plan parameters and the input generators only — no part of
the dedispersion method (no delay tables, no shift-and-sum).  The dispersion law
used to *inject* pulses is the signal model of the synthetic sky (DESIGN.md,
reading A17), typed here independently of both the oracle and the CUDA library.
"""
from .configs import CONFIGS, get_config, plan_args  # noqa: F401
from .filterbank import make_filterbank, pulse_table  # noqa: F401
