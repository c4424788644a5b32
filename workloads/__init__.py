"""Seeded synthetic workloads (inputs only) for the five BASELINE.json configs.

This package is shared by the oracle tests and the CUDA tests/bench.  It holds
none of the method's arithmetic: no mips, no level selection, no traversal, no
line-profile evaluation.  It only draws fields, line parameters, probes and
quadratures (recipe restated in DESIGN.md).
"""
from .gen import Workload, make, CONFIG_NAMES, C_LIGHT_KMS  # noqa: F401
