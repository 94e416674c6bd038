"""Seeded synthetic inputs (serve both the CUDA path's tests/bench and the oracle's tests).

This package holds none of the method's arithmetic: it only manufactures pressure-gradient fields
g = grad P (+ noise) and masks that stand in for the paper's workloads.
"""
from .fields import CONFIGS, make_config, make_field  # noqa: F401
