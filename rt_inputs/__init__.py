"""Seeded synthetic input generators shared by the tests, bench.py and smoke().

This package holds NONE of the method's arithmetic (no directions, no traversal, no transfer
equation): it only produces the kappa / S fields of the five BASELINE.json configs.  Both the
oracle and the CUDA library receive the same fp32 arrays produced here.
"""
from .fields import CONFIGS, ConfigSpec, make_fields, config_spec  # noqa: F401
