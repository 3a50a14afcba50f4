"""Seeded synthetic input generators shared (as data only) by the oracle and the CUDA path."""
from . import rng, configs  # noqa: F401
from .configs import CONFIGS, Workload  # noqa: F401
