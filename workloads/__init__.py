"""Seeded synthetic inputs for the fringe-search hot path (serves both the oracle tests and the
CUDA path; holds none of the method's arithmetic)."""
from .gen import CONFIG_IDS, config, generate, next_pow2  # noqa: F401
