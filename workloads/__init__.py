"""Synthetic workload descriptions + seeded input generators (inputs only, no method arithmetic)."""
from . import shapes, gen  # noqa: F401
