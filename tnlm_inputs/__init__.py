"""Seeded synthetic inputs shared by the oracle-side tests and the CUDA path (no TNLM arithmetic)."""
from .phantoms import CONFIGS, TnlmConfig, make_stack, dynamic_range, random_stack, z_slab
from . import projections

__all__ = ["CONFIGS", "TnlmConfig", "make_stack", "dynamic_range", "random_stack", "z_slab", "projections"]
