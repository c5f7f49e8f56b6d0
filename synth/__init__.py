"""Seeded synthetic input generators shared by the oracle tests and the CUDA tests.

This package holds NO arithmetic of the method (no quantizer, no scoring, no
GEMM): only counter-based random tensors with the shapes and value structure
DESIGN.md "Input recipe" states.  Both `oracle/` and the CUDA path consume its
outputs; neither imports the other.
"""
from .generators import (  # noqa: F401
    gen_weight,
    gen_act,
    gen_calib,
    outlier_channels,
    budget_from_density,
    LayerShape,
    CONFIGS,
    config_shapes,
)
