"""Seeded synthetic workloads (input generators only; no method arithmetic)."""
from .gen import (  # noqa: F401
    BASE_SEED,
    AffineConfig,
    SelectiveConfig,
    config,
    make_affine_inputs,
    make_selective_inputs,
    normal,
    to_f64_numpy,
    uniform,
)
