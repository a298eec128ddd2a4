"""Seeded synthetic inputs for the five BASELINE.json configs.

This package is *data only*: it builds the arrays (orbitals, local potential,
projector functions, projector strengths, occupations, laser samples) that both
the FP64 oracle (`oracle/`) and the CUDA library (`paper_2509_00966_b200/`)
consume.  It contains none of the method's arithmetic (no stencil, no
propagator, no projection) and imports neither of the two.
"""
from .configs import (  # noqa: F401
    DomainConfig,
    CONFIGS,
    get_config,
    generate_domain,
    generate,
    laser_samples,
)
