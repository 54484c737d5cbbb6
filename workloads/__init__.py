"""Seeded synthetic inputs shared by the oracle tests and the CUDA path.

This package holds NO arithmetic of the method (no basis ranking, no matrix
assembly, no sparse product, no Chebyshev/Clenshaw, no Lanczos).  It only draws
the random model parameters of the five BASELINE.json workloads from
``numpy.random.Generator(PCG64(seed))`` and writes them down as a *term list*
(the description of H both sides consume) plus the random start blocks.

Recipe: seed = 1000 + config for the
Hamiltonian parameters, 2000 + config for the start block.
"""
from .configs import (  # noqa: F401
    CONFIGS,
    Workload,
    make_workload,
    start_block,
    xxz_terms,
    fermion_terms,
    quantum_sun_terms,
)
