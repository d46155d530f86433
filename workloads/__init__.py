"""Seeded synthetic input generators shared by the oracle tests and the CUDA path.

This package holds NONE of the method's arithmetic (no FFT of the method, no
half-step, no energy): it only materialises the arrays (psi0, V, Omega, delta)
and the parameter sets of the five workloads of BASELINE.json / SURVEY.md
section 8(d), from a fixed counter-based generator, so that the oracle and the
GPU consume byte-identical inputs.
"""
from .configs import (  # noqa: F401
    CONFIGS,
    Workload,
    make_workload,
    splitmix64,
    uniforms,
    normals,
)
