"""Seeded synthetic input generators for the DNN-SP2-PT hot path.

This module serves BOTH the CUDA path and the CPU oracle and therefore holds
none of the method's arithmetic (no Gershgorin bounds, no SP2 recursion, no
hi/lo split): it only builds symmetric matrices H0, H1 with a known occupation
count.  The recipes stand in for the paper's LATTE water boxes (PAPER.md:546,
569) and Ergo water clusters, which are not available; see
DESIGN.md "Input recipe".
"""
from .hamiltonians import (  # noqa: F401
    Workload,
    CONFIGS,
    seed_for,
    symmetric_gaussian,
    gapped_random_orthogonal,
    tight_binding_cube,
    make_config,
)
