"""Seeded synthetic input generators shared by the oracle tests, the GPU parity tests and bench.py.

This package holds NONE of the method's arithmetic (no reconstruction, no softmax, no quantiser):
it only draws random tensors and tier/flag metadata with the shapes, sizes and value distributions
of BASELINE.json's configs (SURVEY.md §8d recipe, restated in DESIGN.md §5). Both `oracle/` and the
CUDA path consume exactly the tensors produced here; neither imports the other.
"""
from .workloads import (  # noqa: F401
    BASE_SEED,
    Workload,
    WORKLOADS,
    make_routing,
    make_basis,
    make_gates,
    make_q,
    make_coef_chunk,
    make_resid_chunk,
    make_dense_kv_chunk,
    make_omega,
    class_of,
    expected_bytes_per_lht,
)
