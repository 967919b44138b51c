"""Seeded synthetic workload generator (inputs only; holds none of the method's arithmetic).

Serves BOTH the CPU oracle (``oracle/``) and the CUDA path (``paper_2607_02749_b200``) with the same
input arrays: ansatz layouts / op lists, Pauli strings (+ their integer masks as plain data), real
coefficients, parameter batches and parameter masks.  Recipe: DESIGN.md "Input recipe".
"""
from .generator import (  # noqa: F401
    CONFIGS,
    Workload,
    SplitMix64,
    make_workload,
    make_hamiltonian,
    layout_ops,
    num_params,
    shift_rows,
    community_param_mask,
    OP_RY,
    OP_RZ,
    OP_CZ,
    OP_CNOT,
)
