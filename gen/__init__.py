"""Seeded synthetic input generator shared by the oracle and the CUDA path.

Inputs only: this package holds none of ProtoKV's arithmetic (no assignment, no
statistics, no attention).  See gen/workload.py and DESIGN.md "Input recipe".
"""
from .workload import (  # noqa: F401
    WorkloadSpec,
    CONFIGS,
    spec_for,
    frame_kv,
    grid_positions,
    codebooks,
    queries,
    cluster_ids,
    splitmix64,
    standard_normal,
)
