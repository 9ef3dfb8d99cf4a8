"""Seeded synthetic inputs for the block-causal streaming-attention path.

This package holds ONLY input generation (random draws, rounding to the storage
dtype, workload shapes).  It contains none of the method's arithmetic and is the
only code shared by the CPU oracle's tests and the CUDA path's tests/bench.
"""
from .workloads import (  # noqa: F401
    WorkloadSpec,
    Workload,
    SessionInputs,
    CONFIG_SPECS,
    spec_for_config,
    generate,
    modality_tags,
    to_bf16,
    algorithmic_flops,
    algorithmic_bytes,
)
