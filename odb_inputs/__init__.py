"""Seeded synthetic inputs for the ODB group -> align -> collate path.

This package holds ONLY input generation (lengths, masked spans, token ids, the
named workload configurations). It contains none of the method's arithmetic
(no sorting, grouping, alignment or collation) and is the one module that both
the CPU oracle's tests and the CUDA path's tests / bench may import.
"""
from .gen import (  # noqa: F401
    VOCAB,
    Workload,
    bj_config,
    config5_cells,
    make_workload,
    protocol_workload,
    custom_workload,
    audit_distribution,
    AUDIT_KINDS,
    token_ids,
    tokens_for_samples,
    describe,
    split_ranks,
    offline_workload,
)
