"""Seeded synthetic input generators shared by the tests, bench.py and smoke().

This module holds NONE of the method's arithmetic (no copy, no gather/scatter,
no attention, no stage planning): it only draws the random *inputs* — pool
contents, block-id permutations, appended-token values, context lengths,
queries and request-length mixes — that both the CPU oracle (`oracle/`) and the
CUDA path (`paper_2406_03243_b200/`) are then run on.  Neither of those two
imports this module; the callers (tests / bench) pass the arrays in.

The inputs *stand in for* the paper's LLaMA-7B / LLaMA-30B serving workloads
(§6.1 Testbed/Models) and its Table-1 power-law length mixes
(PAPER.md:256-266); the recipe is stated in DESIGN.md §"Input recipe".
"""
from .generators import (  # noqa: F401
    CONFIGS,
    slice_values_f16,
    block_permutation,
    append_values_f16,
    context_lengths,
    queries_f16,
    bounded_pareto_alpha,
    bounded_pareto_lengths,
    batch_request_blocks,
    SENTINEL_U16,
)
