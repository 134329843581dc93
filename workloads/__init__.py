"""Seeded synthetic inputs for the FP8 EAGLE verify step.

This package holds NONE of the method's arithmetic (no E4M3, no scales, no
attention, no acceptance).  It only draws the random bits both sides consume:
model weights (bf16 bit patterns), context ids, draft trees and draft tokens,
with the shapes BASELINE.json's five configs name.  Both the CPU oracle
(`oracle/`) and the CUDA library (`paper_2606_18502_b200/`) are *fed* these
arrays by the tests and by bench.py; neither imports the other.

Recipe:
  * weights: fp32 N(0, 0.02^2) -> bf16 round-to-nearest-even, one independent
    stream per (seed, matrix kind, layer); RMSNorm gains 1.0.
  * context ids / root ids / draft ids: uniform in [0, vocab).
  * trees: chains, or the T-1 cheapest child-rank paths under per-depth caps.
"""
from .configs import CONFIGS, ModelShape, TINY, LLAMA8B, WorkloadSpec  # noqa: F401
from .gen import (  # noqa: F401
    MATRIX_KINDS, matrix_shape, weight_matrix_bf16, gain_vector_bf16,
    chain_parents, tree_parents, tree_depths, context_lengths, context_ids,
    draft_tokens_uniform, calibration_hidden, f32_to_bf16_bits, bf16_bits_to_f32,
)
