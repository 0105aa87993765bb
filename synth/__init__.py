"""Seeded synthetic inputs for the coalesced-chunk hot path.

This package is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA
path (`paper_2606_19271_b200/`).  It holds no arithmetic of the method: it draws
random numbers, rounds them once to bf16 (the input format)
and describes workload structure (shapes, prior lengths, free-list
permutations, the churn event script).  Recipes: DESIGN.md §"Input recipe".
"""
from .bf16 import f32_to_bf16_bits, bf16_bits_to_f32, bf16_bits_to_f64
from .configs import (PoolShape, SessionSpec, Workload, tiny, wan13b_single,
                      wan13b_batch, wan14b_batch, churn_script, attention_flops,
                      attention_pairs, CONFIG_BUILDERS, sched_events)
from .draw import draw_bits, draw_session_tensors

__all__ = [
    "f32_to_bf16_bits", "bf16_bits_to_f32", "bf16_bits_to_f64", "PoolShape", "SessionSpec",
    "Workload", "tiny", "wan13b_single", "wan13b_batch", "wan14b_batch", "churn_script",
    "attention_flops", "attention_pairs", "CONFIG_BUILDERS", "sched_events", "draw_bits", "draw_session_tensors",
]
