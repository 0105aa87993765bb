"""bf16 <-> fp32/fp64 bit conversions on numpy arrays (numpy has no bf16 dtype).

bf16 values travel as uint16 bit patterns: the top 16 bits of the IEEE fp32
encoding.  Rounding fp32 -> bf16 is round-to-nearest-even, done once when the
inputs are drawn; widening is exact.
"""
import numpy as np


def f32_to_bf16_bits(x):
    """fp32 array -> uint16 bf16 bit patterns, round-to-nearest-even. Finite inputs only."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    u = x.view(np.uint32)
    rounding_bias = ((u >> 16) & 1) + np.uint32(0x7FFF)
    return ((u + rounding_bias) >> 16).astype(np.uint16)


def bf16_bits_to_f32(bits):
    """uint16 bf16 bit patterns -> fp32 (exact)."""
    bits = np.ascontiguousarray(bits, dtype=np.uint16)
    return (bits.astype(np.uint32) << 16).view(np.float32)


def bf16_bits_to_f64(bits):
    """uint16 bf16 bit patterns -> fp64 (exact)."""
    return bf16_bits_to_f32(bits).astype(np.float64)
