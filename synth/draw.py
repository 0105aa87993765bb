"""Tensor draws: N(0,1) in fp32, rounded once to bf16 (SURVEY.md §8(d) "Synthetic inputs").

Host path (numpy Generator) is used for configs the oracle runs in full; the
device path (torch CUDA generator) for the large configs, whose drawn tensors
are then copied to the oracle as data.  Draw order per session, in sid order:
prior K, prior V, Q, Kn, Vn.
"""
import numpy as np

from .bf16 import f32_to_bf16_bits


def draw_bits(rng, n_tokens, n_heads, head_dim):
    """[n_tokens, H, D] uint16 bf16 bits from `rng` (numpy Generator)."""
    x = rng.standard_normal((n_tokens, n_heads, head_dim), dtype=np.float32)
    return f32_to_bf16_bits(x)


def draw_session_tensors(rng, shape, spec, layer_count=1):
    """All tensors of one session for one chunk step, host path.

    Returns dict with 'prior_k','prior_v' (lists over layers of [P*T,H,D] bits, fed to
    the pool in 3-frame appends by the caller) and 'q','k','v' ([C,H,D] bits).
    """
    H, D, T = shape.n_heads, shape.head_dim, shape.frame_tokens
    out = {"prior_k": [], "prior_v": []}
    for _ in range(layer_count):
        out["prior_k"].append(draw_bits(rng, spec.prior_frames * T, H, D))
        out["prior_v"].append(draw_bits(rng, spec.prior_frames * T, H, D))
    C = spec.chunk_frames * T
    out["q"] = draw_bits(rng, C, H, D)
    out["k"] = draw_bits(rng, C, H, D)
    out["v"] = draw_bits(rng, C, H, D)
    return out


def draw_bits_torch(gen, n_tokens, n_heads, head_dim, device):
    """Device path: torch bf16 tensor [n_tokens,H,D] drawn with a torch.Generator on `device`."""
    import torch
    x = torch.randn((n_tokens, n_heads, head_dim), generator=gen, device=device, dtype=torch.float32)
    return x.to(torch.bfloat16)   # round-to-nearest-even
