"""Test-side helpers: build an oracle pool for a synth Workload and feed priors in 3-frame appends."""
import numpy as np

import oracle
import synth


def make_oracle_pool(shape, free_order=None, host_pages=None):
    return oracle.OraclePool(shape.n_layers, shape.n_heads, shape.head_dim, shape.page_tokens,
                             shape.n_pages, shape.frame_tokens, shape.window_frames,
                             shape.max_sessions, free_order, host_pages)


def feed_prior(pool, sid, k_layers, v_layers, frame_tokens, frames_per_append=3):
    """Install a prior cache through append (exercises append); commit on the last layer."""
    n_frames = k_layers[0].shape[0] // frame_tokens
    f = 0
    while f < n_frames:
        c = min(frames_per_append, n_frames - f)
        lo, hi = f * frame_tokens, (f + c) * frame_tokens
        for layer in range(len(k_layers)):
            pool.append(layer, [sid], [c], k_layers[layer][lo:hi], v_layers[layer][lo:hi],
                        commit=(layer == len(k_layers) - 1))
        f += c


def build_oracle_workload(w):
    """Open all sessions of `w`, feed priors, return (pool, sids, tensors, q, k, v packed)."""
    pool = make_oracle_pool(w.shape, w.free_order)
    sids = [pool.open() for _ in w.sessions]
    tensors = [synth.draw_session_tensors(w.rng, w.shape, s, w.shape.n_layers) for s in w.sessions]
    for sid, spec, t in zip(sids, w.sessions, tensors):
        if spec.prior_frames:
            feed_prior(pool, sid, t["prior_k"], t["prior_v"], w.shape.frame_tokens)
    q = np.concatenate([t["q"] for t in tensors])
    k = np.concatenate([t["k"] for t in tensors])
    v = np.concatenate([t["v"] for t in tensors])
    return pool, sids, tensors, q, k, v


def rel_l2(a, b):
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))
