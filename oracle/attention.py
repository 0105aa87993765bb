"""Oracle attention: frame-block-causal masked softmax attention in fp64 (TEST INFRASTRUCTURE).

O1 of SURVEY.md §8(c).  PAPER.md:66 (iii) "invokes the model once for the batch": per session,
the chunk's query tokens attend to that session's own persistent KV cache (PAPER.md:261
"temporal or KV-cache states") and to the chunk itself.  The mask, window and shapes are
BASELINE.json north_star's: "a query token sees all KV-cache tokens and all chunk tokens of
frames up to its own", "rolling-window cap" (readings R1, R2, R5, R6 in DESIGN.md).

For session s, head h, chunk token i (frame f_i = i // T):
  visible prior tokens  j in [a*T, L)            with a = max(0, P + c - W)   (W > 0)
  visible chunk tokens  j in [0, C) with j // T <= f_i
  z_j = scale * <q_i, k_j>;  m = max z;  w_j = exp(z_j - m);  o_i = sum w_j v_j / sum w_j;
  lse_i = m + log(sum w_j)                                      (natural log)
Everything in fp64 on exactly-widened bf16 inputs; `scale` is the caller's fp32 value widened.
Two passes, no online softmax.  The only library step is numpy's fp64 matmul.
"""
import numpy as np


def _widen(bits):
    """bf16 bit patterns (uint16) -> fp64, exact."""
    return (np.ascontiguousarray(bits, dtype=np.uint16).astype(np.uint32) << 16).view(np.float32).astype(np.float64)


def _visible_prior(pool, layer, sid, c):
    """K, V (fp64 [n_vis, H, D]) of the visible prior tokens, read through the page table."""
    s = pool.sessions[sid]
    T, B, W = pool.T, pool.B, pool.W
    a = max(0, s.P + c - W) if W > 0 else 0
    j = np.arange(a * T, s.P * T, dtype=np.int64)
    x = s.o + j
    if len(j) == 0:
        z = np.zeros((0, pool.H, pool.D))
        return z, z
    pages = np.asarray(s.PT, dtype=np.int64)[x // B]
    slots = x % B
    return _widen(pool.K[layer, pages, slots]), _widen(pool.V[layer, pages, slots])


def _attend(q, rows, kp, vp, kc, vc, T, scale):
    """q [R, D] fp64, rows [R] chunk-token index of each query; kp/vp [Lv, D] prior; kc/vc [C, D] chunk."""
    C = kc.shape[0]
    z_prior = scale * (q @ kp.T)                                            # every visible prior key
    z_chunk = scale * (q @ kc.T)
    visible = (np.arange(C)[None, :] // T) <= (rows[:, None] // T)          # frame(j) <= frame(i)
    z_chunk = np.where(visible, z_chunk, -np.inf)
    z = np.concatenate([z_prior, z_chunk], axis=1)
    m = z.max(axis=1, keepdims=True)                                        # own frame is always visible: finite
    w = np.exp(z - m)
    denom = w.sum(axis=1, keepdims=True)
    o = (w @ np.concatenate([vp, vc], axis=0)) / denom
    lse = (m + np.log(denom))[:, 0]
    return o, lse


def attention_rows(pool, layer, sid, c, q, kn, vn, scale, head, rows):
    """Selected query rows of one (session, head), each computed in full over all its visible keys.
    q, kn, vn: uint16 [C, H, D] of THIS session's chunk.  Returns (o [R, D], lse [R]) fp64."""
    rows = np.asarray(rows, dtype=np.int64)
    kp, vp = _visible_prior(pool, layer, sid, c)
    s = float(np.float32(scale))
    return _attend(_widen(q[rows, head]), rows, kp[:, head], vp[:, head],
                   _widen(kn[:, head]), _widen(vn[:, head]), pool.T, s)


def chunk_attention(pool, layer, sids, chunk_frames, q, kn, vn, scale):
    """Whole coalesced batch.  q, kn, vn: uint16 bf16 bits [sum C_s, H, D] packed in `sids` order (R15).
    Returns (O fp64 [sum C_s, H, D], LSE fp64 [sum C_s, H]).  No pool state changes (R5)."""
    pool._check_batch(layer, sids, chunk_frames)
    T, H, D = pool.T, pool.H, pool.D
    total = sum(c * T for c in chunk_frames)
    if q.shape != (total, H, D) or kn.shape != q.shape or vn.shape != q.shape:
        from .pool import OracleError, INVALID
        raise OracleError(INVALID, "q/k/v shape")
    s = float(np.float32(scale))
    out = np.zeros((total, H, D), dtype=np.float64)
    lse = np.zeros((total, H), dtype=np.float64)
    off = 0
    for sid, c in zip(sids, chunk_frames):                    # sessions are independent
        C = c * T
        kp, vp = _visible_prior(pool, layer, sid, c)
        qs, ks, vs = _widen(q[off:off + C]), _widen(kn[off:off + C]), _widen(vn[off:off + C])
        rows = np.arange(C, dtype=np.int64)
        for h in range(H):
            o, l = _attend(qs[:, h], rows, kp[:, h], vp[:, h], ks[:, h], vs[:, h], T, s)
            out[off:off + C, h] = o
            lse[off:off + C, h] = l
        off += C
    return out, lse
