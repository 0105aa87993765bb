"""Pins P1-P12 for the CPU oracle.  None of these re-type the oracle's formula
through the same routine: each is brute force, a closed form, an invariant, a reduction to a
library routine, or a hand-worked trace."""
import math
import os

import numpy as np
import pytest
import torch

import oracle
import synth
from helpers import build_oracle_workload, feed_prior, make_oracle_pool, rel_l2

W64 = synth.bf16_bits_to_f64


def small_shape(**kw):
    d = dict(n_layers=1, n_heads=2, head_dim=16, page_tokens=8, n_pages=64, frame_tokens=5,
             window_frames=0, max_sessions=8)
    d.update(kw)
    return synth.PoolShape(**d)


def draw(rng, n, shape):
    return synth.draw_bits(rng, n, shape.n_heads, shape.head_dim)


# ---- P1: brute force on Tiny, explicit visible(i, j), naive exp/sum, logical arrays ----------
def test_p1_brute_force_tiny():
    w = synth.tiny()
    pool, sids, tensors, q, k, v = build_oracle_workload(w)
    cf = [s.chunk_frames for s in w.sessions]
    O, LSE = oracle.chunk_attention(pool, 0, sids, cf, q, k, v, w.scale)
    T, H, D = w.shape.frame_tokens, w.shape.n_heads, w.shape.head_dim
    scale = float(w.scale)
    off = 0
    for spec, t in zip(w.sessions, tensors):
        # logical K/V: prior tokens (as drawn, no page table) then chunk tokens
        Kl = np.concatenate([W64(t["prior_k"][0]), W64(t["k"])])
        Vl = np.concatenate([W64(t["prior_v"][0]), W64(t["v"])])
        Lp = spec.prior_frames * T
        C = spec.chunk_frames * T
        Q = W64(t["q"])

        def visible(i, j):      # i: chunk query index, j: index into [prior | chunk]
            return True if j < Lp else ((j - Lp) // T <= i // T)

        for h in range(H):
            for i in range(C):
                num = [0.0] * D
                den = 0.0
                for j in range(Lp + C):
                    if not visible(i, j):
                        continue
                    dot = 0.0
                    for d in range(D):
                        dot += Q[i, h, d] * Kl[j, h, d]
                    e = math.exp(scale * dot)
                    den += e
                    for d in range(D):
                        num[d] += e * Vl[j, h, d]
                ref = np.array(num) / den
                np.testing.assert_allclose(O[off + i, h], ref, rtol=1e-11, atol=1e-13)
                assert abs(LSE[off + i, h] - math.log(den)) < 1e-11
        off += C


# ---- P2: constant V => output == V ---------------------------------------------------------------
def test_p2_constant_v():
    shape = small_shape()
    rng = np.random.default_rng(11)
    pool = make_oracle_pool(shape, rng.permutation(shape.n_pages))
    sid = pool.open()
    u = draw(rng, 1, shape)                                     # one token's value, all heads
    T = shape.frame_tokens
    feed_prior(pool, sid, [draw(rng, 4 * T, shape)], [np.repeat(u, 4 * T, axis=0)], T)
    q, k = draw(rng, 2 * T, shape), draw(rng, 2 * T, shape)
    O, _ = oracle.chunk_attention(pool, 0, [sid], [2], q, k, np.repeat(u, 2 * T, axis=0), 0.25)
    np.testing.assert_allclose(O, np.broadcast_to(W64(u), O.shape), rtol=0, atol=1e-15)


# ---- P3: single visible key ------------------------------------------------------------------------
def test_p3_single_visible_key():
    shape = small_shape(frame_tokens=1)
    rng = np.random.default_rng(12)
    pool = make_oracle_pool(shape)
    sid = pool.open()
    q, k, v = draw(rng, 4, shape), draw(rng, 4, shape), draw(rng, 4, shape)
    scale = np.float32(0.3)
    O, LSE = oracle.chunk_attention(pool, 0, [sid], [4], q, k, v, scale)
    np.testing.assert_array_equal(O[0], W64(v)[0])              # exactly v_0
    z0 = float(scale) * np.einsum("hd,hd->h", W64(q)[0], W64(k)[0])
    np.testing.assert_allclose(LSE[0], z0, rtol=0, atol=1e-14)
    # the last token of a later frame must differ from v_0 (sees more than one key)
    assert np.abs(O[3] - W64(v)[0]).max() > 1e-3


# ---- P4: placement invariance --------------------------------------------------------------------------
def test_p4_placement_invariance():
    shape = small_shape()
    T = shape.frame_tokens
    outs = []
    for perm_seed in (1, 2):
        rng = np.random.default_rng(13)
        pool = make_oracle_pool(shape, np.random.default_rng(perm_seed).permutation(shape.n_pages))
        a, b = pool.open(), pool.open()
        feed_prior(pool, b, [draw(rng, 3 * T, shape)], [draw(rng, 3 * T, shape)], T)
        feed_prior(pool, a, [draw(rng, 6 * T, shape)], [draw(rng, 6 * T, shape)], T)
        q, k, v = (draw(rng, 4 * T, shape) for _ in range(3))
        outs.append((oracle.chunk_attention(pool, 0, [a, b], [2, 2], q, k, v, 0.25), pool.page_table(a)))
    (O1, L1), pt1 = outs[0]
    (O2, L2), pt2 = outs[1]
    assert pt1 != pt2
    np.testing.assert_array_equal(O1, O2)
    np.testing.assert_array_equal(L1, L2)


# ---- P5: suspend -> resume leaves the logical KV bit-identical --------------------------------
def test_p5_suspend_resume_identity():
    shape = small_shape(n_layers=2, window_frames=6)
    T = shape.frame_tokens
    rng = np.random.default_rng(14)
    pool = make_oracle_pool(shape, rng.permutation(shape.n_pages))
    a, b = pool.open(), pool.open()
    for sid, frames in ((a, 3), (b, 9)):      # b has rolled: head offset != 0
        feed_prior(pool, sid, [draw(rng, frames * T, shape) for _ in range(2)],
                   [draw(rng, frames * T, shape) for _ in range(2)], T)
    assert pool.info(b)["head_off"] != 0
    before = [pool.gather_kv(l, b) for l in range(2)]
    info_before, pt_before = pool.info(b), pool.page_table(b)
    q, k, v = (draw(rng, 2 * T, shape) for _ in range(3))
    O_before = oracle.chunk_attention(pool, 1, [b], [2], q, k, v, 0.25)
    a_before = pool.gather_kv(0, a)
    pool.suspend(b)
    assert pool.info(b)["state"] == oracle.SUSPENDED and pool.page_table(b) == []
    with pytest.raises(oracle.OracleError) as e:
        oracle.chunk_attention(pool, 1, [b], [2], q, k, v, 0.25)
    assert e.value.kind == oracle.STATE
    c = pool.open()                            # steal some pages in between, then give them back
    feed_prior(pool, c, [draw(rng, 2 * T, shape) for _ in range(2)], [draw(rng, 2 * T, shape) for _ in range(2)], T)
    pool.resume(b)
    after = [pool.gather_kv(l, b) for l in range(2)]
    for (k0, v0), (k1, v1) in zip(before, after):
        np.testing.assert_array_equal(k0, k1)
        np.testing.assert_array_equal(v0, v1)
    info_after = pool.info(b)
    assert {x: info_after[x] for x in ("len_tokens", "head_off", "n_pages")} == \
           {x: info_before[x] for x in ("len_tokens", "head_off", "n_pages")}
    assert pool.page_table(b) != pt_before          # physical ids may differ
    O_after = oracle.chunk_attention(pool, 1, [b], [2], q, k, v, 0.25)
    np.testing.assert_array_equal(O_before[0], O_after[0])
    np.testing.assert_array_equal(a_before[0], pool.gather_kv(0, a)[0])   # isolation


# ---- P6: reduction to torch SDPA (fp64, explicit boolean mask) --------------------------------------
def _sdpa(q, k, v, mask, scale):
    tq, tk, tv = (torch.from_numpy(x).permute(1, 0, 2)[None] for x in (q, k, v))   # [1,H,L,D]
    out = torch.nn.functional.scaled_dot_product_attention(tq, tk, tv, attn_mask=torch.from_numpy(mask), scale=scale)
    return out[0].permute(1, 0, 2).numpy()


def test_p6_t1_is_bottom_right_causal():
    shape = small_shape(frame_tokens=1, page_tokens=4)
    rng = np.random.default_rng(15)
    pool = make_oracle_pool(shape, rng.permutation(shape.n_pages))
    sid = pool.open()
    P, C = 11, 7
    pk, pv = draw(rng, P, shape), draw(rng, P, shape)
    feed_prior(pool, sid, [pk], [pv], 1)
    q, k, v = (draw(rng, C, shape) for _ in range(3))
    scale = np.float32(1 / np.sqrt(shape.head_dim))
    O, _ = oracle.chunk_attention(pool, 0, [sid], [C], q, k, v, scale)
    i = np.arange(C)[:, None]
    j = np.arange(P + C)[None, :]
    mask = j <= i + P                                      # bottom-right aligned causal
    ref = _sdpa(W64(q), np.concatenate([W64(pk), W64(k)]), np.concatenate([W64(pv), W64(v)]), mask, float(scale))
    np.testing.assert_allclose(O, ref, rtol=1e-12, atol=1e-14)


def test_p6_single_frame_no_prior_is_plain_sdpa():
    shape = small_shape(frame_tokens=13)
    rng = np.random.default_rng(16)
    pool = make_oracle_pool(shape)
    sid = pool.open()
    q, k, v = (draw(rng, 13, shape) for _ in range(3))
    scale = np.float32(0.2)
    O, LSE = oracle.chunk_attention(pool, 0, [sid], [1], q, k, v, scale)
    ref = _sdpa(W64(q), W64(k), W64(v), np.ones((13, 13), dtype=bool), float(scale))
    np.testing.assert_allclose(O, ref, rtol=1e-12, atol=1e-14)
    z = float(scale) * np.einsum("ihd,jhd->hij", W64(q), W64(k))
    ref_lse = torch.logsumexp(torch.from_numpy(z), dim=-1).numpy().T
    np.testing.assert_allclose(LSE, ref_lse, rtol=1e-12, atol=1e-13)


# ---- P7: chunked == monolithic ---------------------------------------------------------------------------
@pytest.mark.parametrize("chunks", [[3, 3, 3], [1] * 9, [2, 4, 3]])
def test_p7_chunked_equals_monolithic(chunks):
    shape = small_shape(page_tokens=8, frame_tokens=5)
    T = shape.frame_tokens
    rng = np.random.default_rng(17)
    q, k, v = (draw(rng, 9 * T, shape) for _ in range(3))
    mono = make_oracle_pool(shape)
    sid = mono.open()
    O_mono, L_mono = oracle.chunk_attention(mono, 0, [sid], [9], q, k, v, 0.25)
    pool = make_oracle_pool(shape, np.random.default_rng(3).permutation(shape.n_pages))
    sid = pool.open()
    f = 0
    for c in chunks:
        sl = slice(f * T, (f + c) * T)
        O, L = oracle.chunk_attention(pool, 0, [sid], [c], q[sl], k[sl], v[sl], 0.25)
        np.testing.assert_allclose(O, O_mono[sl], rtol=1e-12, atol=1e-14)
        np.testing.assert_allclose(L, L_mono[sl], rtol=1e-12, atol=1e-13)
        pool.append(0, [sid], [c], k[sl], v[sl])
        f += c
        assert len(pool.page_table(sid)) == -(-f * T // shape.page_tokens)
    gk, gv = pool.gather_kv(0, sid)
    np.testing.assert_array_equal(gk, k)
    np.testing.assert_array_equal(gv, v)


# ---- P8: batch-composition invariance ---------------------------------------------------------------------
def test_p8_batch_composition_invariance():
    shape = small_shape(window_frames=7)
    T = shape.frame_tokens
    rng = np.random.default_rng(18)
    priors = {n: (draw(rng, f * T, shape), draw(rng, f * T, shape)) for n, f in (("a", 2), ("b", 6), ("c", 0))}
    chunks = {n: tuple(draw(rng, c * T, shape) for _ in range(3)) for n, c in (("a", 2), ("b", 3), ("c", 1))}
    cf = {"a": 2, "b": 3, "c": 1}

    def run(order):
        pool = make_oracle_pool(shape, np.random.default_rng(5).permutation(shape.n_pages))
        sid = {n: pool.open() for n in order}
        for n in order:
            if priors[n][0].shape[0]:
                feed_prior(pool, sid[n], [priors[n][0]], [priors[n][1]], T)
        q, k, v = (np.concatenate([chunks[n][i] for n in order]) for i in range(3))
        O, L = oracle.chunk_attention(pool, 0, [sid[n] for n in order], [cf[n] for n in order], q, k, v, 0.25)
        pool.append(0, [sid[n] for n in order], [cf[n] for n in order], k, v)
        res, off = {}, 0
        for n in order:
            C = cf[n] * T
            res[n] = (O[off:off + C], L[off:off + C], pool.gather_kv(0, sid[n]), pool.info(sid[n]))
            off += C
        return res

    full = run(["a", "b", "c"])
    for order in (["c", "b", "a"], ["b"], ["a", "c"]):
        part = run(order)
        for n in order:
            np.testing.assert_array_equal(part[n][0], full[n][0])
            np.testing.assert_array_equal(part[n][1], full[n][1])
            np.testing.assert_array_equal(part[n][2][0], full[n][2][0])
            np.testing.assert_array_equal(part[n][2][1], full[n][2][1])
            for key in ("len_tokens", "head_off", "n_pages"):
                assert part[n][3][key] == full[n][3][key]


# ---- P9: softmax invariants and LSE merge --------------------------------------------------------------
def test_p9_softmax_invariants_and_lse_merge():
    shape = small_shape()
    T = shape.frame_tokens
    rng = np.random.default_rng(19)
    pool = make_oracle_pool(shape)
    sid = pool.open()
    pk, pv = draw(rng, 4 * T, shape), draw(rng, 4 * T, shape)
    feed_prior(pool, sid, [pk], [pv], T)
    q, k, v = (draw(rng, 2 * T, shape) for _ in range(3))
    O, L = oracle.chunk_attention(pool, 0, [sid], [2], q, k, v, 0.25)
    allv = np.concatenate([W64(pv), W64(v)])
    for i in range(2 * T):
        vis = allv[: 4 * T + (i // T + 1) * T]
        assert (O[i] <= vis.max(axis=0) + 1e-15).all() and (O[i] >= vis.min(axis=0) - 1e-15).all()
    # chunk-only partial: same chunk on an empty session
    empty = make_oracle_pool(shape)
    e = empty.open()
    Oc, Lc = oracle.chunk_attention(empty, 0, [e], [2], q, k, v, 0.25)
    # prior-only partial: plain softmax over the prior keys, written with logsumexp from scipy
    from scipy.special import logsumexp
    z = 0.25 * np.einsum("ihd,jhd->ihj", W64(q), W64(pk))
    Lp = logsumexp(z, axis=2)
    Op = np.einsum("ihj,jhd->ihd", np.exp(z - Lp[:, :, None]), W64(pv))
    Lj = np.logaddexp(Lp, Lc)
    Oj = Op * np.exp(Lp - Lj)[:, :, None] + Oc * np.exp(Lc - Lj)[:, :, None]
    np.testing.assert_allclose(L, Lj, rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(O, Oj, rtol=1e-11, atol=1e-13)


# ---- P10: window equivalence, page-count closed forms, conservation ---------------------------------
def test_p10_window():
    shape = small_shape(window_frames=7, page_tokens=8, frame_tokens=5)
    T, B, Wn = shape.frame_tokens, shape.page_tokens, shape.window_frames
    rng = np.random.default_rng(20)
    pool = make_oracle_pool(shape, rng.permutation(shape.n_pages))
    sid = pool.open()
    other = pool.open()
    n_frames = 16
    ks, vs = draw(rng, n_frames * T, shape), draw(rng, n_frames * T, shape)
    q, k, v = (draw(rng, 3 * T, shape) for _ in range(3))
    fed = 0
    for c in (3, 3, 2, 3, 1, 3, 1):
        sl = slice(fed * T, (fed + c) * T)
        pool.append(0, [sid], [c], ks[sl], vs[sl])
        fed += c
        info = pool.info(sid)
        P = min(fed, Wn)
        evicted = (fed - P) * T
        assert info["frames"] == P
        assert info["head_off"] == evicted % B                               # o = evicted tokens mod B
        assert info["n_pages"] == -(-(info["head_off"] + P * T) // B)        # ceil((o+L)/B)
        pts = pool.page_table(sid) + pool.page_table(other)
        assert len(pool.free) + len(pts) == shape.n_pages                    # conservation
        assert len(set(pts) | set(pool.free)) == shape.n_pages               # no id twice
        gk, gv = pool.gather_kv(0, sid)
        np.testing.assert_array_equal(gk, ks[(fed - P) * T: fed * T])
        np.testing.assert_array_equal(gv, vs[(fed - P) * T: fed * T])
    assert fed == n_frames and pool.info(sid)["frames"] == Wn
    # attention with P + c > W  ==  fresh session whose prior is the last W - c frames
    O, L = oracle.chunk_attention(pool, 0, [sid], [3], q, k, v, 0.25)
    fresh = make_oracle_pool(shape)
    f = fresh.open()
    lo = (n_frames - (Wn - 3)) * T
    feed_prior(fresh, f, [ks[lo:]], [vs[lo:]], T, frames_per_append=2)
    O2, L2 = oracle.chunk_attention(fresh, 0, [f], [3], q, k, v, 0.25)
    np.testing.assert_array_equal(O, O2)
    np.testing.assert_array_equal(L, L2)


# ---- P11: hand-worked Tiny allocator trace -------------------------------------------------------------------
def _parse_golden(path):
    vals = {}
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        key, rest = line.split(None, 1)
        if "A:" in rest:
            a, b = rest.split("B:")
            a = a.replace("A:", "").strip()
            vals[key] = ([] if a == "-" else [int(x) for x in a.split()], [int(x) for x in b.split()])
        else:
            vals[key] = [int(x) for x in rest.split()]
    return vals


def test_p11_tiny_allocator_trace(golden_dir):
    g = _parse_golden(os.path.join(golden_dir, "tiny_allocator_trace.txt"))
    w = synth.tiny()
    assert w.free_order.tolist() == g["free_order"]
    pool = make_oracle_pool(w.shape, w.free_order)
    a, b = pool.open(), pool.open()
    assert (a, b) == (0, 1)
    ts = [synth.draw_session_tensors(w.rng, w.shape, s) for s in w.sessions]
    feed_prior(pool, b, ts[1]["prior_k"], ts[1]["prior_v"], w.shape.frame_tokens)
    assert (pool.page_table(a), pool.page_table(b)) == g["after_prior"]
    k = np.concatenate([t["k"] for t in ts])
    v = np.concatenate([t["v"] for t in ts])
    pool.append(0, [a, b], [2, 2], k, v)
    assert (pool.page_table(a), pool.page_table(b)) == g["after_append"]
    assert list(pool.free) == g["free_after_append"]
    pool.suspend(b)
    assert list(pool.free) == g["free_after_suspend"]
    pool.resume(b)
    assert (pool.page_table(a), pool.page_table(b)) == g["after_resume"]
    assert list(pool.free) == g["free_after_resume"]


# ---- P12: distribution sanity at a larger shape -----------------------------------------------------------
def test_p12_distribution_sanity():
    shape = synth.PoolShape(1, 2, 128, 64, 64, 200, 0, 2)
    T = shape.frame_tokens
    rng = np.random.default_rng(21)
    pool = make_oracle_pool(shape)
    sid = pool.open()
    feed_prior(pool, sid, [draw(rng, 9 * T, shape)], [draw(rng, 9 * T, shape)], T)
    q, k, v = (draw(rng, 3 * T, shape) for _ in range(3))
    scale = np.float32(1 / np.sqrt(128))
    O, L = oracle.chunk_attention(pool, 0, [sid], [3], q, k, v, scale)
    # last frame rows see n = 12*T keys: logits ~ N(0,1) => LSE ~ log(n) + 1/2, output std ~ sqrt(e/n)
    n = 12 * T
    rows = slice(2 * T, 3 * T)
    assert abs(L[rows].mean() - (np.log(n) + 0.5)) < 0.05
    assert abs(O[rows].std() / np.sqrt(np.e / n) - 1) < 0.1


# ---- error behaviour of the state machine (R12, R13, R16, R18) -------------------------------------------------
def test_state_machine_errors():
    shape = small_shape(n_pages=4, max_sessions=2, window_frames=4)
    T = shape.frame_tokens
    rng = np.random.default_rng(22)
    pool = make_oracle_pool(shape, host_pages=2)
    a, b = pool.open(), pool.open()
    with pytest.raises(oracle.OracleError) as e:
        pool.open()
    assert e.value.kind == oracle.CAPACITY
    k1 = draw(rng, T, shape)
    with pytest.raises(oracle.OracleError) as e:
        pool.append(0, [a, a], [1, 1], np.concatenate([k1, k1]), np.concatenate([k1, k1]))
    assert e.value.kind == oracle.INVALID
    with pytest.raises(oracle.OracleError) as e:
        pool.append(0, [a], [5], draw(rng, 5 * T, shape), draw(rng, 5 * T, shape))
    assert e.value.kind == oracle.INVALID
    pool.append(0, [a], [4], draw(rng, 4 * T, shape), draw(rng, 4 * T, shape))     # 20 tokens = 3 pages
    free_before, pt_before = list(pool.free), pool.page_table(a)
    with pytest.raises(oracle.OracleError) as e:                                   # needs 2, only 1 free
        pool.append(0, [b], [2], draw(rng, 2 * T, shape), draw(rng, 2 * T, shape))
    assert e.value.kind == oracle.NO_PAGES
    assert list(pool.free) == free_before and pool.page_table(a) == pt_before and pool.page_table(b) == []
    with pytest.raises(oracle.OracleError) as e:
        pool.suspend(a)                                                            # 3 pages > host cap 2
    assert e.value.kind == oracle.NO_HOST
    with pytest.raises(oracle.OracleError) as e:
        pool.resume(a)
    assert e.value.kind == oracle.STATE
    pool.close(a)
    assert len(pool.free) == 4
    with pytest.raises(oracle.OracleError) as e:
        pool.close(a)
    assert e.value.kind == oracle.STATE
    assert pool.open() == a                                                        # lowest free id reused


def test_page_demand_is_never_negative():
    """R14: page growth on append is idempotent and a table never shrinks, so a session that already holds more pages than
    a later, smaller append needs contributes ZERO demand - it must not offset another session's demand in the all-or-nothing
    check (found by the random-operation test: the unclamped sum let an append through that then ran out of pages)."""
    shape = small_shape(n_pages=6, max_sessions=2)            # B = 8, T = 5
    T = shape.frame_tokens
    rng = np.random.default_rng(23)
    pool = make_oracle_pool(shape)
    a, b = pool.open(), pool.open()
    pool.append(0, [a], [6], draw(rng, 6 * T, shape), draw(rng, 6 * T, shape), commit=False)   # 30 tokens: 4 pages, P stays 0
    assert len(pool.page_table(a)) == 4 and len(pool.free) == 2
    snap = (list(pool.free), pool.page_table(a), pool.page_table(b))
    # a needs ceil(5 / 8) = 1 page and holds 4 (demand 0, not -3); b needs ceil(20 / 8) = 3 > 2 free
    k = draw(rng, 5 * T, shape)
    with pytest.raises(oracle.OracleError) as e:
        pool.append(0, [a, b], [1, 4], k, k)
    assert e.value.kind == oracle.NO_PAGES
    assert snap == (list(pool.free), pool.page_table(a), pool.page_table(b))
    pool.append(0, [a, b], [1, 3], k[:4 * T], k[:4 * T])      # b: 15 tokens = 2 pages: fits exactly
    assert len(pool.free) == 0 and len(pool.page_table(a)) == 4 and len(pool.page_table(b)) == 2


# ---- P13: attention_rows — the function behind every sampled-row parity check and the timed CPU baseline ----
def _rolled_multihead_pool():
    """W binding (P + c > W), o != 0, permuted pages, 3 heads, a second session sharing the pool."""
    shape = small_shape(n_heads=3, head_dim=16, window_frames=6, page_tokens=8, frame_tokens=5, n_pages=48)
    T = shape.frame_tokens
    rng = np.random.default_rng(31)
    pool = make_oracle_pool(shape, rng.permutation(shape.n_pages))
    other, sid = pool.open(), pool.open()
    prior_k, prior_v = draw(rng, 11 * T, shape), draw(rng, 11 * T, shape)
    fed = 0
    for c in (3, 2, 3, 3):                                   # 11 frames through a 6-frame window: 5 evicted, o = 25 % 8 = 1
        sl = slice(fed * T, (fed + c) * T)
        pool.append(0, [sid], [c], prior_k[sl], prior_v[sl])
        pool.append(0, [other], [1], draw(rng, T, shape), draw(rng, T, shape))   # interleaves the page ids
        fed += c
    info = pool.info(sid)
    assert info["frames"] == 6 and info["head_off"] == 1
    return shape, pool, sid, other, prior_k, prior_v, rng


def _same_up_to_blas_order(a, b):
    # the two entry points hand numpy's fp64 matmul different row counts (gemv / gemm blocking differs), so the sums
    # are taken in a different order: a few ulp, nothing a wrong index or mask could hide behind
    np.testing.assert_allclose(a, b, rtol=1e-12, atol=1e-14)


def test_p13_attention_rows_equals_chunk_attention():
    # (a) rolled-window multi-head pool: arbitrary unsorted, repeated row subsets, every head, O and LSE
    shape, pool, sid, other, _, _, rng = _rolled_multihead_pool()
    T, H = shape.frame_tokens, shape.n_heads
    c = 3
    q, k, v = (draw(rng, c * T, shape) for _ in range(3))
    qo, ko, vo = (draw(rng, 2 * T, shape) for _ in range(3))
    # the session sits SECOND in a two-session batch, so the packed offset of its chunk is not 0
    qa, ka, va = (np.concatenate([x, y]) for x, y in ((qo, q), (ko, k), (vo, v)))
    O, LSE = oracle.chunk_attention(pool, 0, [other, sid], [2, c], qa, ka, va, np.float32(0.21))
    off = 2 * T
    for rows in ([0], [c * T - 1], [7, 2, 11, 2, 14, 0, 5], list(range(c * T))[::-1], rng.permutation(c * T)[:6].tolist()):
        for h in range(H):
            o, l = oracle.attention_rows(pool, 0, sid, c, q, k, v, np.float32(0.21), h, rows)
            _same_up_to_blas_order(o, O[off + np.asarray(rows), h])
            _same_up_to_blas_order(l, LSE[off + np.asarray(rows), h])
    # ... and on Tiny (no window, D = 64, B = T = 16)
    w = synth.tiny()
    tpool, sids, tensors, tq, tk, tv = build_oracle_workload(w)
    cf = [s.chunk_frames for s in w.sessions]
    TO, TL = oracle.chunk_attention(tpool, 0, sids, cf, tq, tk, tv, w.scale)
    off = 0
    for s, spec, t in zip(sids, w.sessions, tensors):
        Cn = spec.chunk_frames * w.shape.frame_tokens
        rows = [Cn - 1, 0, 17, 3, 16, 15]
        for h in range(w.shape.n_heads):
            o, l = oracle.attention_rows(tpool, 0, s, spec.chunk_frames, t["q"], t["k"], t["v"], w.scale, h, rows)
            _same_up_to_blas_order(o, TO[off + np.asarray(rows), h])
            _same_up_to_blas_order(l, TL[off + np.asarray(rows), h])
        off += Cn


def test_p13_attention_rows_brute_force():
    # (b) hand-picked rows against explicit loops over the LOGICAL arrays (as drawn: no page table, no oracle helper):
    # a row of the first frame, one of the middle frame (last token of it) and the very last row, a different head each.
    shape, pool, sid, _, prior_k, prior_v, rng = _rolled_multihead_pool()
    T, D, Wn = shape.frame_tokens, shape.head_dim, shape.window_frames
    c = 3
    q, k, v = (draw(rng, c * T, shape) for _ in range(3))
    scale = np.float32(0.37)
    n_fed = prior_k.shape[0] // T                      # 11 frames were fed; the cache holds the last 6; W - c = 3 are visible
    vis_lo = (n_fed - (Wn - c)) * T
    Kp, Vp = W64(prior_k)[vis_lo:], W64(prior_v)[vis_lo:]
    Q, Kc, Vc = W64(q), W64(k), W64(v)
    assert Kp.shape[0] == (Wn - c) * T
    for row, head in ((2, 0), (2 * T - 1, 1), (c * T - 1, 2)):
        den, num = 0.0, [0.0] * D
        keys = [(Kp[j, head], Vp[j, head]) for j in range(Kp.shape[0])]
        keys += [(Kc[j, head], Vc[j, head]) for j in range(c * T) if j // T <= row // T]
        for kk, vv in keys:
            dot = 0.0
            for d in range(D):
                dot += Q[row, head, d] * kk[d]
            e = math.exp(float(scale) * dot)
            den += e
            for d in range(D):
                num[d] += e * vv[d]
        o, l = oracle.attention_rows(pool, 0, sid, c, q, k, v, scale, head, [row])
        np.testing.assert_allclose(o[0], np.array(num) / den, rtol=1e-11, atol=1e-13)
        assert abs(l[0] - math.log(den)) < 1e-11
    # a transposed head axis or rows-as-positions slip would show here: the three rows differ from each other's heads
    o_wrong, _ = oracle.attention_rows(pool, 0, sid, c, q, k, v, scale, 1, [2])
    o_right, _ = oracle.attention_rows(pool, 0, sid, c, q, k, v, scale, 0, [2])
    assert np.abs(o_wrong - o_right).max() > 1e-3


# ---- P14: the bf16 conversions against a library (torch.bfloat16 on CPU) ----------------------------------
def test_p14_bf16_widening_all_patterns_vs_torch():
    from oracle.attention import _widen
    bits = np.arange(65536, dtype=np.uint32).astype(np.uint16)
    ref32 = torch.from_numpy(bits.view(np.int16)).view(torch.bfloat16).to(torch.float32).numpy()
    ref64 = torch.from_numpy(bits.view(np.int16)).view(torch.bfloat16).to(torch.float64).numpy()
    for got, ref in ((synth.bf16_bits_to_f32(bits), ref32), (synth.bf16_bits_to_f64(bits), ref64), (_widen(bits), ref64)):
        assert got.dtype == ref.dtype
        nan = np.isnan(ref)
        assert np.array_equal(np.isnan(got), nan)
        # bit-for-bit on every non-NaN pattern (incl. +-0, subnormals, +-inf)
        view = np.uint32 if ref.dtype == np.float32 else np.uint64
        assert np.array_equal(got[~nan].view(view), ref[~nan].view(view))
    assert int(np.isnan(ref32).sum()) == 2 * 127                       # sanity: the NaN patterns were in the sweep


def test_p14_f32_to_bf16_rne_vs_torch():
    rng = np.random.default_rng(41)
    x = rng.standard_normal(1_000_000, dtype=np.float32) * np.float32(3.0)
    # exact ties (low 16 bits == 0x8000) with even and odd kept mantissas, values just below / above a tie, a mantissa carry
    # into the exponent (0x3F7FFFFF -> 1.0), signed zeros, subnormals, the largest finite fp32 that stays finite in bf16
    u = rng.integers(0, 0x7F000000, size=200_000, dtype=np.uint32)
    ties = (u & np.uint32(0xFFFF0000)) | np.uint32(0x8000)
    near = np.concatenate([ties - np.uint32(1), ties + np.uint32(1)])
    special = np.array([0x3F7FFFFF, 0x3F7F8000, 0x3F808000, 0x3F818000, 0x00000000, 0x80000000, 0x00000001, 0x00008000,
                        0x00018000, 0x7F7F0000, 0x7F7F7FFF, 0xBF7FFFFF], dtype=np.uint32)
    allu = np.concatenate([x.view(np.uint32), ties, ties | np.uint32(0x80000000), near, special])
    xs = allu.view(np.float32)
    assert np.isfinite(xs).all()
    ref = torch.from_numpy(xs.copy()).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    got = synth.f32_to_bf16_bits(xs)
    assert np.array_equal(got, ref)
    # round trip: widening the rounded value and rounding again is the identity
    assert np.array_equal(synth.f32_to_bf16_bits(synth.bf16_bits_to_f32(got)), got)
