"""Parity of the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.
Integer / byte work is bit-exact; attention is within max-abs 2e-2 and rel-L2 5e-3 of fp64
(BASELINE.json north_star)."""
import numpy as np
import pytest
import torch

import oracle
import synth
from helpers import DualPool, bits_to_dev, dev_to_bits, rel_l2

pytestmark = pytest.mark.gpu


def shape_of(**kw):
    d = dict(n_layers=1, n_heads=2, head_dim=128, page_tokens=256, n_pages=64, frame_tokens=200,
             window_frames=0, max_sessions=8)
    d.update(kw)
    return synth.PoolShape(**d)


def draw(rng, n, shape):
    return synth.draw_bits(rng, n, shape.n_heads, shape.head_dim)


def scale_of(shape):
    return np.float32(1.0 / np.sqrt(np.float32(shape.head_dim)))


# ---- configs[0]: Tiny, the whole sequence of BASELINE.json --------------------------------------------------
def test_config0_tiny_full_sequence():
    w = synth.tiny()
    dp = DualPool(w.shape, w.free_order, host_pages=8)
    sids = [dp.open() for _ in w.sessions]
    tensors = [synth.draw_session_tensors(w.rng, w.shape, s) for s in w.sessions]
    dp.feed_prior(sids[1], tensors[1]["prior_k"], tensors[1]["prior_v"])
    dp.check_state(sids)
    q, k, v = (np.concatenate([t[n] for t in tensors]) for n in ("q", "k", "v"))
    cf = [s.chunk_frames for s in w.sessions]
    dp.attention(0, sids, cf, q, k, v, w.scale)
    dp.append(0, sids, cf, k, v)
    dp.check_state(sids)
    dp.suspend(sids[1])
    dp.check_state(sids)
    dp.resume(sids[1])
    dp.check_state(sids)
    assert dp.g.ts_session_page_table(sids[1]) == [5, 14, 12, 6, 9]       # tests/golden/tiny_allocator_trace.txt
    dp.attention(0, sids, [1, 1], q[:32], k[:32], v[:32], w.scale)        # after the round trip


# ---- configs[1]: Wan-1.3B-shaped single session, full oracle ------------------------------------------------
def test_config1_wan13b_single():
    w = synth.wan13b_single()
    dp = DualPool(w.shape, w.free_order)
    sid = dp.open()
    t = synth.draw_session_tensors(w.rng, w.shape, w.sessions[0])
    dp.feed_prior(sid, t["prior_k"], t["prior_v"])
    dp.check_state([sid])
    o_gpu, o_ref = dp.attention(0, [sid], [3], t["q"], t["k"], t["v"], w.scale)
    # P12: output std ~ sqrt(e/n) for the last frame's rows
    n = 9 * 1560
    assert abs(o_gpu[2 * 1560:].std() / np.sqrt(np.e / n) - 1) < 0.1
    dp.append(0, [sid], [3], t["k"], t["v"])
    dp.check_state([sid])


# ---- ragged coalesced batch: different priors, window clamp, evicted head offset, T not a multiple of 128 --
@pytest.mark.parametrize("head_dim,page_tokens", [(128, 256), (64, 256), (128, 64), (64, 16), (128, 1024)])
def test_ragged_batch_window_and_offsets(head_dim, page_tokens):
    shape = shape_of(head_dim=head_dim, page_tokens=page_tokens, n_heads=3, frame_tokens=203, window_frames=7,
                     n_pages=max(64, 8 * 1800 // page_tokens), max_sessions=8)
    rng = np.random.default_rng(100 + head_dim + page_tokens)
    dp = DualPool(shape, rng.permutation(shape.n_pages), host_pages=shape.n_pages)
    T = shape.frame_tokens
    priors = [0, 2, 5, 7, 11]            # 7 and 11 frames: window is full / has rolled (head offset != 0)
    chunks = [3, 1, 2, 3, 3]
    sids = [dp.open() for _ in priors]
    for sid, P in zip(sids, priors):
        if P:
            dp.feed_prior(sid, [draw(rng, P * T, shape)], [draw(rng, P * T, shape)])
    assert dp.g.ts_session_info(sids[4])["head_off"] != 0
    dp.check_state(sids)
    total = sum(chunks) * T
    q, k, v = (draw(rng, total, shape) for _ in range(3))
    dp.attention(0, sids, chunks, q, k, v, scale_of(shape))
    dp.append(0, sids, chunks, k, v)
    dp.check_state(sids)
    # suspend two sessions, run the rest, resume, run all again (event ordering across streams)
    dp.suspend(sids[2])
    dp.suspend(sids[4])
    rest = [sids[0], sids[1], sids[3]]
    q2, k2, v2 = (draw(rng, 3 * T, shape) for _ in range(3))
    dp.attention(0, rest, [1, 1, 1], q2, k2, v2, scale_of(shape))
    dp.resume(sids[4])
    dp.resume(sids[2])
    dp.check_state(sids)
    dp.attention(0, sids, chunks, q, k, v, scale_of(shape))


# ---- small / degenerate shapes ------------------------------------------------------------------------------
@pytest.mark.parametrize("frame_tokens,chunk,prior", [(1, 5, 0), (1, 1, 0), (7, 1, 0), (128, 2, 1), (129, 3, 2),
                                                       (100, 1, 0), (300, 1, 3), (257, 2, 0)])
def test_degenerate_shapes(frame_tokens, chunk, prior):
    shape = shape_of(frame_tokens=frame_tokens, page_tokens=32, n_pages=128)
    rng = np.random.default_rng(7 * frame_tokens + chunk)
    dp = DualPool(shape, rng.permutation(shape.n_pages))
    sid = dp.open()
    T = frame_tokens
    if prior:
        dp.feed_prior(sid, [draw(rng, prior * T, shape)], [draw(rng, prior * T, shape)])
    q, k, v = (draw(rng, chunk * T, shape) for _ in range(3))
    dp.attention(0, [sid], [chunk], q, k, v, np.float32(0.11))
    dp.append(0, [sid], [chunk], k, v)
    dp.check_state([sid])


def test_single_visible_key_and_constant_v_on_gpu():
    shape = shape_of(frame_tokens=1, page_tokens=16, n_pages=16)
    rng = np.random.default_rng(5)
    dp = DualPool(shape)
    sid = dp.open()
    q, k, v = (draw(rng, 4, shape) for _ in range(3))
    o_gpu, _ = dp.attention(0, [sid], [4], q, k, v, np.float32(0.3))
    np.testing.assert_array_equal(o_gpu[0], synth.bf16_bits_to_f64(v)[0])          # P3: exactly v_0
    u = draw(rng, 1, shape)
    vc = np.repeat(u, 4, axis=0)
    o_gpu, _ = dp.attention(0, [sid], [4], q, k, vc, np.float32(0.3))
    np.testing.assert_allclose(o_gpu, np.broadcast_to(synth.bf16_bits_to_f64(u), o_gpu.shape), rtol=2 ** -8)


# ---- multi-layer step (configs[3]-shaped, scaled down): growth once, commit on the last layer --------------
def test_multilayer_commit_on_last_layer():
    shape = shape_of(n_layers=3, n_heads=5, frame_tokens=150, window_frames=6, n_pages=64, page_tokens=128)
    rng = np.random.default_rng(9)
    dp = DualPool(shape, rng.permutation(shape.n_pages), host_pages=40)
    T = shape.frame_tokens
    sids = [dp.open(), dp.open()]
    for step in range(3):                      # 3 chunk steps of 3 frames: window (6) rolls on the third
        qs = [draw(rng, 6 * T, shape) for _ in range(3)]
        ks = [draw(rng, 6 * T, shape) for _ in range(3)]
        vs = [draw(rng, 6 * T, shape) for _ in range(3)]
        for layer in range(3):
            dp.attention(layer, sids, [3, 3], qs[layer], ks[layer], vs[layer], scale_of(shape))
            dp.append(layer, sids, [3, 3], ks[layer], vs[layer], commit=(layer == 2))
        dp.check_state(sids)
    dp.suspend(sids[0])
    dp.check_state(sids)
    dp.resume(sids[0])
    dp.check_state(sids)


# ---- batch-composition invariance on the GPU: bitwise ------------------------------------------------------
def test_gpu_batch_composition_invariance():
    shape = shape_of(n_heads=2, frame_tokens=180, window_frames=9, page_tokens=64, n_pages=256)
    rng = np.random.default_rng(11)
    T = shape.frame_tokens
    priors = {0: 4, 1: 0, 2: 6}
    pk = {s: draw(rng, P * T, shape) for s, P in priors.items()}
    pv = {s: draw(rng, P * T, shape) for s, P in priors.items()}
    ch = {s: tuple(draw(rng, 3 * T, shape) for _ in range(3)) for s in priors}

    def run(order):
        dp = DualPool(shape, np.random.default_rng(1).permutation(shape.n_pages))
        sid = {s: dp.open() for s in order}
        for s in order:
            if priors[s]:
                dp.feed_prior(sid[s], [pk[s]], [pv[s]])
        q, k, v = (np.concatenate([ch[s][i] for s in order]) for i in range(3))
        dq, dk, dv = bits_to_dev(q), bits_to_dev(k), bits_to_dev(v)
        out = torch.empty_like(dq)
        dp.g.ts_chunk_attention(0, [sid[s] for s in order], [3] * len(order), dq, dk, dv, out, None, 0.09)
        torch.cuda.synchronize()
        bits = dev_to_bits(out)
        return {s: bits[i * 3 * T:(i + 1) * 3 * T] for i, s in enumerate(order)}

    full = run([0, 1, 2])
    for order in ([2, 1, 0], [1], [0, 2]):
        part = run(order)
        for s in order:
            np.testing.assert_array_equal(part[s], full[s])


# ---- error behaviour through the ABI ---------------------------------------------------------------------------
def test_error_codes_and_all_or_nothing():
    import paper_2606_19271_b200 as tc
    shape = shape_of(n_pages=8, max_sessions=2, window_frames=4, frame_tokens=100, page_tokens=64)
    rng = np.random.default_rng(13)
    dp = DualPool(shape, host_pages=2)
    a, b = dp.open(), dp.open()
    with pytest.raises(tc.TurboChunkError) as e:
        dp.g.ts_session_open()
    assert e.value.code == tc.TS_ERR_CAPACITY
    k1 = bits_to_dev(draw(rng, 200, shape))
    with pytest.raises(tc.TurboChunkError) as e:
        dp.g.ts_kv_append(0, [a, a], [1, 1], k1, k1)
    assert e.value.code == tc.TS_ERR_INVALID
    with pytest.raises(tc.TurboChunkError) as e:
        dp.g.ts_kv_append(0, [a], [5], k1, k1)
    assert e.value.code == tc.TS_ERR_INVALID
    with pytest.raises(tc.TurboChunkError) as e:
        dp.g.ts_kv_append(3, [a], [1], k1, k1)
    assert e.value.code == tc.TS_ERR_INVALID
    big = draw(rng, 400, shape)
    dp.append(0, [a], [4], big, big)                       # 400 tokens = 7 pages of 64
    free_before = dp.g.ts_pool_free_list()
    with pytest.raises(tc.TurboChunkError) as e:           # needs 2 pages, 1 free
        dp.g.ts_kv_append(0, [b], [1], k1, k1)
    assert e.value.code == tc.TS_ERR_NO_PAGES
    with pytest.raises(oracle.OracleError) as eo:
        dp.o.append(0, [b], [1], big[:100], big[:100])
    assert eo.value.kind == oracle.NO_PAGES
    assert dp.g.ts_pool_free_list() == free_before and dp.g.ts_session_page_table(b) == []
    with pytest.raises(tc.TurboChunkError) as e:
        dp.g.ts_session_suspend(a)                         # 7 pages > 2 host pages
    assert e.value.code == tc.TS_ERR_NO_HOST
    with pytest.raises(tc.TurboChunkError) as e:
        dp.g.ts_session_resume(a)
    assert e.value.code == tc.TS_ERR_STATE
    q = bits_to_dev(draw(rng, 100, shape))
    out = torch.empty_like(q)
    with pytest.raises(tc.TurboChunkError) as e:
        dp.g.ts_chunk_attention(0, [a], [1], q, q, q, out, None, -1.0)
    assert e.value.code == tc.TS_ERR_INVALID
    dp.g.ts_chunk_attention(0, [], [], None, None, None, None, None, 1.0)     # n == 0: no-op
    dp.g.ts_kv_append(0, [], [], None, None)
    dp.close(a)
    dp.check_state([b])
    with pytest.raises(tc.TurboChunkError) as e:
        dp.g.ts_session_close(a)
    assert e.value.code == tc.TS_ERR_STATE
    assert dp.open() == a


# ---- configs[4]-style churn, scaled down: integers at every step, KV bytes and attention sampled -----------
def test_churn_scaled_down():
    shape = shape_of(n_heads=2, head_dim=128, frame_tokens=40, window_frames=9, page_tokens=16,
                     n_pages=12 * 36, max_sessions=40)
    steps = synth.churn_script(seed=4, n_steps=60, cap=12, mean_off=2.0, mean_on=9.0)
    rng = np.random.default_rng(4)
    dp = DualPool(shape, rng.permutation(shape.n_pages), host_pages=40 * 36)
    T = shape.frame_tokens
    sid_of = {}
    for it, ev in enumerate(steps):
        for u in ev["suspend"]:
            dp.suspend(sid_of[u])
        for u in ev["resume"]:
            dp.resume(sid_of[u])
        for u in ev["open"]:
            sid_of[u] = dp.open()
        batch = [sid_of[u] for u in ev["batch"]]
        cf = ev["chunk_frames"]
        if batch:
            n_tok = sum(cf) * T
            q, k, v = (draw(rng, n_tok, shape) for _ in range(3))
            if it % 5 == 0:
                dp.attention(0, batch, cf, q, k, v, scale_of(shape))
            dp.append(0, batch, cf, k, v)
        for u in ev["close"]:
            dp.close(sid_of.pop(u))
        dp.check_state(list(sid_of.values()), kv=(it % 10 == 9))
    assert max(len(e["batch"]) for e in steps) > 8


# ---- configs[2] at full size, in the launch configuration bench.py times: sampled rows ----------------------
def test_config2_full_size_sampled_rows():
    w = synth.wan13b_batch()
    shape = w.shape
    T, H, D = shape.frame_tokens, shape.n_heads, shape.head_dim
    dp = DualPool(shape, w.free_order)
    gen = torch.Generator(device="cuda")
    gen.manual_seed(w.seed)
    sids = [dp.open() for _ in w.sessions]
    from synth.draw import draw_bits_torch
    chunks = []
    for sid, spec in zip(sids, w.sessions):
        P = spec.prior_frames
        for f in range(0, P, 3):
            dk = draw_bits_torch(gen, 3 * T, H, D, "cuda")
            dv = draw_bits_torch(gen, 3 * T, H, D, "cuda")
            dp.append(0, [sid], [3], dev_to_bits(dk), dev_to_bits(dv), dev=(dk, dv))
        chunks.append(tuple(draw_bits_torch(gen, 3 * T, H, D, "cuda") for _ in range(3)))
    dp.check_state(sids, kv=False)
    dq, dk, dv = (torch.cat([c[i] for c in chunks]) for i in range(3))
    out = torch.full_like(dq, float("nan"))
    lse = torch.empty(dq.shape[:2], dtype=torch.float32, device="cuda")
    cf = [3] * len(sids)
    dp.g.ts_chunk_attention(0, sids, cf, dq, dk, dv, out, lse, float(w.scale))
    torch.cuda.synchronize()
    o_gpu = out.double().cpu().numpy()
    assert np.isfinite(o_gpu).all()
    rs = np.random.default_rng(0)
    C = 3 * T
    errs, refs = [], []
    for b, sid in enumerate(sids):
        qb, kb, vb = (dev_to_bits(c) for c in chunks[b])
        for _ in range(3):
            h = int(rs.integers(0, H))
            rows = np.unique(np.concatenate([rs.integers(0, C, size=24), [0, T - 1, T, 2 * T - 1, 2 * T, C - 1]]))
            o_ref, l_ref = oracle.attention_rows(dp.o, 0, sid, 3, qb, kb, vb, w.scale, h, rows)
            got = o_gpu[b * C + rows, h]
            errs.append(got - o_ref)
            refs.append(o_ref)
            assert np.abs(lse[b * C + rows, h].double().cpu().numpy() - l_ref).max() <= 2e-3
    err, ref = np.concatenate(errs), np.concatenate(refs)
    assert np.abs(err).max() <= 2e-2
    assert np.linalg.norm(err) / np.linalg.norm(ref) <= 5e-3
    # the launch configuration bench.py times: ts_chunk_step, attention + append in ONE launch.  flags = 0 (as in the timed
    # loop) leaves the state alone and must reproduce the attention-only output bit for bit (every work item is computed
    # the same way whichever cluster takes it); with TS_COMMIT the appended bytes read back bit-exact (a property that
    # holds at any size) and the page tables match the oracle's.
    import paper_2606_19271_b200 as tc
    out2 = torch.full_like(dq, float("nan"))
    lse2 = torch.empty_like(lse)
    dp.g.ts_chunk_step(0, sids, cf, dq, dk, dv, out2, lse2, float(w.scale), 0)
    torch.cuda.synchronize()
    assert torch.equal(out.view(torch.int16), out2.view(torch.int16)) and torch.equal(lse, lse2)
    out3 = torch.full_like(dq, float("nan"))
    dp.o.append(0, sids, cf, dev_to_bits(dk), dev_to_bits(dv))
    dp.g.ts_chunk_step(0, sids, cf, dq, dk, dv, out3, None, float(w.scale), tc.TS_COMMIT)
    torch.cuda.synchronize()
    assert torch.equal(out.view(torch.int16), out3.view(torch.int16))
    dp.check_state(sids, kv=False)
    dp.check_state(sids[:2], kv=True)


# ---- configs[3] (Wan-14B shape: 4 sessions x 40 heads, full 21-frame window): sampled rows on 2 distinct layers ----
def _sampled_rows_check(dp, layer, sids, chunks, o_gpu, lse, w, rs, heads_per_session=2, rows_per_head=16):
    shape = w.shape
    T, H = shape.frame_tokens, shape.n_heads
    C = 3 * T
    errs, refs = [], []
    for b, sid in enumerate(sids):
        qb, kb, vb = (dev_to_bits(c) for c in chunks[b])
        for _ in range(heads_per_session):
            h = int(rs.integers(0, H))
            rows = np.unique(np.concatenate([rs.integers(0, C, size=rows_per_head), [0, T - 1, T, 2 * T, C - 1]]))
            o_ref, l_ref = oracle.attention_rows(dp.o, layer, sid, 3, qb, kb, vb, w.scale, h, rows)
            errs.append(o_gpu[b * C + rows, h] - o_ref)
            refs.append(o_ref)
            assert np.abs(lse[b * C + rows, h].double().cpu().numpy() - l_ref).max() <= 2e-3
    err, ref = np.concatenate(errs), np.concatenate(refs)
    assert np.abs(err).max() <= 2e-2
    assert np.linalg.norm(err) / np.linalg.norm(ref) <= 5e-3


def test_config3_wan14b_two_layers_sampled_rows():
    from synth.draw import draw_bits_torch
    w = synth.wan14b_batch(n_layers=2)
    shape = w.shape
    T, H, D = shape.frame_tokens, shape.n_heads, shape.head_dim
    dp = DualPool(shape, w.free_order)
    gen = torch.Generator(device="cuda")
    gen.manual_seed(w.seed)
    sids = [dp.open() for _ in w.sessions]
    for sid, spec in zip(sids, w.sessions):
        for f in range(0, spec.prior_frames, 3):
            for layer in range(2):
                dk = draw_bits_torch(gen, 3 * T, H, D, "cuda")
                dv = draw_bits_torch(gen, 3 * T, H, D, "cuda")
                dp.append(layer, [sid], [3], dev_to_bits(dk), dev_to_bits(dv), commit=(layer == 1), dev=(dk, dv))
    dp.check_state(sids, kv=False)
    assert all(dp.g.ts_session_info(s)["frames"] == 18 for s in sids)
    rs = np.random.default_rng(3)
    cf = [3] * len(sids)
    for layer in range(2):
        chunks = [tuple(draw_bits_torch(gen, 3 * T, H, D, "cuda") for _ in range(3)) for _ in sids]
        dq, dk, dv = (torch.cat([c[i] for c in chunks]) for i in range(3))
        out = torch.full_like(dq, float("nan"))
        lse = torch.empty(dq.shape[:2], dtype=torch.float32, device="cuda")
        dp.g.ts_chunk_attention(layer, sids, cf, dq, dk, dv, out, lse, float(w.scale))
        torch.cuda.synchronize()
        o_gpu = out.double().cpu().numpy()
        assert np.isfinite(o_gpu).all()
        _sampled_rows_check(dp, layer, sids, chunks, o_gpu, lse, w, rs)
        del out, o_gpu
    # append + commit rolls the full window (21 -> 24 -> 21 frames): page tables, offsets and sampled KV bytes
    dp.append(0, sids, cf, dev_to_bits(dk), dev_to_bits(dv), commit=False, dev=(dk, dv))
    dp.append(1, sids, cf, dev_to_bits(dk), dev_to_bits(dv), commit=True, dev=(dk, dv))
    dp.check_state(sids[:1], kv=True)
    dp.check_state(sids[1:], kv=False)
    dp.g.close()


def test_config3_forty_layers_back_to_back():
    """configs[3] at NL=40 (107 GB of KV slab): layer addressing and the 40-layer chunk step.  No oracle at this
    size - checked by properties: identical K/V in every layer gives bit-identical attention output on every layer,
    appended bytes read back bit-exact from the last layer, other layers untouched."""
    import time
    from synth.draw import draw_bits_torch
    from paper_2606_19271_b200 import TS_COMMIT, TurboChunkPool
    torch.cuda.empty_cache()
    free_b, _ = torch.cuda.mem_get_info()
    w = synth.wan14b_batch(n_layers=40)
    sh = w.shape
    T, H, D, NL = sh.frame_tokens, sh.n_heads, sh.head_dim, sh.n_layers
    need = sh.n_pages * NL * 2 * H * sh.page_tokens * D * 2
    if free_b < need + (8 << 30):
        pytest.skip(f"needs {need >> 30} GiB of free HBM for the 40-layer slab")
    pool = TurboChunkPool(NL, H, D, sh.page_tokens, sh.n_pages, T, sh.window_frames, sh.max_sessions, free_order=w.free_order)
    gen = torch.Generator(device="cuda")
    gen.manual_seed(w.seed)
    sids = [pool.ts_session_open() for _ in w.sessions]
    cf = [3] * len(sids)
    n_tok = 3 * T * len(sids)
    for f in range(0, 18, 3):
        dk = draw_bits_torch(gen, n_tok, H, D, "cuda")
        dv = draw_bits_torch(gen, n_tok, H, D, "cuda")
        for layer in range(NL):
            pool.ts_kv_append(layer, sids, cf, dk, dv, TS_COMMIT if layer == NL - 1 else 0)
    q, k, v = (draw_bits_torch(gen, n_tok, H, D, "cuda") for _ in range(3))
    outs = {}
    for layer in (0, 17, 39):
        out = torch.empty_like(q)
        pool.ts_chunk_attention(layer, sids, cf, q, k, v, out, None, float(w.scale))
        outs[layer] = out
    torch.cuda.synchronize()
    assert torch.isfinite(outs[0].float()).all()
    assert torch.equal(outs[0].view(torch.int16), outs[17].view(torch.int16))
    assert torch.equal(outs[0].view(torch.int16), outs[39].view(torch.int16))
    # one full 40-layer chunk step (attention + append per layer, commit on the last): the per-chunk latency of cfg[3]
    out = torch.empty_like(q)
    times = []
    for rep in range(3):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for layer in range(NL):
            pool.ts_chunk_attention(layer, sids, cf, q, k, v, out, None, float(w.scale))
            pool.ts_kv_append(layer, sids, cf, k, v, 0)     # flags=0: every repetition runs on the same window state
        torch.cuda.synchronize()
        times.append((time.perf_counter() - t0) * 1e3)
    flops = synth.attention_flops(sh, w.sessions) * NL
    print(f"\n[configs[3]] 40-layer chunk step: {min(times):.1f} ms best of 3 ({max(times):.1f} max), "
          f"{flops / min(times) / 1e9:.0f} TFLOP/s attention-equivalent")
    # appended bytes of the last layer read back bit-exact; layer 0 still holds the prior only
    pool.ts_kv_append(NL - 1, sids, cf, k, v, TS_COMMIT)
    gk, gv = pool.ts_gather_kv(NL - 1, sids[2])
    torch.cuda.synchronize()
    C = 3 * T
    assert torch.equal(gk[-C:].view(torch.int16), k[2 * C:3 * C].view(torch.int16))
    assert torch.equal(gv[-C:].view(torch.int16), v[2 * C:3 * C].view(torch.int16))
    assert pool.ts_session_info(sids[2])["frames"] == 21
    pool.close()
    del pool
    torch.cuda.empty_cache()


# ---- configs[4] at full size: 200-step bursty churn, Wan-1.3B attention shape, up to 32 sessions per step ----------
def test_config4_churn_full_size():
    """Page tables, free list, lengths and offsets against the oracle at EVERY step (integers); logical KV bytes and
    attention rows on sampled (step, session, head, row) tuples; suspend/resume through the pinned arena throughout.
    Prints per-chunk latency p50/max of the coalesced step (attention + append, stream completion) and offload GB/s."""
    import time
    from synth.draw import draw_bits_torch
    shape = shape_of(n_heads=12, head_dim=128, frame_tokens=1560, window_frames=21, page_tokens=256,
                     n_pages=4000, max_sessions=128)
    steps = synth.churn_script()          # seed 4, 200 steps, cap 32, MMPP 4 / 24
    rng = np.random.default_rng(4)
    dp = DualPool(shape, rng.permutation(shape.n_pages), host_pages=5400)
    gen = torch.Generator(device="cuda")
    gen.manual_seed(4)
    T, H, D = shape.frame_tokens, shape.n_heads, shape.head_dim
    C = 3 * T
    scale = scale_of(shape)
    sid_of = {}
    lat, flops, off_bytes, off_ms = [], [], 0, 0.0
    for it, ev in enumerate(steps):
        for u in ev["suspend"]:
            dp.o.suspend(sid_of[u])
        for u in ev["resume"]:
            dp.o.resume(sid_of[u])
        if ev["suspend"] or ev["resume"]:
            torch.cuda.synchronize()
            t_off = time.perf_counter()
            for u in ev["suspend"]:
                off_bytes += dp.g.ts_session_info(sid_of[u])["n_pages"] * dp.g.page_bytes
                dp.g.ts_session_suspend(sid_of[u])
            for u in ev["resume"]:
                dp.g.ts_session_resume(sid_of[u])
                off_bytes += dp.g.ts_session_info(sid_of[u])["n_pages"] * dp.g.page_bytes
            dp.g.ts_offload_sync()
            off_ms += (time.perf_counter() - t_off) * 1e3
        for u in ev["open"]:
            sid_of[u] = dp.open()
        batch = [sid_of[u] for u in ev["batch"]]
        cf = ev["chunk_frames"]
        if batch:
            n_tok = len(batch) * C
            dq, dk, dv = (draw_bits_torch(gen, n_tok, H, D, "cuda") for _ in range(3))
            out = torch.empty_like(dq)
            lse = torch.empty(dq.shape[:2], dtype=torch.float32, device="cuda")
            prior = [dp.o.info(s)["frames"] for s in batch]
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            dp.g.ts_chunk_attention(0, batch, cf, dq, dk, dv, out, lse, float(scale))
            dp.g.ts_kv_append(0, batch, cf, dk, dv)
            torch.cuda.synchronize()
            lat.append((time.perf_counter() - t0) * 1e3)
            flops.append(4 * D * H * sum(synth.attention_pairs(p, 3, T, shape.window_frames) for p in prior))
            kb, vb = dev_to_bits(dk), dev_to_bits(dv)
            if it % 20 == 3:      # sampled attention rows, before the oracle appends this chunk
                o_gpu = out.double().cpu().numpy()
                assert np.isfinite(o_gpu).all()
                qb = dev_to_bits(dq)
                errs, refs = [], []
                for b in sorted({0, len(batch) // 2, len(batch) - 1}):
                    h = int(rng.integers(0, H))
                    rows = np.unique(np.concatenate([rng.integers(0, C, size=12), [0, T, C - 1]]))
                    sl = slice(b * C, (b + 1) * C)
                    o_ref, l_ref = oracle.attention_rows(dp.o, 0, batch[b], 3, qb[sl], kb[sl], vb[sl], scale, h, rows)
                    errs.append(o_gpu[b * C + rows, h] - o_ref)
                    refs.append(o_ref)
                    assert np.abs(lse[b * C + rows, h].double().cpu().numpy() - l_ref).max() <= 2e-3
                err, ref = np.concatenate(errs), np.concatenate(refs)
                assert np.abs(err).max() <= 2e-2
                assert np.linalg.norm(err) / np.linalg.norm(ref) <= 5e-3
            dp.o.append(0, batch, cf, kb, vb, commit=True)
        for u in ev["close"]:
            dp.close(sid_of.pop(u))
        live = list(sid_of.values())
        dp.check_state(live, kv=False)
        if it % 25 == 7 and live:
            dp.check_state(live[:1] + live[-1:], kv=True)
    assert max(len(e["batch"]) for e in steps) == 32
    lat_a = np.array(lat)
    tfl = np.array(flops) / lat_a / 1e9
    print(f"\n[configs[4]] {len(lat)} served steps: per-chunk latency p50 {np.median(lat_a):.2f} ms, max {lat_a.max():.2f} ms; "
          f"attention {np.sum(flops) / np.sum(lat_a) / 1e9:.0f} TFLOP/s over the run (best step {tfl.max():.0f}); "
          f"offload {off_bytes / 1e9:.1f} GB in {off_ms:.0f} ms = {off_bytes / max(off_ms, 1e-9) / 1e6:.1f} GB/s")
    dp.g.close()


# ---- latency model l_hat(n): the sweep runs through the C ABI and is monotone in n ---------
def test_latency_model_sweep_small():
    from paper_2606_19271_b200 import latency_model
    rows = [latency_model.measure(n, 6, 4, 128, 520, 21, 256, reps=3) for n in (1, 4)]
    for attn_ms, app_ms, tfl in rows:
        assert attn_ms > 0 and app_ms > 0 and tfl > 0
    assert rows[1][0] > rows[0][0]          # four sessions take longer than one


def test_latency_model_is_linear_in_n_at_full_size():
    """l_hat(n) on the Wan-1.3B shape at the full 21-frame window (the one quantity the controllers take from the
    runtime): attention time per layer is linear in the number of co-located sessions - every n within +-10 % of the
    per-session time fitted through the sweep - and the values are in the band the B200 can produce at all (0.55-1.0 ms
    per session-layer = 1100-1700 TFLOP/s ... a plausibility band, not a performance claim)."""
    from paper_2606_19271_b200 import latency_model
    ns = (2, 4, 8, 16)
    ms = [latency_model.measure(n, 18, 12, 128, 1560, 21, 256, reps=5)[0] for n in ns]
    per = float(np.sum(np.array(ms) * np.array(ns)) / np.sum(np.array(ns) ** 2))        # least squares through the origin
    for n, t in zip(ns, ms):
        assert abs(t / (per * n) - 1.0) <= 0.10, (n, t, per)
    assert 0.55 <= per <= 1.0, per


def test_resumed_session_is_served_by_the_next_step_without_a_host_wait():
    """PAPER.md:76 (iii) "restored ... before chunk generation resumes": a full-window session is resumed while the other
    sessions' step is being enqueued and is in the NEXT step's batch.  The host never waits for the copy (both calls return in
    a small fraction of the 4 ms the 201 MB copy takes; the step's launch waits for the resume's event on the stream), and the
    output of the step that serves it matches the oracle."""
    import time
    from synth.draw import draw_bits_torch
    from paper_2606_19271_b200 import TS_COMMIT
    shape = shape_of(n_heads=12, head_dim=128, frame_tokens=1560, window_frames=21, page_tokens=256, n_pages=3 * 140,
                     max_sessions=4)
    rng = np.random.default_rng(60)
    dp = DualPool(shape, rng.permutation(shape.n_pages), host_pages=140)
    gen = torch.Generator(device="cuda")
    gen.manual_seed(60)
    T, H, D = shape.frame_tokens, shape.n_heads, shape.head_dim
    a, b = dp.open(), dp.open()
    for _ in range(6):                                           # both at the full window (18 prior frames)
        for sid in (a, b):
            dk, dv = draw_bits_torch(gen, 3 * T, H, D, "cuda"), draw_bits_torch(gen, 3 * T, H, D, "cuda")
            dp.append(0, [sid], [3], dev_to_bits(dk), dev_to_bits(dv), dev=(dk, dv))
    dp.suspend(b)
    dp.g.ts_offload_sync()
    qa, ka, va = (draw_bits_torch(gen, 3 * T, H, D, "cuda") for _ in range(3))
    qb, kb, vb = (draw_bits_torch(gen, 3 * T, H, D, "cuda") for _ in range(3))
    q2, k2, v2 = (torch.cat([x, y]) for x, y in ((qa, qb), (ka, kb), (va, vb)))
    out1, out2 = torch.empty_like(qa), torch.full_like(q2, float("nan"))
    scale = float(scale_of(shape))
    dp.o.resume(b)
    torch.cuda.synchronize()
    side = dp.g.side_stream
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.perf_counter()
    e0.record(side)
    dp.g.ts_session_resume(b)                                    # step t: the resume of b is enqueued ...
    e1.record(side)
    dp.g.ts_chunk_step(0, [a], [3], qa, ka, va, out1, None, scale, 0)          # ... while a is served
    dp.g.ts_chunk_step(0, [a, b], [3, 3], q2, k2, v2, out2, None, scale, 0)    # step t + 1 serves b
    host_ms = (time.perf_counter() - t0) * 1e3
    torch.cuda.synchronize()
    copy_ms = e0.elapsed_time(e1)
    assert copy_ms > 2.0, copy_ms                                # 201 MB over the host link
    assert host_ms < 0.5 * copy_ms, (host_ms, copy_ms)           # the host was back long before the copy had finished
    rs = np.random.default_rng(61)
    C = 3 * T
    o_gpu = out2.double().cpu().numpy()
    assert np.isfinite(o_gpu).all()
    errs, refs = [], []
    for i, (sid, (qq, kk, vv)) in enumerate(((a, (qa, ka, va)), (b, (qb, kb, vb)))):
        rows = np.unique(np.concatenate([rs.integers(0, C, size=12), [0, T, C - 1]]))
        h = int(rs.integers(0, H))
        o_ref, _ = oracle.attention_rows(dp.o, 0, sid, 3, dev_to_bits(qq), dev_to_bits(kk), dev_to_bits(vv), scale_of(shape), h, rows)
        errs.append(o_gpu[i * C + rows, h] - o_ref)
        refs.append(o_ref)
    err, ref = np.concatenate(errs), np.concatenate(refs)
    assert np.abs(err).max() <= 2e-2 and np.linalg.norm(err) / np.linalg.norm(ref) <= 5e-3
    dp.o.append(0, [a], [3], dev_to_bits(ka), dev_to_bits(va), commit=False)       # the two uncommitted appends of the steps
    dp.o.append(0, [a, b], [3, 3], dev_to_bits(k2), dev_to_bits(v2), commit=False)
    dp.check_state([a, b], kv=False)
    dp.g.close()


# ---- ts_chunk_step_host: the host-buffer entry point (H2D, attention, append, D2H), two pipelined steps ------------
def test_chunk_step_host_two_steps():
    from paper_2606_19271_b200 import TS_COMMIT
    shape = shape_of(n_heads=3, head_dim=128, frame_tokens=200, window_frames=6, page_tokens=64, n_pages=96)
    rng = np.random.default_rng(11)
    dp = DualPool(shape, rng.permutation(shape.n_pages))
    T = shape.frame_tokens
    sids = [dp.open(), dp.open()]
    k0, v0 = draw(rng, 2 * T, shape), draw(rng, 2 * T, shape)
    dp.append(0, [sids[1]], [2], k0, v0)
    outs, refs = [], []
    hosts = []
    for step in range(3):                      # three steps back to back: both staging sets are reused
        cf = [2, 1]
        n_tok = sum(cf) * T
        q, k, v = (draw(rng, n_tok, shape) for _ in range(3))
        o_ref, _ = oracle.chunk_attention(dp.o, 0, sids, cf, q, k, v, scale_of(shape))
        hq, hk, hv = (torch.from_numpy(x.view(np.int16)).pin_memory() for x in (q, k, v))
        hout = torch.zeros_like(hq).pin_memory()
        hosts.append((hq, hk, hv, hout))       # keep the host buffers alive until the stream is done
        dp.g.ts_chunk_step_host(0, sids, cf, hq, hk, hv, hout, float(scale_of(shape)), TS_COMMIT)
        dp.o.append(0, sids, cf, k, v, commit=True)
        refs.append(o_ref)
    torch.cuda.synchronize()
    for (hq, hk, hv, hout), o_ref in zip(hosts, refs):
        o_gpu = hout.view(torch.bfloat16).double().numpy()
        assert np.abs(o_gpu - o_ref).max() <= 2e-2
        assert rel_l2(o_gpu, o_ref) <= 5e-3
    dp.check_state(sids, kv=True)
    # a packed host buffer [3][tokens][H][D] (one H2D) and a larger batch than before (the staging grows, no device sync)
    cf = [3, 3]
    n_tok = sum(cf) * T
    q, k, v = (draw(rng, n_tok, shape) for _ in range(3))
    o_ref, _ = oracle.chunk_attention(dp.o, 0, sids, cf, q, k, v, scale_of(shape))
    packed = torch.from_numpy(np.stack([q, k, v]).view(np.int16)).pin_memory()
    assert packed[0].numel() * 2 % 1024 == 0                   # tensors sit 1024-byte aligned behind each other
    hout = torch.zeros_like(packed[0]).pin_memory()
    dp.g.ts_chunk_step_host(0, sids, cf, packed[0], packed[1], packed[2], hout, float(scale_of(shape)), TS_COMMIT)
    dp.o.append(0, sids, cf, k, v, commit=True)
    torch.cuda.synchronize()
    o_gpu = hout.view(torch.bfloat16).double().numpy()
    assert np.abs(o_gpu - o_ref).max() <= 2e-2 and rel_l2(o_gpu, o_ref) <= 5e-3
    dp.check_state(sids, kv=True)
    dp.g.close()


def test_chunk_step_host_is_all_or_nothing():
    """TS_ERR_NO_PAGES from the host-buffer step: nothing was enqueued (out_host keeps its sentinel, no kernel was
    launched), no table or free-list entry changed, and the next valid call runs as if the failed one had not happened."""
    import paper_2606_19271_b200 as tc
    shape = shape_of(n_heads=2, head_dim=128, frame_tokens=100, window_frames=0, page_tokens=64, n_pages=7)
    rng = np.random.default_rng(12)
    dp = DualPool(shape, None)
    T = shape.frame_tokens
    a, b = dp.open(), dp.open()
    scale = float(scale_of(shape))

    def host(bits):
        return torch.from_numpy(bits.view(np.int16)).pin_memory()

    q, k, v = (draw(rng, 2 * T, shape) for _ in range(3))       # a: 1 frame, b: 1 frame -> 2 + 2 pages: fits
    o_ref, _ = oracle.chunk_attention(dp.o, 0, [a, b], [1, 1], q, k, v, scale_of(shape))
    h1 = [host(x) for x in (q, k, v)] + [torch.zeros(2 * T, 2, 128, dtype=torch.int16).pin_memory()]
    dp.g.ts_chunk_step_host(0, [a, b], [1, 1], *h1, scale, tc.TS_COMMIT)
    dp.o.append(0, [a, b], [1, 1], k, v, commit=True)
    torch.cuda.synchronize()
    launches = dp.g.ts_pool_launch_count()
    q2, k2, v2 = (draw(rng, 4 * T, shape) for _ in range(3))    # 2 + 2 more frames: 300 tokens each = 5 pages each > 7
    sentinel = torch.full((4 * T, 2, 128), 0x1234, dtype=torch.int16).pin_memory()
    h2 = [host(x) for x in (q2, k2, v2)]
    with pytest.raises(tc.TurboChunkError) as e:
        dp.g.ts_chunk_step_host(0, [a, b], [2, 2], *h2, sentinel, scale, tc.TS_COMMIT)
    assert e.value.code == tc.TS_ERR_NO_PAGES
    torch.cuda.synchronize()
    assert dp.g.ts_pool_launch_count() == launches and bool((sentinel == 0x1234).all())
    dp.check_state([a, b])
    q3, k3, v3 = (draw(rng, 2 * T, shape) for _ in range(3))    # one more frame for a only: fits
    o3, _ = oracle.chunk_attention(dp.o, 0, [a], [2], q3, k3, v3, scale_of(shape))
    h3 = [host(x) for x in (q3, k3, v3)] + [torch.zeros(2 * T, 2, 128, dtype=torch.int16).pin_memory()]
    dp.g.ts_chunk_step_host(0, [a], [2], *h3, scale, tc.TS_COMMIT)
    dp.o.append(0, [a], [2], k3, v3, commit=True)
    torch.cuda.synchronize()
    for hout, ref in ((h1[3], o_ref), (h3[3], o3)):
        o_gpu = hout.view(torch.bfloat16).double().numpy()
        assert np.abs(o_gpu - ref).max() <= 2e-2 and rel_l2(o_gpu, ref) <= 5e-3
    dp.check_state([a, b])
    dp.g.close()


# ---- cluster scheduling edge cases: the two CTAs of a cluster share K/V loads of one (session, head) stream ---------
@pytest.mark.parametrize("n_heads,priors,chunks", [
    (1, [0], [3]),            # one stream, q-pair KV lengths 3,5,8,8 tiles: an equal pair + a mismatched multicast pair
    (1, [2], [1]),            # one stream, two q-pairs of different length: one mismatched pair, nothing else
    (1, [0], [4]),            # 5 q-pairs: pairs + one odd item that shares a cluster with nothing
    (3, [0, 4, 1], [3, 2, 4]),   # odd items of different streams share clusters without sharing loads
    (2, [5], [1]),            # rolled window (head offset != 0), lone query tiles only
])
def test_cluster_pairing_shapes(n_heads, priors, chunks):
    shape = shape_of(n_heads=n_heads, head_dim=128, frame_tokens=300, window_frames=5, page_tokens=64,
                     n_pages=160, max_sessions=4)
    rng = np.random.default_rng(1000 + n_heads + sum(priors) + 7 * sum(chunks))
    dp = DualPool(shape, rng.permutation(shape.n_pages))
    T = shape.frame_tokens
    sids = [dp.open() for _ in priors]
    for sid, P in zip(sids, priors):
        if P:
            dp.feed_prior(sid, [draw(rng, P * T, shape)], [draw(rng, P * T, shape)])
    total = sum(chunks) * T
    for rep in range(2):      # the second call reuses the cached schedule
        q, k, v = (draw(rng, total, shape) for _ in range(3))
        dp.attention(0, sids, chunks, q, k, v, scale_of(shape))
    dp.append(0, sids, chunks, k, v)
    dp.check_state(sids)
    q, k, v = (draw(rng, total, shape) for _ in range(3))
    dp.attention(0, sids, [min(c, 2) for c in chunks], *(x[:sum(min(c, 2) for c in chunks) * T] for x in (q, k, v)),
                 scale_of(shape))


# ---- ts_chunk_step: attention + append as one call, the append running under the attention on a pool stream --------
def test_chunk_step_fused_equals_sequence():
    from paper_2606_19271_b200 import TS_COMMIT
    shape = shape_of(n_heads=3, head_dim=128, frame_tokens=203, window_frames=5, page_tokens=64, n_pages=128)
    rng = np.random.default_rng(21)
    dp = DualPool(shape, rng.permutation(shape.n_pages))
    T = shape.frame_tokens
    sids = [dp.open(), dp.open(), dp.open()]
    cf = [2, 1, 3]
    n_tok = sum(cf) * T
    for step in range(4):                      # the window of the 3-frame session fills and rolls at step 2
        q, k, v = (draw(rng, n_tok, shape) for _ in range(3))
        o_ref, _ = oracle.chunk_attention(dp.o, 0, sids, cf, q, k, v, scale_of(shape))
        dq, dk, dv = bits_to_dev(q), bits_to_dev(k), bits_to_dev(v)
        out = torch.full_like(dq, float("nan"))
        dp.g.ts_chunk_step(0, sids, cf, dq, dk, dv, out, None, float(scale_of(shape)), TS_COMMIT)
        dp.o.append(0, sids, cf, k, v, commit=True)
        torch.cuda.synchronize()
        o_gpu = out.double().cpu().numpy()
        assert np.abs(o_gpu - o_ref).max() <= 2e-2 and rel_l2(o_gpu, o_ref) <= 5e-3
        dp.check_state(sids, kv=True)
    # all-or-nothing: a step that cannot get its pages changes nothing and enqueues nothing
    big = shape_of(n_heads=3, head_dim=128, frame_tokens=203, window_frames=0, page_tokens=64, n_pages=8)
    dq2 = DualPool(big, None)
    s0 = dq2.open()
    q, k, v = (draw(rng, 3 * T, big) for _ in range(3))
    import paper_2606_19271_b200 as tc
    with pytest.raises(tc.TurboChunkError) as e:
        dq2.g.ts_chunk_step(0, [s0], [3], bits_to_dev(q), bits_to_dev(k), bits_to_dev(v), torch.empty(3 * T, 3, 128, dtype=torch.bfloat16, device="cuda"), None, 0.1, TS_COMMIT)
    assert e.value.code == tc.TS_ERR_NO_PAGES
    dq2.check_state([s0])


# ---- the lazy-rescale path and the split-tile merge under large score jumps (N(0,1) inputs almost never take them) -----------
@pytest.mark.parametrize("pattern", ["ramp_up", "ramp_down", "spikes", "masked_spike"])
@pytest.mark.parametrize("page_tokens", [64, 256])
def test_lazy_rescale_and_outliers(pattern, page_tokens):
    """Scores that jump by far more than the rescale threshold (2^8) from tile to tile, in both directions, inside either
    64-key half of a tile, in the chunk, and behind the frame mask: every rescale of O in TMEM, the (m, l) merge of a split
    lone tile and the mask must hold against the fp64 oracle."""
    f32_to_bf16_bits = synth.f32_to_bf16_bits
    T, H, D, prior, c = 160, 2, 128, 6, 2
    shape = shape_of(n_heads=H, head_dim=D, page_tokens=page_tokens, frame_tokens=T, n_pages=64, window_frames=0)
    rng = np.random.default_rng(len(pattern) * 37 + page_tokens)
    dp = DualPool(shape, rng.permutation(shape.n_pages))
    sid = dp.open()
    Lp, C = prior * T, c * T
    u = np.ones(D, dtype=np.float32) / np.sqrt(np.float32(D))
    a = np.zeros(Lp + C, dtype=np.float32)                       # boost of key j along u
    if pattern == "ramp_up":
        a[:] = 0.125 * np.arange(Lp + C)                         # +5.6 nats per 128-key tile, logits up to ~56 nats
    elif pattern == "ramp_down":
        a[:] = 0.125 * np.arange(Lp + C)[::-1]
    elif pattern == "spikes":
        for j in (5, 100, 128 + 70, 3 * 128 + 64, 5 * 128 + 127, Lp - 1, Lp + 3, Lp + 130, Lp + T - 1):
            a[j] = 150.0 + j % 7                                  # isolated keys ~50 nats above the rest
    else:                                                         # a huge key in the chunk's SECOND frame: frame-0 queries
        a[Lp + T + 17] = 400.0                                    # must not see it, frame-1 queries are dominated by it
        a[Lp + 2 * T - 1] = 380.0
    noise = lambda n: rng.standard_normal((n, H, D)).astype(np.float32) * 0.5
    k_all = noise(Lp + C) + a[:, None, None] * u[None, None, :]
    v_all = rng.standard_normal((Lp + C, H, D)).astype(np.float32)
    q = noise(C) + 4.0 * u[None, None, :]
    kb, vb, qb = f32_to_bf16_bits(k_all), f32_to_bf16_bits(v_all), f32_to_bf16_bits(q)
    dp.feed_prior(sid, [kb[:Lp]], [vb[:Lp]])
    o_gpu, o_ref = dp.attention(0, [sid], [c], qb, kb[Lp:], vb[Lp:], scale_of(shape))
    if pattern == "masked_spike":
        # frame-0 rows ignore the spike entirely; frame-1 rows are (almost) exactly v of the spike key
        v_spike = synth.bf16_bits_to_f64(vb[Lp + T + 17])
        assert np.abs(o_gpu[T:] - v_spike[None]).max() < 0.15     # the second, smaller spike keeps a weight of ~1 %
        assert np.abs(o_gpu[:T] - v_spike[None]).max() > 0.5
    # a second session in the same batch with plain N(0,1) inputs must be unaffected (isolation inside one launch)
    other = dp.open()
    dp.feed_prior(other, [draw(rng, 3 * T, shape)], [draw(rng, 3 * T, shape)])
    q2, k2, v2 = (draw(rng, 3 * T, shape) for _ in range(3))
    dp.attention(0, [other, sid], [3, c], np.concatenate([q2, qb]), np.concatenate([k2, kb[Lp:]]),
                 np.concatenate([v2, vb[Lp:]]), scale_of(shape))


def test_output_alignment_is_checked():
    """`out` is written with 256-bit stores: a pointer that is 16- but not 32-byte aligned is TS_ERR_INVALID, not a fault."""
    import paper_2606_19271_b200 as tc
    shape = shape_of(n_heads=1, head_dim=64, frame_tokens=16, window_frames=0, page_tokens=16, n_pages=8)
    dp = DualPool(shape)
    sid = dp.open()
    rng = np.random.default_rng(1)
    q, k, v = (bits_to_dev(draw(rng, 16, shape)) for _ in range(3))
    raw = torch.empty(16 * 64 + 16, dtype=torch.bfloat16, device="cuda")
    assert raw.data_ptr() % 32 == 0
    bad = raw[8:8 + 16 * 64].view(16, 1, 64)                     # 16 bytes past a 32-byte boundary
    for call in (lambda o: dp.g.ts_chunk_attention(0, [sid], [1], q, k, v, o, None, 0.125),
                 lambda o: dp.g.ts_chunk_step(0, [sid], [1], q, k, v, o, None, 0.125, tc.TS_COMMIT)):
        with pytest.raises(tc.TurboChunkError) as e:
            call(bad)
        assert e.value.code == tc.TS_ERR_INVALID
    dp.check_state([sid])
    good = raw[:16 * 64].view(16, 1, 64)
    dp.g.ts_chunk_attention(0, [sid], [1], q, k, v, good, None, 0.125)
    torch.cuda.synchronize()
    assert torch.isfinite(good.float()).all()
    dp.g.close()


@pytest.mark.parametrize("fused", [False, True])
def test_batch_with_resumes_in_flight_runs_ready_sessions_first(fused):
    """PAPER.md:76 (iii): sessions 1 and 3 of a five-session batch are resumed right before the call (their copies - ~10 MB
    each - are still in flight when it is made): the call runs as two launches (ready sessions 0, 2, 4 first, then 1 and 3
    behind their copy events; the groups are NOT contiguous in the packed tensors) and the result is that of one launch:
    output against the oracle, appended bytes, page tables."""
    import paper_2606_19271_b200 as tc
    shape = shape_of(n_heads=4, head_dim=128, frame_tokens=200, window_frames=9, page_tokens=64, n_pages=5 * 40, max_sessions=8)
    rng = np.random.default_rng(70 + int(fused))
    dp = DualPool(shape, rng.permutation(shape.n_pages), host_pages=2 * 40)
    T = shape.frame_tokens
    sids = [dp.open() for _ in range(5)]
    for i, sid in enumerate(sids):
        n_frames = (6, 6, 2, 6, 0)[i]
        if n_frames:
            dp.feed_prior(sid, [draw(rng, n_frames * T, shape)], [draw(rng, n_frames * T, shape)])
    cf = [2, 3, 1, 2, 3]
    scale = scale_of(shape)
    for step in range(3):
        for sid in (sids[1], sids[3]):
            dp.suspend(sid)
        dp.g.ts_offload_sync()
        torch.cuda.synchronize()
        before = dp.g.ts_pool_split_batches()
        # a long copy in front of the resumes on the side stream, so that they are certainly still pending at call time
        blocker_h = torch.empty(256 << 20, dtype=torch.uint8).pin_memory()
        blocker_d = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
        q, k, v = (draw(rng, sum(cf) * T, shape) for _ in range(3))
        # the oracle's side first (it takes seconds); then the GPU calls back to back, so that the resumes are still in flight
        for sid in (sids[1], sids[3]):
            dp.o.resume(sid)
        o_ref, _ = oracle.chunk_attention(dp.o, 0, sids, cf, q, k, v, scale)
        dp.o.append(0, sids, cf, k, v, commit=True)
        dq, dk, dv = bits_to_dev(q), bits_to_dev(k), bits_to_dev(v)
        out = torch.full_like(dq, float("nan"))
        torch.cuda.synchronize()
        with torch.cuda.stream(dp.g.side_stream):
            blocker_d.copy_(blocker_h, non_blocking=True)
        for sid in (sids[1], sids[3]):
            dp.g.ts_session_resume(sid)
        if fused:
            dp.g.ts_chunk_step(0, sids, cf, dq, dk, dv, out, None, float(scale), tc.TS_COMMIT)
        else:
            dp.g.ts_chunk_attention(0, sids, cf, dq, dk, dv, out, None, float(scale))
            dp.g.ts_kv_append(0, sids, cf, dk, dv, tc.TS_COMMIT)
        torch.cuda.synchronize()
        o_gpu = out.double().cpu().numpy()
        assert np.isfinite(o_gpu).all()
        assert np.abs(o_gpu - o_ref).max() <= 2e-2 and rel_l2(o_gpu, o_ref) <= 5e-3
        assert dp.g.ts_pool_split_batches() == before + 1
        dp.check_state(sids)
    dp.g.close()
