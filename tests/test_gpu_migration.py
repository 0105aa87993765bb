"""Parity of ts_session_migrate (GPU-GPU session migration, reading R22) against the oracle's
`OraclePool.migrate_to` on the same seeded inputs: ids, page tables, free lists and logical KV bytes bit-exact on
both pools; attention on the target within the north_star tolerance.  The two pools live on the one GPU of the
box (the fetch kernel reads the source slab through an ordinary device pointer there; across two GPUs the same
pointer is a peer mapping)."""
import dataclasses
import os

import numpy as np
import pytest
import torch

import oracle
import synth
from helpers import DualPool, bits_to_dev, dev_to_bits
from test_oracle_migration_pins import parse_trace

pytestmark = pytest.mark.gpu


def shape_of(**kw):
    d = dict(n_layers=1, n_heads=2, head_dim=128, page_tokens=64, n_pages=64, frame_tokens=100,
             window_frames=0, max_sessions=8)
    d.update(kw)
    return synth.PoolShape(**d)


def draw(rng, n, shape):
    return synth.draw_bits(rng, n, shape.n_heads, shape.head_dim)


def scale_of(shape):
    return np.float32(1.0 / np.sqrt(np.float32(shape.head_dim)))


def migrate(src, sid, dst):
    """The same move on the oracle pair and on the CUDA pair; the new ids must agree."""
    a = src.o.migrate_to(sid, dst.o)
    b = src.g.ts_session_migrate(sid, dst.g)
    assert a == b
    return a


def add_frames(dp, sid, rng, frames):
    sh = dp.shape
    n = frames * sh.frame_tokens
    dp.feed_prior(sid, [draw(rng, n, sh) for _ in range(sh.n_layers)], [draw(rng, n, sh) for _ in range(sh.n_layers)])


def test_migration_hand_worked_trace_on_gpu(golden_dir):
    g = parse_trace(os.path.join(golden_dir, "migration_trace.txt"))
    rng = np.random.default_rng(50)
    kw = dict(head_dim=64, page_tokens=16, frame_tokens=16, max_sessions=4)
    src = DualPool(shape_of(n_pages=8, **kw), g["src_free_order"])
    dst = DualPool(shape_of(n_pages=6, **kw), g["dst_free_order"])
    a = src.open()
    add_frames(src, a, rng, 2)
    s = src.open()
    add_frames(src, s, rng, 3)
    x = dst.open()
    add_frames(dst, x, rng, 1)
    s2 = migrate(src, s, dst)
    assert [s2] == g["migrated_sid"]
    assert dst.g.ts_session_page_table(s2) == g["dst_after_migrate"]["S"]
    assert dst.g.ts_pool_free_list() == g["dst_free_after_migrate"]
    assert src.g.ts_pool_free_list() == g["src_free_after_migrate"]
    src.check_state([a])
    dst.check_state([x, s2])
    c = src.open()
    assert c == s
    add_frames(src, c, rng, 1)
    s3 = migrate(dst, s2, src)
    assert [s3] == g["returned_sid"]
    assert src.g.ts_session_page_table(s3) == g["src_after_return"]["S"]
    assert src.g.ts_pool_free_list() == g["src_free_after_return"]
    assert dst.g.ts_pool_free_list() == g["dst_free_after_return"]
    src.check_state([a, c, s3])
    dst.check_state([x])


@pytest.mark.parametrize("head_dim,page_tokens,n_layers", [(128, 256, 2), (64, 16, 1), (128, 64, 3)])
def test_migration_parity_window_offsets_layers(head_dim, page_tokens, n_layers):
    """A rolled window (head offset != 0), several layers, permuted pools of different sizes: migrate, attend and
    append on the target, migrate back."""
    T = 203
    per = -(-9 * T // page_tokens) + 2
    rng = np.random.default_rng(60 + head_dim + page_tokens)
    ssh = shape_of(head_dim=head_dim, page_tokens=page_tokens, n_layers=n_layers, n_heads=3, frame_tokens=T,
                   window_frames=7, n_pages=3 * per)
    dsh = shape_of(head_dim=head_dim, page_tokens=page_tokens, n_layers=n_layers, n_heads=3, frame_tokens=T,
                   window_frames=7, n_pages=2 * per + 3)
    src = DualPool(ssh, rng.permutation(ssh.n_pages), host_pages=per)
    dst = DualPool(dsh, rng.permutation(dsh.n_pages))
    stay, s = src.open(), src.open()
    add_frames(src, stay, rng, 2)
    add_frames(src, s, rng, 11)                                   # window 7: rolled twice
    assert src.g.ts_session_info(s)["head_off"] != 0
    other = dst.open()
    add_frames(dst, other, rng, 4)
    # suspend + resume right before: the fetch must also wait for a resume that is still copying in
    src.suspend(s)
    src.resume(s)
    new = migrate(src, s, dst)
    src.check_state([stay])
    dst.check_state([other, new])
    q, k, v = (draw(rng, 5 * T, dsh) for _ in range(3))
    for layer in range(n_layers):
        dst.attention(layer, [other, new], [2, 3], q, k, v, scale_of(dsh))
        dst.append(layer, [other, new], [2, 3], k, v, commit=(layer == n_layers - 1))
    dst.check_state([other, new])
    back = migrate(dst, new, src)
    src.check_state([stay, back])
    dst.check_state([other])
    q, k, v = (draw(rng, 4 * T, ssh) for _ in range(3))
    src.attention(n_layers - 1, [back, stay], [3, 1], q, k, v, scale_of(ssh))


def test_migration_is_stream_ordered_without_host_sync():
    """(i) the fetch follows the chunk step already enqueued on the session; (ii) attention on the target follows the
    fetch; (iii) the source's pages are rewritten by a later append only after the fetch - no host wait anywhere."""
    import paper_2606_19271_b200 as tc
    T = 520
    sh = shape_of(head_dim=128, page_tokens=256, n_heads=12, frame_tokens=T, window_frames=21, n_pages=48, max_sessions=4)
    rng = np.random.default_rng(70)
    src = DualPool(sh, rng.permutation(48))
    dst = DualPool(sh, rng.permutation(48))
    s = src.open()
    add_frames(src, s, rng, 15)                                   # 7800 tokens = 31 pages (37 after the step): 11 left in the source
    q, k, v = (draw(rng, 3 * T, sh) for _ in range(3))
    dq, dk, dv = bits_to_dev(q), bits_to_dev(k), bits_to_dev(v)
    k2, v2 = draw(rng, 18 * T, sh), draw(rng, 18 * T, sh)         # 9360 tokens = 37 pages: 11 untouched + 26 of the freed ones
    dk2, dv2 = bits_to_dev(k2), bits_to_dev(v2)
    out = torch.full_like(dq, float("nan"))
    out2 = torch.full_like(dq, float("nan"))
    torch.cuda.synchronize()
    # ---- enqueue everything back to back
    src.g.ts_chunk_step(0, [s], [3], dq, dk, dv, out, None, float(scale_of(sh)), tc.TS_COMMIT)
    new = src.g.ts_session_migrate(s, dst.g)
    dst.g.ts_chunk_attention(0, [new], [3], dq, dk, dv, out2, None, float(scale_of(sh)))
    fresh = src.g.ts_session_open()
    src.g.ts_kv_append(0, [fresh], [18], dk2, dv2)                # overwrites pages the fetch is reading
    torch.cuda.synchronize()
    # ---- the same on the oracle
    o1, _ = oracle.chunk_attention(src.o, 0, [s], [3], q, k, v, scale_of(sh))
    src.o.append(0, [s], [3], k, v)
    former = set(src.o.page_table(s))
    assert src.o.migrate_to(s, dst.o) == new
    o2, _ = oracle.chunk_attention(dst.o, 0, [new], [3], q, k, v, scale_of(sh))
    assert src.o.open() == fresh
    src.o.append(0, [fresh], [18], k2, v2)
    assert len(former & set(src.o.page_table(fresh))) == 26      # the append did rewrite pages the fetch had to read first
    src.check_state([fresh])
    dst.check_state([new])                                        # bit-exact: nothing was overwritten under the fetch
    for got, want in ((out, o1), (out2, o2)):
        got = got.double().cpu().numpy()
        assert np.isfinite(got).all()
        assert np.abs(got - want).max() <= DualPool.MAX_ABS
        assert np.linalg.norm(got - want) / np.linalg.norm(want) <= DualPool.REL_L2


def test_migration_error_codes_and_all_or_nothing():
    import paper_2606_19271_b200 as tc
    rng = np.random.default_rng(80)
    sh = shape_of(head_dim=64, page_tokens=16, frame_tokens=10, n_pages=12, max_sessions=2)
    src = DualPool(sh, rng.permutation(12), host_pages=8)
    dst = DualPool(sh, rng.permutation(12))
    s0, s1 = src.open(), src.open()
    add_frames(src, s0, rng, 4)                                   # 40 tokens = 3 pages
    add_frames(src, s1, rng, 6)                                   # 60 tokens = 4 pages
    d0 = dst.open()
    add_frames(dst, d0, rng, 14)                                  # 140 tokens = 9 pages: 3 free

    def both_fail(src_dp, sid, dst_dp, code, kind):
        with pytest.raises(tc.TurboChunkError) as e:
            src_dp.g.ts_session_migrate(sid, dst_dp.g)
        assert e.value.code == code
        with pytest.raises(oracle.OracleError) as eo:
            src_dp.o.migrate_to(sid, dst_dp.o)
        assert eo.value.kind == kind
        src.check_state([s0, s1])
        dst.check_state([d0])

    both_fail(src, s1, dst, tc.TS_ERR_NO_PAGES, oracle.NO_PAGES)
    both_fail(src, s1, src, tc.TS_ERR_INVALID, oracle.INVALID)
    odd = DualPool(shape_of(head_dim=64, page_tokens=32, frame_tokens=10, n_pages=12, max_sessions=2))
    both_fail(src, s1, odd, tc.TS_ERR_INVALID, oracle.INVALID)
    with pytest.raises(tc.TurboChunkError) as e:
        src.g.ts_session_migrate(7, dst.g)
    assert e.value.code == tc.TS_ERR_STATE
    src.suspend(s1)
    both_fail(src, s1, dst, tc.TS_ERR_STATE, oracle.STATE)
    src.resume(s1)
    d1 = dst.open()
    with pytest.raises(tc.TurboChunkError) as e:
        src.g.ts_session_migrate(s0, dst.g)
    assert e.value.code == tc.TS_ERR_CAPACITY
    with pytest.raises(oracle.OracleError) as eo:
        src.o.migrate_to(s0, dst.o)
    assert eo.value.kind == oracle.CAPACITY
    dst.close(d1)
    new = migrate(src, s0, dst)                                   # 3 pages: fits exactly
    assert dst.g.ts_pool_stats()["free_pages"] == 0
    src.check_state([s1])
    dst.check_state([d0, new])
    empty = src.open()                                            # a session without pages migrates too (no kernel)
    dst.close(d0)
    e2 = migrate(src, empty, dst)
    dst.check_state([new, e2])
    src.check_state([s1])


def test_migration_full_window_wan13b():
    """BASELINE.json configs[1]-[2] session shape at the full 21-frame window: 128-129 pages, 201 MB; ping-pong."""
    w = synth.wan13b_single()
    sh = dataclasses.replace(w.shape, n_pages=160, max_sessions=2)
    rng = np.random.default_rng(90)
    a = DualPool(sh, rng.permutation(sh.n_pages))
    b = DualPool(sh, rng.permutation(sh.n_pages))
    s = a.open()
    T = sh.frame_tokens
    gen = torch.Generator(device="cuda").manual_seed(90)
    for _ in range(8):                                            # 24 frames through a 21-frame window: rolled once
        k = torch.randn((3 * T, sh.n_heads, sh.head_dim), generator=gen, device="cuda").to(torch.bfloat16)
        v = torch.randn((3 * T, sh.n_heads, sh.head_dim), generator=gen, device="cuda").to(torch.bfloat16)
        a.append(0, [s], [3], dev_to_bits(k), dev_to_bits(v), dev=(k, v))
    assert a.g.ts_session_info(s)["frames"] == 21 and a.g.ts_session_info(s)["n_pages"] >= 128
    x = migrate(a, s, b)
    b.check_state([x])
    y = migrate(b, x, a)
    a.check_state([y])
    times = []
    pools, sid = (a, b), y
    for i in range(6):
        src, dst = pools[i & 1], pools[(i & 1) ^ 1]
        st = dst.g.side_stream
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        want = src.o.migrate_to(sid, dst.o)                       # the oracle's move first: host time stays outside the events
        e0.record(st)
        sid = src.g.ts_session_migrate(sid, dst.g)
        e1.record(st)
        assert sid == want
        torch.cuda.synchronize()
        times.append(e0.elapsed_time(e1))
    a.check_state([sid])
    nbytes = a.g.ts_session_info(sid)["n_pages"] * a.g.page_bytes
    print(f"migrate {nbytes / 1e6:.0f} MB: {np.median(times) * 1e3:.0f} us, {2 * nbytes / np.median(times) / 1e6:.0f} GB/s read+write")


# ---- two devices: the fetch kernel runs on the target GPU and reads the source slab through the peer mapping (NVLink) ----
@pytest.mark.skipif(torch.cuda.device_count() < 2, reason="needs two GPUs with peer access (one-GPU boxes run the same "
                    "kernel with both pools on one device: every other test of this file)")
def test_migration_between_two_devices():
    """Pools on devices 0 and 1 of this process; a session migrates 0 -> 1, is served there, migrates back 1 -> 0 and is
    served again: ids, page tables, free lists, logical KV bytes against the oracle on both devices, attention on the
    target within tolerance."""
    if not (torch.cuda.can_device_access_peer(0, 1) and torch.cuda.can_device_access_peer(1, 0)):
        pytest.skip("no peer access between devices 0 and 1")
    sh = shape_of(n_heads=3, head_dim=128, page_tokens=64, frame_tokens=130, window_frames=6, n_pages=48, n_layers=2)
    rng = np.random.default_rng(77)
    pools = [DualPool(sh, rng.permutation(sh.n_pages), device=d) for d in (0, 1)]
    T = sh.frame_tokens
    sid = pools[0].open()
    other = [pools[0].open(), pools[1].open()]                 # bystanders on both devices
    add_frames(pools[0], sid, rng, 5)
    add_frames(pools[0], other[0], rng, 2)
    add_frames(pools[1], other[1], rng, 3)
    where = 0
    for hop in range(4):                                       # 0 -> 1 -> 0 -> 1 -> 0, the window rolling on the way
        src, dst = pools[where], pools[where ^ 1]
        sid = migrate(src, sid, dst)
        where ^= 1
        dst.check_state([sid, other[where]])
        src.check_state([other[where ^ 1]])
        with torch.cuda.device(where):
            for layer in range(sh.n_layers):
                q, k, v = (draw(rng, 3 * T, sh) for _ in range(3))
                dst.fused_step(layer, [sid, other[where]], [2, 1], q, k, v, scale_of(sh), commit=(layer == sh.n_layers - 1))
        dst.check_state([sid, other[where]])
    for p in pools:
        p.g.close()
