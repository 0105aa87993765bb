"""Pins M1-M4 for the oracle's GPU-GPU migration (O4, `OraclePool.migrate_to`, reading R22).
None re-types the routine: M1 is a hand-worked id trace, M2 composes the already pinned suspend / resume (P5,
P11) by hand, M3 is a round-trip identity plus attention invariance, M4 are conservation laws."""
import copy
import os

import numpy as np
import pytest

import oracle
import synth
from helpers import feed_prior, make_oracle_pool


def shape_of(n_pages, **kw):
    d = dict(n_layers=1, n_heads=2, head_dim=16, page_tokens=16, n_pages=n_pages, frame_tokens=16,
             window_frames=0, max_sessions=4)
    d.update(kw)
    return synth.PoolShape(**d)


def draw(rng, n, shape):
    return synth.draw_bits(rng, n, shape.n_heads, shape.head_dim)


def add_frames(pool, sid, rng, shape, frames):
    T = shape.frame_tokens
    ks = [draw(rng, frames * T, shape) for _ in range(shape.n_layers)]
    vs = [draw(rng, frames * T, shape) for _ in range(shape.n_layers)]
    feed_prior(pool, sid, ks, vs, T)
    return ks, vs


def parse_trace(path):
    vals = {}
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        key, rest = line.split(None, 1)
        if ":" in rest:      # "A: 3 1   S: 4 0 5" -> {"A": [3, 1], "S": [4, 0, 5]}
            tables, name = {}, None
            for tok in rest.split():
                if tok.endswith(":"):
                    name = tok[:-1]
                    tables[name] = []
                else:
                    tables[name].append(int(tok))
            vals[key] = tables
        else:
            vals[key] = [int(x) for x in rest.split()]
    return vals


# ---- M1: hand-worked trace (tests/golden/migration_trace.txt) ---------------------------------------------
def test_m1_hand_worked_trace(golden_dir):
    g = parse_trace(os.path.join(golden_dir, "migration_trace.txt"))
    rng = np.random.default_rng(40)
    ssh, dsh = shape_of(8), shape_of(6)
    src = make_oracle_pool(ssh, g["src_free_order"])
    dst = make_oracle_pool(dsh, g["dst_free_order"])
    a = src.open()
    add_frames(src, a, rng, ssh, 2)
    s = src.open()
    add_frames(src, s, rng, ssh, 3)
    assert {"A": src.page_table(a), "S": src.page_table(s)} == g["src_after_setup"]
    assert list(src.free) == g["src_free_after_setup"]
    x = dst.open()
    add_frames(dst, x, rng, dsh, 1)
    assert {"X": dst.page_table(x)} == g["dst_after_setup"]
    assert list(dst.free) == g["dst_free_after_setup"]

    s2 = src.migrate_to(s, dst)
    assert [s2] == g["migrated_sid"]
    assert {"X": dst.page_table(x), "S": dst.page_table(s2)} == g["dst_after_migrate"]
    assert list(dst.free) == g["dst_free_after_migrate"]
    assert list(src.free) == g["src_free_after_migrate"]
    with pytest.raises(oracle.OracleError) as e:
        src.info(s)                                   # ownership flipped: the source no longer knows the session
    assert e.value.kind == oracle.STATE

    c = src.open()
    assert c == s                                     # the id is reusable on the source
    add_frames(src, c, rng, ssh, 1)
    assert {"A": src.page_table(a), "C": src.page_table(c)} == g["src_after_reopen"]
    s3 = dst.migrate_to(s2, src)
    assert [s3] == g["returned_sid"]
    assert {"A": src.page_table(a), "C": src.page_table(c), "S": src.page_table(s3)} == g["src_after_return"]
    assert list(src.free) == g["src_free_after_return"]
    assert list(dst.free) == g["dst_free_after_return"]


# ---- M2: migration == suspend on the source + carrying the host copy over + resume on the target ------------
def test_m2_equals_suspend_transplant_resume():
    rng = np.random.default_rng(41)
    ssh = shape_of(24, n_layers=2, page_tokens=8, frame_tokens=5, window_frames=6)
    dsh = shape_of(20, n_layers=2, page_tokens=8, frame_tokens=5, window_frames=6)
    src = make_oracle_pool(ssh, rng.permutation(24))
    dst = make_oracle_pool(dsh, rng.permutation(20))
    other = src.open()
    add_frames(src, other, rng, ssh, 2)
    s = src.open()
    add_frames(src, s, rng, ssh, 8)                   # window 6: two frames evicted, head offset o = 10 % 8 = 2
    assert src.info(s)["head_off"] == 2 and src.info(s)["frames"] == 6
    y = dst.open()
    add_frames(dst, y, rng, dsh, 3)
    src_b, dst_b = copy.deepcopy(src), copy.deepcopy(dst)

    new = src.migrate_to(s, dst)

    # the same move spelled out with the pinned primitives: suspend (source), open + adopt the host copy + resume (target)
    src_b.suspend(s)
    host = src_b.sessions[s].host
    P, o = src_b.sessions[s].P, src_b.sessions[s].o
    src_b.close(s)
    new_b = dst_b.open()
    t = dst_b.sessions[new_b]
    t.P, t.o, t.host, t.state = P, o, host, oracle.SUSPENDED
    dst_b.host_pages_used += host[2]
    dst_b.resume(new_b)

    assert new == new_b
    assert list(src.free) == list(src_b.free) and list(dst.free) == list(dst_b.free)
    assert dst.page_table(new) == dst_b.page_table(new_b)
    assert dst.info(new) == dst_b.info(new_b)
    assert sorted(src.sessions) == sorted(src_b.sessions)
    for layer in range(2):
        for got, want in zip(dst.gather_kv(layer, new), dst_b.gather_kv(layer, new_b)):
            np.testing.assert_array_equal(got, want)
    np.testing.assert_array_equal(dst.K, dst_b.K)     # whole pages, incl. dead head/tail slots (R11)
    np.testing.assert_array_equal(dst.V, dst_b.V)


# ---- M3: round trip identity; attention and later appends do not see the move -------------------------------
def test_m3_round_trip_and_attention_invariance():
    rng = np.random.default_rng(42)
    sh = shape_of(32, n_layers=2, page_tokens=8, frame_tokens=5, window_frames=7)
    a = make_oracle_pool(sh, rng.permutation(32))
    b = make_oracle_pool(sh, rng.permutation(32))
    stay = make_oracle_pool(sh, rng.permutation(32))      # the same session history, never migrated
    sa, ss = a.open(), stay.open()
    T = sh.frame_tokens
    ks = [draw(rng, 5 * T, sh) for _ in range(2)]
    vs = [draw(rng, 5 * T, sh) for _ in range(2)]
    feed_prior(a, sa, ks, vs, T)
    feed_prior(stay, ss, ks, vs, T)
    filler = b.open()
    add_frames(b, filler, rng, sh, 2)
    q, kn, vn = (draw(rng, 3 * T, sh) for _ in range(3))
    before = [a.gather_kv(l, sa) for l in range(2)]
    o_before = oracle.chunk_attention(a, 1, [sa], [3], q, kn, vn, 0.25)

    sb = a.migrate_to(sa, b)
    o_there = oracle.chunk_attention(b, 1, [sb], [3], q, kn, vn, 0.25)
    for x, y in zip(o_before, o_there):
        np.testing.assert_array_equal(x, y)
    # the session keeps living on the target: a committed append rolls the window there exactly as it would have at home
    for layer in range(2):
        b.append(layer, [sb], [3], kn, vn, commit=(layer == 1))
        stay.append(layer, [ss], [3], kn, vn, commit=(layer == 1))
    assert {k: v for k, v in b.info(sb).items()} == {k: v for k, v in stay.info(ss).items()}
    back = b.migrate_to(sb, a)
    for layer in range(2):
        for got, want in zip(a.gather_kv(layer, back), stay.gather_kv(layer, ss)):
            np.testing.assert_array_equal(got, want)
    assert a.info(back) == stay.info(ss)
    # ... and before the append the round trip alone changed no logical byte
    c = make_oracle_pool(sh, rng.permutation(32))
    d = make_oracle_pool(sh, rng.permutation(32))
    sc = c.open()
    feed_prior(c, sc, ks, vs, T)
    sc2 = d.migrate_to(c.migrate_to(sc, d), c)
    for layer in range(2):
        for got, want in zip(c.gather_kv(layer, sc2), before[layer]):
            np.testing.assert_array_equal(got, want)


# ---- M4: conservation, isolation, all-or-nothing errors ----------------------------------------------------
def conserved(pool):
    held = [p for s in pool.sessions.values() for p in s.PT]
    ids = held + list(pool.free)
    return sorted(ids) == list(range(pool.n_pages))


def test_m4_conservation_isolation_errors():
    rng = np.random.default_rng(43)
    sh = shape_of(12, page_tokens=8, frame_tokens=5, max_sessions=2)
    src = make_oracle_pool(sh, rng.permutation(12))
    dst = make_oracle_pool(sh, rng.permutation(12))
    s0, s1 = src.open(), src.open()
    add_frames(src, s0, rng, sh, 4)                   # 20 tokens = 3 pages
    add_frames(src, s1, rng, sh, 6)                   # 30 tokens = 4 pages
    d0 = dst.open()
    add_frames(dst, d0, rng, sh, 14)                  # 70 tokens = 9 pages: 3 free on the target
    keep = [src.gather_kv(0, s0), dst.gather_kv(0, d0)]
    snap = (list(src.free), list(dst.free), src.page_table(s1), sorted(src.sessions), sorted(dst.sessions))

    def unchanged():
        return snap == (list(src.free), list(dst.free), src.page_table(s1), sorted(src.sessions), sorted(dst.sessions))

    with pytest.raises(oracle.OracleError) as e:
        src.migrate_to(s1, dst)                       # 4 pages needed, 3 free
    assert e.value.kind == oracle.NO_PAGES and unchanged()
    with pytest.raises(oracle.OracleError) as e:
        src.migrate_to(s1, src)
    assert e.value.kind == oracle.INVALID and unchanged()
    other = make_oracle_pool(shape_of(12, page_tokens=16, frame_tokens=5, max_sessions=2))
    with pytest.raises(oracle.OracleError) as e:
        src.migrate_to(s1, other)                     # different page size
    assert e.value.kind == oracle.INVALID and unchanged()
    src.host_pages_cap = None
    src.suspend(s1)
    with pytest.raises(oracle.OracleError) as e:
        src.migrate_to(s1, dst)                       # only a resident (frozen, live) state moves
    assert e.value.kind == oracle.STATE
    src.resume(s1)
    d1 = dst.open()
    with pytest.raises(oracle.OracleError) as e:
        src.migrate_to(s0, dst)                       # the target's session table is full
    assert e.value.kind == oracle.CAPACITY
    dst.close(d1)

    new = src.migrate_to(s0, dst)                     # 3 pages: fits exactly
    assert conserved(src) and conserved(dst) and len(dst.free) == 0
    assert sorted(src.sessions) == [s1] and sorted(dst.sessions) == [d0, new]
    # isolation: nobody else's logical bytes moved
    for got, want in zip(dst.gather_kv(0, new), keep[0]):
        np.testing.assert_array_equal(got, want)
    for got, want in zip(dst.gather_kv(0, d0), keep[1]):
        np.testing.assert_array_equal(got, want)
