"""Session migration between two WORKER PROCESSES (PAPER.md:66, :271 one worker per GPU; :263-265 registration, freeze,
one-sided fetch + verify, ownership flip) against the oracle's `OraclePool.migrate_to`: ids, page tables, free lists and
logical KV bytes bit-exact on both workers; attention on the target within the north_star tolerance.

Two processes (paper_2606_19271_b200.worker), each with its own CUDA context and pool on the one GPU of the box; the source
slab reaches the target's fetch kernel through CUDA IPC; "state frozen" and "installed" are interprocess events, so neither
process waits on the host anywhere in a move.  The parent plays the control plane and holds the oracle pools.  Both worker
slabs are NaN-poisoned and sit between guard bands."""
import numpy as np
import pytest

import oracle
import synth
from helpers import make_oracle_pool, rel_l2

pytestmark = pytest.mark.gpu

MAX_ABS, REL_L2 = 2e-2, 5e-3
NAN_BF16 = 0x7FC0


class Side:
    """One worker process + the oracle pool that mirrors it."""

    def __init__(self, shape, free_order, host_pages=32):
        from paper_2606_19271_b200 import worker
        self.shape = shape
        self.o = make_oracle_pool(shape, free_order, host_pages)
        self.w = worker.spawn(device=0)
        self.w.call("create", n_layers=shape.n_layers, n_heads=shape.n_heads, head_dim=shape.head_dim,
                    page_tokens=shape.page_tokens, n_pages=shape.n_pages, frame_tokens=shape.frame_tokens,
                    window_frames=shape.window_frames, max_sessions=shape.max_sessions, free_order=free_order,
                    host_pages=host_pages, guard_bytes=1 << 20, poison=NAN_BF16)

    def open(self):
        a, b = self.o.open(), self.w.call("pool", "ts_session_open")
        assert a == b
        return a

    def append(self, sids, cf, rng, sync=True):
        """One committed chunk per session of `sids` on every layer (commit on the last)."""
        from paper_2606_19271_b200 import TS_COMMIT
        sh = self.shape
        n = sum(cf) * sh.frame_tokens
        for layer in range(sh.n_layers):
            k, v = (synth.draw_bits(rng, n, sh.n_heads, sh.head_dim) for _ in range(2))
            last = layer == sh.n_layers - 1
            self.o.append(layer, sids, cf, k, v, commit=last)
            self.w.call("append", layer, sids, cf, k, v, TS_COMMIT if last else 0)

    def check(self, sids):
        assert self.w.call("pool", "ts_pool_free_list") == [int(x) for x in self.o.free]
        for sid in sids:
            assert self.w.call("pool", "ts_session_page_table", sid) == self.o.page_table(sid)
            info = self.w.call("pool", "ts_session_info", sid)
            oi = self.o.info(sid)
            assert (info["frames"], info["head_off"], info["n_pages"]) == (oi["frames"], oi["head_off"], oi["n_pages"])
            for layer in range(self.shape.n_layers):
                gk, gv = self.w.call("gather", layer, sid)
                ok, ov = self.o.gather_kv(layer, sid)
                assert np.array_equal(gk.reshape(ok.shape), ok) and np.array_equal(gv.reshape(ov.shape), ov)
        assert self.w.call("pool", "check_guards"), "a library write strayed outside the KV slab"

    def attention(self, layer, sids, cf, rng, scale):
        sh = self.shape
        n = sum(cf) * sh.frame_tokens
        q, k, v = (synth.draw_bits(rng, n, sh.n_heads, sh.head_dim) for _ in range(3))
        ref, _ = oracle.chunk_attention(self.o, layer, sids, cf, q, k, v, scale)
        bits = self.w.call("attention", layer, sids, cf, q, k, v, float(scale))
        got = synth.bf16_bits_to_f64(bits).reshape(ref.shape)
        assert np.isfinite(got).all()
        assert float(np.abs(got - ref).max()) <= MAX_ABS and rel_l2(got, ref) <= REL_L2

    def close(self):
        self.w.close()


def move(src, sid, dst, peer_src_on_dst, peer_dst_on_src):
    """freeze -> ticket -> import -> "enqueued" -> release, no synchronisation anywhere; the oracle does migrate_to."""
    ticket = src.w.call("pool", "ts_session_freeze", sid)
    assert ticket["pages"] == src.o.page_table(sid)
    new = dst.w.call("pool", "ts_session_import", peer_src_on_dst, ticket)
    src.w.call("pool", "ts_session_release", sid, peer_dst_on_src)
    assert new == src.o.migrate_to(sid, dst.o)
    return new


def _ipc_call(side, *call):
    """Registration calls: a box whose driver refuses CUDA IPC (a container without a shared IPC namespace) skips these tests
    instead of failing them - the library reports it as TS_ERR_CUDA; everything else still fails loudly."""
    from paper_2606_19271_b200 import TS_ERR_CUDA
    from paper_2606_19271_b200.worker import WorkerError
    try:
        return side.w.call(*call)
    except WorkerError as exc:
        if exc.code == TS_ERR_CUDA:
            pytest.skip(f"CUDA IPC is not available on this box: {exc}")
        raise


def register(side):
    return _ipc_call(side, "pool", "ts_pool_export")


def open_peer(side, blob):
    return _ipc_call(side, "pool", "ts_peer_open", blob)


@pytest.fixture
def pair():
    sides, peers = [], []

    def make(shape_a, order_a, shape_b, order_b):
        sides.append(Side(shape_a, order_a))
        sides.append(Side(shape_b, order_b))
        a, b = sides
        blob_a, blob_b = register(a), register(b)
        assert isinstance(blob_a, bytes) and len(blob_a) == 320
        peers.extend([(b, open_peer(b, blob_a)), (a, open_peer(a, blob_b))])
        return a, b, peers[0][1], peers[1][1]

    yield make
    for side, peer in peers:        # every mapping of a slab goes before the pool that exported it
        side.w.call("pool", "ts_peer_close", peer)
    for s in sides:
        s.close()


def test_session_moves_between_two_worker_processes_and_back(pair):
    NL, H, D, T, B, W = 2, 3, 128, 100, 64, 7
    rng = np.random.default_rng(60)
    sh_a = synth.PoolShape(NL, H, D, B, 72, T, W, 6)
    sh_b = synth.PoolShape(NL, H, D, B, 56, T, W, 4)      # another pool size: page ids differ on the two sides
    a, b, a_on_b, b_on_a = pair(sh_a, rng.permutation(72), sh_b, rng.permutation(56))
    scale = np.float32(1.0 / np.sqrt(D))
    s0, s1, s2 = a.open(), a.open(), a.open()
    x0 = b.open()
    a.append([s0, s1, s2], [2, 3, 1], rng)
    a.append([s1], [3], rng)                       # s1: 6 frames, window 7
    b.append([x0], [2], rng)
    a.check([s0, s1, s2])
    b.check([x0])

    # the move is requested right behind a committed append on the session: "state frozen" has to cover it
    a.append([s1], [1], rng)                       # 7 frames: the window is full
    t1 = move(a, s1, b, a_on_b, b_on_a)
    b.check([x0, t1])
    a.check([s0, s2])
    b.attention(1, [t1, x0], [2, 1], rng, scale)   # the migrated session serves its next chunk on the target
    # the freed pages of the source are handed out again at once (appends on other sessions), the freed id too
    a.append([s0, s2], [3, 3], rng)
    s3 = a.open()
    assert s3 == s1
    a.append([s3], [2], rng)
    a.check([s0, s2, s3])
    # the session lives on at the target: the window rolls (pages return to the target's free list), then it moves back
    b.append([t1, x0], [2, 1], rng)
    b.check([x0, t1])
    back = move(b, t1, a, b_on_a, a_on_b)
    a.check([s0, s2, s3, back])
    b.check([x0])
    a.attention(0, [back, s0, s3], [1, 2, 3], rng, scale)
    # a frozen session is held: every other call on it is refused, and the move can be called off
    from paper_2606_19271_b200 import TS_ERR_STATE
    from paper_2606_19271_b200.worker import WorkerError
    ticket = a.w.call("pool", "ts_session_freeze", s0)
    for call in (("pool", "ts_session_suspend", s0), ("pool", "ts_session_close", s0), ("pool", "ts_session_freeze", s0)):
        with pytest.raises(WorkerError) as err:
            a.w.call(*call)
        assert err.value.code == TS_ERR_STATE
    a.w.call("pool", "ts_session_unfreeze", s0)
    a.attention(0, [s0], [1], rng, scale)
    a.check([s0, s2, s3, back])
    del ticket


def test_import_verifies_the_ticket_and_leaves_the_target_unchanged_on_refusal(pair):
    from paper_2606_19271_b200 import TS_ERR_INVALID, TS_ERR_NO_PAGES
    from paper_2606_19271_b200.worker import WorkerError
    H, D, T, B = 2, 64, 40, 16
    rng = np.random.default_rng(61)
    sh_a = synth.PoolShape(1, H, D, B, 40, T, 0, 4)
    sh_b = synth.PoolShape(1, H, D, B, 12, T, 0, 4)       # too small for the 6-frame session (15 pages)
    a, b, a_on_b, b_on_a = pair(sh_a, None, sh_b, None)
    s = a.open()
    a.append([s], [3], rng)
    a.append([s], [3], rng)
    x = b.open()
    b.append([x], [1], rng)
    ticket = a.w.call("pool", "ts_session_freeze", s)
    with pytest.raises(WorkerError) as err:
        b.w.call("pool", "ts_session_import", a_on_b, ticket)
    assert err.value.code == TS_ERR_NO_PAGES
    for bad in (dict(ticket, head_off=B), dict(ticket, frames=ticket["frames"] + 4), dict(ticket, pages=[0, 1, 40]),
                dict(ticket, pages=[-1] + ticket["pages"][1:])):
        with pytest.raises(WorkerError) as err:
            b.w.call("pool", "ts_session_import", a_on_b, bad)
        assert err.value.code == TS_ERR_INVALID
    b.check([x])                                          # nothing changed on the target
    a.w.call("pool", "ts_session_unfreeze", s)            # the move is called off: the session serves on at the source
    a.append([s], [1], rng)
    a.check([s])
    # a geometry mismatch is caught at registration
    c = Side(synth.PoolShape(1, H, D, 32, 12, T, 0, 4), None)
    try:
        with pytest.raises(WorkerError) as err:
            c.w.call("pool", "ts_peer_open", a.w.call("pool", "ts_pool_export"))
        assert err.value.code == TS_ERR_INVALID
    finally:
        c.close()


def test_many_moves_with_chunks_in_between(pair):
    """Three sessions wander between the two workers for 30 moves while they keep generating chunks (windows roll, page
    tables wrap around both free lists, freed ids and pages are reused at once); state and bytes against the oracle every
    tenth move and at the end, attention on both workers at the end."""
    from paper_2606_19271_b200 import TS_ERR_STATE
    from paper_2606_19271_b200.worker import WorkerError
    NL, H, D, T, B, W = 1, 2, 64, 50, 16, 5
    rng = np.random.default_rng(62)
    sh = synth.PoolShape(NL, H, D, B, 80, T, W, 4)
    a, b, a_on_b, b_on_a = pair(sh, rng.permutation(80), sh, rng.permutation(80))
    sides = [a, b]
    peer_of_src_on = {0: b_on_a, 1: a_on_b}     # peer handle held by side i for the OTHER side's pool
    where = {}                                  # session tag -> (side index, sid)
    for tag in range(3):
        sid = a.open()
        a.append([sid], [int(rng.integers(1, 4))], rng)
        where[tag] = (0, sid)
    scale = np.float32(1.0 / np.sqrt(D))
    for mv in range(30):
        tag = int(rng.integers(0, 3))
        i, sid = where[tag]
        src, dst = sides[i], sides[1 - i]
        if rng.random() < 0.6:
            src.append([sid], [int(rng.integers(1, 3))], rng)          # the move follows a chunk without any wait
        if rng.random() < 0.2:                                         # a suspended session does not move
            src.w.call("pool", "ts_session_suspend", sid)
            src.o.suspend(sid)
            with pytest.raises(WorkerError) as err:
                src.w.call("pool", "ts_session_freeze", sid)
            assert err.value.code == TS_ERR_STATE
            src.w.call("pool", "ts_session_resume", sid)
            src.o.resume(sid)
        new = move(src, sid, dst, peer_of_src_on[1 - i], peer_of_src_on[i])
        where[tag] = (1 - i, new)
        if mv % 10 == 9:
            for k, side in enumerate(sides):
                side.check(sorted(s for (w, s) in where.values() if w == k))
    for k, side in enumerate(sides):
        mine = sorted(s for (w, s) in where.values() if w == k)
        side.check(mine)
        if mine:
            side.attention(0, mine, [1] * len(mine), rng, scale)


def test_scheduler_drives_three_worker_processes():
    """TurboServe in miniature, deployed as the paper deploys it: a session manager (this
    process: the ownership table, the closed-loop scheduler of Algorithm 1) and three GPU worker PROCESSES.  Every decision
    epoch the scheduler places the sessions and sets the budget; the manager carries the decisions out over the pipes -
    open / close, suspend of idle sessions, resume, freeze -> import -> release for every net migration - and every worker
    then runs one coalesced chunk step (one fused launch) for its active sessions.  The oracle (SchedulerOracle + one
    OraclePool per worker) is driven by the same events: decisions, page tables, free lists and KV bytes identical,
    attention within the north_star tolerance."""
    import paper_2606_19271_b200 as tc
    from test_scheduler_parity import event_stream, same
    T, K, M_max = 96, 3, 3
    shape = synth.PoolShape(n_layers=1, n_heads=2, head_dim=128, page_tokens=64, n_pages=K * 12 + 8, frame_tokens=T,
                            window_frames=6, max_sessions=K + 2)
    rng = np.random.default_rng(12)
    workers = [Side(shape, rng.permutation(shape.n_pages), host_pages=40 * 9) for _ in range(M_max)]
    peers = {}
    try:
        blobs = [register(w) for w in workers]
        for i in range(M_max):                    # peers[(i, j)]: worker j's pool as seen from worker i
            for j in range(M_max):
                if i != j:
                    peers[(i, j)] = open_peer(workers[i], blobs[j])
        cfg = dict(K=K, M_max=M_max, M0=1, l_hat=[0, 90, 174, 267], rho_hat=0.7, delta=0.1, eta=0.01, kappa_alpha=5.0,
                   kappa_beta=0.05)
        so, sg = oracle.SchedulerOracle(**cfg), tc.TurboSched(**cfg)
        scale = np.float32(1.0 / np.sqrt(128.0))
        where, suspended = {}, set()              # the ownership table: session uid -> (worker, local sid)
        n_mig = n_steps = n_resume = 0
        for it, ev in enumerate(event_stream(seed=5, n_events=60, cap=K * M_max, mean_on=2.0, mean_off=0.5, p_leave=0.06)):
            a, b = so.event(ev), sg.ts_sched_event(ev)
            same(a, b)
            live = {uid for uid, _, _ in ev}
            for uid in [u for u in where if u not in live]:                     # terminated
                w, sid = where.pop(uid)
                workers[w].o.close(sid)
                workers[w].w.call("pool", "ts_session_close", sid)
                suspended.discard(uid)
            for uid, alpha, _ in ev:
                g = b["phi"][uid]
                if uid not in where:
                    if g >= 0:
                        where[uid] = (g, workers[g].open())
                    continue
                w, sid = where[uid]
                if g < 0:
                    if uid not in suspended and not alpha:                      # went idle: offload, release the slot
                        workers[w].o.suspend(sid)
                        workers[w].w.call("pool", "ts_session_suspend", sid)
                        suspended.add(uid)
                    continue
                if uid in suspended:                                            # reactivated: restore where the copy is ...
                    workers[w].o.resume(sid)
                    workers[w].w.call("pool", "ts_session_resume", sid)
                    suspended.discard(uid)
                    n_resume += 1
                if g != w:                                                      # ... and move to the worker PLACE chose
                    where[uid] = (g, move(workers[w], sid, workers[g], peers[(g, w)], peers[(w, g)]))
                    n_mig += 1
            for g in b["alive"]:                                                # one coalesced chunk step per worker
                batch = sorted(sid for uid, (w, sid) in where.items() if w == g and b["phi"].get(uid, -1) == g)
                if not batch:
                    continue
                cf = [int(rng.integers(1, 3)) for _ in batch]
                q, k, v = (synth.draw_bits(rng, sum(cf) * T, shape.n_heads, shape.head_dim) for _ in range(3))
                side = workers[g]
                ref, _ = oracle.chunk_attention(side.o, 0, batch, cf, q, k, v, scale)
                side.o.append(0, batch, cf, k, v)
                got = synth.bf16_bits_to_f64(side.w.call("chunk_step", 0, batch, cf, q, k, v, float(scale), tc.TS_COMMIT))
                got = got.reshape(ref.shape)
                assert float(np.abs(got - ref).max()) <= MAX_ABS and rel_l2(got, ref) <= REL_L2
                n_steps += 1
            if it % 6 == 5 or it == 59:
                for g, side in enumerate(workers):
                    side.check([sid for uid, (w, sid) in where.items() if w == g and uid not in suspended])
        assert n_mig >= 3 and n_resume >= 2 and n_steps >= 40, (n_mig, n_resume, n_steps)
    finally:
        for (i, j), peer in peers.items():
            try:
                workers[i].w.call("pool", "ts_peer_close", peer)
            except Exception:
                pass
        for w in workers:
            w.close()
