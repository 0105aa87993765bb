"""Differential state-machine test: seeded random sequences of every lifecycle operation (open, close, append with and
without commit, attention, fused step, suspend, resume, migrate between two pools, and calls that must fail) applied to the
CUDA pools and to the oracle pools in lockstep.  Integers (ids, page tables, free lists, stats) are compared after every
operation, KV bytes at checkpoints, attention within tolerance, error codes by kind."""
import numpy as np
import pytest
import torch

import oracle
import synth
from helpers import DualPool, bits_to_dev

pytestmark = pytest.mark.gpu

KIND_OF = {-1: oracle.INVALID, -2: oracle.STATE, -3: oracle.NO_PAGES, -4: oracle.NO_HOST, -5: oracle.CAPACITY}


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_random_operation_sequences(seed):
    import paper_2606_19271_b200 as tc
    rng = np.random.default_rng(seed)
    T = int(rng.choice([24, 40, 130]))
    shape = synth.PoolShape(n_layers=2, n_heads=2, head_dim=int(rng.choice([64, 128])), page_tokens=int(rng.choice([16, 64])),
                            n_pages=96, frame_tokens=T, window_frames=5, max_sessions=5)
    pools = [DualPool(shape, rng.permutation(shape.n_pages), host_pages=40) for _ in range(2)]
    live = [dict(), dict()]                       # per pool: sid -> "R" | "S"
    scale = np.float32(1.0 / np.sqrt(shape.head_dim))
    n_fail = n_mig = n_att = 0

    def both(w, name, o_call, g_call):
        """Run the same operation on both sides; either both succeed (returning equal values) or both fail alike."""
        nonlocal n_fail
        try:
            a = o_call()
            err = None
        except oracle.OracleError as e:
            a, err = None, e.kind
        if err is None:
            b = g_call()
            assert a == b or a is None, (name, a, b)
            return True, a
        with pytest.raises(tc.TurboChunkError) as ex:
            g_call()
        assert KIND_OF[ex.value.code] == err, (name, ex.value.code, err)
        n_fail += 1
        return False, None

    for step in range(140):
        w = int(rng.integers(0, 2))
        dp, mine = pools[w], live[w]
        resident = sorted(s for s, st in mine.items() if st == "R")
        op = rng.choice(["open", "close", "append", "attend", "step", "suspend", "resume", "migrate", "bad"],
                        p=[0.12, 0.06, 0.2, 0.1, 0.14, 0.1, 0.1, 0.12, 0.06])
        if op == "open":
            ok, sid = both(w, op, dp.o.open, dp.g.ts_session_open)
            if ok:
                mine[sid] = "R"
        elif op == "close" and mine:
            sid = int(rng.choice(sorted(mine)))
            both(w, op, lambda: dp.o.close(sid), lambda: dp.g.ts_session_close(sid))
            del mine[sid]
        elif op in ("append", "attend", "step") and resident:
            k = int(rng.integers(1, len(resident) + 1))
            batch = [int(x) for x in rng.permutation(resident)[:k]]
            cf = [int(rng.integers(1, 4)) for _ in batch]
            n_tok = sum(cf) * T
            q, kk, vv = (synth.draw_bits(rng, n_tok, shape.n_heads, shape.head_dim) for _ in range(3))
            if op == "attend":
                dp.attention(int(rng.integers(0, 2)), batch, cf, q, kk, vv, scale, with_lse=bool(rng.integers(0, 2)))
                n_att += 1
            else:
                # one step of the protocol (R14): the same batch on every layer, TS_COMMIT (if at all) on the last one
                commit = bool(rng.integers(0, 2))
                dq, dk, dv = bits_to_dev(q), bits_to_dev(kk), bits_to_dev(vv)
                out = torch.empty_like(dq)
                for layer in range(shape.n_layers):
                    last = commit and layer == shape.n_layers - 1
                    flags = tc.TS_COMMIT if last else 0
                    if op == "append":
                        g_call = lambda: dp.g.ts_kv_append(layer, batch, cf, dk, dv, flags)
                    else:
                        g_call = lambda: dp.g.ts_chunk_step(layer, batch, cf, dq, dk, dv, out, None, float(scale), flags)
                    ok, _ = both(w, op, lambda: dp.o.append(layer, batch, cf, kk, vv, commit=last), g_call)
                    if not ok:
                        break
        elif op == "suspend" and resident:
            sid = int(rng.choice(resident))
            ok, _ = both(w, op, lambda: dp.o.suspend(sid), lambda: dp.g.ts_session_suspend(sid))
            if ok:
                mine[sid] = "S"
        elif op == "resume" and any(st == "S" for st in mine.values()):
            sid = int(rng.choice(sorted(s for s, st in mine.items() if st == "S")))
            ok, _ = both(w, op, lambda: dp.o.resume(sid), lambda: dp.g.ts_session_resume(sid))
            if ok:
                mine[sid] = "R"
        elif op == "migrate" and mine:
            sid = int(rng.choice(sorted(mine)))             # also suspended ones: must fail alike with STATE
            other = pools[1 - w]
            ok, new = both(w, op, lambda: dp.o.migrate_to(sid, other.o), lambda: dp.g.ts_session_migrate(sid, other.g))
            if ok:
                del mine[sid]
                live[1 - w][new] = "R"
                n_mig += 1
        elif op == "bad":
            sid = int(rng.integers(0, shape.max_sessions))  # often closed or suspended
            kk = synth.draw_bits(rng, T, shape.n_heads, shape.head_dim)
            dk = bits_to_dev(kk)
            both(w, op, lambda: dp.o.append(0, [sid, sid], [1, 1], np.concatenate([kk, kk]), np.concatenate([kk, kk])),
                 lambda: dp.g.ts_kv_append(0, [sid, sid], [1, 1], torch.cat([dk, dk]), torch.cat([dk, dk])))
        for x, l in zip(pools, live):
            x.check_state(sorted(l), kv=(step % 20 == 19 or step == 139))
    assert n_fail >= 5 and n_mig >= 3 and n_att >= 5
