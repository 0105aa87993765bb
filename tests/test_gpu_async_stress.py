"""Stream-ordering stress: a long seeded sequence of chunk steps, suspends, resumes, closes and migrations on two tight pools
is ENQUEUED WITHOUT ANY HOST SYNCHRONISATION (the oracle is driven afterwards from the recorded script), so every hazard the
event timelines must cover is live: pages released by a suspend or a migration are immediately taken by the next append while
the copy out of them may still be running, a resumed session is attended to while its pages are still arriving, a migrated
session is stepped on the target while the source rewrites its old pages.  After one final synchronisation every logical
KV byte, page table and free list must equal the oracle's and every attention output must be within tolerance."""
import numpy as np
import pytest
import torch

import oracle
import synth
from helpers import DualPool, bits_to_dev

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("seed", [0, 1])
def test_enqueue_everything_then_compare(seed):
    import paper_2606_19271_b200 as tc
    rng = np.random.default_rng(300 + seed)
    T, H, D, B = 256, 12, 128, 64                       # 393 KB pages: copies take long enough to overlap what follows
    shape = synth.PoolShape(1, H, D, B, 150, T, 6, 5)
    pools = [DualPool(shape, rng.permutation(shape.n_pages), host_pages=200) for _ in range(2)]
    scale = np.float32(1.0 / np.sqrt(D))
    state = [dict(), dict()]                            # per pool: sid -> "R" / "S"
    script, outs = [], []
    torch.cuda.synchronize()
    for step in range(110):
        w = int(rng.integers(0, 2))
        g, mine = pools[w].g, state[w]
        res = sorted(s for s, st in mine.items() if st == "R")
        r = rng.random()
        try:
            if (r < 0.12 or step < 6) and len(mine) < shape.max_sessions:
                sid = g.ts_session_open()
                mine[sid] = "R"
                script.append(("open", w, sid))
            elif r < 0.55 and res:
                batch = [int(x) for x in rng.permutation(res)[:int(rng.integers(1, len(res) + 1))]]
                cf = [int(rng.integers(1, 4)) for _ in batch]
                q, k, v = (synth.draw_bits(rng, sum(cf) * T, H, D) for _ in range(3))
                dq, dk, dv = bits_to_dev(q), bits_to_dev(k), bits_to_dev(v)
                out = torch.full_like(dq, float("nan"))
                g.ts_chunk_step(0, batch, cf, dq, dk, dv, out, None, float(scale), tc.TS_COMMIT)
                script.append(("step", w, batch, cf, q, k, v))
                outs.append((len(script) - 1, out, (dq, dk, dv)))
            elif r < 0.70 and res:
                sid = int(rng.choice(res))
                g.ts_session_suspend(sid)
                mine[sid] = "S"
                script.append(("suspend", w, sid))
            elif r < 0.85 and any(st == "S" for st in mine.values()):
                sid = int(rng.choice(sorted(s for s, st in mine.items() if st == "S")))
                g.ts_session_resume(sid)
                mine[sid] = "R"
                script.append(("resume", w, sid))
            elif r < 0.95 and res and len(state[1 - w]) < shape.max_sessions:
                sid = int(rng.choice(res))
                new = g.ts_session_migrate(sid, pools[1 - w].g)
                del mine[sid]
                state[1 - w][new] = "R"
                script.append(("migrate", w, sid, new))
            elif mine:
                sid = int(rng.choice(sorted(mine)))
                g.ts_session_close(sid)
                del mine[sid]
                script.append(("close", w, sid))
        except tc.TurboChunkError as e:                 # out of pages / arena: nothing changed on the GPU side, skip
            assert e.code in (tc.TS_ERR_NO_PAGES, tc.TS_ERR_NO_HOST), e
    torch.cuda.synchronize()                            # ---- the only synchronisation
    refs = {}
    for i, op in enumerate(script):
        o = pools[op[1]].o
        if op[0] == "open":
            assert o.open() == op[2]
        elif op[0] == "step":
            _, _, batch, cf, q, k, v = op
            refs[i] = oracle.chunk_attention(o, 0, batch, cf, q, k, v, scale)[0]
            o.append(0, batch, cf, k, v)
        elif op[0] == "suspend":
            o.suspend(op[2])
        elif op[0] == "resume":
            o.resume(op[2])
        elif op[0] == "migrate":
            assert o.migrate_to(op[2], pools[1 - op[1]].o) == op[3]
        else:
            o.close(op[2])
    kinds = [op[0] for op in script]
    assert kinds.count("step") >= 12 and kinds.count("suspend") >= 3 and kinds.count("resume") >= 2 and kinds.count("migrate") >= 2
    for i, out, _ in outs:
        got = out.double().cpu().numpy()
        assert np.isfinite(got).all(), (i, script[i][2])
        assert np.abs(got - refs[i]).max() <= DualPool.MAX_ABS
        assert np.linalg.norm(got - refs[i]) / np.linalg.norm(refs[i]) <= DualPool.REL_L2
    for dp, mine in zip(pools, state):
        dp.check_state(sorted(mine))
