"""The pieces together on one B200: three pools stand for three GPU workers; the closed-loop scheduler (ts_sched_event,
PAPER.md Algorithm 1) decides placement and budget from a seeded bursty event stream, the runtime carries its decisions
out - open / close, suspend of idle sessions, resume, ts_session_migrate for every net migration - and every worker then
runs one coalesced chunk step (ts_chunk_step) for its active sessions.  The oracle pair (SchedulerOracle + one OraclePool
per worker) is driven by the same events; decisions, page tables, free lists and KV bytes must be identical, attention
within the north_star tolerance."""
import numpy as np
import pytest
import torch

import oracle
import synth
from helpers import DualPool, bits_to_dev
from test_scheduler_parity import event_stream, same

pytestmark = pytest.mark.gpu


def test_scheduler_drives_three_workers():
    import paper_2606_19271_b200 as tc
    T, K, M_max = 96, 3, 3
    shape = synth.PoolShape(n_layers=1, n_heads=2, head_dim=128, page_tokens=64, n_pages=K * 12 + 8, frame_tokens=T,
                            window_frames=6, max_sessions=K + 2)
    rng = np.random.default_rng(11)
    workers = [DualPool(shape, rng.permutation(shape.n_pages), host_pages=40 * 9) for _ in range(M_max)]
    cfg = dict(K=K, M_max=M_max, M0=1, l_hat=[0, 90, 174, 267], rho_hat=0.7, delta=0.1, eta=0.01, kappa_alpha=5.0,
               kappa_beta=0.05)
    so, sg = oracle.SchedulerOracle(**cfg), tc.TurboSched(**cfg)
    scale = np.float32(1.0 / np.sqrt(128.0))
    where = {}                      # session uid -> (worker index, local sid); the session's pages or host copy live there
    suspended = set()
    n_mig = n_steps = n_resume = 0
    for it, ev in enumerate(event_stream(seed=3, n_events=70, cap=K * M_max, mean_on=2.0, mean_off=0.5, p_leave=0.06)):
        a, b = so.event(ev), sg.ts_sched_event(ev)
        same(a, b)
        live = {uid for uid, _, _ in ev}
        for uid in [u for u in where if u not in live]:                         # terminated
            w, sid = where.pop(uid)
            workers[w].close(sid)
            suspended.discard(uid)
        for uid, alpha, _ in ev:
            g = b["phi"][uid]
            if uid not in where:
                if g >= 0:                                                      # new session: initialisation on its GPU
                    where[uid] = (g, workers[g].open())
                continue
            w, sid = where[uid]
            if g < 0:
                if uid not in suspended and not alpha:                          # went idle: offload, release the slot
                    workers[w].suspend(sid)
                    suspended.add(uid)
                continue
            if uid in suspended:                                                # reactivated: restore where the copy is ...
                workers[w].resume(sid)
                suspended.discard(uid)
                n_resume += 1
            if g != w:                                                          # ... and move to the GPU PLACE chose
                new = workers[w].o.migrate_to(sid, workers[g].o)
                assert workers[w].g.ts_session_migrate(sid, workers[g].g) == new
                where[uid] = (g, new)
                n_mig += 1
        for g in b["alive"]:                                                    # one coalesced chunk step per worker
            batch = sorted(sid for uid, (w, sid) in where.items() if w == g and b["phi"].get(uid, -1) == g)
            if not batch:
                continue
            cf = [int(rng.integers(1, 3)) for _ in batch]
            n_tok = sum(cf) * T
            q, k, v = (synth.draw_bits(rng, n_tok, shape.n_heads, shape.head_dim) for _ in range(3))
            dp = workers[g]
            if it % 4 == 0:
                dp.attention(0, batch, cf, q, k, v, scale, with_lse=False)
            dq, dk, dv = bits_to_dev(q), bits_to_dev(k), bits_to_dev(v)
            out = torch.empty_like(dq)
            dp.o.append(0, batch, cf, k, v)
            dp.g.ts_chunk_step(0, batch, cf, dq, dk, dv, out, None, float(scale), tc.TS_COMMIT)
            n_steps += 1
        if it % 6 == 5 or it == 69:
            for g, dp in enumerate(workers):
                dp.check_state([sid for uid, (w, sid) in where.items() if w == g])
    assert n_mig >= 3 and n_resume >= 3 and n_steps >= 60
