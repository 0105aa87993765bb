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


# ---------------------------------------------------------------------------------------------------------
# GPU-side helpers (imported lazily so that the CPU-only tests never touch the CUDA binding)
# ---------------------------------------------------------------------------------------------------------
def bits_to_dev(bits, device="cuda"):
    """uint16 bf16 bit patterns (numpy) -> torch bf16 tensor on the device (no value change)."""
    import torch
    return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).to(device).view(torch.bfloat16)


def dev_to_bits(t):
    """torch bf16 tensor -> numpy uint16 bit patterns."""
    import torch
    return t.contiguous().view(torch.int16).cpu().numpy().view(np.uint16)


class DualPool:
    """Drives the oracle pool and the CUDA pool with the same operations and compares what is unique:
    page tables, free list, (len, head_off, n_pages), logical KV bytes (bit-exact) and attention output
    (max-abs <= 2e-2, rel-L2 <= 5e-3 against fp64 — BASELINE.json north_star)."""

    MAX_ABS, REL_L2 = 2e-2, 5e-3
    NAN_BF16, HUGE_BF16 = 0x7FC0, 0x7F7F

    def __init__(self, shape, free_order=None, host_pages=0, poison=NAN_BF16, device=0):
        """Every test pool starts with its whole KV slab filled with bf16 NaN (`poison`; None: torch.empty), and every state
        check refills the pages on the free list: a result that depends on a byte the library has not written itself (a
        stale page behind a grown table, a recycled page) turns into a NaN in the output instead of passing by luck."""
        from paper_2606_19271_b200 import TurboChunkPool
        self.shape = shape
        self.dev = f"cuda:{device}"
        self.o = make_oracle_pool(shape, free_order, host_pages if host_pages else None)
        self.g = TurboChunkPool(shape.n_layers, shape.n_heads, shape.head_dim, shape.page_tokens, shape.n_pages,
                                shape.frame_tokens, shape.window_frames, shape.max_sessions,
                                free_order=free_order, host_pages=host_pages, guard_bytes=1 << 20, poison=poison,
                                device=device)

    def open(self):
        a, b = self.o.open(), self.g.ts_session_open()
        assert a == b
        return a

    def close(self, sid):
        self.o.close(sid)
        self.g.ts_session_close(sid)

    def append(self, layer, sids, cf, k_bits, v_bits, commit=True, dev=None):
        from paper_2606_19271_b200 import TS_COMMIT
        self.o.append(layer, sids, cf, k_bits, v_bits, commit=commit)
        dk, dv = dev if dev is not None else (bits_to_dev(k_bits, self.dev), bits_to_dev(v_bits, self.dev))
        self.g.ts_kv_append(layer, sids, cf, dk, dv, TS_COMMIT if commit else 0)

    def feed_prior(self, sid, k_layers, v_layers, frames_per_append=3):
        T = self.shape.frame_tokens
        n_frames = k_layers[0].shape[0] // T
        f = 0
        while f < n_frames:
            c = min(frames_per_append, n_frames - f)
            lo, hi = f * T, (f + c) * T
            for layer in range(len(k_layers)):
                self.append(layer, [sid], [c], k_layers[layer][lo:hi], v_layers[layer][lo:hi],
                            commit=(layer == len(k_layers) - 1))
            f += c

    def suspend(self, sid):
        self.o.suspend(sid)
        self.g.ts_session_suspend(sid)

    def resume(self, sid):
        self.o.resume(sid)
        self.g.ts_session_resume(sid)

    def attention(self, layer, sids, cf, q_bits, k_bits, v_bits, scale, check=True, with_lse=True):
        import torch
        o_ref, lse_ref = oracle.chunk_attention(self.o, layer, sids, cf, q_bits, k_bits, v_bits, scale)
        dq, dk, dv = (bits_to_dev(x, self.dev) for x in (q_bits, k_bits, v_bits))
        out = torch.full_like(dq, float("nan"))
        lse = torch.full(dq.shape[:2], float("nan"), dtype=torch.float32, device=dq.device) if with_lse else None
        self.g.ts_chunk_attention(layer, sids, cf, dq, dk, dv, out, lse, float(scale))
        torch.cuda.synchronize(self.dev)
        o_gpu = out.double().cpu().numpy()
        if check:
            assert np.isfinite(o_gpu).all()
            max_abs = float(np.abs(o_gpu - o_ref).max())
            rl2 = rel_l2(o_gpu, o_ref)
            assert max_abs <= self.MAX_ABS and rl2 <= self.REL_L2, (max_abs, rl2)
            if with_lse:
                l_gpu = lse.double().cpu().numpy()
                assert np.abs(l_gpu - lse_ref).max() <= 2e-3, float(np.abs(l_gpu - lse_ref).max())
        return o_gpu, o_ref

    def fused_step(self, layer, sids, cf, q_bits, k_bits, v_bits, scale, commit=True, dev=None):
        """ts_chunk_step (attention + append in one launch) against oracle attention followed by oracle append; the fused
        launch's `out` is compared like a plain attention's."""
        import torch
        from paper_2606_19271_b200 import TS_COMMIT
        o_ref, _ = oracle.chunk_attention(self.o, layer, sids, cf, q_bits, k_bits, v_bits, scale)
        self.o.append(layer, sids, cf, k_bits, v_bits, commit=commit)
        dq, dk, dv = dev if dev is not None else tuple(bits_to_dev(x, self.dev) for x in (q_bits, k_bits, v_bits))
        out = torch.full_like(dq, float("nan"))
        self.g.ts_chunk_step(layer, sids, cf, dq, dk, dv, out, None, float(scale), TS_COMMIT if commit else 0)
        torch.cuda.synchronize(self.dev)
        o_gpu = out.double().cpu().numpy()
        assert np.isfinite(o_gpu).all(), "fused step: non-finite output (a masked operand read bytes the library never wrote)"
        max_abs = float(np.abs(o_gpu - o_ref).max())
        rl2 = rel_l2(o_gpu, o_ref)
        assert max_abs <= self.MAX_ABS and rl2 <= self.REL_L2, (max_abs, rl2)
        return o_gpu, o_ref

    def plan_step(self, sids, cf, q_bits, k_bits, v_bits, scale, n_layers, passes=1):
        """A whole multi-layer chunk step through ts_step_plan_* (one buffer set, the same tensors on every layer; attention-only
        launches for all passes but the last, which also appends; TS_COMMIT) against the oracle's attention per layer, appends on
        every layer and the commit on the last."""
        import torch
        from paper_2606_19271_b200 import TS_COMMIT, TS_RUN_APPEND
        refs = [oracle.chunk_attention(self.o, l, sids, cf, q_bits, k_bits, v_bits, scale)[0] for l in range(n_layers)]
        for l in range(n_layers):
            self.o.append(l, sids, cf, k_bits, v_bits, commit=(l == n_layers - 1))
        dq, dk, dv = (bits_to_dev(x, self.dev) for x in (q_bits, k_bits, v_bits))
        outs = [torch.full_like(dq, float("nan")) for _ in range(n_layers)]
        plan = self.g.ts_step_plan_create(sids, cf, n_slots=n_layers)
        for l in range(n_layers):
            plan.ts_step_plan_bind(l, dq, dk, dv, outs[l], None)
        plan.ts_step_plan_prepare()
        for p in range(passes):
            for l in range(n_layers):
                plan.ts_step_plan_run(l, l, float(scale), TS_RUN_APPEND if p == passes - 1 else 0)
        plan.ts_step_plan_commit(TS_COMMIT)
        torch.cuda.synchronize(self.dev)
        plan.close()
        for l in range(n_layers):
            o_gpu = outs[l].double().cpu().numpy()
            assert np.isfinite(o_gpu).all(), "step plan: non-finite output"
            max_abs, rl2 = float(np.abs(o_gpu - refs[l]).max()), rel_l2(o_gpu, refs[l])
            assert max_abs <= self.MAX_ABS and rl2 <= self.REL_L2, (l, max_abs, rl2)

    def check_state(self, sids, layers=None, kv=True):
        import torch
        # compute-sanitizer is closed on the GPU pool: 1 MiB guard bands around the slab and the pinned arena stand in for it
        assert self.g.check_guards(), "a library write strayed outside the KV slab or the pinned arena"
        assert list(self.o.free) == self.g.ts_pool_free_list()
        st_o, st_g = self.o.stats(), self.g.ts_pool_stats()
        for key in ("free_pages", "resident", "suspended", "host_pages_used"):
            assert st_o[key] == st_g[key], (key, st_o, st_g)
        for sid in sids:
            io, ig = self.o.info(sid), self.g.ts_session_info(sid)
            assert ig["state"] == (1 if io["state"] == oracle.RESIDENT else 2)
            for key in ("frames", "len_tokens", "head_off", "n_pages"):
                assert io[key] == ig[key], (sid, key, io, ig)
            assert self.o.page_table(sid) == self.g.ts_session_page_table(sid)
            if kv and io["state"] == oracle.RESIDENT:
                for layer in (layers if layers is not None else range(self.shape.n_layers)):
                    gk, gv = self.g.ts_gather_kv(layer, sid)
                    torch.cuda.synchronize(self.dev)
                    ok, ov = self.o.gather_kv(layer, sid)
                    assert np.array_equal(dev_to_bits(gk), ok), f"K bytes differ sid={sid} layer={layer}"
                    assert np.array_equal(dev_to_bits(gv), ov), f"V bytes differ sid={sid} layer={layer}"
        self.g.poison_free_pages()
