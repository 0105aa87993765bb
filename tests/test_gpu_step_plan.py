"""ts_step_plan_*: the capture-safe multi-layer chunk step (PAPER.md:66 (iii) "invokes the model
once for the batch ... writes ... updated states back").  Against the oracle: attention of every layer and pass, appended
bytes, page tables and the window roll - run eagerly and as ONE CUDA graph captured at the first chunk step and replayed
for the later ones (the page tables, windows and schedules change between replays; the graph does not)."""
import numpy as np
import pytest
import torch

import oracle
import synth
from helpers import DualPool, bits_to_dev, rel_l2

pytestmark = pytest.mark.gpu


def draw(rng, n, shape):
    return synth.draw_bits(rng, n, shape.n_heads, shape.head_dim)


def _step_inputs(rng, shape, n_tok, NL):
    return [tuple(draw(rng, n_tok, shape) for _ in range(3)) for _ in range(NL)]


def _oracle_step(dp, sids, cf, layers_qkv, scale, passes):
    """Oracle: every pass attends on the unchanged caches (R5); the append of the last pass writes, commit on the last layer."""
    NL = len(layers_qkv)
    refs = []
    for layer, (q, k, v) in enumerate(layers_qkv):
        o_ref, l_ref = oracle.chunk_attention(dp.o, layer, sids, cf, q, k, v, scale)
        refs.append((o_ref, l_ref))
    for layer, (q, k, v) in enumerate(layers_qkv):
        dp.o.append(layer, sids, cf, k, v, commit=(layer == NL - 1))
    return refs


def _check_outputs(bufs, refs):
    torch.cuda.synchronize()
    for (dq, dk, dv, out, lse), (o_ref, l_ref) in zip(bufs, refs):
        o_gpu = out.double().cpu().numpy()
        assert np.isfinite(o_gpu).all()
        assert np.abs(o_gpu - o_ref).max() <= DualPool.MAX_ABS and rel_l2(o_gpu, o_ref) <= DualPool.REL_L2
        assert np.abs(lse.double().cpu().numpy() - l_ref).max() <= 2e-3


@pytest.mark.parametrize("page_tokens,use_graph", [(64, False), (256, False), (32, True), (256, True)])
def test_multilayer_step_plan_matches_oracle(page_tokens, use_graph):
    import paper_2606_19271_b200 as tc
    NL, H, D, T, W = 3, 3, 128, 90, 7
    shape = synth.PoolShape(NL, H, D, page_tokens, 64 * 256 // page_tokens, T, W, 4)
    rng = np.random.default_rng(100 + page_tokens + int(use_graph))
    dp = DualPool(shape, rng.permutation(shape.n_pages), host_pages=shape.n_pages)
    sids = [dp.open(), dp.open(), dp.open()]
    cf = [3, 1, 2]
    n_tok = sum(cf) * T
    scale = np.float32(1.0 / np.sqrt(D))
    passes = 2
    # one buffer set per layer (slot = layer); the graph is captured on these addresses, later steps copy new data in
    bufs = []
    plan = dp.g.ts_step_plan_create(sids, cf, n_slots=NL)
    for layer in range(NL):
        dq, dk, dv = (torch.empty(n_tok, H, D, dtype=torch.bfloat16, device="cuda") for _ in range(3))
        out = torch.full_like(dq, float("nan"))
        lse = torch.full((n_tok, H), float("nan"), dtype=torch.float32, device="cuda")
        plan.ts_step_plan_bind(layer, dq, dk, dv, out, lse)
        bufs.append((dq, dk, dv, out, lse))
    assert plan.ts_step_plan_block_bytes() > 0
    graph = None
    stream = torch.cuda.Stream()
    launches0 = dp.g.ts_pool_launch_count()

    def enqueue_runs(s):
        for p in range(passes):
            for layer in range(NL):
                plan.ts_step_plan_run(layer, layer, scale, tc.TS_RUN_APPEND if p == passes - 1 else 0, stream=s)

    for step in range(5):                                   # the 7-frame window binds from step 2 on and rolls every step
        layers_qkv = _step_inputs(rng, shape, n_tok, NL)
        refs = _oracle_step(dp, sids, cf, layers_qkv, scale, passes)
        for (dq, dk, dv, out, lse), (q, k, v) in zip(bufs, layers_qkv):
            dq.copy_(bits_to_dev(q)); dk.copy_(bits_to_dev(k)); dv.copy_(bits_to_dev(v))
            out.fill_(float("nan")); lse.fill_(float("nan"))
        torch.cuda.synchronize()
        with torch.cuda.stream(stream):
            plan.ts_step_plan_prepare(stream=stream)
            # inside a prepared step the sessions belong to the plan
            with pytest.raises(tc.TurboChunkError) as e:
                dp.g.ts_session_suspend(sids[0])
            assert e.value.code == tc.TS_ERR_STATE
            with pytest.raises(tc.TurboChunkError) as e:
                dp.g.ts_kv_append(0, sids[:1], cf[:1], bufs[0][1], bufs[0][2])
            assert e.value.code == tc.TS_ERR_STATE
            if not use_graph:
                enqueue_runs(stream)
            elif graph is None:
                graph = torch.cuda.CUDAGraph()
                stream.synchronize()
                with torch.cuda.graph(graph, stream=stream, capture_error_mode="thread_local"):
                    enqueue_runs(torch.cuda.current_stream())
                graph.replay()                              # capturing does not execute
            else:
                graph.replay()
            plan.ts_step_plan_commit(tc.TS_COMMIT, stream=stream)
        stream.synchronize()
        _check_outputs(bufs, refs)
        dp.check_state(sids)
    if use_graph:
        # the capture recorded NL * passes launches once; the four replays launched nothing through the host path
        assert dp.g.ts_pool_launch_count() - launches0 < 5 * NL * passes + 5 * (NL * 3 * 2 + 1)   # (check_state's gathers and uploads count too)
    # a suspended session in the batch: prepare fails with TS_ERR_STATE and changes nothing
    dp.suspend(sids[1])
    with pytest.raises(tc.TurboChunkError) as e:
        plan.ts_step_plan_prepare()
    assert e.value.code == tc.TS_ERR_STATE
    dp.check_state(sids)
    dp.resume(sids[1])
    # commit(0) abandons a prepared step: tables stay grown (as after an uncommitted append), nothing advances
    before = [dp.g.ts_session_info(s)["frames"] for s in sids]
    plan.ts_step_plan_prepare()
    plan.ts_step_plan_commit(0)
    assert [dp.g.ts_session_info(s)["frames"] for s in sids] == before
    torch.cuda.synchronize()
    plan.close()
    dp.g.close()


def test_step_plan_no_pages_changes_nothing():
    import paper_2606_19271_b200 as tc
    H, D, T = 2, 64, 100
    shape = synth.PoolShape(1, H, D, 64, 6, T, 0, 2)          # 6 pages of 64 tokens: a 3-frame chunk needs 5
    dp = DualPool(shape, None)
    a, b = dp.open(), dp.open()
    rng = np.random.default_rng(3)
    plan = dp.g.ts_step_plan_create([a, b], [3, 3])
    t = [torch.zeros(6 * T, H, D, dtype=torch.bfloat16, device="cuda") for _ in range(4)]
    plan.ts_step_plan_bind(0, *t)
    with pytest.raises(tc.TurboChunkError) as e:
        plan.ts_step_plan_prepare()
    assert e.value.code == tc.TS_ERR_NO_PAGES
    dp.check_state([a, b])
    with pytest.raises(tc.TurboChunkError) as e:
        plan.ts_step_plan_run(0, 0, 0.1)
    assert e.value.code == tc.TS_ERR_STATE                    # not prepared
    plan.close()
    dp.g.close()


def test_config3_two_layers_through_one_graph_sampled_rows():
    """configs[3] shape (4 sessions x 40 heads, full 21-frame window, B = 256) at NL = 2: the whole step (2 layers, attention
    + append each) captured as one graph; sampled rows of both layers against the oracle, appended bytes and the rolled
    window exact."""
    import paper_2606_19271_b200 as tc
    from helpers import dev_to_bits
    from synth.draw import draw_bits_torch
    from test_gpu_parity import _sampled_rows_check
    w = synth.wan14b_batch(n_layers=2)
    shape = w.shape
    T, H, D = shape.frame_tokens, shape.n_heads, shape.head_dim
    dp = DualPool(shape, w.free_order)
    gen = torch.Generator(device="cuda")
    gen.manual_seed(w.seed + 1)
    sids = [dp.open() for _ in w.sessions]
    for sid, spec in zip(sids, w.sessions):
        for f in range(0, spec.prior_frames, 3):
            for layer in range(2):
                dk = draw_bits_torch(gen, 3 * T, H, D, "cuda")
                dv = draw_bits_torch(gen, 3 * T, H, D, "cuda")
                dp.append(layer, [sid], [3], dev_to_bits(dk), dev_to_bits(dv), commit=(layer == 1), dev=(dk, dv))
    cf = [3] * len(sids)
    plan = dp.g.ts_step_plan_create(sids, cf, n_slots=2)
    bufs, chunks = [], []
    for layer in range(2):
        ch = [tuple(draw_bits_torch(gen, 3 * T, H, D, "cuda") for _ in range(3)) for _ in sids]
        dq, dk, dv = (torch.cat([c[i] for c in ch]) for i in range(3))
        out = torch.full_like(dq, float("nan"))
        lse = torch.empty(dq.shape[:2], dtype=torch.float32, device="cuda")
        plan.ts_step_plan_bind(layer, dq, dk, dv, out, lse)
        bufs.append((dq, dk, dv, out, lse))
        chunks.append(ch)
    stream = torch.cuda.Stream()
    torch.cuda.synchronize()
    with torch.cuda.stream(stream):
        plan.ts_step_plan_prepare(stream=stream)
        stream.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=stream, capture_error_mode="thread_local"):
            for layer in range(2):
                plan.ts_step_plan_run(layer, layer, float(w.scale), tc.TS_RUN_APPEND, stream=torch.cuda.current_stream())
        graph.replay()
        plan.ts_step_plan_commit(tc.TS_COMMIT, stream=stream)
    stream.synchronize()
    rs = np.random.default_rng(33)
    for layer in range(2):                                   # the oracle pool still holds the pre-step state
        dq, dk, dv, out, lse = bufs[layer]
        o_gpu = out.double().cpu().numpy()
        assert np.isfinite(o_gpu).all()
        _sampled_rows_check(dp, layer, sids, chunks[layer], o_gpu, lse, w, rs)
    for layer in range(2):
        dq, dk, dv, out, lse = bufs[layer]
        dp.o.append(layer, sids, cf, dev_to_bits(dk), dev_to_bits(dv), commit=(layer == 1))
    dp.check_state(sids[:1], kv=True)
    dp.check_state(sids[1:], kv=False)
    plan.close()
    dp.g.close()
