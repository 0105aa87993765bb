"""Seeded shape fuzz of the coalesced step against the oracle: frame sizes from 1 token to several tiles, page sizes from 16
to 512 tokens, 1-12 heads, both head dims, 1-8 sessions with ragged priors and chunk lengths, windows that clamp and roll,
one or two layers, three softmax scales, on a NaN-poisoned slab.  Each case runs attention (tolerance of the north_star), the fused
step on every layer with the commit on the last (its output against the oracle; page tables, free list, KV bytes exact) and a second attention over the grown caches in reversed
batch order.  The work-tile scheduler sees pairs, odd items, lone tiles, single-tile plans and unrelated items sharing a
cluster across these cases."""
import numpy as np
import pytest
import torch

import synth
from helpers import DualPool, bits_to_dev

pytestmark = pytest.mark.gpu


def run_case(seed, large, use_plan=False):
    import paper_2606_19271_b200 as tc
    rng = np.random.default_rng(1000 + seed)
    if large:
        T = int(rng.choice([64, 128, 130, 200, 257, 390, 520, 777]))
        H, n, W = int(rng.integers(1, 13)), int(rng.integers(1, 9)), int(rng.choice([0, 6, 9, 21]))
        priors_hi = 16
    else:
        T = int(rng.choice([1, 3, 17, 64, 100, 128, 130, 200, 257, 390]))
        H, n, W = int(rng.integers(1, 5)), int(rng.integers(1, 6)), int(rng.choice([0, 4, 6, 9]))
        priors_hi = 11
    D = int(rng.choice([64, 128]))
    B = int(rng.choice([16, 32, 64, 128, 256, 512]))
    NL = int(rng.integers(1, 3))
    cmax = 3 if W == 0 else min(3, W)
    cf = [int(rng.integers(1, cmax + 1)) for _ in range(n)]
    priors = [int(rng.integers(0, priors_hi)) for _ in range(n)]
    n_pages = sum(-(-(p + c + 1) * T // B) + 2 for p, c in zip(priors, cf)) + 8
    shape = synth.PoolShape(NL, H, D, B, n_pages, T, W, n + 1)
    dp = DualPool(shape, rng.permutation(n_pages))
    sids = [dp.open() for _ in range(n)]
    for sid, P in zip(sids, priors):
        if P:
            dp.feed_prior(sid, [synth.draw_bits(rng, P * T, H, D) for _ in range(NL)],
                          [synth.draw_bits(rng, P * T, H, D) for _ in range(NL)], frames_per_append=int(rng.integers(1, cmax + 1)))
    q, k, v = (synth.draw_bits(rng, sum(cf) * T, H, D) for _ in range(3))
    scale = np.float32(rng.choice([0.05, 1.0 / np.sqrt(D), 0.3]))
    layer = int(rng.integers(0, NL))
    dp.attention(layer, sids, cf, q, k, v, scale)
    dev = (bits_to_dev(q), bits_to_dev(k), bits_to_dev(v))
    if use_plan:        # the same step through the capture-safe plan calls (one prepare, NL x 2 launches, one commit)
        dp.plan_step(sids, cf, q, k, v, scale, NL, passes=2)
    for l in range(0 if use_plan else NL):
        # layer l > 0 runs on page tables that layer 0's uncommitted append has already grown: the slab is NaN-poisoned
        # (DualPool), so a gather that strays onto a not-yet-written page shows up in `out`, which is compared here
        dp.fused_step(l, sids, cf, q, k, v, scale, commit=(l == NL - 1), dev=dev)
    dp.check_state(sids)
    q2, k2, v2 = (synth.draw_bits(rng, n * T, H, D) for _ in range(3))
    dp.attention(layer, sids[::-1], [1] * n, q2, k2, v2, scale)
    dp.g.close()


@pytest.mark.parametrize("seed", range(0, 24))
def test_small_shapes(seed):
    run_case(seed, large=False)


@pytest.mark.parametrize("seed", range(200, 208))
def test_larger_shapes(seed):
    run_case(seed, large=True)


@pytest.mark.parametrize("seed", range(400, 412))
def test_shapes_through_step_plan(seed):
    run_case(seed, large=(seed % 3 == 0), use_plan=True)
