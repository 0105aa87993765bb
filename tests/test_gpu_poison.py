"""The library needs no initialised KV slab (include/turbochunk.h): no result may depend on a byte it has not written itself.

Every DualPool of the suite starts NaN-filled and re-poisons its free pages at each state check; the cases here aim at the
places where a masked operand could still reach such bytes ("isolated per-session state regions"):
  * page tables grown BEFORE the attention that runs on them - the fused ts_chunk_step, and layers > 0 of a multi-layer step
    whose layer-0 append has already popped the new pages (their bytes in layer l are stale until layer l's own append);
  * page sizes below the 128-key tile (B = 16, 32, 64), where the last cache tile spans several table entries;
  * pages recycled from a closed / suspended / migrated session;
  * the target pool of a migration.
Two poisons: bf16 NaN (0 x NaN = NaN inside the MMA) and the largest finite bf16 (a masked weight that is tiny instead of
exactly zero would leak 3.4e38 x 2^-125 ~ 8 into the output)."""
import numpy as np
import pytest
import torch

import oracle
import synth
from helpers import DualPool, bits_to_dev, rel_l2

pytestmark = pytest.mark.gpu

POISONS = [DualPool.NAN_BF16, DualPool.HUGE_BF16]


def draw(rng, n, shape):
    return synth.draw_bits(rng, n, shape.n_heads, shape.head_dim)


@pytest.mark.parametrize("poison", POISONS)
@pytest.mark.parametrize("page_tokens", [16, 32, 64, 256])
@pytest.mark.parametrize("fused", [False, True])
def test_multilayer_step_on_grown_tables(poison, page_tokens, fused):
    """Three layers; layer 0's (uncommitted) append grows the page tables, then layers 1 and 2 attend on the grown tables."""
    NL, H, D, T = 3, 3, 128, 50       # 50 tokens per frame: the last cache tile is partial for every prior length used here
    shape = synth.PoolShape(NL, H, D, page_tokens, 40 * 256 // page_tokens, T, 7, 4)
    rng = np.random.default_rng(page_tokens + int(fused))
    dp = DualPool(shape, rng.permutation(shape.n_pages), poison=poison)
    sids = [dp.open(), dp.open(), dp.open()]
    cf = [2, 1, 3]
    scale = np.float32(1.0 / np.sqrt(D))
    for step in range(5):                                     # the window (7) binds and rolls from step 2 on
        n_tok = sum(cf) * T
        for layer in range(NL):
            q, k, v = (draw(rng, n_tok, shape) for _ in range(3))
            if fused:
                dp.fused_step(layer, sids, cf, q, k, v, scale, commit=(layer == NL - 1))
            else:
                dp.attention(layer, sids, cf, q, k, v, scale)
                dp.append(layer, sids, cf, k, v, commit=(layer == NL - 1))
        dp.check_state(sids)
    dp.g.close()


@pytest.mark.parametrize("poison", POISONS)
def test_recycled_pages_and_migration_target(poison):
    """Pages that return to the free list are re-poisoned (check_state), then handed to other sessions by append, resume and
    migration; every attention that follows must be finite and within tolerance."""
    H, D, T, B = 2, 64, 37, 32
    shape = synth.PoolShape(2, H, D, B, 96, T, 6, 6)
    rng = np.random.default_rng(5)
    src = DualPool(shape, rng.permutation(shape.n_pages), host_pages=96, poison=poison)
    dst = DualPool(shape, rng.permutation(shape.n_pages), poison=poison)
    scale = np.float32(0.2)

    def step(dp, sids, cf):
        n_tok = sum(cf) * T
        for layer in range(2):
            q, k, v = (draw(rng, n_tok, shape) for _ in range(3))
            dp.fused_step(layer, sids, cf, q, k, v, scale, commit=(layer == 1))
        dp.check_state(sids)

    a, b, c = src.open(), src.open(), src.open()
    for _ in range(3):
        step(src, [a, b, c], [2, 3, 1])
    src.close(b)                                              # b's pages go back, poisoned at the next check
    src.suspend(c)
    src.check_state([a, c])
    step(src, [a], [3])                                       # a grows into recycled pages
    src.resume(c)
    step(src, [c, a], [1, 2])
    # migrate a into the (entirely poisoned) target pool and keep stepping there
    new_o = src.o.migrate_to(a, dst.o)
    new_g = src.g.ts_session_migrate(a, dst.g)
    assert new_o == new_g
    dst.check_state([new_g])
    src.check_state([c])
    other = dst.open()
    step(dst, [new_g, other], [2, 3])
    step(dst, [other, new_g], [3, 3])
    src.g.close()
    dst.g.close()


@pytest.mark.parametrize("poison", POISONS)
def test_single_tile_plans_and_lone_tiles_under_poison(poison):
    """One small session: the scheduler takes single-tile items (lone tiles split over both TMEM slots); B = 16."""
    H, D, T, B = 1, 128, 72, 16
    shape = synth.PoolShape(1, H, D, B, 128, T, 0, 2)
    rng = np.random.default_rng(8)
    dp = DualPool(shape, rng.permutation(shape.n_pages), poison=poison)
    sid = dp.open()
    scale = np.float32(0.09)
    for cf in (1, 3, 2, 1, 3):
        q, k, v = (draw(rng, cf * T, shape) for _ in range(3))
        dp.fused_step(0, [sid], [cf], q, k, v, scale)
        dp.check_state([sid])
    dp.g.close()
