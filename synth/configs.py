"""Workload structure for BASELINE.json configs[0..4].

Only structure lives here: shapes, per-session prior lengths, the free-list
permutation ("pages at random pool slots" is injected as DATA, SURVEY.md §8(c)
R9), the churn event script, and FLOP counting for reporting.  Structure draws
come first from one `numpy.random.default_rng(seed)`: per-session prior lengths
(cfg[2] only), then `free_order = rng.permutation(n_pages)`; the same `rng` is
then handed to `synth.draw` for the tensors (host path).
"""
from dataclasses import dataclass, field
from typing import List

import numpy as np


@dataclass(frozen=True)
class PoolShape:
    n_layers: int
    n_heads: int
    head_dim: int
    page_tokens: int      # B
    n_pages: int
    frame_tokens: int     # T
    window_frames: int    # W; 0 = no cap
    max_sessions: int


@dataclass(frozen=True)
class SessionSpec:
    prior_frames: int     # P_s
    chunk_frames: int     # c_s


@dataclass
class Workload:
    name: str
    seed: int
    shape: PoolShape
    sessions: List[SessionSpec]
    free_order: np.ndarray              # int32 permutation of 0..n_pages-1
    scale: np.float32                   # softmax scale, fp32 (R2)
    rng: np.random.Generator = field(repr=False, default=None)   # positioned after the structure draws


def _scale(head_dim):
    return np.float32(1.0 / np.sqrt(np.float32(head_dim)))


def tiny(seed=0):
    """configs[0]: 2 sessions, H=2, D=64, T=16, c=2, B=16, priors 0 and 3 frames, permuted pages."""
    shape = PoolShape(n_layers=1, n_heads=2, head_dim=64, page_tokens=16, n_pages=16,
                      frame_tokens=16, window_frames=0, max_sessions=4)
    rng = np.random.default_rng(seed)
    free_order = rng.permutation(shape.n_pages).astype(np.int32)
    sessions = [SessionSpec(0, 2), SessionSpec(3, 2)]
    return Workload("tiny", seed, shape, sessions, free_order, _scale(64), rng)


def wan13b_single(seed=1):
    """configs[1]: one session, H=12, D=128, T=1560, c=3, P=6, B=256, identity placement."""
    shape = PoolShape(n_layers=1, n_heads=12, head_dim=128, page_tokens=256, n_pages=64,
                      frame_tokens=1560, window_frames=21, max_sessions=4)
    rng = np.random.default_rng(seed)
    free_order = np.arange(shape.n_pages, dtype=np.int32)
    return Workload("wan13b_single", seed, shape, [SessionSpec(6, 3)], free_order, _scale(128), rng)


def wan13b_batch(seed=2, n_sessions=8, extra_pages=0):
    """configs[2]: 8 sessions, priors 3*U{0..6} frames, W=21, pages permuted."""
    n_pages = 129 * (n_sessions + 1) + extra_pages
    shape = PoolShape(n_layers=1, n_heads=12, head_dim=128, page_tokens=256, n_pages=n_pages,
                      frame_tokens=1560, window_frames=21, max_sessions=32)
    rng = np.random.default_rng(seed)
    priors = 3 * rng.integers(0, 7, size=n_sessions)
    free_order = rng.permutation(shape.n_pages).astype(np.int32)
    sessions = [SessionSpec(int(p), 3) for p in priors]
    return Workload("wan13b_batch", seed, shape, sessions, free_order, _scale(128), rng)


def wan14b_batch(seed=3, n_layers=40):
    """configs[3]: 4 sessions, H=40, P=18 (full window), NL layers with distinct slabs."""
    shape = PoolShape(n_layers=n_layers, n_heads=40, head_dim=128, page_tokens=256, n_pages=4 * 129 + 4,
                      frame_tokens=1560, window_frames=21, max_sessions=8)
    rng = np.random.default_rng(seed)
    free_order = np.arange(shape.n_pages, dtype=np.int32)
    sessions = [SessionSpec(18, 3) for _ in range(4)]
    return Workload("wan14b_batch", seed, shape, sessions, free_order, _scale(128), rng)


CONFIG_BUILDERS = {"tiny": tiny, "wan13b_single": wan13b_single, "wan13b_batch": wan13b_batch,
                   "wan14b_batch": wan14b_batch}


def attention_pairs(prior_frames, chunk_frames, frame_tokens, window_frames):
    """Visible (query, key) pairs per head for one session (SURVEY.md §8(d) formula):
    sum_f T * (min(P, W-c)*T + (f+1)*T); masked pairs are not counted."""
    T, c = frame_tokens, chunk_frames
    vis_prior = prior_frames if window_frames <= 0 else min(prior_frames, window_frames - c)
    return sum(T * (vis_prior * T + (f + 1) * T) for f in range(c))


def attention_flops(shape, sessions):
    """4*D FLOP per visible pair per head (QK^T 2D + PV 2D); exp/max/rescale not counted."""
    pairs = sum(attention_pairs(s.prior_frames, s.chunk_frames, shape.frame_tokens, shape.window_frames)
                for s in sessions)
    return 4 * shape.head_dim * shape.n_heads * pairs


def churn_script(seed=4, n_steps=200, cap=32, mean_off=4.0, mean_on=24.0, p_off_on=0.05, p_on_off=0.10,
                 chunk_frames=3, lifetime_mu=2.0, lifetime_sigma=1.0):
    """configs[4]: seeded on/off Markov-modulated Poisson session churn (SURVEY.md §8(d) cfg[4]).

    Sessions are named by a monotonically increasing uid (the runner maps uid -> library sid).
    Per step the script lists, in execution order:
      'suspend': uids (resident since the previous step) suspended before this step runs,
      'resume': uids to resume, 'open': uids to open, 'batch': uids served this step (attention +
      append/commit, in this order), 'close': uids closed after the step (lifetime exhausted).
    Rules: mode chain off<->on; n_t = min(cap, Poisson(mean)); the active set keeps still-alive
    previously-active sessions (lowest uid first) up to n_t, the surplus is suspended; a deficit is
    filled by a fair coin between resuming the longest-suspended session and opening a new one (new
    when none is suspended); lifetime in chunks = ceil(lognormal(mu, sigma)), decremented per served
    chunk, close at 0.
    """
    rng = np.random.default_rng(seed)
    mode_on = False
    next_uid = 0
    life = {}
    active = []        # uids resident and served last step
    suspended = []     # FIFO, longest-suspended first
    steps = []
    for _ in range(n_steps):
        flip = rng.random()
        if mode_on and flip < p_on_off:
            mode_on = False
        elif (not mode_on) and flip < p_off_on:
            mode_on = True
        n_t = int(min(cap, rng.poisson(mean_on if mode_on else mean_off)))
        ev = {"suspend": [], "resume": [], "open": [], "batch": [], "close": []}
        active.sort()
        keep, surplus = active[:n_t], active[n_t:]
        ev["suspend"] = list(surplus)
        suspended.extend(surplus)
        batch = list(keep)
        while len(batch) < n_t:
            take_old = bool(suspended) and rng.random() < 0.5
            if take_old:
                u = suspended.pop(0)
                ev["resume"].append(u)
            else:
                u = next_uid
                next_uid += 1
                life[u] = int(np.ceil(rng.lognormal(lifetime_mu, lifetime_sigma)))
                ev["open"].append(u)
            batch.append(u)
        ev["batch"] = list(batch)
        ev["chunk_frames"] = [chunk_frames] * len(batch)
        nxt = []
        for u in batch:
            life[u] -= 1
            if life[u] <= 0:
                ev["close"].append(u)
            else:
                nxt.append(u)
        active = nxt
        ev["mode_on"] = mode_on
        steps.append(ev)
    return steps


def sched_events(seed, n_events, cap, p_on=0.05, p_off=0.10, mean_off=0.4, mean_on=3.0, p_leave=0.04, p_flip=0.15):
    """Seeded event stream for the closed-loop scheduler (§5.1 "event-driven scheduling"): per event the list of
    live sessions `(id, alpha, state size in MB)`.  Structure: bursty on/off arrivals (an off/on Markov chain modulating a
    Poisson arrival count, the shape PAPER.md:36-38 describes), departures, active <-> idle flips; now and then the
    sessions are listed in a shuffled order.  The paper's production traces are not available; this stands in for them."""
    rng = np.random.default_rng(seed)
    live, next_id, on = {}, 0, False
    for _ in range(n_events):
        on = (rng.random() < p_on) if not on else (rng.random() >= p_off)
        for sid in list(live):
            u = rng.random()
            if u < p_leave:
                del live[sid]
            elif u < p_leave + p_flip:
                live[sid] = (1 - live[sid][0], live[sid][1])
        for _ in range(rng.poisson(mean_on if on else mean_off)):
            if len(live) < cap:
                live[next_id] = (1, float(rng.integers(30, 210)) + 0.25 * float(rng.integers(0, 4)))
                next_id += 1
        order = sorted(live) if rng.random() < 0.8 else [int(x) for x in rng.permutation(sorted(live))]
        yield [(sid, live[sid][0], live[sid][1]) for sid in order]
