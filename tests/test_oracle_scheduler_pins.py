"""Pins S1-S6 for the oracle of the closed-loop scheduler (oracle/scheduler.py; §5.2, Algorithm 1, App. A).
Closed forms from the paper's own formulas with hand-computed numbers, exhaustive search on tiny instances (the paper's
"placement oracle"), hand-worked move sequences, invariants of Eq. (1), and numpy.std for Eq. (6)."""
import itertools

import numpy as np

from oracle import SchedulerOracle

LHAT5 = [0, 90, 174, 267, 350, 441]      # ms, the measured l_hat(n) of DESIGN.md §7.2 (30 layers x 4 passes), n = 0..5


def sess(ids, active=True, mb=200.0):
    return [(i, 1 if active else 0, mb) for i in ids]


# ---- S1: M_tar = ceil(N_req / (K rho_hat)) and the hysteresis band, numbers worked by hand ------------
def test_s1_proportional_target_and_hysteresis():
    s = SchedulerOracle(K=5, M_max=64, M0=1, l_hat=LHAT5, rho_hat=0.7, delta=0.1)
    # scale-out: rho_max = 1.0 > 0.8.  10 / 3.5 = 2.857 -> 3 ; 23 / 3.5 = 6.571 -> 7 ; 35 / 3.5 = 10 exactly -> 10
    assert s.scale(1.0, 1, 10) == 3
    assert s.scale(1.0, 1, 23) == 7
    assert s.scale(1.0, 1, 35) == 10
    # scale-in: rho_max = 0.4 < 0.6.  7 / 3.5 = 2 -> 2
    assert s.scale(0.4, 6, 7) == 2
    # inside the band [0.6, 0.8]: the budget stays, whatever the proportional target says
    assert s.scale(0.6, 6, 7) == 6 and s.scale(0.8, 6, 7) == 6 and s.scale(0.7, 1, 23) == 1
    # R29: a scale-out trigger never shrinks, a scale-in trigger never grows, M_max caps, feasibility floors
    assert s.scale(1.0, 9, 10) == 9 and s.scale(0.2, 1, 23) == 1
    assert s.scale(1.0, 1, 1000) == 64
    s2 = SchedulerOracle(K=5, M_max=64, M0=1, l_hat=LHAT5, rho_hat=0.5, delta=0.1)
    assert s2.scale(1.0, 1, 7) == 3          # 7 / 2.5 = 2.8 -> 3


# ---- S2: Eq. (3) assignment from an empty cluster reaches the exhaustive-search optimum ----------------------------------
def test_s2_assignment_matches_exhaustive_search():
    for M, N, K in [(2, 5, 3), (3, 7, 3), (3, 6, 5), (4, 6, 2)]:
        l_hat = [0.0] + [10.0 * n * n + 1 for n in range(1, K + 1)]
        best = min(max(l_hat[c] for c in np.bincount(p, minlength=M))
                   for p in itertools.product(range(M), repeat=N) if np.bincount(p, minlength=M).max() <= K)
        s = SchedulerOracle(K=K, M_max=M, M0=M, l_hat=l_hat, rho_hat=1.0, delta=1.0)      # band so wide that M never moves
        r = s.event(sess(range(N)))
        loads = np.bincount(list(r["phi"].values()), minlength=M)
        assert r["L"] == best == l_hat[-(-N // M)]
        assert loads.max() - loads.min() <= 1 and r["migrations"] == [] and r["unplaced"] == []


# ---- S3: hand-worked rebalancing sequence (Eq. 4, eta = 0) ---------------------------------------------------------------
def test_s3_rebalancing_hand_worked():
    s = SchedulerOracle(K=5, M_max=3, M0=3, l_hat=LHAT5, rho_hat=1.0, delta=1.0)
    s.phi = {0: 0, 1: 0, 2: 0, 3: 0, 4: 0, 5: 1, 6: 2}            # loads (5, 1, 1)
    s.known = set(range(7))
    r = s.event(sess(range(7)))
    # move 1: any session of GPU 0 to GPU 1 or 2 gives L' = l(4): tie -> lowest session id 0, equal loads -> lowest GPU id 1
    # move 2: loads (4, 2, 1): both targets give L' = l(3): tie -> session 1, less-loaded target GPU 2 -> (3, 2, 2)
    # then every move leaves L at l(3): Gamma = 0, stop.  ceil(7 / 3) = 3 is the optimum.
    assert r["moves"] == [(0, 0, 1), (1, 0, 2)] and r["migrations"] == r["moves"]
    assert r["L"] == LHAT5[3] and sorted(np.bincount(list(r["phi"].values())).tolist()) == [2, 2, 3]
    # the plateau the paper's local search cannot leave: (3, 3, 1, 1) -> no single move lowers the bottleneck
    s = SchedulerOracle(K=5, M_max=4, M0=4, l_hat=LHAT5, rho_hat=1.0, delta=1.0)
    s.phi = {0: 0, 1: 0, 2: 0, 3: 1, 4: 1, 5: 1, 6: 2, 7: 3}
    s.known = set(range(8))
    r = s.event(sess(range(8)))
    assert r["moves"] == [] and r["migrations"] == [] and r["L"] == LHAT5[3]


# ---- S4: the gain threshold Gamma = L - L' - eta * kappa > 0 and the alpha-beta cost ----------------------------------------
def test_s4_gain_threshold_and_kappa():
    l_hat = [0.0, 100.0, 200.0, 300.0]
    def run(eta, sizes):
        s = SchedulerOracle(K=3, M_max=2, M0=2, l_hat=l_hat, rho_hat=1.0, delta=1.0, eta=eta, kappa_alpha=10.0, kappa_beta=0.1)
        s.phi = {0: 0, 1: 0, 2: 0, 3: 1}
        s.known = {0, 1, 2, 3}
        return s.event([(i, 1, sizes[i]) for i in range(4)])["moves"]
    # L = 300, L' = 200; kappa = 10 + 0.1 * 200 = 30.  eta = 3: Gamma = 100 - 90 = 10 > 0 -> move.  eta = 3.4: -2 -> none.
    assert run(3.0, [200.0] * 4) == [(0, 0, 1)]
    assert run(3.4, [200.0] * 4) == []
    assert run(100.0 / 30.0, [200.0] * 4) == []                    # Gamma = 0 is not > 0
    # the cheapest state moves: session 2 is the small one (kappa 15 against 30)
    assert run(3.0, [200.0, 200.0, 50.0, 200.0]) == [(2, 0, 1)]


# ---- S5: Algorithm 1 on a seeded event stream: constraints of Eq. (1), scale-in / scale-out order, move bookkeeping ---------
def test_s5_algorithm1_invariants_on_event_stream():
    rng = np.random.default_rng(5)
    K, M_max = 5, 12
    s = SchedulerOracle(K=K, M_max=M_max, M0=2, l_hat=LHAT5, rho_hat=0.7, delta=0.1, eta=0.01, kappa_alpha=1.0, kappa_beta=0.01)
    live, next_id, on = {}, 0, False
    seen_out = seen_in = 0
    for t in range(300):
        on = (rng.random() < 0.05) if not on else (rng.random() >= 0.10)
        for sid in list(live):
            if rng.random() < 0.04:
                del live[sid]                                     # departure
            elif rng.random() < 0.15:
                live[sid] = (1 - live[sid][0], live[sid][1])     # active <-> idle
        for _ in range(rng.poisson(3.0 if on else 0.4)):
            if len(live) < 40:
                live[next_id] = (1, float(rng.integers(50, 250)))
                next_id += 1
        ev = [(sid, a, mb) for sid, (a, mb) in sorted(live.items())]
        phi_prev, alive_prev = dict(s.phi), [j for j in range(M_max) if s.alive[j]]
        r = s.event(ev)
        loads = np.bincount([g for g in r["phi"].values() if g >= 0], minlength=M_max)
        assert loads.max(initial=0) <= K                                                       # Eq. (1), capacity
        assert all(loads[j] == 0 for j in range(M_max) if j not in r["alive"])
        n_active = sum(a for _, a, _ in ev)
        if n_active <= K * r["M"]:
            assert r["unplaced"] == []                                                         # Eq. (1), alpha = 1 => placed
        assert all(r["phi"][sid] == -1 for sid, a, _ in ev if not a)                           # R25
        assert r["rho_max"] == loads.max(initial=0) / K and r["L"] == LHAT5[loads.max(initial=0)]
        # the net migrations are exactly the sessions placed before and after on different GPUs ...
        want = [(sid, g, r["phi"][sid]) for sid, g in sorted(phi_prev.items()) if r["phi"].get(sid, -1) >= 0 and r["phi"][sid] != g]
        assert r["migrations"] == want
        # ... and the move log, replayed on the old placement, leads every such session from its old GPU to its new one
        pos = dict(phi_prev)
        for sid, a, b in r["moves"]:
            if sid in pos:
                assert pos[sid] == a, (t, sid, a, b, pos[sid])
                pos[sid] = b
        for sid, g in r["phi"].items():
            if g >= 0 and sid in phi_prev:
                assert pos[sid] == g
        seen_out += r["M"] > len(alive_prev)
        seen_in += r["M"] < len(alive_prev)
        if r["M"] < len(alive_prev):
            assert set(r["alive"]) < set(alive_prev)                                           # scale-in only removes
        if r["M"] > len(alive_prev):
            assert set(r["alive"]) > set(alive_prev) and loads[[j for j in r["alive"] if j not in alive_prev]].sum() >= 0
    assert seen_out >= 3 and seen_in >= 3


# ---- S6: volatility sigma(t) of Eq. (6) is numpy.std over the window; measure -> quantise -> look up -> replace --------------
def test_s6_volatility_mapping():
    s = SchedulerOracle(K=5, M_max=8, M0=8, l_hat=LHAT5, rho_hat=0.9, delta=0.1, vol_window=4, vol_bounds=[1.0, 3.0],
                        vol_rho=[0.9, 0.7, 0.5])
    # activations per event 0, 4, 0, 4: mean 2, sigma = 2 exactly -> level 1 -> rho_hat 0.7
    nxt, live = 0, []
    sig = []
    for n_new in [0, 4, 0, 4]:
        live = live + list(range(nxt, nxt + n_new))
        nxt += n_new
        sig.append(s.event(sess(live))["sigma"])
    assert sig[-1] == 2.0 and s.rho_hat == 0.7
    rng = np.random.default_rng(6)
    s = SchedulerOracle(K=5, M_max=60, M0=60, l_hat=LHAT5, vol_window=6, vol_bounds=[0.5, 1.5, 2.5], vol_rho=[0.95, 0.8, 0.65, 0.5])
    a_hist, nxt, live = [], 0, []
    for _ in range(40):
        n_new = int(rng.poisson(2.0))
        live = live[int(rng.integers(0, 3)):] + list(range(nxt, nxt + n_new))
        nxt += n_new
        a_hist.append(n_new)
        r = s.event(sess(live))
        want = float(np.std(a_hist[-6:]))
        assert abs(r["sigma"] - want) < 1e-12
        assert r["rho_hat"] == [0.95, 0.8, 0.65, 0.5][int(np.searchsorted([0.5, 1.5, 2.5], r["sigma"], side="right"))]
