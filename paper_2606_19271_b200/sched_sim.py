"""Replay of a seeded bursty event stream through the closed-loop scheduler (ts_sched_event; Algorithm 1), driven by
the per-GPU latency model l_hat(n) that `latency_model.py` measures on the B200.

    python -m paper_2606_19271_b200.sched_sim [--events 2000] [--seed 1] [--K 5] [--M-max 16]

Prints one JSON line per configuration of the SAME controller: the full closed loop, the loop without migration (eta so
large that no move has a positive gain, Eq. 4) and without autoscaling (a fixed budget), the two ablations of the
paper's §7.3.  Metrics as in PAPER.md §7.1: worst-case per-chunk latency (max over events of L(t) = max_j l_hat(n_j)) and GPU
operating cost (sum over events of M(t), in GPU-events).  The paper's own numbers come from production traces on real
clusters and are not reproducible here; this is the controller's behaviour on synthetic events, not a comparison with them.
Host code only.
"""
import argparse
import json

# l_hat(n) in ms for n = 0..5 co-located Wan-1.3B sessions at the full 21-frame window, 30 layers x (4 attention passes +
# 1 append), measured through the C ABI on one B200
LHAT_WAN13B_MS = [0.0, 90.0, 174.0, 267.0, 350.0, 441.0]


def replay(events, K, M_max, M0, l_hat, rho_hat, delta, eta, kappa_alpha=23.0, kappa_beta=0.0, vol=None):
    from . import TurboSched
    kw = dict(K=K, M_max=M_max, M0=M0, l_hat=l_hat, rho_hat=rho_hat, delta=delta, eta=eta, kappa_alpha=kappa_alpha,
              kappa_beta=kappa_beta)
    if vol:
        kw.update(vol)
    s = TurboSched(**kw)
    worst, sum_L, cost, moves, unplaced, n = 0.0, 0.0, 0, 0, 0, 0
    for ev in events:
        r = s.ts_sched_event(ev)
        worst = max(worst, r["L"])
        sum_L += r["L"]
        cost += r["M"]
        moves += len(r["migrations"])
        unplaced += r["n_unplaced"]
        n += 1
    s.close()
    return {"worst_case_latency_ms": worst, "mean_bottleneck_latency_ms": round(sum_L / max(n, 1), 2), "gpu_events": cost,
            "mean_gpus": round(cost / max(n, 1), 3), "migrations": moves, "unplaced_session_events": unplaced, "events": n}


def main():
    import synth
    ap = argparse.ArgumentParser()
    ap.add_argument("--events", type=int, default=2000)
    ap.add_argument("--seed", type=int, default=1)
    ap.add_argument("--K", type=int, default=5)
    ap.add_argument("--M-max", type=int, default=16)
    args = ap.parse_args()
    l_hat = LHAT_WAN13B_MS[:args.K + 1]
    stream = lambda: synth.sched_events(args.seed, args.events, cap=args.K * args.M_max)
    # kappa: the paper's measured migration overhead, 23 ms; eta small (footnote 3 of PAPER.md:213)
    full = replay(stream(), args.K, args.M_max, 1, l_hat, 0.7, 0.1, eta=0.05)
    fixed = max(1, round(full["mean_gpus"]))
    runs = {
        "closed_loop": full,
        "no_migration": replay(stream(), args.K, args.M_max, 1, l_hat, 0.7, 0.1, eta=1e9),
        "no_autoscaling_same_mean_budget": replay(stream(), args.K, fixed, fixed, l_hat, 0.7, 10.0, eta=0.05),
        "no_autoscaling_peak_budget": replay(stream(), args.K, args.M_max, args.M_max, l_hat, 0.7, 10.0, eta=0.05),
    }
    for name, r in runs.items():
        print(json.dumps({"config": name, **r}))


if __name__ == "__main__":
    main()
