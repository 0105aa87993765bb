"""Measured per-GPU latency model l_hat(n) of the coalesced chunk step.

TurboServe's placement and autoscaling controllers consume one quantity from the per-GPU runtime: the per-chunk
latency l_hat_j(n_j) of a GPU that co-locates n_j sessions (Eq. 3-4), and the per-GPU session cap K
 is the largest n that still meets the latency SLO (670 ms in the paper's appendix study,
PAPER.md:466).  This script measures the part of that curve this library owns - attention + KV append per layer, as
a function of the number of coalesced sessions - on synthetic Wan-1.3B-shaped inputs, through the C ABI:

    python -m paper_2606_19271_b200.latency_model [--layers 30] [--passes 4] [--slo-ms 670] [--prior-frames 18]

One JSON line per batch size n: attention and append time of ONE layer (CUDA events, median of --reps), the chunk
step extrapolated to `layers x passes` attention calls + `layers` appends (the rest of the model - projections, MLP -
is not part of this library, so this is a lower bound of l_hat), and a last line with the largest n under the SLO.
No CPU fallback: needs the CUDA library and an sm_100 device.
"""
import argparse
import json
import sys

import numpy as np


def measure(n, prior_frames, heads, head_dim, frame_tokens, window, page_tokens, reps, device=0, seed=7):
    """Returns (attention_ms, append_ms, attention_tflops) for one layer with n co-located sessions."""
    import torch

    from . import TS_COMMIT, TurboChunkPool

    dev = torch.device("cuda", device)
    pages_per_session = (window + 3) * frame_tokens // page_tokens + 2
    pool = TurboChunkPool(1, heads, head_dim, page_tokens, pages_per_session * n + 8, frame_tokens, window, max(n, 1),
                          device=device)
    gen = torch.Generator(device=dev)
    gen.manual_seed(seed)
    draw = lambda: torch.randn((3 * frame_tokens * n, heads, head_dim), generator=gen, device=dev).to(torch.bfloat16)
    sids = [pool.ts_session_open() for _ in range(n)]
    cf = [3] * n
    kv = draw()
    for _ in range(0, prior_frames, 3):
        pool.ts_kv_append(0, sids, cf, kv, kv, TS_COMMIT)
    q = draw()
    out = torch.empty_like(q)
    scale = float(1.0 / np.sqrt(head_dim))
    for _ in range(3):
        pool.ts_chunk_attention(0, sids, cf, q, kv, kv, out, None, scale)
        pool.ts_kv_append(0, sids, cf, kv, kv, 0)        # flags=0: the window state stays the same for every repetition
    torch.cuda.synchronize(dev)
    t_attn, t_app = [], []
    for _ in range(reps):
        e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        e[0].record()
        pool.ts_chunk_attention(0, sids, cf, q, kv, kv, out, None, scale)
        e[1].record()
        pool.ts_kv_append(0, sids, cf, kv, kv, 0)
        e[2].record()
        torch.cuda.synchronize(dev)
        t_attn.append(e[0].elapsed_time(e[1]))
        t_app.append(e[1].elapsed_time(e[2]))
    vis = min(prior_frames, window - 3) if window > 0 else prior_frames
    pairs = sum(frame_tokens * (vis * frame_tokens + (f + 1) * frame_tokens) for f in range(3))
    flops = 4 * head_dim * heads * n * pairs
    attn_ms, app_ms = float(np.median(t_attn)), float(np.median(t_app))
    pool.close()
    del pool, q, out, kv
    torch.cuda.empty_cache()
    return attn_ms, app_ms, flops / attn_ms / 1e9


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--sessions", type=int, nargs="*", default=[1, 2, 3, 4, 5, 8, 12, 16, 24, 32])
    ap.add_argument("--prior-frames", type=int, default=18)
    ap.add_argument("--layers", type=int, default=30, help="attention layers per model pass (Wan-1.3B: 30)")
    ap.add_argument("--passes", type=int, default=4, help="denoising passes per chunk (Self-Forcing-style: 4)")
    ap.add_argument("--slo-ms", type=float, default=670.0, help="per-chunk latency SLO (PAPER.md:466)")
    ap.add_argument("--heads", type=int, default=12)
    ap.add_argument("--head-dim", type=int, default=128)
    ap.add_argument("--frame-tokens", type=int, default=1560)
    ap.add_argument("--window", type=int, default=21)
    ap.add_argument("--page-tokens", type=int, default=256)
    ap.add_argument("--reps", type=int, default=8)
    args = ap.parse_args(argv)
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("latency_model needs a CUDA device: the library has no CPU fallback")
    best = 0
    for n in args.sessions:
        attn_ms, app_ms, tfl = measure(n, args.prior_frames, args.heads, args.head_dim, args.frame_tokens, args.window,
                                       args.page_tokens, args.reps)
        step_ms = args.layers * (args.passes * attn_ms + app_ms)
        if step_ms <= args.slo_ms:
            best = max(best, n)
        print(json.dumps({"n_sessions": n, "prior_frames": args.prior_frames, "attention_ms_per_layer": round(attn_ms, 4),
                          "append_ms_per_layer": round(app_ms, 4), "attention_tflops": round(tfl, 1),
                          "chunk_step_ms_lower_bound": round(step_ms, 2)}), flush=True)
    print(json.dumps({"slo_ms": args.slo_ms, "layers": args.layers, "passes": args.passes,
                      "largest_n_under_slo": best,
                      "note": "attention + KV append only; projections and MLP of the model are outside this library"}))
    return 0


if __name__ == "__main__":
    sys.exit(main())
