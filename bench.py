#!/usr/bin/env python
"""bench.py — coalesced chunk step on BASELINE.json configs[2] (Wan-1.3B-shaped 8-session batch).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

One JSON line on stdout (rank 0).  A "step" is one pass of the hot path over one coalesced batch:
    resume(idle session X) on the side stream                      (a6)
    open + close of a transient session                            (a7)
    ts_chunk_step(batch of 8, flags=0)    scheduler + attention (a1, a2) and paged scatter (a3) in ONE launch: the
                                          scatter is done by the two role-less warps of every attention CTA
    suspend(X) on the side stream                                  (a5)
flags=0 keeps every timed step on the identical drawn state of configs[2]; the window roll (a4) is host
integer arithmetic inside ts_kv_append(TS_COMMIT), exercised by the tests, not by the timed loop.
`value` = attention FLOPs of the batch / step time (all ranks); `roofline` (attention) and `append` are the two
kernels timed alone with CUDA events, one after the other, in a second loop over the same steps;
`e2e` is the same step through ts_chunk_step_host with pinned HOST buffers (H2D of Q/K/V and D2H of O inside
the timed region).  N > 1 runs N independent replicas (sessions are independent units).
`--impl reference` times the CPU oracle (oracle/) on a bounded sample of the same workload.
"""
import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "coalesced chunk-attn TFLOP/s"
UNIT = "TFLOP/s"
WORKLOAD = "configs[2] wan13b_batch: 8 sessions x 12 heads x D128, T=1560, 3-frame chunks, W=21, B=256"
NOMINAL_BF16_TFLOPS = 2250.0
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}
# dram__bytes_read.sum + dram__bytes_write.sum of one attention launch on this workload, from the ncu --set full
# capture summarised in profiles/ (None until a capture exists).
ATTENTION_DRAM_TRAFFIC_BYTES = 1037573888  # 934.57 MB read + 103.00 MB write (attention-only launch), profiles/r1_final_build.txt


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f), "measured"
    return dict(FALLBACK_PEAKS), "fallback"


class ClockSampler:
    """Samples SM clock and throttle reasons while the timed region runs (B200_PROFILING.md clocks line)."""

    def __init__(self, index):
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        names = {
            "hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
            "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4),
        }
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for name, bit in names.items():
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop.wait(0.02)

    def __enter__(self):
        if self.nv is not None:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()
        return self

    def __exit__(self, *exc):
        self._stop.set()
        if self._thread is not None:
            self._thread.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons)}


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


def aggregate(ms_local, units_local, world, backend_device):
    """max-over-ranks time, sum-over-ranks units (weak scaling: replicas).  Works with gloo (CPU) and nccl."""
    import torch
    import torch.distributed as dist
    if world == 1:
        return ms_local, units_local
    t = torch.tensor([ms_local], dtype=torch.float64, device=backend_device)
    u = torch.tensor([units_local], dtype=torch.float64, device=backend_device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


# ------------------------------------------------------------------------------------------------ workload
def build_workload(device, with_oracle):
    """configs[2] on `device`: returns dict with the CUDA pool, sids, chunk tensors and (optionally) an oracle
    pool fed with copies of the same drawn tensors (inputs are data, shared)."""
    import torch

    import synth
    from synth.draw import draw_bits_torch
    from paper_2606_19271_b200 import TS_COMMIT, TurboChunkPool

    w = synth.wan13b_batch()
    sh = w.shape
    T, H, D = sh.frame_tokens, sh.n_heads, sh.head_dim
    idle_frames = 3
    host_pages = 32
    pool = TurboChunkPool(sh.n_layers, H, D, sh.page_tokens, sh.n_pages, T, sh.window_frames, sh.max_sessions,
                          free_order=w.free_order, host_pages=host_pages, device=device.index)
    opool = None
    if with_oracle:
        import oracle
        opool = oracle.OraclePool(sh.n_layers, H, D, sh.page_tokens, sh.n_pages, T, sh.window_frames,
                                  sh.max_sessions, w.free_order, host_pages)
    gen = torch.Generator(device=device)
    gen.manual_seed(w.seed)
    to_bits = lambda t: t.contiguous().view(torch.int16).cpu().numpy().view(np.uint16)
    sids, chunks = [], []
    for spec in w.sessions:
        sid = pool.ts_session_open()
        if opool is not None:
            assert opool.open() == sid
        for _ in range(0, spec.prior_frames, 3):
            dk = draw_bits_torch(gen, 3 * T, H, D, device)
            dv = draw_bits_torch(gen, 3 * T, H, D, device)
            pool.ts_kv_append(0, [sid], [3], dk, dv, TS_COMMIT)
            if opool is not None:
                opool.append(0, [sid], [3], to_bits(dk), to_bits(dv))
        chunks.append(tuple(draw_bits_torch(gen, 3 * T, H, D, device) for _ in range(3)))
        sids.append(sid)
    q, k, v = (torch.cat([c[i] for c in chunks]) for i in range(3))
    # the idle session X that is resumed / suspended every step on the side stream
    x = pool.ts_session_open()
    xk = draw_bits_torch(gen, idle_frames * T, H, D, device)
    pool.ts_kv_append(0, [x], [idle_frames], xk, xk, TS_COMMIT)
    pool.ts_session_suspend(x)
    pool.ts_offload_sync()
    torch.cuda.synchronize(device)
    return {"w": w, "pool": pool, "opool": opool, "sids": sids, "cf": [3] * len(sids), "q": q, "k": k, "v": v,
            "x": x, "x_pages": pool.ts_session_info(x)["n_pages"], "chunks": chunks, "to_bits": to_bits}


def step_device(wl, out):
    """One coalesced chunk step, inputs resident in HBM."""
    pool = wl["pool"]
    pool.ts_session_resume(wl["x"])
    t = pool.ts_session_open()
    pool.ts_session_close(t)
    pool.ts_chunk_step(0, wl["sids"], wl["cf"], wl["q"], wl["k"], wl["v"], out, None, float(wl["w"].scale), 0)
    pool.ts_session_suspend(wl["x"])


def step_kernels(wl, out, ev):
    """The same step with attention and append as separate calls on one stream, for per-kernel timing."""
    pool = wl["pool"]
    pool.ts_session_resume(wl["x"])
    ev[0].record()
    pool.ts_chunk_attention(0, wl["sids"], wl["cf"], wl["q"], wl["k"], wl["v"], out, None, float(wl["w"].scale))
    ev[1].record()
    pool.ts_kv_append(0, wl["sids"], wl["cf"], wl["k"], wl["v"], 0)
    ev[2].record()
    pool.ts_session_suspend(wl["x"])


def step_host(wl, hq, hk, hv, hout):
    pool = wl["pool"]
    pool.ts_session_resume(wl["x"])
    pool.ts_chunk_step_host(0, wl["sids"], wl["cf"], hq, hk, hv, hout, float(wl["w"].scale), 0)
    pool.ts_session_suspend(wl["x"])


def join_side(pool):
    """Make the current stream wait for the pool's side stream (the step ends when both are done)."""
    import torch
    torch.cuda.current_stream().wait_stream(pool.side_stream)


# ------------------------------------------------------------------------------------------------ CPU baseline
def oracle_sample(w, opool, sids, chunk_bits, n_heads_per_session=1):
    """Bounded sample of the workload for the oracle: `n_heads_per_session` whole heads (all 4680 query rows, each
    over all its visible keys) of every session.  Returns (seconds, flops, description)."""
    import oracle
    import synth
    sh = w.shape
    T = sh.frame_tokens
    rows = np.arange(3 * T)
    flops = 0
    t0 = time.perf_counter()
    for b, sid in enumerate(sids):
        qb, kb, vb = chunk_bits[b]
        for h in range(n_heads_per_session):
            oracle.attention_rows(opool, 0, sid, 3, qb, kb, vb, w.scale, (b + h) % sh.n_heads, rows)
        spec = w.sessions[b]
        flops += 4 * sh.head_dim * n_heads_per_session * synth.attention_pairs(spec.prior_frames, 3, T, sh.window_frames)
    dt = time.perf_counter() - t0
    return dt, flops, (f"{n_heads_per_session} of {sh.n_heads} heads of each of the {len(sids)} sessions, "
                       "all 4680 query rows over all visible keys, fp64 numpy")


def cpu_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [p["num_threads"] for p in threadpool_info() if p.get("user_api") == "blas"]
        if n:
            return max(n)
    except Exception:
        pass
    return os.cpu_count()


# ------------------------------------------------------------------------------------------------ main
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    rank, world, local = dist_env()

    import torch

    import synth

    if args.impl == "reference":
        if rank != 0:
            return 0
        run_reference(args)
        return 0

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    device = torch.device("cuda", local)
    torch.cuda.set_device(device)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=device)
    peaks, peaks_kind = load_peaks()

    wl = build_workload(device, with_oracle=(rank == 0 and world == 1))
    pool, w = wl["pool"], wl["w"]
    sh = w.shape
    flops_step = synth.attention_flops(sh, w.sessions)
    tokens = wl["q"].shape[0]
    append_bytes = 4 * tokens * sh.n_heads * sh.head_dim * 2            # read K,V + write K,V
    out = torch.empty_like(wl["q"])

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize(device)

    # ---- device-resident timing
    for _ in range(args.warmup):
        step_device(wl, out)
        join_side(pool)
    barrier()
    t_begin, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    step_evs = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(args.steps)]
    launches0 = pool.ts_pool_launch_count()
    with ClockSampler(device.index if device.index is not None else 0) as clocks:
        t_begin.record()
        for i in range(args.steps):
            step_evs[i][0].record()
            step_device(wl, out)
            join_side(pool)
            step_evs[i][1].record()
        t_end.record()
        barrier()
    launches = pool.ts_pool_launch_count() - launches0
    ms_total = t_begin.elapsed_time(t_end)
    step_ms_max = float(max(e[0].elapsed_time(e[1]) for e in step_evs))

    # ---- the two kernels alone (same steps, attention and append as separate calls on one stream).  The GPU is
    # power-capped: a short idle gap lets this loop start from the same power state as the timed loop above.
    time.sleep(0.5)
    for _ in range(args.warmup):
        step_kernels(wl, out, [torch.cuda.Event(enable_timing=True) for _ in range(3)])
        join_side(pool)
    barrier()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    for i in range(args.steps):
        step_kernels(wl, out, evs[i])
        join_side(pool)
    barrier()
    attn_ms = float(np.mean([e[0].elapsed_time(e[1]) for e in evs]))
    append_ms = float(np.mean([e[1].elapsed_time(e[2]) for e in evs]))

    # ---- offload leg (side stream, timed alone): suspend / resume of a full-window session
    off = measure_offload(wl)
    off["scattered"] = {k: v for k, v in measure_offload(wl, permuted=True).items() if k in ("d2h", "h2d", "placement")}
    mig = measure_migration(wl, peaks["hbm_gbs"])

    # ---- end to end through ts_chunk_step_host with pinned host buffers
    hq, hk, hv = (t.cpu().pin_memory() for t in (wl["q"], wl["k"], wl["v"]))
    hout = torch.empty_like(hq).pin_memory()
    for _ in range(3):
        step_host(wl, hq, hk, hv, hout)
        join_side(pool)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        step_host(wl, hq, hk, hv, hout)
        join_side(pool)
    e1.record()
    barrier()
    e2e_ms = e0.elapsed_time(e1)
    h2d = 3 * hq.numel() * 2 + wl["x_pages"] * pool.page_bytes
    d2h = hq.numel() * 2 + wl["x_pages"] * pool.page_bytes

    backend_dev = device
    ms_total_all, flops_all = aggregate(ms_total, flops_step * args.steps, world, backend_dev)
    e2e_ms_all, _ = aggregate(e2e_ms, 0.0, world, backend_dev)
    if rank != 0:
        return 0

    value = flops_all / (ms_total_all * 1e-3) / 1e12
    achieved = flops_step / (attn_ms * 1e-3) / 1e12
    peak = peaks["bf16_tflops"]
    result = {
        "metric": METRIC, "value": round(value, 2), "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": round(ms_total_all / args.steps, 4), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "config": {"workload": WORKLOAD, "prior_frames": [s.prior_frames for s in w.sessions],
                   "attention_tflop_per_step": round(flops_step / 1e12, 4), "append_flags": 0,
                   "l2": "inputs larger than L2 (Q/K/V 345 MB + KV cache 1.1 GB per step vs 126 MB L2)",
                   "parallelism": f"replicas x{world} (sessions are independent; no collective)"},
        "max_chunk_latency_ms": round(step_ms_max, 4),
        "roofline": {"bound": "tensor", "kernel": "chunk_attention_kernel<128>", "achieved": round(achieved, 2),
                     "peak": peak, "unit": "TFLOP/s", "frac": round(achieved / peak, 4),
                     "peak_kind": f"{peaks_kind} burst cuBLAS bf16 (MEASURED_PEAKS.json)",
                     "frac_of_sustained": round(achieved / peaks.get("bf16_tflops_sustained", peak), 4),
                     "frac_of_nominal_2250": round(achieved / NOMINAL_BF16_TFLOPS, 4),
                     "ms_per_launch": round(attn_ms, 4), "traffic": ATTENTION_DRAM_TRAFFIC_BYTES},
        "append": {"bound": "hbm", "kernel": "kv_append_kernel", "bytes_per_launch": append_bytes,
                   "ms_per_launch": round(append_ms, 4), "achieved": round(append_bytes / (append_ms * 1e-3) / 1e9, 1),
                   "peak": peaks["hbm_gbs"], "unit": "GB/s",
                   "frac": round(append_bytes / (append_ms * 1e-3) / 1e9 / peaks["hbm_gbs"], 4)},
        "offload": off,
        "migrate": mig,
        "e2e": {"value": round(flops_step * args.steps * world / (e2e_ms_all * 1e-3) / 1e12, 2), "unit": UNIT,
                "ms_per_step": round(e2e_ms_all / args.steps, 4), "h2d_bytes_per_step": int(h2d),
                "d2h_bytes_per_step": int(d2h), "api": "ts_chunk_step_host (pinned host Q/K/V/O)"},
        "gpu_launches": int(launches),
        "clocks": clocks.summary(),
    }
    if world == 1:
        chunk_bits = [tuple(wl["to_bits"](t) for t in c) for c in wl["chunks"]]
        dt, fl, desc = oracle_sample(w, wl["opool"], wl["sids"], chunk_bits)
        result["cpu_baseline"] = {"value": round(fl / dt / 1e12, 5), "unit": UNIT, "cores": cpu_threads(),
                                  "kind": "oracle", "sample": desc, "seconds": round(dt, 2)}
    print(json.dumps(result))
    pool.close()
    return 0


def measure_offload(wl, permuted=False):
    """Suspend / resume of a full-window (21-frame) session on the side stream, timed with events on that stream,
    against a plain pinned cudaMemcpy of the same bytes measured in the same run."""
    import torch
    from synth.draw import draw_bits_torch
    from paper_2606_19271_b200 import TS_COMMIT, TurboChunkPool
    w = wl["w"]
    sh = w.shape
    T, H, D = sh.frame_tokens, sh.n_heads, sh.head_dim
    dev = wl["q"].device
    # FIFO allocation from an untouched pool keeps the session's pages adjacent (suspend / resume then move them in a few
    # large copies); `permuted` scatters them over the pool as configs[2] asks: one copy per 1.57 MB page
    order = np.random.default_rng(97).permutation(160) if permuted else None
    pool = TurboChunkPool(1, H, D, sh.page_tokens, 160, T, sh.window_frames, 2, free_order=order, host_pages=130,
                          device=dev.index)
    gen = torch.Generator(device=dev)
    gen.manual_seed(99)
    sid = pool.ts_session_open()
    for _ in range(7):
        kk = draw_bits_torch(gen, 3 * T, H, D, dev)
        pool.ts_kv_append(0, [sid], [3], kk, kk, TS_COMMIT)
    n_pages = pool.ts_session_info(sid)["n_pages"]
    nbytes = n_pages * pool.page_bytes
    side = pool.side_stream
    res = {}
    torch.cuda.synchronize()
    times = {"d2h": [], "h2d": []}
    for it in range(7):
        a, b, c = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        a.record(side)
        pool.ts_session_suspend(sid)
        b.record(side)
        pool.ts_session_resume(sid)
        c.record(side)
        side.synchronize()
        if it:
            times["d2h"].append(a.elapsed_time(b))
            times["h2d"].append(b.elapsed_time(c))
    # reference: one large pinned copy each way
    dbuf = torch.empty(nbytes, dtype=torch.uint8, device=dev)
    hbuf = torch.empty(nbytes, dtype=torch.uint8).pin_memory()
    ref = {}
    for name, (dst, src) in {"d2h": (hbuf, dbuf), "h2d": (dbuf, hbuf)}.items():
        best = 1e9
        for _ in range(6):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            with torch.cuda.stream(side):
                a.record(side)
                dst.copy_(src, non_blocking=True)
                b.record(side)
            side.synchronize()
            best = min(best, a.elapsed_time(b))
        ref[name] = nbytes / (best * 1e-3) / 1e9
    for name in ("d2h", "h2d"):
        gbs = nbytes / (float(np.min(times[name])) * 1e-3) / 1e9      # best of 6, like the reference copy (best of 6)
        res[name] = {"achieved": round(gbs, 2), "peak": round(ref[name], 2), "unit": "GB/s",
                     "frac": round(gbs / ref[name], 4)}
    res["bytes"] = int(nbytes)
    res["pages"] = int(n_pages)
    res["peak_kind"] = "one pinned cudaMemcpyAsync of the same bytes, same run; both sides best of 6 (the host link is shared with other tenants of the box)"
    res["placement"] = "pages scattered (one copy per page)" if permuted else "pages adjacent (FIFO allocation): runs of pages merge into one copy"
    pool.close()
    return res


def measure_migration(wl, hbm_peak):
    """ts_session_migrate of a full-window (21-frame) session between two pools, ping-pong, 8 moves enqueued back to
    back behind a blocker copy (so that the host's enqueue time is not in the events).  Both pools sit on this one GPU,
    where the fetch kernel is HBM-bound (read + write of the session's pages); between two GPUs the same kernel reads
    the source slab over NVLink - not measurable on a 1-GPU box."""
    import torch
    from synth.draw import draw_bits_torch
    from paper_2606_19271_b200 import TS_COMMIT, TurboChunkPool
    sh = wl["w"].shape
    T, H, D = sh.frame_tokens, sh.n_heads, sh.head_dim
    dev = wl["q"].device
    pools = [TurboChunkPool(1, H, D, sh.page_tokens, 160, T, sh.window_frames, 2, device=dev.index) for _ in range(2)]
    gen = torch.Generator(device=dev)
    gen.manual_seed(98)
    sid = pools[0].ts_session_open()
    for _ in range(7):
        kk = draw_bits_torch(gen, 3 * T, H, D, dev)
        pools[0].ts_kv_append(0, [sid], [3], kk, kk, TS_COMMIT)
    n_pages = pools[0].ts_session_info(sid)["n_pages"]
    nbytes = n_pages * pools[0].page_bytes
    blocker_src = torch.empty(1 << 30, dtype=torch.uint8, device=dev)
    blocker_dst = torch.empty_like(blocker_src)
    n_moves, best = 8, 1e9
    torch.cuda.synchronize()
    for _ in range(3):
        first = pools[1].side_stream
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with torch.cuda.stream(first):
            blocker_dst.copy_(blocker_src, non_blocking=True)
        e0.record(first)
        for i in range(n_moves):
            src, dst = pools[i & 1], pools[(i & 1) ^ 1]
            sid = src.ts_session_migrate(sid, dst)
        e1.record(pools[(n_moves - 1) & 1 ^ 1].side_stream)
        torch.cuda.synchronize()
        best = min(best, e0.elapsed_time(e1) / n_moves)
    gbs = 2 * nbytes / (best * 1e-3) / 1e9
    for p in pools:
        p.close()
    return {"bound": "hbm", "kernel": "page_pull_kernel", "bytes_moved": int(nbytes), "pages": int(n_pages),
            "algorithmic_bytes_per_launch": int(2 * nbytes), "ms_per_move": round(best, 4), "achieved": round(gbs, 1),
            "peak": hbm_peak, "unit": "GB/s", "frac": round(gbs / hbm_peak, 4),
            "note": "both pools on this GPU (read + write in HBM); across GPUs the fetch reads over NVLink"}


def run_reference(args):
    """The CPU oracle as it stands, on the same config/metric; each step is a bounded sample of the workload.
    Inputs are drawn on the host (numpy path of synth/) so that this arm needs no GPU."""
    import oracle
    import synth
    w = synth.wan13b_batch()
    sh = w.shape
    T, H, D = sh.frame_tokens, sh.n_heads, sh.head_dim
    opool = oracle.OraclePool(sh.n_layers, H, D, sh.page_tokens, sh.n_pages, T, sh.window_frames, sh.max_sessions,
                              w.free_order)
    sids, chunk_bits = [], []
    for spec in w.sessions:
        sid = opool.open()
        for _ in range(0, spec.prior_frames, 3):
            opool.append(0, [sid], [3], synth.draw_bits(w.rng, 3 * T, H, D), synth.draw_bits(w.rng, 3 * T, H, D))
        chunk_bits.append(tuple(synth.draw_bits(w.rng, 3 * T, H, D) for _ in range(3)))
        sids.append(sid)
    steps = max(1, min(args.steps, 3))
    oracle_sample(w, opool, sids, chunk_bits)          # warm-up
    tot_t, tot_f, desc = 0.0, 0, ""
    for _ in range(steps):
        dt, fl, desc = oracle_sample(w, opool, sids, chunk_bits)
        tot_t += dt
        tot_f += fl
    value = tot_f / tot_t / 1e12
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": round(value, 5), "unit": UNIT, "n_gpus": 1, "steps": steps,
        "warmup": 1, "ms_per_step": round(tot_t / steps * 1e3, 2), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD, "prior_frames": [s.prior_frames for s in w.sessions]},
        "cpu_baseline": {"value": round(value, 5), "unit": UNIT, "kind": "oracle", "cores": cpu_threads(), "sample": desc},
        "e2e": {"value": round(value, 5), "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


if __name__ == "__main__":
    sys.exit(main())
