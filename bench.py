#!/usr/bin/env python
"""bench.py — coalesced chunk step on BASELINE.json configs[2] (Wan-1.3B-shaped 8-session batch).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--no-extras]

One JSON line on stdout (rank 0).  A "step" is one pass of the hot path over one coalesced batch:
    resume(idle session X) on the side stream                      (a6)   (suspends run on a second offload stream)
    open + close of a transient session                            (a7)
    every COMMIT_EVERY-th step: the transient session's first chunk as a real committed step - page growth, a
        schedule build for it AND (single-entry schedule cache) a rebuild for the main batch, commit (a1, a3, a4)
    ts_chunk_step(batch of 8, flags=0)    scheduler + attention (a1, a2) and paged scatter (a3) in ONE launch: the
                                          scatter is done by the two role-less warps of every attention CTA
    suspend(X) on the side stream                                  (a5)
flags=0 on the main batch keeps every timed step on the identical drawn state of configs[2].
`value` = attention FLOPs of all launches / time of the K steps (all ranks).  `roofline` comes from the SAME loop:
CUDA events around every fused launch of the main batch on the launching stream (so ms_per_launch <= ms_per_step),
with the SM clock measured inside the kernel (clock64 / globaltimer, ts_pool_clock_probe).  `sustained` repeats
the step back to back for >= 2 s.  `kernels_alone` times attention and append as separate launches (the append's
roofline).  `e2e` is the same step through ts_chunk_step_host with pinned HOST buffers (H2D of Q/K/V and D2H of O
inside the timed region).  `configs` carries configs[1], [3] (one layer, and the 40-layer step eager and as one CUDA
graph) and [4] (200-step churn); `overlap` the cost of a full-window offload under the step (NEXT-1); `latency_model`
the measured l_hat(n).  N > 1 runs N independent replicas (sessions are independent units).
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
COMMIT_EVERY = 4
# dram__bytes_read.sum + dram__bytes_write.sum of one attention launch on this workload, from the ncu --set full
# capture summarised in the file named beside it (not a measurement of this run).
IDLE_BEFORE_LOOP_S = 0.5   # both burst loops start from an idle GPU
ATTENTION_DRAM_TRAFFIC = {"bytes": 1543272000, "from": "profiles/r2_attention.txt (ncu --set full, final build, the fused launch: 1.2028 GB read + 340.5 MB "
                                                          "written; attention-only launch 1.038 GB, profiles/r1_final_build.txt)"}


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f), "measured"
    return dict(FALLBACK_PEAKS), "fallback"


def config_dict(w, world):
    """The workload description both arms print (the driver compares them key by key)."""
    import synth
    return {"workload": WORKLOAD, "prior_frames": [s.prior_frames for s in w.sessions],
            "attention_tflop_per_step": round(synth.attention_flops(w.shape, w.sessions) / 1e12, 4),
            "l2": "inputs larger than L2 (Q/K/V 345 MB + KV cache 1.1 GB per step vs 126 MB L2)",
            "parallelism": f"replicas x{world} (sessions are independent; no collective)"}


class ClockSampler:
    """Samples SM clock and throttle reasons while the timed region runs (B200_PROFILING.md clocks line).  NVML reports
    the clock BETWEEN launches of a few ms; the clock under the kernel is measured in the kernel (clock probe)."""

    def __init__(self, index, period=0.005):
        self.index, self.samples, self.reasons, self.max_mhz, self.period = index, [], set(), None, period
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
            self._stop.wait(self.period)

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
        return {"sm_mhz": float(np.median(self.samples)), "sm_min_mhz": float(np.min(self.samples)),
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "nvml_samples": len(self.samples)}


class KernelClock:
    """SM clock under the attention kernel itself: CTA 0 accumulates clock64 cycles and globaltimer nanoseconds."""

    def __init__(self, pool, device):
        import torch
        self.pool = pool
        self.buf = torch.zeros(2, dtype=torch.int64, device=device)

    def __enter__(self):
        self.buf.zero_()
        self.pool.ts_pool_clock_probe(self.buf)
        return self

    def __exit__(self, *exc):
        self.pool.ts_pool_clock_probe(None)

    def mhz(self):
        import torch
        torch.cuda.synchronize()
        cyc, ns = (int(x) for x in self.buf.tolist())
        return round(cyc / ns * 1e3, 1) if ns > 0 else None


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
    # the transient session's first chunk (1 frame): q = k = v of the first T tokens
    tq = q[:T].contiguous()
    torch.cuda.synchronize(device)
    return {"w": w, "pool": pool, "opool": opool, "sids": sids, "cf": [3] * len(sids), "q": q, "k": k, "v": v,
            "x": x, "x_pages": pool.ts_session_info(x)["n_pages"], "chunks": chunks, "to_bits": to_bits,
            "tq": tq, "tout": torch.empty_like(tq),
            "t_flops": 4 * D * H * synth.attention_pairs(0, 1, T, sh.window_frames)}


def step_device(wl, out, i=0, ev=None):
    """One coalesced chunk step, inputs resident in HBM.  Returns the attention FLOPs it launched."""
    from paper_2606_19271_b200 import TS_COMMIT
    pool = wl["pool"]
    scale = float(wl["w"].scale)
    flops = wl["flops_step"]
    pool.ts_session_resume(wl["x"])
    t = pool.ts_session_open()
    if i % COMMIT_EVERY == COMMIT_EVERY - 1:
        pool.ts_chunk_step(0, [t], [1], wl["tq"], wl["tq"], wl["tq"], wl["tout"], None, scale, TS_COMMIT)
        flops += wl["t_flops"]
    pool.ts_session_close(t)
    if ev is not None:
        ev[0].record()
    pool.ts_chunk_step(0, wl["sids"], wl["cf"], wl["q"], wl["k"], wl["v"], out, None, scale, 0)
    if ev is not None:
        ev[1].record()
    pool.ts_session_suspend(wl["x"])
    return flops


def step_kernels(wl, out, ev):
    """The same batch with attention and append as separate launches on one stream, for per-kernel timing."""
    pool = wl["pool"]
    ev[0].record()
    pool.ts_chunk_attention(0, wl["sids"], wl["cf"], wl["q"], wl["k"], wl["v"], out, None, float(wl["w"].scale))
    ev[1].record()
    pool.ts_kv_append(0, wl["sids"], wl["cf"], wl["k"], wl["v"], 0)
    ev[2].record()


def step_host(wl, hq, hk, hv, hout):
    pool = wl["pool"]
    pool.ts_session_resume(wl["x"])
    pool.ts_chunk_step_host(0, wl["sids"], wl["cf"], hq, hk, hv, hout, float(wl["w"].scale), 0)
    pool.ts_session_suspend(wl["x"])


def join_side(pool):
    """Make the current stream wait for the pool's side stream (the step ends when both are done)."""
    import torch
    torch.cuda.current_stream().wait_stream(pool.side_stream)
    torch.cuda.current_stream().wait_stream(pool.suspend_stream)


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
    ap.add_argument("--power-table", action="store_true",
                    help="print the clock / power table of profiles/r2_power_table.md (attention kernel vs cuBLAS bf16, burst "
                         "and sustained) instead of the bench line")
    ap.add_argument("--no-extras", action="store_true",
                    help="only the timed loop, the roofline and e2e (skips sustained / configs / overlap / latency_model)")
    args = ap.parse_args()
    rank, world, local = dist_env()

    import torch

    import synth

    if args.impl == "reference":
        if rank != 0:
            return 0
        run_reference(args, world)
        return 0

    if args.warmup < 3:
        args.warmup = 3                     # timing rule: at least 3 warm-up steps on the GPU
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    device = torch.device("cuda", local)
    torch.cuda.set_device(device)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=device)
    peaks, peaks_kind = load_peaks()
    extras = (world == 1) and not args.no_extras

    if args.power_table:
        print(json.dumps(power_table(device, peaks), indent=1))
        return 0
    wl = build_workload(device, with_oracle=(rank == 0 and world == 1))
    pool, w = wl["pool"], wl["w"]
    sh = w.shape
    flops_step = synth.attention_flops(sh, w.sessions)
    wl["flops_step"] = flops_step
    tokens = wl["q"].shape[0]
    append_bytes = 4 * tokens * sh.n_heads * sh.head_dim * 2            # read K,V + write K,V
    out = torch.empty_like(wl["q"])
    kclock = KernelClock(pool, device)

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize(device)

    # ---- device-resident timing: `value` and the attention roofline come from this one loop.  Like the separate-kernel loop
    # below it starts after a short idle gap (the workload set-up has just run thousands of small kernels): both 20-step loops
    # are bursts from an idle GPU - `step.idle_before_loop_s` says so in the line, `sustained` is the power-capped regime
    time.sleep(IDLE_BEFORE_LOOP_S)
    for i in range(args.warmup):
        step_device(wl, out, i)
        join_side(pool)
    barrier()
    t_begin, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    step_evs = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(args.steps)]
    launch_evs = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(args.steps)]
    launches0, builds0 = pool.ts_pool_launch_count(), pool.ts_pool_sched_builds()
    flops_loop, host_s = 0.0, 0.0
    with ClockSampler(device.index if device.index is not None else 0) as clocks, kclock:
        t_begin.record()
        for i in range(args.steps):
            step_evs[i][0].record()
            h0 = time.perf_counter()
            flops_loop += step_device(wl, out, i, launch_evs[i])
            host_s += time.perf_counter() - h0
            join_side(pool)
            step_evs[i][1].record()
        t_end.record()
        barrier()
        clock_in_kernel = kclock.mhz()
    launches = pool.ts_pool_launch_count() - launches0
    builds = pool.ts_pool_sched_builds() - builds0
    # host cost of a step's calls with an empty queue behind them (in the loop above the host runs ahead of the GPU until
    # the 8-deep staging ring pushes back, so its wall time there is mostly waiting)
    host_unblocked = []
    for i in range(2 * COMMIT_EVERY):
        torch.cuda.synchronize(device)
        h0 = time.perf_counter()
        step_device(wl, out, i)
        host_unblocked.append((time.perf_counter() - h0) * 1e3)
        join_side(pool)
    torch.cuda.synchronize(device)
    ms_total = t_begin.elapsed_time(t_end)
    step_ms_max = float(max(e[0].elapsed_time(e[1]) for e in step_evs))
    attn_ms = float(np.mean([e[0].elapsed_time(e[1]) for e in launch_evs]))

    backend_dev = device
    ms_total_all, flops_all = aggregate(ms_total, flops_loop, world, backend_dev)

    # ---- the two kernels as separate launches (the append's roofline).  The GPU is power-capped: a short idle gap
    # lets this loop start from the same power state as the timed loop above.
    time.sleep(IDLE_BEFORE_LOOP_S)
    for _ in range(args.warmup):
        step_kernels(wl, out, [torch.cuda.Event(enable_timing=True) for _ in range(3)])
    barrier()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    for i in range(args.steps):
        step_kernels(wl, out, evs[i])
    barrier()
    attn_alone_ms = float(np.mean([e[0].elapsed_time(e[1]) for e in evs]))
    append_ms = float(np.mean([e[1].elapsed_time(e[2]) for e in evs]))

    # ---- end to end through ts_chunk_step_host with pinned host buffers (one packed [3][tokens][H][D] input buffer)
    hin = torch.stack([t.cpu() for t in (wl["q"], wl["k"], wl["v"])]).pin_memory()
    hq, hk, hv = hin[0], hin[1], hin[2]
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
    e2e_ms_all, _ = aggregate(e2e_ms, 0.0, world, backend_dev)
    link = measure_link(device, h2d, d2h) if rank == 0 else None

    if rank != 0:
        if world > 1:
            torch.distributed.barrier()       # rank 0's migrate_p2p leg runs while the others wait here
        return 0

    value = flops_all / (ms_total_all * 1e-3) / 1e12
    achieved = flops_step / (attn_ms * 1e-3) / 1e12
    peak = peaks["bf16_tflops"]
    sust_peak = peaks.get("bf16_tflops_sustained", peak)
    clk = clocks.summary()
    clk["sm_mhz_in_kernel"] = clock_in_kernel
    clk["note"] = "sm_mhz: NVML between launches; sm_mhz_in_kernel: clock64/globaltimer inside the attention kernel"
    result = {
        "metric": METRIC, "value": round(value, 2), "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": round(ms_total_all / args.steps, 4), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "config": config_dict(w, world),
        "step": {"append_flags_main_batch": 0, "commit_every": COMMIT_EVERY,
                 "committed_step": "transient session, 1 frame, P=0: page growth + schedule build + commit; evicts the "
                                   "single-entry schedule cache, so the main batch's schedule is rebuilt too",
                 "idle_before_loop_s": IDLE_BEFORE_LOOP_S,
                 "sched_builds_in_timed_loop": int(builds), "host_ms_per_step_in_loop": round(host_s / args.steps * 1e3, 4),
                 "host_ms_per_step_unblocked": {"cached_schedule": round(float(np.min(host_unblocked)), 4),
                                                "with_committed_step_and_rebuild": round(float(np.max(host_unblocked)), 4)}},
        "max_chunk_latency_ms": round(step_ms_max, 4),
        "roofline": {"bound": "tensor", "kernel": "chunk_attention_kernel<128> (fused: + the batch's KV append)",
                     "achieved": round(achieved, 2), "peak": peak, "unit": "TFLOP/s", "frac": round(achieved / peak, 4),
                     "peak_kind": f"{peaks_kind} burst cuBLAS bf16 (MEASURED_PEAKS.json)",
                     "frac_of_sustained": round(achieved / sust_peak, 4),
                     "frac_of_nominal_2250": round(achieved / NOMINAL_BF16_TFLOPS, 4),
                     "ms_per_launch": round(attn_ms, 4), "timed_in": "the loop `value` comes from (events around each launch)",
                     "sm_mhz_in_kernel": clock_in_kernel,
                     # FLOP per SM clock against the tensor pipe's 8192 per SM: does not depend on the clock the box grants
                     "tensor_frac_of_cycles": (round(achieved * 1e12 / (148 * 8192 * clock_in_kernel * 1e6), 4)
                                               if clock_in_kernel else None),
                     "traffic": ATTENTION_DRAM_TRAFFIC["bytes"], "traffic_from": ATTENTION_DRAM_TRAFFIC["from"]},
        "kernels_alone": {"note": "separate launches, second loop after a 0.5 s idle gap (another power state)",
                          "attention_ms": round(attn_alone_ms, 4),
                          "attention_tflops": round(flops_step / (attn_alone_ms * 1e-3) / 1e12, 2)},
        "append": {"bound": "hbm", "kernel": "kv_append_kernel", "bytes_per_launch": append_bytes,
                   "ms_per_launch": round(append_ms, 4), "achieved": round(append_bytes / (append_ms * 1e-3) / 1e9, 1),
                   "peak": peaks["hbm_gbs"], "unit": "GB/s",
                   "frac": round(append_bytes / (append_ms * 1e-3) / 1e9 / peaks["hbm_gbs"], 4)},
        "e2e": {"value": round(flops_step * args.steps * world / (e2e_ms_all * 1e-3) / 1e12, 2), "unit": UNIT,
                "ms_per_step": round(e2e_ms_all / args.steps, 4), "h2d_bytes_per_step": int(h2d),
                "d2h_bytes_per_step": int(d2h),
                "api": "ts_chunk_step_host (pinned host Q/K/V packed in one buffer, O; one fused launch per step)",
                "link": e2e_link(link, h2d, d2h, e2e_ms_all / args.steps)},
        "gpu_launches": int(launches),
        "clocks": clk,
    }
    # ---- legs that do not feed `value` (single GPU only)
    result["offload"] = measure_offload(wl)
    result["offload"]["scattered"] = {k: v for k, v in measure_offload(wl, permuted=True).items()
                                      if k in ("d2h", "h2d", "placement")}
    result["migrate"] = measure_migration(wl, peaks["hbm_gbs"])
    if extras:
        try:      # two extra processes and CUDA IPC: a box that refuses either must not cost the run its headline line
            result["migrate_ipc"] = measure_migration_ipc(wl, peaks["hbm_gbs"])
        except Exception as exc:
            result["migrate_ipc"] = {"unavailable": f"{type(exc).__name__}: {exc}"[:300]}
    if world > 1 and torch.cuda.device_count() >= 2:
        result["migrate_p2p"] = measure_migration_p2p(wl)
    if extras:
        result["sustained"] = measure_sustained(wl, out, kclock, device, sust_peak, peak)
        result["static_entry"] = measure_static_entry(wl, out)
        result["overlap"] = measure_overlap(wl, out)
        pool.close()
        wl["pool"] = None
        torch.cuda.empty_cache()
        result["latency_model"] = measure_latency_model()
        result["configs"] = {"configs[1]": run_config1(device, peak), "configs[3]": run_config3(device, peak),
                             "configs[4]": run_config4(device, peak)}
    if world == 1:
        chunk_bits = [tuple(wl["to_bits"](t) for t in c) for c in wl["chunks"]]
        dt, fl, desc = oracle_sample(w, wl["opool"], wl["sids"], chunk_bits)
        result["cpu_baseline"] = {"value": round(fl / dt / 1e12, 5), "unit": UNIT, "cores": cpu_threads(),
                                  "kind": "oracle", "sample": desc, "seconds": round(dt, 2)}
    print(json.dumps(result))
    if wl["pool"] is not None:
        wl["pool"].close()
    if world > 1:
        torch.distributed.barrier()
    return 0


# ------------------------------------------------------------------------------------------------ power table
class PowerSampler(ClockSampler):
    """ClockSampler that also records board power (NVML, mW)."""

    def _run(self):
        nv = self.nv
        self.power = []
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1e3)
                mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                if mask & getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4):
                    self.reasons.add("sw_power_cap")
            except Exception:
                pass
            self._stop.wait(self.period)


def power_table(device, peaks):
    """What bounds the attention kernel on this box: SM clock under the kernel (in-kernel probe), SM cycles per launch
    (independent of the clock), board power, against cuBLAS bf16 8192^3 in the same two regimes (burst: 20 launches after
    an idle second; sustained: back to back for 3 s)."""
    import torch
    import synth
    wl = build_workload(device, False)
    pool, w = wl["pool"], wl["w"]
    flops = synth.attention_flops(w.shape, w.sessions)
    out = torch.empty_like(wl["q"])
    scale = float(w.scale)
    probe = torch.zeros(2, dtype=torch.int64, device=device)
    idx = device.index or 0
    peak_per_mhz = 148 * 8192 / 1e6            # TFLOP/s per MHz of SM clock at 100 % tensor-pipe activity (8192 FLOP/clk/SM)

    def attn():
        pool.ts_chunk_attention(0, wl["sids"], wl["cf"], wl["q"], wl["k"], wl["v"], out, None, scale)

    a = torch.randn(8192, 8192, device=device, dtype=torch.bfloat16)
    b = torch.randn(8192, 8192, device=device, dtype=torch.bfloat16)
    c = torch.empty_like(a)
    mm_flops = 2 * 8192 ** 3

    def mm():
        torch.matmul(a, b, out=c)

    def run(fn, fl, n=None, seconds=None, probe_on=False):
        for _ in range(3):
            fn()
        torch.cuda.synchronize(device)
        time.sleep(1.0)
        if probe_on:
            probe.zero_()
            pool.ts_pool_clock_probe(probe)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        count = 0
        with PowerSampler(idx, period=0.005) as ps:
            e0.record()
            if n is not None:
                for _ in range(n):
                    fn()
                count = n
            else:
                t0 = time.perf_counter()
                while time.perf_counter() - t0 < seconds:
                    for _ in range(50):
                        fn()
                    count += 50
                    torch.cuda.synchronize(device)
            e1.record()
            torch.cuda.synchronize(device)
        ms = e0.elapsed_time(e1)
        row = {"launches": count, "ms_per_launch": round(ms / count, 4), "tflops": round(fl * count / ms / 1e9, 1),
               "nvml_sm_mhz_median": float(np.median(ps.samples)) if ps.samples else None,
               "nvml_power_w_median": round(float(np.median(ps.power)), 1) if ps.power else None,
               "nvml_power_w_max": round(float(np.max(ps.power)), 1) if ps.power else None,
               "reasons": sorted(ps.reasons)}
        if probe_on:
            pool.ts_pool_clock_probe(None)
            cyc, ns = (int(x) for x in probe.tolist())
            mhz = cyc / ns * 1e3
            row.update({"sm_mhz_in_kernel": round(mhz, 1), "mcycles_per_launch": round(cyc / count / 1e6, 4),
                        "tensor_pipe_floor_mcycles": round(fl / (148 * 8192) / 1e6, 4),
                        "tensor_frac_of_cycles": round(fl / (148 * 8192) / (cyc / count), 4),
                        "peak_at_this_clock_tflops": round(peak_per_mhz * mhz, 1)})
        else:
            # cuBLAS cannot be probed from inside: the clock it must at least have run at, were its tensor pipe 100 % active
            row["implied_min_sm_mhz"] = round(row["tflops"] / peak_per_mhz, 1)
        if row["nvml_power_w_median"]:
            row["joule_per_launch"] = round(row["nvml_power_w_median"] * ms / count / 1e3, 3)
            row["pj_per_flop"] = round(row["nvml_power_w_median"] * ms * 1e-3 / (fl * count) * 1e12, 3)
        return row

    table = {"workload": WORKLOAD + " (attention-only launches, 3.14 TFLOP each)",
             "attention_burst_20": run(attn, flops, n=20, probe_on=True),
             "attention_sustained_3s": run(attn, flops, seconds=3.0, probe_on=True),
             "cublas_bf16_8192_burst_20": run(mm, mm_flops, n=20),
             "cublas_bf16_8192_sustained_3s": run(mm, mm_flops, seconds=3.0),
             "measured_peaks": {k: peaks.get(k) for k in ("bf16_tflops", "bf16_tflops_sustained")}}
    tgt = 0.6 * NOMINAL_BF16_TFLOPS
    for key in ("attention_burst_20", "attention_sustained_3s"):
        r = table[key]
        r["tensor_frac_needed_for_1350_at_this_clock"] = round(tgt / r["peak_at_this_clock_tflops"], 4)
    pool.close()
    return table


# ------------------------------------------------------------------------------------------------ legs
def measure_link(device, h2d_bytes, d2h_bytes):
    """The host link of this box, this run: one pinned copy each way alone, and both at once with the step's byte mix."""
    import torch
    n_in, n_out = int(h2d_bytes), int(d2h_bytes)
    hin = torch.empty(n_in, dtype=torch.uint8).pin_memory()
    hout = torch.empty(n_out, dtype=torch.uint8).pin_memory()
    din = torch.empty(n_in, dtype=torch.uint8, device=device)
    dout = torch.empty(n_out, dtype=torch.uint8, device=device)
    s_in, s_out = torch.cuda.Stream(device), torch.cuda.Stream(device)
    res = {}

    def run(do_in, do_out):
        best = 1e9
        for _ in range(5):
            torch.cuda.synchronize(device)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            s_in.wait_event(a)
            s_out.wait_event(a)
            if do_in:
                with torch.cuda.stream(s_in):
                    din.copy_(hin, non_blocking=True)
            if do_out:
                with torch.cuda.stream(s_out):
                    hout.copy_(dout, non_blocking=True)
            torch.cuda.current_stream().wait_stream(s_in)
            torch.cuda.current_stream().wait_stream(s_out)
            b.record()
            torch.cuda.synchronize(device)
            best = min(best, a.elapsed_time(b))
        return best
    res["h2d_alone_gbs"] = n_in / (run(True, False) * 1e-3) / 1e9
    res["d2h_alone_gbs"] = n_out / (run(False, True) * 1e-3) / 1e9
    res["both_ms"] = run(True, True)
    return res


def e2e_link(link, h2d, d2h, ms_per_step):
    if link is None:
        return None
    return {"h2d_gbs_in_step": round(h2d / (ms_per_step * 1e-3) / 1e9, 2),
            "h2d_alone_gbs": round(link["h2d_alone_gbs"], 2), "d2h_alone_gbs": round(link["d2h_alone_gbs"], 2),
            "frac_of_h2d_alone": round(h2d / (ms_per_step * 1e-3) / 1e9 / link["h2d_alone_gbs"], 4),
            "both_directions_ms": round(link["both_ms"], 4),
            "frac_of_both_directions": round(link["both_ms"] / ms_per_step, 4),
            "note": "the step moves h2d and d2h bytes at once; `both_directions_ms` is the same byte mix as two plain "
                    "pinned copies running concurrently (the link's own limit for this step), best of 5, same run"}


def measure_sustained(wl, out, kclock, device, sust_peak, burst_peak, seconds=2.0):
    """The step back to back for >= `seconds`: the power-capped regime."""
    import torch
    pool = wl["pool"]
    time.sleep(0.5)
    for i in range(3):
        step_device(wl, out, i)
        join_side(pool)
    torch.cuda.synchronize(device)
    n_guess = max(50, int(seconds * 1e3 / 2.4))
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    flops, steps, ms = 0.0, 0, 0.0
    with ClockSampler(device.index if device.index is not None else 0, period=0.02) as clocks, kclock:
        while ms < seconds * 1e3:
            a.record()
            for i in range(n_guess):
                flops += step_device(wl, out, steps + i)
                join_side(pool)
            b.record()
            torch.cuda.synchronize(device)
            ms += a.elapsed_time(b)
            steps += n_guess
            n_guess = 100
        mhz = kclock.mhz()
    tfl = flops / (ms * 1e-3) / 1e12
    c = clocks.summary()
    return {"seconds": round(ms / 1e3, 3), "steps": steps, "value": round(tfl, 2), "unit": UNIT,
            "ms_per_step": round(ms / steps, 4), "peak": sust_peak,
            "frac": round(tfl / sust_peak, 4), "frac_of_burst": round(tfl / burst_peak, 4),
            "frac_of_nominal_2250": round(tfl / NOMINAL_BF16_TFLOPS, 4), "sm_mhz_in_kernel": mhz,
            "nvml": {"sm_mhz_median": c.get("sm_mhz"), "sm_mhz_min": c.get("sm_min_mhz"), "reasons": c.get("reasons")},
            "peak_kind": "bf16_tflops_sustained (MEASURED_PEAKS.json): cuBLAS back to back for 4 s"}


def measure_static_entry(wl, out, reps=20):
    """ts_chunk_attention_static (no allocation: the schedule block in the library's static device array, copied there from
    pageable host memory) against ts_chunk_attention on the same batch: ms per call, calls back to back, events on the
    compute stream.  Outputs are compared bit for bit."""
    import torch
    pool = wl["pool"]
    scale = float(wl["w"].scale)
    args = (0, wl["sids"], wl["cf"], wl["q"], wl["k"], wl["v"])
    out2 = torch.empty_like(out)
    res = {}
    for name, fn, o in (("ts_chunk_attention", pool.ts_chunk_attention, out),
                        ("ts_chunk_attention_static", pool.ts_chunk_attention_static, out2)):
        for _ in range(3):
            fn(*args, o, None, scale)
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        a.record()
        for _ in range(reps):
            fn(*args, o, None, scale)
        b.record()
        host_ms = (time.perf_counter() - t0) * 1e3 / reps
        torch.cuda.synchronize()
        res[name] = {"ms_per_call": round(a.elapsed_time(b) / reps, 4), "host_ms_per_call": round(host_ms, 4)}
    res["bit_identical"] = bool(torch.equal(out.view(torch.int16), out2.view(torch.int16)))
    res["static_scratch_bytes"] = 256 * 1024
    res["note"] = ("the static entry copies its block from pageable host memory (no pinned staging to allocate): the driver "
                   "stages this batch's 53 KB at call time; ts_chunk_attention's host time is the wait for a free slot of its "
                   "8-deep staging ring when calls are enqueued faster than the GPU runs them")
    return res


def measure_overlap(wl, out, reps=12):
    """SURVEY.md §8(f) NEXT-1 (PAPER.md:76 (iii), :160): the configs[2] step alone, and the same step while a FULL-window
    (21-frame, 201 MB) idle session is resumed and another suspended on the side stream.  Step time by events on the
    compute stream, offload rate by events on the side stream; `resume_done_before_step_end` says whether a session
    resumed at the start of step t is ready when step t ends (it is served in step t+1 without a wait)."""
    import torch
    from synth.draw import draw_bits_torch
    from paper_2606_19271_b200 import TS_COMMIT, TurboChunkPool
    w = wl["w"]
    sh = w.shape
    T, H, D = sh.frame_tokens, sh.n_heads, sh.head_dim
    dev = wl["q"].device
    # a second pool for the two idle full-window sessions would not share the step's free list; use the main pool's twin:
    # same geometry, the batch of configs[2] re-created in it plus two full-window idle sessions Y, Z
    n_pages = sh.n_pages + 2 * 130
    pool = TurboChunkPool(1, H, D, sh.page_tokens, n_pages, T, sh.window_frames, sh.max_sessions,
                          free_order=np.random.default_rng(5).permutation(n_pages), host_pages=2 * 130, device=dev.index)
    gen = torch.Generator(device=dev)
    gen.manual_seed(w.seed)
    sids = []
    for spec in w.sessions:
        sid = pool.ts_session_open()
        for _ in range(0, spec.prior_frames, 3):
            dk = draw_bits_torch(gen, 3 * T, H, D, dev)
            pool.ts_kv_append(0, [sid], [3], dk, dk, TS_COMMIT)
        sids.append(sid)
    idle = []
    for _ in range(2):
        s = pool.ts_session_open()
        for _ in range(7):
            dk = draw_bits_torch(gen, 3 * T, H, D, dev)
            pool.ts_kv_append(0, [s], [3], dk, dk, TS_COMMIT)
        idle.append(s)
    y, z = idle
    pool.ts_session_suspend(y)
    pool.ts_offload_sync()
    nbytes = pool.ts_session_info(y)["n_pages"] * pool.page_bytes
    side = pool.side_stream
    scale = float(w.scale)
    cur = torch.cuda.current_stream()

    def step():
        pool.ts_chunk_step(0, sids, wl["cf"], wl["q"], wl["k"], wl["v"], out, None, scale, 0)

    for _ in range(3):
        step()
    torch.cuda.synchronize()
    # steady state: `n_steps` steps back to back (the host runs ahead, as in serving), alone and under continuous offload
    n_steps, alone, loaded, h2d_ms, d2h_ms = 8, [], [], [], []
    for r in range(reps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(n_steps):
            step()
        b.record()
        torch.cuda.synchronize()
        alone.append(a.elapsed_time(b) / n_steps)
    out_s = pool.suspend_stream
    for r in range(reps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev_in = [torch.cuda.Event(enable_timing=True) for _ in range(6)]
        ev_out = [torch.cuda.Event(enable_timing=True) for _ in range(6)]
        a.record()
        side.wait_event(a)                     # the offload starts with the first step
        out_s.wait_event(a)
        for i in range(3):                     # 3 x (resume 201 MB H2D, suspend 201 MB D2H): the two directions run at once
            ev_in[2 * i].record(side)
            pool.ts_session_resume(y)
            ev_in[2 * i + 1].record(side)
            ev_out[2 * i].record(out_s)
            pool.ts_session_suspend(z)
            ev_out[2 * i + 1].record(out_s)
            y, z = z, y
        for _ in range(n_steps):
            step()
        b.record()
        torch.cuda.synchronize()
        loaded.append(a.elapsed_time(b) / n_steps)
        h2d_ms += [ev_in[2 * i].elapsed_time(ev_in[2 * i + 1]) for i in range(3)]
        d2h_ms += [ev_out[2 * i].elapsed_time(ev_out[2 * i + 1]) for i in range(3)]
    pool.close()
    alone_ms, loaded_ms = float(np.median(alone)), float(np.median(loaded))
    h2d, d2h = float(np.median(h2d_ms)), float(np.median(d2h_ms))
    return {"steps_back_to_back": n_steps, "step_alone_ms": round(alone_ms, 4), "step_with_offload_ms": round(loaded_ms, 4),
            "step_slowdown": round(loaded_ms / alone_ms - 1.0, 4), "offload_bytes_each_way": int(nbytes),
            "resume_h2d_gbs_under_load": round(nbytes / (h2d * 1e-3) / 1e9, 2),
            "suspend_d2h_gbs_under_load": round(nbytes / (d2h * 1e-3) / 1e9, 2),
            "resume_ms": round(h2d, 4), "steps_to_hide_one_resume": round(h2d / loaded_ms, 2),
            "resume_done_within_steps": int(np.ceil(h2d / loaded_ms)),
            "note": "a full-window (201 MB) resume takes `resume_ms` at the link rate, i.e. `steps_to_hide_one_resume` steps of "
                    "this batch: a session whose resume is enqueued at the start of step t is served in step "
                    "t + resume_done_within_steps without any host wait (the step's launch waits on the resume's event), "
                    "and the steps it hides behind run `step_slowdown` slower"}


def measure_latency_model(ns=(1, 2, 4, 5, 6, 7, 8, 16, 32), layers=30, passes=4, slo_ms=670.0):
    """l_hat(n): per-layer attention + append time against the number of co-located full-window sessions,
    and the largest n whose 30-layer x 4-pass lower bound meets the 670 ms SLO."""
    from paper_2606_19271_b200.latency_model import measure
    rows, best = [], 0
    for n in ns:
        attn_ms, app_ms, tfl = measure(n, 18, 12, 128, 1560, 21, 256, reps=5)
        step_ms = layers * (passes * attn_ms + app_ms)
        if step_ms <= slo_ms:
            best = max(best, n)
        rows.append({"n": n, "attention_ms_per_layer": round(attn_ms, 4), "append_ms_per_layer": round(app_ms, 4),
                     "attention_tflops": round(tfl, 1), "chunk_step_ms_lower_bound": round(step_ms, 1)})
    per = [r["attention_ms_per_layer"] / r["n"] for r in rows]
    return {"shape": "Wan-1.3B attention, every session at the full 21-frame window, one layer", "l_hat": rows,
            "ms_per_session_layer_min_max": [round(min(per), 4), round(max(per), 4)],
            "model": f"{layers} layers x ({passes} passes attention + 1 append); projections/MLP are outside this library",
            "slo_ms": slo_ms, "largest_n_under_slo": best}


def _timed(fn, reps, device):
    import torch
    ts = []
    for _ in range(reps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        fn()
        b.record()
        torch.cuda.synchronize(device)
        ts.append(a.elapsed_time(b))
    return ts


def run_config1(device, peak):
    """configs[1]: one session, 12 heads, P = 6, c = 3."""
    import torch
    import synth
    from synth.draw import draw_bits_torch
    from paper_2606_19271_b200 import TS_COMMIT, TurboChunkPool
    w = synth.wan13b_single()
    sh = w.shape
    T, H, D = sh.frame_tokens, sh.n_heads, sh.head_dim
    pool = TurboChunkPool(1, H, D, sh.page_tokens, sh.n_pages, T, sh.window_frames, sh.max_sessions, device=device.index)
    gen = torch.Generator(device=device)
    gen.manual_seed(w.seed)
    sid = pool.ts_session_open()
    for _ in range(2):
        dk = draw_bits_torch(gen, 3 * T, H, D, device)
        pool.ts_kv_append(0, [sid], [3], dk, dk, TS_COMMIT)
    q, k, v = (draw_bits_torch(gen, 3 * T, H, D, device) for _ in range(3))
    out = torch.empty_like(q)
    fn = lambda: pool.ts_chunk_step(0, [sid], [3], q, k, v, out, None, float(w.scale), 0)
    for _ in range(3):
        fn()
    ts = _timed(fn, 20, device)                       # one call at a time on an idle GPU: host enqueue time included
    flops = synth.attention_flops(sh, w.sessions)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize(device)
    a.record()
    for _ in range(20):                               # back to back: the host runs ahead, as in a multi-layer step
        fn()
    b.record()
    torch.cuda.synchronize(device)
    ms_b2b = a.elapsed_time(b) / 20
    ms = float(np.median(ts))
    pool.close()
    return {"workload": "1 session x 12 heads, P=6, c=3 (444 query tiles on 148 SMs)",
            "ms_per_step": round(ms_b2b, 4), "tflops": round(flops / ms_b2b / 1e9, 1), "frac": round(flops / ms_b2b / 1e9 / peak, 4),
            "single_call_on_idle_gpu": {"ms": round(ms, 4), "max_ms": round(max(ts), 4),
                                        "note": "event before the call to completion: includes the host's enqueue time (tensor-map encodes, "
                                                "descriptor upload) that back-to-back calls hide behind the previous launch"}}


def run_config3(device, peak):
    """configs[3]: 4 sessions x 40 heads at the full window; one layer, and the 40-layer chunk step - 40 eager
    ts_chunk_step calls against ONE CUDA graph of 40 ts_step_plan_run launches (NEXT-2)."""
    import torch
    import synth
    from synth.draw import draw_bits_torch
    from paper_2606_19271_b200 import TS_COMMIT, TS_RUN_APPEND, TurboChunkPool
    torch.cuda.empty_cache()
    free_b, _ = torch.cuda.mem_get_info(device)
    NL = 40
    w = synth.wan14b_batch(n_layers=NL)
    sh = w.shape
    per_layer = sh.n_pages * 2 * sh.n_heads * sh.page_tokens * sh.head_dim * 2
    while NL > 1 and per_layer * NL + (6 << 30) > free_b:
        NL //= 2
    if NL != 40:
        w = synth.wan14b_batch(n_layers=NL)
        sh = w.shape
    T, H, D = sh.frame_tokens, sh.n_heads, sh.head_dim
    pool = TurboChunkPool(NL, H, D, sh.page_tokens, sh.n_pages, T, sh.window_frames, sh.max_sessions, device=device.index)
    gen = torch.Generator(device=device)
    gen.manual_seed(w.seed)
    sids = [pool.ts_session_open() for _ in w.sessions]
    cf = [3] * len(sids)
    n_tok = 3 * T * len(sids)
    for _ in range(0, 18, 3):
        dk = draw_bits_torch(gen, n_tok, H, D, device)
        dv = draw_bits_torch(gen, n_tok, H, D, device)
        for layer in range(NL):
            pool.ts_kv_append(layer, sids, cf, dk, dv, TS_COMMIT if layer == NL - 1 else 0)
    q, k, v = (draw_bits_torch(gen, n_tok, H, D, device) for _ in range(3))
    out = torch.empty_like(q)
    scale = float(w.scale)
    flops = synth.attention_flops(sh, w.sessions)
    one = lambda: pool.ts_chunk_step(0, sids, cf, q, k, v, out, None, scale, 0)
    for _ in range(2):
        one()
    t_one = _timed(one, 5, device)

    def eager():
        for layer in range(NL):
            pool.ts_chunk_step(layer, sids, cf, q, k, v, out, None, scale, 0)
    eager()
    torch.cuda.synchronize(device)
    host_eager, t_eager = [], []
    for _ in range(3):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        h0 = time.perf_counter()
        a.record()
        eager()
        b.record()
        host_eager.append((time.perf_counter() - h0) * 1e3)
        torch.cuda.synchronize(device)
        t_eager.append(a.elapsed_time(b))
    # the same step as one graph: prepare (host + one upload), one graph launch, commit
    plan = pool.ts_step_plan_create(sids, cf, n_slots=1)
    plan.ts_step_plan_bind(0, q, k, v, out, None)
    stream = torch.cuda.Stream(device)
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(stream):
        plan.ts_step_plan_prepare(stream=stream)
        stream.synchronize()
        with torch.cuda.graph(graph, stream=stream, capture_error_mode="thread_local"):
            for layer in range(NL):
                plan.ts_step_plan_run(layer, 0, scale, TS_RUN_APPEND, stream=torch.cuda.current_stream())
        graph.replay()
        plan.ts_step_plan_commit(0, stream=stream)
        stream.synchronize()
        host_graph, t_graph = [], []
        for _ in range(3):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            h0 = time.perf_counter()
            a.record(stream)
            plan.ts_step_plan_prepare(stream=stream)
            graph.replay()
            plan.ts_step_plan_commit(0, stream=stream)
            b.record(stream)
            host_graph.append((time.perf_counter() - h0) * 1e3)
            stream.synchronize()
            t_graph.append(a.elapsed_time(b))
    plan.close()
    pool.close()
    del pool, q, k, v, out
    torch.cuda.empty_cache()
    ms1 = float(np.median(t_one))
    return {"workload": f"4 sessions x 40 heads, P=18 (full 21-frame window), {NL} layers"
                        + ("" if NL == 40 else " (fewer than 40: not enough free HBM for the 107 GB slab)"),
            "one_layer": {"ms": round(ms1, 4), "tflops": round(flops / ms1 / 1e9, 1), "frac": round(flops / ms1 / 1e9 / peak, 4)},
            "chunk_step_eager": {"layers": NL, "calls": NL, "ms": round(min(t_eager), 2), "max_ms": round(max(t_eager), 2),
                                 "host_ms": round(float(np.median(host_eager)), 3),
                                 "tflops": round(flops * NL / min(t_eager) / 1e9, 1)},
            "chunk_step_graph": {"layers": NL, "graph_launches": 1, "ms": round(min(t_graph), 2),
                                 "max_ms": round(max(t_graph), 2), "host_ms": round(float(np.median(host_graph)), 3),
                                 "tflops": round(flops * NL / min(t_graph) / 1e9, 1),
                                 "frac": round(flops * NL / min(t_graph) / 1e9 / peak, 4),
                                 "what": "ts_step_plan_prepare + cudaGraphLaunch(40 x ts_step_plan_run) + ts_step_plan_commit"}}


def run_config4(device, peak):
    """configs[4]: 200-step bursty churn (synth.churn_script, seed 4), Wan-1.3B attention shape, up to 32 sessions per step;
    idle sessions suspended to the pinned arena and resumed on reactivation, all on the side stream.  Per-chunk latency =
    wall clock from the first call of a step to the completion of its fused launch (a resume the batch waits for included)."""
    import torch
    import synth
    from synth.draw import draw_bits_torch
    from paper_2606_19271_b200 import TS_COMMIT, TurboChunkPool
    T, H, D, B, Wn = 1560, 12, 128, 256, 21
    steps = synth.churn_script()
    rng = np.random.default_rng(4)
    n_pages = 4000
    pool = TurboChunkPool(1, H, D, B, n_pages, T, Wn, 128, free_order=rng.permutation(n_pages), host_pages=5400,
                          device=device.index)
    gen = torch.Generator(device=device)
    gen.manual_seed(4)
    C = 3 * T
    cap = max(len(e["batch"]) for e in steps)
    q, k, v = (draw_bits_torch(gen, cap * C, H, D, device) for _ in range(3))
    out = torch.empty_like(q)
    scale = float(1.0 / np.sqrt(D))
    side = pool.side_stream
    sid_of, frames = {}, {}
    lat, flops, off_bytes, off_ms, n_served = [], [], 0, 0.0, []
    for ev in steps:
        torch.cuda.synchronize(device)
        t0 = time.perf_counter()
        moved = 0
        s0, s1, s2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        s0.record()                                        # everything is idle here: the offload of the step starts now
        for u in ev["suspend"]:
            moved += pool.ts_session_info(sid_of[u])["n_pages"] * pool.page_bytes
            pool.ts_session_suspend(sid_of[u])
        for u in ev["resume"]:
            pool.ts_session_resume(sid_of[u])
            moved += pool.ts_session_info(sid_of[u])["n_pages"] * pool.page_bytes
        s1.record(side)
        s2.record(pool.suspend_stream)
        for u in ev["open"]:
            sid_of[u] = pool.ts_session_open()
            frames[u] = 0
        batch = [sid_of[u] for u in ev["batch"]]
        if batch:
            n_tok = len(batch) * C
            pool.ts_chunk_step(0, batch, ev["chunk_frames"], q[:n_tok], k[:n_tok], v[:n_tok], out[:n_tok], None, scale, TS_COMMIT)
            torch.cuda.current_stream().synchronize()
            lat.append((time.perf_counter() - t0) * 1e3)
            flops.append(4 * D * H * sum(synth.attention_pairs(frames[u], 3, T, Wn) for u in ev["batch"]))
            n_served.append(len(batch))
            for u in ev["batch"]:
                frames[u] = min(Wn, frames[u] + 3)
        torch.cuda.synchronize(device)
        if moved:
            off_bytes += moved
            off_ms += max(s0.elapsed_time(s1), s0.elapsed_time(s2))   # the two directions run at the same time
        for u in ev["close"]:
            pool.ts_session_close(sid_of.pop(u))
            frames.pop(u)
    n_split = pool.ts_pool_split_batches()
    pool.close()
    lat_a, fl = np.array(lat), np.array(flops)
    return {"workload": "200-step MMPP churn (mean 4 / 24 sessions, cap 32), suspend/resume through pinned host memory",
            "served_steps": len(lat), "max_batch": int(max(n_served)), "steps_run_as_two_launches": int(n_split), "latency_ms_p50": round(float(np.median(lat_a)), 3),
            "latency_ms_p99": round(float(np.percentile(lat_a, 99)), 3), "latency_ms_max": round(float(lat_a.max()), 3),
            "attention_tflops": round(float(fl.sum() / lat_a.sum() / 1e9), 1),
            "attention_tflops_best_step": round(float((fl / lat_a).max() / 1e9), 1),
            "frac": round(float(fl.sum() / lat_a.sum() / 1e9) / peak, 4),
            "offload_gb": round(off_bytes / 1e9, 2), "offload_gbs": round(off_bytes / max(off_ms, 1e-9) / 1e6, 2),
            "note": "latency includes the host calls and any resume the batch waits for; offload rate = bytes moved in both directions / time "
                    "until both offload streams are done (suspends and resumes run on two streams, at the same time)"}


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
    side, out_s = pool.side_stream, pool.suspend_stream
    res = {}
    torch.cuda.synchronize()
    times = {"d2h": [], "h2d": []}
    for it in range(7):
        a, b, b2, c = (torch.cuda.Event(enable_timing=True) for _ in range(4))
        a.record(out_s)
        pool.ts_session_suspend(sid)                      # device -> host on the suspend stream
        b.record(out_s)
        side.wait_event(b)
        b2.record(side)
        pool.ts_session_resume(sid)                       # host -> device on the side stream
        c.record(side)
        side.synchronize()
        if it:
            times["d2h"].append(a.elapsed_time(b))
            times["h2d"].append(b2.elapsed_time(c))
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
    the source slab over NVLink (`migrate_p2p`, --gpus >= 2)."""
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


def measure_migration_ipc(wl, hbm_peak):
    """The same full-window session moved between two WORKER PROCESSES on this GPU (paper_2606_19271_b200.worker: one pool
    each, the source slab mapped through CUDA IPC, "state frozen" / "installed" as interprocess events; PAPER.md:263-265,
    :271).  Reported: the device time of the fetches (4 sessions fetched back to back, events on the target's side stream)
    and the wall-clock time of one whole move as the control plane sees it (freeze -> ticket -> import -> release: three
    pipe round trips between three Python processes; no host synchronisation with the GPU in either worker)."""
    import time
    from paper_2606_19271_b200 import TS_COMMIT, worker
    sh = wl["w"].shape
    geo = dict(n_layers=1, n_heads=sh.n_heads, head_dim=sh.head_dim, page_tokens=sh.page_tokens, n_pages=4 * 132,
               frame_tokens=sh.frame_tokens, window_frames=sh.window_frames, max_sessions=4)
    ws = [worker.spawn(device=wl["q"].device.index or 0) for _ in range(2)]
    try:
        for w in ws:
            w.post("create", **geo)
        for w in ws:
            w.result()
        blobs = [w.call("pool", "ts_pool_export") for w in ws]
        peers = [ws[0].call("pool", "ts_peer_open", blobs[1]), ws[1].call("pool", "ts_peer_open", blobs[0])]   # peer of the OTHER side
        sids = [ws[0].call("pool", "ts_session_open") for _ in range(4)]
        for i in range(7):
            ws[0].call("append_random", 0, sids, [3] * 4, 200 + i, TS_COMMIT)
        ws[0].call("sync")
        n_pages = ws[0].call("pool", "ts_session_info", sids[0])["n_pages"]
        nbytes = n_pages * ws[0].call("pool", "ts_pool_stats")["page_bytes"]
        best_ms, walls = 1e9, []
        where = 0
        for rep in range(8):
            src, dst = ws[where], ws[where ^ 1]
            if rep < 4:      # device time: the four fetches enqueued back to back, events on the target's side stream
                tickets = [src.call("pool", "ts_session_freeze", s) for s in sids]
                new, ms = dst.call("timed_imports", peers[where ^ 1], tickets)
                for s in sids:
                    src.call("pool", "ts_session_release", s, peers[where])
                if rep > 0:
                    best_ms = min(best_ms, ms / len(sids))
            else:            # control-plane time: whole moves one after the other, nothing waits for the GPU
                new = []
                for s in sids:
                    t0 = time.perf_counter()
                    ticket = src.call("pool", "ts_session_freeze", s)
                    new.append(dst.call("pool", "ts_session_import", peers[where ^ 1], ticket))
                    src.call("pool", "ts_session_release", s, peers[where])
                    walls.append(time.perf_counter() - t0)
            sids, where = new, where ^ 1
        for w in ws:
            w.call("sync")
        for w, peer in zip(ws, peers):   # mappings go before the pools that exported them
            w.call("pool", "ts_peer_close", peer)
    finally:
        for w in ws:
            w.close()
    gbs = 2 * nbytes / (best_ms * 1e-3) / 1e9
    return {"bound": "hbm", "kernel": "page_pull_kernel (source slab through CUDA IPC)", "bytes_moved": int(nbytes),
            "pages": int(n_pages), "algorithmic_bytes_per_launch": int(2 * nbytes), "ms_per_move_device": round(best_ms, 4),
            "achieved": round(gbs, 1), "peak": hbm_peak, "unit": "GB/s", "frac": round(gbs / hbm_peak, 4),
            "ms_per_move_control_plane": {"median": round(1e3 * sorted(walls)[len(walls) // 2], 3), "max": round(1e3 * max(walls), 3)},
            "note": "two worker processes on this one GPU; device time = fetches of 4 sessions back to back on the target's "
                    "side stream; control-plane time = wall clock of freeze + import + release per session through the "
                    "parent's pipes (Python), no host-GPU synchronisation in the workers"}


def measure_migration_p2p(wl, peer_peak_gbs=770.0):
    """--gpus >= 2, rank 0 only (the other ranks wait at a barrier): a full-window session moved between a pool on device 0
    and a pool on device 1 of THIS process, both ways.  The fetch kernel runs on the target and reads the source slab
    through the peer mapping (NVLink); timed by events on the target's side stream."""
    import torch
    from synth.draw import draw_bits_torch
    from paper_2606_19271_b200 import TS_COMMIT, TurboChunkPool
    sh = wl["w"].shape
    T, H, D = sh.frame_tokens, sh.n_heads, sh.head_dim
    pools = [TurboChunkPool(1, H, D, sh.page_tokens, 160, T, sh.window_frames, 2, device=d) for d in (0, 1)]
    dev0 = torch.device("cuda", 0)
    gen = torch.Generator(device=dev0)
    gen.manual_seed(98)
    with torch.cuda.device(0):
        sid = pools[0].ts_session_open()
        for _ in range(7):
            kk = draw_bits_torch(gen, 3 * T, H, D, dev0)
            pools[0].ts_kv_append(0, [sid], [3], kk, kk, TS_COMMIT)
    nbytes = pools[0].ts_session_info(sid)["n_pages"] * pools[0].page_bytes
    torch.cuda.synchronize(0)
    times = []
    for i in range(8):
        src, dst = pools[i & 1], pools[(i & 1) ^ 1]
        with torch.cuda.device((i & 1) ^ 1):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(dst.side_stream)
            sid = src.ts_session_migrate(sid, dst)
            b.record(dst.side_stream)
            dst.side_stream.synchronize()
            times.append(a.elapsed_time(b))
    for p in pools:
        p.close()
    torch.cuda.set_device(0)
    best = float(np.min(times[2:]))
    gbs = nbytes / (best * 1e-3) / 1e9
    return {"bound": "nvlink", "kernel": "page_pull_kernel (peer loads)", "bytes_moved": int(nbytes),
            "ms_per_move": round(best, 4), "achieved": round(gbs, 1), "peak": peer_peak_gbs, "unit": "GB/s",
            "frac": round(gbs / peer_peak_gbs, 4),
            "peak_kind": "measured peer copy on this pool, 770 GB/s per direction (B200_PROFILING.md); nominal 900"}


def run_reference(args, world):
    """The CPU oracle as it stands, on the same config/metric; each step is a bounded sample of the workload.
    Inputs are drawn on the host (numpy path of synth/) so that this arm needs no GPU."""
    import oracle
    import synth
    w = synth.wan13b_batch()
    sh = w.shape
    T, H, D = sh.frame_tokens, sh.n_heads, sh.head_dim
    cfg = config_dict(w, world)
    opool = oracle.OraclePool(sh.n_layers, H, D, sh.page_tokens, sh.n_pages, T, sh.window_frames, sh.max_sessions,
                              w.free_order)
    sids, chunk_bits = [], []
    for spec in w.sessions:
        sid = opool.open()
        for _ in range(0, spec.prior_frames, 3):
            opool.append(0, [sid], [3], synth.draw_bits(w.rng, 3 * T, H, D), synth.draw_bits(w.rng, 3 * T, H, D))
        chunk_bits.append(tuple(synth.draw_bits(w.rng, 3 * T, H, D) for _ in range(3)))
        sids.append(sid)
    steps, warmup = max(1, args.steps), max(1, args.warmup)
    # each step = a bounded sample of the workload, sized so that warmup + steps end within a few minutes: one whole head
    # of as many sessions as a per-step budget allows (the batch's sessions in order, wrapping around)
    t_probe, _, _ = oracle_sample(w, opool, sids[:1], chunk_bits[:1])
    budget_s = 150.0 / (steps + warmup)
    per_step = int(max(1, min(len(sids), budget_s / max(t_probe, 1e-3))))
    tot_t, tot_f, desc, cursor = 0.0, 0, "", 0
    for it in range(warmup + steps):
        pick = [(cursor + j) % len(sids) for j in range(per_step)]
        cursor += per_step
        dt, fl, desc = oracle_sample(w, opool, [sids[j] for j in pick], [chunk_bits[j] for j in pick])
        if it >= warmup:
            tot_t += dt
            tot_f += fl
    value = tot_f / tot_t / 1e12
    sample = f"per step: one whole head (all 4680 query rows over all visible keys) of {per_step} of the 8 sessions, fp64 numpy"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": round(value, 5), "unit": UNIT, "n_gpus": world, "steps": steps,
        "warmup": warmup, "ms_per_step": round(tot_t / steps * 1e3, 2), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": cfg,
        "cpu_baseline": {"value": round(value, 5), "unit": UNIT, "kind": "oracle", "cores": cpu_threads(), "sample": sample},
        "e2e": {"value": round(value, 5), "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


if __name__ == "__main__":
    sys.exit(main())
