"""A minimal GPU worker process: one TurboChunkPool behind a pipe (one worker per GPU).

The paper's runtime keeps one worker process per GPU and moves sessions between them.  This module is the
smallest such worker: it owns one pool on one device and executes commands that arrive over a `multiprocessing` connection.
Everything that crosses the pipe is plain data (ints, lists, bytes, numpy uint16 arrays holding bf16 bit patterns), which is
also all the cross-process migration calls of include/turbochunk.h need (`ts_pool_export` blob, freeze ticket).
It is argument marshalling only, like binding.py; tests/test_gpu_ipc_migration.py and bench.py's `migrate_ipc` leg drive it.

    w = spawn(device=0); w.call("create", n_layers=..., ...); sid = w.call("pool", "ts_session_open"); ...; w.close()
"""
import multiprocessing as mp
import traceback

import numpy as np


def _to_dev(bits, device):
    import torch
    return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).to(device).view(torch.bfloat16)


def _to_bits(t):
    import torch
    return t.contiguous().view(torch.int16).cpu().numpy().view(np.uint16)


def serve(conn, device):
    """Command loop of the worker process.  Replies ("ok", value) or ("err", text, status code or None)."""
    import torch
    from . import binding
    pool = None
    dev = f"cuda:{device}"
    while True:
        try:
            msg = conn.recv()
        except EOFError:
            break
        op, args, kw = msg[0], msg[1], msg[2]
        try:
            if op == "exit":
                conn.send(("ok", None))
                break
            if op == "create":
                pool = binding.TurboChunkPool(device=device, **kw)
                res = None
            elif op == "pool":            # any binding method whose arguments and result are plain data
                res = getattr(pool, args[0])(*args[1:], **kw)
            elif op == "append":          # (layer, sids, cf, k_bits, v_bits, flags)
                layer, sids, cf, k, v, flags = args
                pool.ts_kv_append(layer, sids, cf, _to_dev(k, dev), _to_dev(v, dev), flags)
                res = None
            elif op == "append_random":   # (layer, sids, cf, seed, flags): K = V = seeded N(0,1) bf16 drawn on the device
                layer, sids, cf, seed, flags = args
                gen = torch.Generator(device=dev)
                gen.manual_seed(int(seed))
                n = sum(cf) * pool.shape[5]
                kk = torch.randn((n, pool.shape[1], pool.shape[2]), generator=gen, device=dev, dtype=torch.float32).to(torch.bfloat16)
                pool.ts_kv_append(layer, sids, cf, kk, kk, flags)
                res = None
            elif op == "attention":       # (layer, sids, cf, q_bits, k_bits, v_bits, scale) -> out bits
                layer, sids, cf, q, k, v, scale = args
                dq = _to_dev(q, dev)
                out = torch.full_like(dq, float("nan"))
                pool.ts_chunk_attention(layer, sids, cf, dq, _to_dev(k, dev), _to_dev(v, dev), out, None, float(scale))
                torch.cuda.synchronize(dev)
                res = _to_bits(out)
            elif op == "chunk_step":      # (layer, sids, cf, q_bits, k_bits, v_bits, scale, flags) -> out bits (one fused launch)
                layer, sids, cf, q, k, v, scale, flags = args
                dq = _to_dev(q, dev)
                out = torch.full_like(dq, float("nan"))
                pool.ts_chunk_step(layer, sids, cf, dq, _to_dev(k, dev), _to_dev(v, dev), out, None, float(scale), flags)
                torch.cuda.synchronize(dev)
                res = _to_bits(out)
            elif op == "gather":          # (layer, sid) -> (k bits, v bits) in logical order
                gk, gv = pool.ts_gather_kv(*args)
                torch.cuda.synchronize(dev)
                res = (_to_bits(gk), _to_bits(gv))
            elif op == "sync":
                torch.cuda.synchronize(dev)
                res = None
            elif op == "timed_imports":   # (peer, tickets) -> (new sids, ms on the side stream for all fetches)
                peer, tickets = args
                side = torch.cuda.ExternalStream(binding.lib.ts_pool_side_stream(pool._h), device=dev)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(side)
                new = [pool.ts_session_import(peer, t) for t in tickets]
                e1.record(side)
                e1.synchronize()
                res = (new, e0.elapsed_time(e1))
            else:
                raise ValueError(f"unknown worker command {op!r}")
            conn.send(("ok", res))
        except Exception as exc:   # the parent decides what an error means; the worker keeps serving
            conn.send(("err", "".join(traceback.format_exception_only(type(exc), exc)).strip(), getattr(exc, "code", None)))
    if pool is not None:
        pool.close()
    conn.close()


class WorkerError(RuntimeError):
    def __init__(self, text, code):
        super().__init__(text)
        self.code = code


class Worker:
    """Parent-side handle of a worker process."""

    def __init__(self, proc, conn):
        self.proc, self.conn = proc, conn

    def call(self, op, *args, **kw):
        self.conn.send((op, args, kw))
        return self.result()

    def post(self, op, *args, **kw):
        """Send without waiting for the reply (collect it with result()): lets two workers run side by side."""
        self.conn.send((op, args, kw))

    def result(self, timeout=180):
        if not self.conn.poll(timeout):
            raise WorkerError("worker did not answer", None)
        rep = self.conn.recv()
        if rep[0] == "err":
            raise WorkerError(rep[1], rep[2])
        return rep[1]

    def close(self):
        try:
            self.call("exit")
        except Exception:
            pass
        self.proc.join(timeout=30)
        if self.proc.is_alive():
            self.proc.kill()


def spawn(device=0):
    """Starts a worker process for `device` (spawn context: a fresh CUDA context of its own)."""
    ctx = mp.get_context("spawn")
    parent, child = ctx.Pipe()
    proc = ctx.Process(target=serve, args=(child, device), daemon=True)
    proc.start()
    child.close()
    return Worker(proc, parent)
