"""ctypes binding of include/turbochunk.h.  Same names as the C ABI; marshalling only.

Tensors are torch tensors (bf16 or any 16-bit dtype for K/V/Q/O, fp32 for LSE); device memory for the KV
slab and pinned memory for the offload arena are allocated with torch and handed to the library as raw
pointers.  No step of the path is computed in Python.
"""
import ctypes as C
import os

import torch

HERE = os.path.dirname(os.path.abspath(__file__))
lib_path = os.path.join(HERE, "libturbochunk.so")

TS_OK, TS_ERR_INVALID, TS_ERR_STATE, TS_ERR_NO_PAGES, TS_ERR_NO_HOST, TS_ERR_CAPACITY, TS_ERR_CUDA = 0, -1, -2, -3, -4, -5, -6
TS_SESSION_CLOSED, TS_SESSION_RESIDENT, TS_SESSION_SUSPENDED = 0, 1, 2
TS_COMMIT = 1
TS_RUN_APPEND = 1

EXPORTED_SYMBOLS = [
    "ts_pool_page_bytes", "ts_pool_slab_bytes", "ts_pool_create", "ts_pool_destroy", "ts_session_open",
    "ts_session_close", "ts_chunk_attention", "ts_kv_append", "ts_chunk_step", "ts_chunk_step_host", "ts_session_suspend",
    "ts_session_resume", "ts_session_migrate", "ts_offload_sync", "ts_session_info", "ts_session_page_table", "ts_gather_kv",
    "ts_pool_free_list", "ts_pool_stats", "ts_pool_side_stream", "ts_pool_suspend_stream", "ts_pool_launch_count", "ts_pool_sched_builds", "ts_pool_split_batches",
    "ts_pool_clock_probe", "ts_strerror",
    "ts_last_cuda_error", "ts_version",
    "ts_step_plan_create", "ts_step_plan_bind", "ts_step_plan_prepare", "ts_step_plan_run", "ts_step_plan_commit",
    "ts_step_plan_destroy", "ts_step_plan_block_bytes",
    "ts_chunk_attention_static", "ts_static_scratch_bytes",
    "ts_pool_export", "ts_peer_open", "ts_peer_close", "ts_session_freeze", "ts_session_unfreeze", "ts_session_import",
    "ts_session_release",
    "ts_sched_create", "ts_sched_destroy", "ts_sched_event", "ts_sched_moves", "ts_sched_alive",
]


class ts_pool_config(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("n_heads", C.c_int32), ("head_dim", C.c_int32), ("page_tokens", C.c_int32),
                ("n_pages", C.c_int32), ("frame_tokens", C.c_int32), ("window_frames", C.c_int32),
                ("max_sessions", C.c_int32), ("device", C.c_int32), ("reserved", C.c_int32),
                ("free_order", C.POINTER(C.c_int32)), ("kv_slab", C.c_void_p), ("kv_slab_bytes", C.c_int64),
                ("host_arena", C.c_void_p), ("host_bytes", C.c_int64), ("side_stream", C.c_void_p)]


class ts_session_info_t(C.Structure):
    _fields_ = [("state", C.c_int32), ("frames", C.c_int32), ("len_tokens", C.c_int64), ("head_off", C.c_int32),
                ("n_pages", C.c_int32)]


class ts_pool_export_t(C.Structure):
    _fields_ = [("bytes", C.c_ubyte * 320)]


class ts_migration_ticket_t(C.Structure):
    _fields_ = [("sid", C.c_int32), ("frames", C.c_int32), ("head_off", C.c_int32), ("n_pages", C.c_int32)]


class ts_pool_stats_t(C.Structure):
    _fields_ = [("free_pages", C.c_int32), ("resident", C.c_int32), ("suspended", C.c_int32),
                ("host_pages_used", C.c_int32), ("host_pages_cap", C.c_int32), ("reserved", C.c_int32),
                ("page_bytes", C.c_int64)]


class ts_sched_config(C.Structure):
    _fields_ = [("K", C.c_int32), ("M_max", C.c_int32), ("M0", C.c_int32), ("vol_window", C.c_int32),
                ("rho_hat", C.c_double), ("delta", C.c_double), ("eta", C.c_double), ("kappa_alpha", C.c_double),
                ("kappa_beta", C.c_double), ("l_hat", C.POINTER(C.c_double)), ("n_levels", C.c_int32),
                ("reserved", C.c_int32), ("vol_bounds", C.POINTER(C.c_double)), ("vol_rho", C.POINTER(C.c_double))]


class ts_sched_result(C.Structure):
    _fields_ = [("M", C.c_int32), ("n_migrations", C.c_int32), ("n_moves", C.c_int32), ("n_unplaced", C.c_int32),
                ("n_req", C.c_int32), ("reserved", C.c_int32), ("rho_max", C.c_double), ("L", C.c_double),
                ("rho_hat", C.c_double), ("sigma", C.c_double)]


def _load():
    if not os.path.exists(lib_path):
        raise ImportError(f"{lib_path} is missing: run `python -m paper_2606_19271_b200.build` "
                          "(or __graft_entry__.build()). There is no fallback path.")
    L = C.CDLL(lib_path)
    P = C.c_void_p
    I32P = C.POINTER(C.c_int32)
    L.ts_pool_page_bytes.restype = C.c_int64
    L.ts_pool_page_bytes.argtypes = [C.POINTER(ts_pool_config)]
    L.ts_pool_slab_bytes.restype = C.c_int64
    L.ts_pool_slab_bytes.argtypes = [C.POINTER(ts_pool_config)]
    L.ts_pool_create.argtypes = [C.POINTER(ts_pool_config), C.POINTER(P)]
    L.ts_pool_destroy.argtypes = [P]
    L.ts_session_open.argtypes = [P, I32P]
    L.ts_session_close.argtypes = [P, C.c_int32]
    L.ts_chunk_attention.argtypes = [P, C.c_int32, C.c_int32, I32P, I32P, P, P, P, P, P, C.c_float, P]
    L.ts_chunk_attention_static.argtypes = [P, C.c_int32, C.c_int32, I32P, I32P, P, P, P, P, P, C.c_float, P]
    L.ts_static_scratch_bytes.restype = C.c_int64
    L.ts_static_scratch_bytes.argtypes = []
    L.ts_kv_append.argtypes = [P, C.c_int32, C.c_int32, I32P, I32P, P, P, C.c_uint32, P]
    L.ts_chunk_step.argtypes = [P, C.c_int32, C.c_int32, I32P, I32P, P, P, P, P, P, C.c_float, C.c_uint32, P]
    L.ts_chunk_step_host.argtypes = [P, C.c_int32, C.c_int32, I32P, I32P, P, P, P, P, C.c_float, C.c_uint32, P]
    L.ts_session_suspend.argtypes = [P, C.c_int32]
    L.ts_session_resume.argtypes = [P, C.c_int32]
    L.ts_session_migrate.argtypes = [P, C.c_int32, P, I32P]
    L.ts_offload_sync.argtypes = [P]
    L.ts_pool_export.argtypes = [P, C.POINTER(ts_pool_export_t)]
    L.ts_peer_open.argtypes = [P, C.POINTER(ts_pool_export_t), C.POINTER(P)]
    L.ts_peer_close.argtypes = [P]
    L.ts_session_freeze.argtypes = [P, C.c_int32, C.POINTER(ts_migration_ticket_t), I32P, C.c_int32]
    L.ts_session_unfreeze.argtypes = [P, C.c_int32]
    L.ts_session_import.argtypes = [P, P, C.POINTER(ts_migration_ticket_t), I32P, I32P]
    L.ts_session_release.argtypes = [P, C.c_int32, P]
    L.ts_session_info.argtypes = [P, C.c_int32, C.POINTER(ts_session_info_t)]
    L.ts_session_page_table.argtypes = [P, C.c_int32, I32P, C.c_int32, I32P]
    L.ts_gather_kv.argtypes = [P, C.c_int32, C.c_int32, P, P, P]
    L.ts_pool_free_list.argtypes = [P, I32P, C.c_int32, I32P]
    L.ts_pool_stats.argtypes = [P, C.POINTER(ts_pool_stats_t)]
    L.ts_pool_side_stream.restype = P
    L.ts_pool_side_stream.argtypes = [P]
    L.ts_pool_suspend_stream.restype = P
    L.ts_pool_suspend_stream.argtypes = [P]
    L.ts_pool_launch_count.restype = C.c_int64
    L.ts_pool_launch_count.argtypes = [P]
    L.ts_pool_sched_builds.restype = C.c_int64
    L.ts_pool_sched_builds.argtypes = [P]
    L.ts_pool_clock_probe.argtypes = [P, P]
    L.ts_pool_split_batches.restype = C.c_int64
    L.ts_pool_split_batches.argtypes = [P]
    L.ts_step_plan_create.argtypes = [P, C.c_int32, I32P, I32P, C.c_int32, C.POINTER(P)]
    L.ts_step_plan_bind.argtypes = [P, C.c_int32, P, P, P, P, P]
    L.ts_step_plan_prepare.argtypes = [P, P]
    L.ts_step_plan_run.argtypes = [P, C.c_int32, C.c_int32, C.c_float, C.c_uint32, P]
    L.ts_step_plan_commit.argtypes = [P, C.c_uint32, P]
    L.ts_step_plan_destroy.argtypes = [P]
    L.ts_step_plan_block_bytes.restype = C.c_int64
    L.ts_step_plan_block_bytes.argtypes = [P]
    DP = C.POINTER(C.c_double)
    L.ts_sched_create.argtypes = [C.POINTER(ts_sched_config), C.POINTER(P)]
    L.ts_sched_destroy.argtypes = [P]
    L.ts_sched_event.argtypes = [P, C.c_int32, I32P, I32P, DP, I32P, C.POINTER(ts_sched_result)]
    L.ts_sched_moves.argtypes = [P, C.c_int32, I32P, I32P, I32P, C.c_int32, I32P]
    L.ts_sched_alive.argtypes = [P, I32P]
    L.ts_strerror.restype = C.c_char_p
    L.ts_strerror.argtypes = [C.c_int]
    L.ts_last_cuda_error.restype = C.c_char_p
    L.ts_version.restype = C.c_char_p
    return L


lib = _load()


class TurboChunkError(RuntimeError):
    def __init__(self, code, where):
        detail = lib.ts_last_cuda_error().decode() if code == TS_ERR_CUDA else ""
        super().__init__(f"{where}: {lib.ts_strerror(code).decode()} ({code}) {detail}".strip())
        self.code = code


def _check(code, where):
    if code != TS_OK:
        raise TurboChunkError(code, where)


def _i32(values):
    arr = (C.c_int32 * max(1, len(values)))(*[int(x) for x in values])
    return arr


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else C.c_void_p(0)


def _stream(stream, device=None):
    if stream is None:
        stream = torch.cuda.current_stream(device)      # the current stream of the POOL's device, not of the current device
    return C.c_void_p(stream.cuda_stream)


class TurboChunkPool:
    """Owns a ts_pool and the torch memory behind it.  Methods mirror the C ABI one to one."""

    def __init__(self, n_layers, n_heads, head_dim, page_tokens, n_pages, frame_tokens, window_frames,
                 max_sessions, free_order=None, host_pages=0, device=0, guard_bytes=0, poison=None):
        """guard_bytes > 0 (tests): the KV slab and the pinned arena sit between two guard bands of that many bytes filled
        with 0xA5; `check_guards()` tells whether any library write strayed outside them.
        poison (tests): a 16-bit pattern (0x7FC0 = bf16 NaN, 0x7F7F = the largest finite bf16) the whole slab is filled
        with before ts_pool_create; `poison_free_pages()` refills the pages on the free list.  The library needs no
        initialised slab (turbochunk.h): a result must never depend on bytes it has not written itself."""
        cfg = ts_pool_config()
        cfg.n_layers, cfg.n_heads, cfg.head_dim, cfg.page_tokens = n_layers, n_heads, head_dim, page_tokens
        cfg.n_pages, cfg.frame_tokens, cfg.window_frames, cfg.max_sessions = n_pages, frame_tokens, window_frames, max_sessions
        cfg.device = device
        page_bytes = lib.ts_pool_page_bytes(C.byref(cfg))
        if page_bytes < 0:
            raise TurboChunkError(int(page_bytes), "ts_pool_page_bytes")
        self.page_bytes = int(page_bytes)
        slab_bytes = int(lib.ts_pool_slab_bytes(C.byref(cfg)))
        self.device = torch.device("cuda", device)
        # device memory and pinned memory come from torch (PyTorch is the allocator, not the product)
        guard = (int(guard_bytes) + 1023) // 1024 * 1024
        self._guard = guard
        self._slab = torch.empty(slab_bytes + 1024 + 2 * guard, dtype=torch.uint8, device=self.device)
        base = self._slab.data_ptr()
        aligned = (base + guard + 1023) // 1024 * 1024
        self._slab_off = aligned - base
        cfg.kv_slab = aligned
        cfg.kv_slab_bytes = slab_bytes
        self._slab_bytes = slab_bytes
        if guard:
            self._slab[:self._slab_off].fill_(0xA5)
            self._slab[self._slab_off + slab_bytes:].fill_(0xA5)
        self._poison = poison
        if poison is not None:
            self._slab[self._slab_off:self._slab_off + slab_bytes].view(torch.int16).fill_(int(poison) - (1 << 16 if poison >= 1 << 15 else 0))
        self._host = None
        if host_pages > 0:
            self._host = torch.empty(host_pages * self.page_bytes + 2 * guard, dtype=torch.uint8, pin_memory=True)
            if guard:
                self._host[:guard].fill_(0xA5)
                self._host[guard + host_pages * self.page_bytes:].fill_(0xA5)
            cfg.host_arena = self._host.data_ptr() + guard
            cfg.host_bytes = host_pages * self.page_bytes
        self._free_order = None
        if free_order is not None:
            self._free_order = _i32(list(free_order))
            cfg.free_order = C.cast(self._free_order, C.POINTER(C.c_int32))
        self._side = torch.cuda.Stream(device=self.device)
        cfg.side_stream = self._side.cuda_stream
        self.cfg = cfg
        self.shape = (n_layers, n_heads, head_dim, page_tokens, n_pages, frame_tokens, window_frames, max_sessions)
        handle = C.c_void_p()
        _check(lib.ts_pool_create(C.byref(cfg), C.byref(handle)), "ts_pool_create")
        self._h = handle
        self._peers = []     # ts_peer handles opened on this pool (closed with it)

    def check_guards(self):
        """True if the guard bands around the KV slab and the pinned arena still hold their fill pattern."""
        if not self._guard:
            return True
        torch.cuda.synchronize(self.device)
        ok = bool((self._slab[:self._slab_off] == 0xA5).all()) and \
            bool((self._slab[self._slab_off + self._slab_bytes:] == 0xA5).all())
        if self._host is not None:
            n = self._host.numel()
            ok = ok and bool((self._host[:self._guard] == 0xA5).all()) and bool((self._host[n - self._guard:] == 0xA5).all())
        return ok

    def poison_free_pages(self):
        """(tests) Refill every page on the free list with the poison pattern.  Synchronises the device first: a page on
        the free list may still be the source of a suspend's copy or the operand of an enqueued kernel."""
        if self._poison is None:
            return
        torch.cuda.synchronize(self.device)
        body = self._slab[self._slab_off:self._slab_off + self._slab_bytes].view(torch.int16).view(-1, self.page_bytes // 2)
        ids = self.ts_pool_free_list()
        if ids:
            body[torch.tensor(ids, dtype=torch.long, device=self.device)] = int(self._poison) - (1 << 16 if self._poison >= 1 << 15 else 0)
        torch.cuda.synchronize(self.device)

    # ---- lifecycle
    def close(self):
        if getattr(self, "_h", None):
            for peer in list(getattr(self, "_peers", [])):
                lib.ts_peer_close(C.c_void_p(peer))
            self._peers = []
            lib.ts_pool_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def ts_session_open(self):
        sid = C.c_int32(-1)
        _check(lib.ts_session_open(self._h, C.byref(sid)), "ts_session_open")
        return sid.value

    def ts_session_close(self, sid):
        _check(lib.ts_session_close(self._h, sid), "ts_session_close")

    # ---- hot path
    def ts_chunk_attention(self, layer, sids, chunk_frames, q, k, v, out, lse=None, scale=1.0, stream=None):
        _check(lib.ts_chunk_attention(self._h, layer, len(sids), _i32(sids), _i32(chunk_frames), _ptr(q), _ptr(k),
                                      _ptr(v), _ptr(out), _ptr(lse), C.c_float(float(scale)), _stream(stream, self.device)),
               "ts_chunk_attention")

    def ts_chunk_attention_static(self, layer, sids, chunk_frames, q, k, v, out, lse=None, scale=1.0, stream=None):
        """ts_chunk_attention without any allocation: the schedule block lives in the library's static device array."""
        rc = lib.ts_chunk_attention_static(self._h, layer, len(sids), _i32(sids), _i32(chunk_frames), _ptr(q), _ptr(k),
                                           _ptr(v), _ptr(out), _ptr(lse), C.c_float(float(scale)),
                                           _stream(stream, self.device))
        if rc == TS_ERR_CAPACITY:   # the library says which size exceeded which limit
            raise TurboChunkError(rc, lib.ts_last_cuda_error().decode())
        _check(rc, "ts_chunk_attention_static")

    def ts_kv_append(self, layer, sids, chunk_frames, k, v, flags=TS_COMMIT, stream=None):
        _check(lib.ts_kv_append(self._h, layer, len(sids), _i32(sids), _i32(chunk_frames), _ptr(k), _ptr(v),
                                C.c_uint32(flags), _stream(stream, self.device)), "ts_kv_append")

    def ts_chunk_step(self, layer, sids, chunk_frames, q, k, v, out, lse=None, scale=1.0, flags=TS_COMMIT, stream=None):
        _check(lib.ts_chunk_step(self._h, layer, len(sids), _i32(sids), _i32(chunk_frames), _ptr(q), _ptr(k), _ptr(v),
                                 _ptr(out), _ptr(lse), C.c_float(float(scale)), C.c_uint32(flags), _stream(stream, self.device)),
               "ts_chunk_step")

    def ts_chunk_step_host(self, layer, sids, chunk_frames, q_host, k_host, v_host, out_host, scale, flags=TS_COMMIT,
                           stream=None):
        _check(lib.ts_chunk_step_host(self._h, layer, len(sids), _i32(sids), _i32(chunk_frames), _ptr(q_host),
                                      _ptr(k_host), _ptr(v_host), _ptr(out_host), C.c_float(float(scale)),
                                      C.c_uint32(flags), _stream(stream, self.device)), "ts_chunk_step_host")

    def ts_step_plan_create(self, sids, chunk_frames, n_slots=1):
        """A capture-safe multi-layer step plan for this batch (include/turbochunk.h); returns a StepPlan."""
        return StepPlan(self, sids, chunk_frames, n_slots)

    def ts_session_suspend(self, sid):
        _check(lib.ts_session_suspend(self._h, sid), "ts_session_suspend")

    def ts_session_resume(self, sid):
        _check(lib.ts_session_resume(self._h, sid), "ts_session_resume")

    def ts_session_migrate(self, sid, dst):
        """Move RESIDENT session `sid` of this pool to pool `dst`; returns its id there."""
        new = C.c_int32(-1)
        _check(lib.ts_session_migrate(self._h, sid, dst._h, C.byref(new)), "ts_session_migrate")
        return new.value

    def ts_offload_sync(self):
        _check(lib.ts_offload_sync(self._h), "ts_offload_sync")

    # ---- migration between worker processes (include/turbochunk.h): everything that crosses the process boundary is
    #      plain Python data (bytes, ints, lists), so it can go through any pipe or socket
    def ts_pool_export(self):
        """This pool's registration blob (bytes) for the other worker's ts_peer_open."""
        blob = ts_pool_export_t()
        _check(lib.ts_pool_export(self._h, C.byref(blob)), "ts_pool_export")
        return bytes(blob.bytes)

    def ts_peer_open(self, blob):
        """Maps the pool another process exported; returns an opaque peer handle (int) for import / release."""
        b = ts_pool_export_t()
        C.memmove(b.bytes, bytes(blob), len(b.bytes))
        peer = C.c_void_p()
        _check(lib.ts_peer_open(self._h, C.byref(b), C.byref(peer)), "ts_peer_open")
        self._peers.append(peer.value)
        return peer.value

    def ts_peer_close(self, peer):
        self._peers.remove(peer)
        _check(lib.ts_peer_close(C.c_void_p(peer)), "ts_peer_close")

    def ts_session_freeze(self, sid):
        """(i) freeze: returns the ticket {"sid", "frames", "head_off", "pages"} to send to the target worker."""
        cap = max(1, self.ts_session_info(sid)["n_pages"])
        t = ts_migration_ticket_t()
        pages = (C.c_int32 * cap)()
        _check(lib.ts_session_freeze(self._h, sid, C.byref(t), pages, cap), "ts_session_freeze")
        return {"sid": t.sid, "frames": t.frames, "head_off": t.head_off, "pages": list(pages[:t.n_pages])}

    def ts_session_unfreeze(self, sid):
        _check(lib.ts_session_unfreeze(self._h, sid), "ts_session_unfreeze")

    def ts_session_import(self, peer, ticket):
        """(ii) fetch + verify on the target: returns the session's id in this pool."""
        t = ts_migration_ticket_t(int(ticket["sid"]), int(ticket["frames"]), int(ticket["head_off"]), len(ticket["pages"]))
        new = C.c_int32(-1)
        _check(lib.ts_session_import(self._h, C.c_void_p(peer), C.byref(t), _i32(ticket["pages"]), C.byref(new)),
               "ts_session_import")
        return new.value

    def ts_session_release(self, sid, peer=None):
        """(iii) ownership flip on the source, after the target has returned from ts_session_import."""
        _check(lib.ts_session_release(self._h, sid, C.c_void_p(peer) if peer is not None else C.c_void_p(0)),
               "ts_session_release")

    # ---- introspection
    def ts_session_info(self, sid):
        info = ts_session_info_t()
        _check(lib.ts_session_info(self._h, sid, C.byref(info)), "ts_session_info")
        return {"state": info.state, "frames": info.frames, "len_tokens": info.len_tokens,
                "head_off": info.head_off, "n_pages": info.n_pages}

    def ts_session_page_table(self, sid):
        n = C.c_int32(0)
        _check(lib.ts_session_page_table(self._h, sid, None, 0, C.byref(n)), "ts_session_page_table")
        buf = (C.c_int32 * max(1, n.value))()
        _check(lib.ts_session_page_table(self._h, sid, buf, n.value, C.byref(n)), "ts_session_page_table")
        return [buf[i] for i in range(n.value)]

    def ts_pool_free_list(self):
        n = C.c_int32(0)
        _check(lib.ts_pool_free_list(self._h, None, 0, C.byref(n)), "ts_pool_free_list")
        buf = (C.c_int32 * max(1, n.value))()
        _check(lib.ts_pool_free_list(self._h, buf, n.value, C.byref(n)), "ts_pool_free_list")
        return [buf[i] for i in range(n.value)]

    def ts_gather_kv(self, layer, sid, stream=None):
        info = self.ts_session_info(sid)
        H, D = self.shape[1], self.shape[2]
        k = torch.empty((info["len_tokens"], H, D), dtype=torch.bfloat16, device=self.device)
        v = torch.empty_like(k)
        _check(lib.ts_gather_kv(self._h, layer, sid, _ptr(k), _ptr(v), _stream(stream, self.device)), "ts_gather_kv")
        return k, v

    def ts_pool_stats(self):
        st = ts_pool_stats_t()
        _check(lib.ts_pool_stats(self._h, C.byref(st)), "ts_pool_stats")
        return {f: getattr(st, f) for f, _ in ts_pool_stats_t._fields_ if f != "reserved"}

    def ts_pool_launch_count(self):
        return int(lib.ts_pool_launch_count(self._h))

    def ts_pool_sched_builds(self):
        return int(lib.ts_pool_sched_builds(self._h))

    def ts_pool_split_batches(self):
        return int(lib.ts_pool_split_batches(self._h))

    def ts_pool_clock_probe(self, buf):
        """buf: torch int64[2] on the pool's device (zeroed by the caller), or None to switch the probe off."""
        _check(lib.ts_pool_clock_probe(self._h, _ptr(buf)), "ts_pool_clock_probe")
        self._probe = buf

    @property
    def side_stream(self):
        """The stream resumes (and migration fetches) run on."""
        return self._side

    @property
    def suspend_stream(self):
        """The stream suspends run on (owned by the library), as a torch stream for event timing."""
        if getattr(self, "_out", None) is None:
            self._out = torch.cuda.ExternalStream(int(lib.ts_pool_suspend_stream(self._h)), device=self.device)
        return self._out


class StepPlan:
    """ctypes view of the ts_step_plan_* calls; keeps the bound tensors alive.  Marshalling only."""

    def __init__(self, pool, sids, chunk_frames, n_slots=1):
        h = C.c_void_p()
        _check(lib.ts_step_plan_create(pool._h, len(sids), _i32(sids), _i32(chunk_frames), n_slots, C.byref(h)),
               "ts_step_plan_create")
        self._h, self._pool, self._keep = h, pool, {}

    def ts_step_plan_bind(self, slot, q, k, v, out, lse=None):
        _check(lib.ts_step_plan_bind(self._h, slot, _ptr(q), _ptr(k), _ptr(v), _ptr(out), _ptr(lse)), "ts_step_plan_bind")
        self._keep[slot] = (q, k, v, out, lse)

    def ts_step_plan_prepare(self, stream=None):
        _check(lib.ts_step_plan_prepare(self._h, _stream(stream, self._pool.device)), "ts_step_plan_prepare")

    def ts_step_plan_run(self, layer, slot, scale, run_flags=TS_RUN_APPEND, stream=None):
        _check(lib.ts_step_plan_run(self._h, layer, slot, C.c_float(float(scale)), C.c_uint32(run_flags), _stream(stream, self._pool.device)),
               "ts_step_plan_run")

    def ts_step_plan_commit(self, flags=TS_COMMIT, stream=None):
        _check(lib.ts_step_plan_commit(self._h, C.c_uint32(flags), _stream(stream, self._pool.device)), "ts_step_plan_commit")

    def ts_step_plan_block_bytes(self):
        return int(lib.ts_step_plan_block_bytes(self._h))

    def close(self):
        if getattr(self, "_h", None):
            lib.ts_step_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            if getattr(self._pool, "_h", None):    # the pool must still exist: the plan points into it
                self.close()
        except Exception:
            pass


class TurboSched:
    """ctypes view of include/turbochunk_sched.h (the closed-loop scheduler, §5.2).  Host code only."""

    def __init__(self, K, M_max, M0, l_hat, rho_hat=0.7, delta=0.1, eta=0.0, kappa_alpha=0.0, kappa_beta=0.0,
                 vol_window=0, vol_bounds=(), vol_rho=()):
        cfg = ts_sched_config()
        cfg.K, cfg.M_max, cfg.M0, cfg.vol_window = K, M_max, M0, vol_window
        cfg.rho_hat, cfg.delta, cfg.eta, cfg.kappa_alpha, cfg.kappa_beta = rho_hat, delta, eta, kappa_alpha, kappa_beta
        self._l_hat = (C.c_double * len(l_hat))(*[float(x) for x in l_hat])
        cfg.l_hat = C.cast(self._l_hat, C.POINTER(C.c_double))
        cfg.n_levels = len(vol_rho)
        self._vb = (C.c_double * max(1, len(vol_bounds)))(*[float(x) for x in vol_bounds])
        self._vr = (C.c_double * max(1, len(vol_rho)))(*[float(x) for x in vol_rho])
        cfg.vol_bounds = C.cast(self._vb, C.POINTER(C.c_double))
        cfg.vol_rho = C.cast(self._vr, C.POINTER(C.c_double))
        if len(l_hat) != K + 1 or (vol_window and len(vol_bounds) != len(vol_rho) - 1):
            raise TurboChunkError(TS_ERR_INVALID, "ts_sched_create")
        self.M_max = M_max
        h = C.c_void_p()
        _check(lib.ts_sched_create(C.byref(cfg), C.byref(h)), "ts_sched_create")
        self._h = h

    def close(self):
        if getattr(self, "_h", None):
            lib.ts_sched_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _moves(self, which):
        n = C.c_int32(0)
        _check(lib.ts_sched_moves(self._h, which, None, None, None, 0, C.byref(n)), "ts_sched_moves")
        a, b, c = ((C.c_int32 * max(1, n.value))() for _ in range(3))
        _check(lib.ts_sched_moves(self._h, which, a, b, c, n.value, C.byref(n)), "ts_sched_moves")
        return [(a[i], b[i], c[i]) for i in range(n.value)]

    def ts_sched_event(self, sessions):
        """sessions: list of (session id, alpha, state_mb) in event order; returns the decision of Algorithm 1."""
        n = len(sessions)
        ids = _i32([s[0] for s in sessions])
        act = _i32([s[1] for s in sessions])
        mb = (C.c_double * max(1, n))(*[float(s[2]) for s in sessions])
        phi = (C.c_int32 * max(1, n))()
        res = ts_sched_result()
        _check(lib.ts_sched_event(self._h, n, ids, act, mb, phi, C.byref(res)), "ts_sched_event")
        alive = (C.c_int32 * self.M_max)()
        _check(lib.ts_sched_alive(self._h, alive), "ts_sched_alive")
        return {"M": res.M, "alive": [j for j in range(self.M_max) if alive[j]], "rho_max": res.rho_max, "L": res.L,
                "phi": {sessions[i][0]: phi[i] for i in range(n)}, "migrations": self._moves(0), "moves": self._moves(1),
                "n_unplaced": res.n_unplaced, "rho_hat": res.rho_hat, "sigma": res.sigma, "n_req": res.n_req}
