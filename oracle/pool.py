"""Oracle state model: paged KV pool, per-session page tables, lifecycle (TEST INFRASTRUCTURE).

Follows SURVEY.md §8(c) "Oracle state", O2 (append + window roll), O3 (suspend / resume /
open / close).  Paper passages: PAPER.md:66 step (iii) "writes the generated chunks and updated
states back to their corresponding sessions"; :74 three session states and lifecycle operations;
:76 offloading steps (i)-(iii); :261 isolated per-session state regions + ownership table.
Readings of what the paper leaves open (R5-R16, R18) are listed in DESIGN.md.

Notation: H heads, D head_dim, B page_tokens, T frame_tokens, W window_frames,
NL layers; per session P (cached frames), L = P*T cached tokens, o (dead slots at the start of
the first page, 0 <= o < B), PT (physical page ids in logical order).
Logical token j of a session lives at page PT[(o+j) // B], slot (o+j) % B   (R7).
"""
from collections import deque

import numpy as np

INVALID, STATE, NO_PAGES, NO_HOST, CAPACITY = "INVALID", "STATE", "NO_PAGES", "NO_HOST", "CAPACITY"
RESIDENT, SUSPENDED = "RESIDENT", "SUSPENDED"


class OracleError(Exception):
    def __init__(self, kind, msg=""):
        super().__init__(f"{kind}: {msg}")
        self.kind = kind


class _Session:
    def __init__(self):
        self.state = RESIDENT
        self.P = 0          # committed cached frames
        self.o = 0          # dead slots at the head of PT[0]
        self.PT = []        # physical page ids, logical order
        self.host = None    # (K pages, V pages, n_pages) while SUSPENDED


class OraclePool:
    def __init__(self, n_layers, n_heads, head_dim, page_tokens, n_pages, frame_tokens,
                 window_frames, max_sessions, free_order=None, host_pages=None):
        self.NL, self.H, self.D = n_layers, n_heads, head_dim
        self.B, self.n_pages, self.T, self.W = page_tokens, n_pages, frame_tokens, window_frames
        self.max_sessions = max_sessions
        order = np.arange(n_pages) if free_order is None else np.asarray(free_order)
        if sorted(order.tolist()) != list(range(n_pages)):
            raise OracleError(INVALID, "free_order is not a permutation")
        self.free = deque(int(p) for p in order)          # FIFO: pop front to allocate, push back to free (R8)
        # bf16 bit patterns; layout [layer][page][slot][head][dim] (private: only logical gathers are compared)
        self.K = np.zeros((n_layers, n_pages, page_tokens, n_heads, head_dim), dtype=np.uint16)
        self.V = np.zeros_like(self.K)
        self.sessions = {}
        self.host_pages_cap = host_pages          # None = unbounded
        self.host_pages_used = 0

    # ---- lifecycle -------------------------------------------------------------
    def open(self):
        """initialization: lowest unused id, P = o = 0, empty PT, RESIDENT (R13)."""
        for sid in range(self.max_sessions):
            if sid not in self.sessions:
                self.sessions[sid] = _Session()
                return sid
        raise OracleError(CAPACITY, "no free session id")

    def close(self, sid):
        """termination: all resources released (PAPER.md:74 (iii)). Legal from RESIDENT or SUSPENDED."""
        s = self._get(sid)
        if s.state == RESIDENT:
            self.free.extend(s.PT)                 # logical order, to the back
        else:
            self.host_pages_used -= s.host[2]
        del self.sessions[sid]

    def suspend(self, sid):
        """PAPER.md:76 (i)-(ii): copy persistent state GPU->host, mark suspended, release the GPU slot.
        Whole pages of every layer, in logical order (R11); ids go to the back of `free` in logical order."""
        s = self._get(sid)
        if s.state != RESIDENT:
            raise OracleError(STATE, "suspend of a non-resident session")
        n = len(s.PT)
        if self.host_pages_cap is not None and self.host_pages_used + n > self.host_pages_cap:
            raise OracleError(NO_HOST, "pinned arena full")
        idx = np.asarray(s.PT, dtype=np.int64)
        s.host = (self.K[:, idx].copy(), self.V[:, idx].copy(), n)
        self.host_pages_used += n
        self.free.extend(s.PT)
        s.PT = []
        s.state = SUSPENDED

    def resume(self, sid):
        """PAPER.md:76 (iii): restore the state to the GPU before generation resumes."""
        s = self._get(sid)
        if s.state != SUSPENDED:
            raise OracleError(STATE, "resume of a non-suspended session")
        hk, hv, n = s.host
        if n > len(self.free):
            raise OracleError(NO_PAGES, "resume needs more pages than are free")
        s.PT = [self.free.popleft() for _ in range(n)]
        idx = np.asarray(s.PT, dtype=np.int64)
        self.K[:, idx] = hk
        self.V[:, idx] = hv
        self.host_pages_used -= n
        s.host = None
        s.state = RESIDENT

    # ---- GPU-GPU migration (O4; "migrates only the corresponding per-session state region";
    #      :265 consistency protocol (i) freeze at a chunk boundary, (ii) target fetches and verifies that the
    #      buffers are installed, (iii) ownership flips only after the transfer) ---------------------------
    def migrate_to(self, sid, dst):
        """Move RESIDENT session `sid` of this pool (the source worker) to pool `dst` (the target worker).
        Reading R22 (the paper fixes neither ids nor page order): the target installs the session exactly as
        a resume would - lowest unused id, |PT| pages popped from the FRONT of its free list, whole pages of
        every layer copied in logical order (R11), same (P, o); the source then releases the session exactly
        as a close would - its page ids go to the BACK of its free list in logical order and the id becomes
        reusable.  All-or-nothing: every check comes before any change to either pool.  Returns the new id."""
        s = self._get(sid)
        if dst is self:
            raise OracleError(INVALID, "migration to the same pool")
        if (self.NL, self.H, self.D, self.B, self.T, self.W) != (dst.NL, dst.H, dst.D, dst.B, dst.T, dst.W):
            raise OracleError(INVALID, "pools differ in geometry")
        if s.state != RESIDENT:
            raise OracleError(STATE, "migration of a non-resident session")   # (i): only a live, frozen state moves
        new_sid = next((i for i in range(dst.max_sessions) if i not in dst.sessions), None)
        if new_sid is None:
            raise OracleError(CAPACITY, "no free session id on the target")
        if len(s.PT) > len(dst.free):
            raise OracleError(NO_PAGES, "target has too few free pages")
        t = _Session()
        t.P, t.o = s.P, s.o
        t.PT = [dst.free.popleft() for _ in range(len(s.PT))]
        for a, b in zip(s.PT, t.PT):                   # (ii) fetch: page by page, logical order, every layer
            dst.K[:, b] = self.K[:, a]
            dst.V[:, b] = self.V[:, a]
        dst.sessions[new_sid] = t                      # (iii) ownership: installed on the target ...
        self.free.extend(s.PT)                         # ... released on the source
        del self.sessions[sid]
        return new_sid

    # ---- append + window roll (O2; PAPER.md:66 (iii)) --------------------------------------------
    def append(self, layer, sids, chunk_frames, kn, vn, commit=True):
        """kn, vn: uint16 bf16 bits [sum C_s, H, D], sessions concatenated in `sids` order (R15)."""
        self._check_batch(layer, sids, chunk_frames)
        B, T = self.B, self.T
        total = sum(c * T for c in chunk_frames)
        if kn.shape != (total, self.H, self.D) or vn.shape != kn.shape:
            raise OracleError(INVALID, "k/v shape")
        need = []
        for sid, c in zip(sids, chunk_frames):
            s = self.sessions[sid]
            end = s.o + s.P * T + c * T
            need.append(max(0, -(-end // B) - len(s.PT)))       # R14: growth is idempotent, a table never shrinks on append
        if sum(need) > len(self.free):
            raise OracleError(NO_PAGES, "append needs more pages than are free")   # all-or-nothing
        off = 0
        for sid, c, nd in zip(sids, chunk_frames, need):
            s = self.sessions[sid]
            for _ in range(nd):
                s.PT.append(self.free.popleft())
            L = s.P * T
            for t in range(c * T):
                x = s.o + L + t
                page, slot = s.PT[x // B], x % B
                self.K[layer, page, slot] = kn[off + t]
                self.V[layer, page, slot] = vn[off + t]
            off += c * T
            if commit:
                s.P += c
                e = max(0, s.P - self.W) if self.W > 0 else 0     # evict oldest WHOLE frames (R6 ii, R10)
                s.P -= e
                s.o += e * T
                while s.o >= B:
                    self.free.append(s.PT.pop(0))                 # page fully dead -> back of the free list
                    s.o -= B

    # ---- introspection -------------------------------------------------------------------------
    def info(self, sid):
        s = self._get(sid)
        n_pages = len(s.PT) if s.state == RESIDENT else s.host[2]
        return {"state": s.state, "len_tokens": s.P * self.T, "head_off": s.o, "n_pages": n_pages,
                "frames": s.P}

    def page_table(self, sid):
        return list(self._get(sid).PT)

    def gather_kv(self, layer, sid):
        """Logical K, V of a RESIDENT session: uint16 [L, H, D]."""
        s = self._get(sid)
        if s.state != RESIDENT:
            raise OracleError(STATE, "gather of a non-resident session")
        L = s.P * self.T
        x = s.o + np.arange(L, dtype=np.int64)
        pages = np.asarray(s.PT, dtype=np.int64)[x // self.B] if L else np.zeros(0, dtype=np.int64)
        slots = x % self.B
        return self.K[layer, pages, slots].copy(), self.V[layer, pages, slots].copy()

    def stats(self):
        res = sum(1 for s in self.sessions.values() if s.state == RESIDENT)
        return {"free_pages": len(self.free), "resident": res, "suspended": len(self.sessions) - res,
                "host_pages_used": self.host_pages_used}

    # ---- helpers ---------------------------------------------------------------------------------
    def _get(self, sid):
        if sid not in self.sessions:
            raise OracleError(STATE, f"session {sid} is not open")
        return self.sessions[sid]

    def _check_batch(self, layer, sids, chunk_frames):
        if not (0 <= layer < self.NL):
            raise OracleError(INVALID, "layer")
        if len(sids) != len(chunk_frames):
            raise OracleError(INVALID, "sids/chunk_frames length")
        if len(sids) > self.max_sessions:
            raise OracleError(CAPACITY, "batch larger than max_sessions")
        if len(set(sids)) != len(sids):
            raise OracleError(INVALID, "duplicate session in batch")
        for c in chunk_frames:
            if c < 1 or (self.W > 0 and c > self.W):
                raise OracleError(INVALID, "chunk_frames out of [1, W]")      # R18
        for sid in sids:
            if self._get(sid).state != RESIDENT:
                raise OracleError(STATE, "session in batch is not resident")  # R12
