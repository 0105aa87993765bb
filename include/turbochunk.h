/*
 * turbochunk.h — C ABI of the B200-native coalesced chunk-processing library.
 *
 * The library implements, for ONE GPU, the data-parallel hot path of TurboServe
 * (arxiv/paper_2606_19271): coalesced chunk processing over persistent per-session
 * state.  Citations are PAPER.md:<line> (+ section) or SURVEY.md §8 readings (Rn),
 * which DESIGN.md lists.
 *
 *   PAPER.md:66  §3.1  coalesced execution: (i) collect ready sessions, (ii) group them
 *                      into one coalesced chunk batch, (iii) invoke the model once and write
 *                      the generated chunks and updated states back per session.
 *   PAPER.md:74  §3.1  session states execution / suspend / terminate; lifecycle operations
 *                      initialization, suspension, resumption, termination.
 *   PAPER.md:76  §3.1  GPU-CPU state offloading: copy state to host, mark suspended and release
 *                      the GPU slot, restore before generation resumes.
 *   PAPER.md:261 §6.1  isolated per-session state regions (incl. "temporal or KV-cache states")
 *                      and a session ownership table.
 *
 * Conventions
 *   - Every call returns TS_OK (0) or a negative ts_status.  No C++ exception crosses the ABI.
 *   - All-or-nothing: a call validates its whole batch and its page demand before it mutates
 *     anything; on error no host or device state has changed.
 *   - Host metadata (page tables, lengths, states, free list) mutates synchronously, in program
 *     order, at call time.  Device effects are stream-ordered: the library orders its side
 *     (offload) stream against the caller's compute stream with events, never with host waits
 *     (ts_offload_sync excepted).
 *   - Threading: one caller thread per pool.  Compute calls of one pool that are issued on
 *     different streams must be ordered by the caller.
 *   - Pointers named *device* are CUDA device pointers on the pool's device; *host* are host
 *     pointers.  bf16 tensors are raw 16-bit patterns.  The caller owns Q/K/V/O/LSE buffers and
 *     must keep them alive until the stream reaches the call.
 *   - No fallback: an unsupported shape is TS_ERR_INVALID, never a slow path.  Without a CUDA
 *     device every compute call fails with TS_ERR_CUDA.
 *
 * Notation: H heads, D head_dim, B page_tokens, T frame_tokens, W window_frames,
 * NL layers.  Per session: P cached frames, L = P*T cached tokens, o = dead slots at the head of
 * the first page (0 <= o < B), PT = page table (physical ids, logical order).  Logical token j
 * lives at page PT[(o+j) div B], slot (o+j) mod B  (R7).
 */
#ifndef TURBOCHUNK_H_
#define TURBOCHUNK_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ts_pool ts_pool; /* opaque */

typedef enum ts_status {
  TS_OK = 0,
  TS_ERR_INVALID = -1,  /* null pointer, bad shape/layer, duplicate sid in a batch, chunk_frames < 1 or > W */
  TS_ERR_STATE = -2,    /* session closed / not RESIDENT for attention, append, suspend / not SUSPENDED for resume */
  TS_ERR_NO_PAGES = -3, /* device page demand exceeds the free list */
  TS_ERR_NO_HOST = -4,  /* pinned host arena cannot hold the suspended pages */
  TS_ERR_CAPACITY = -5, /* no free session id, or batch larger than max_sessions */
  TS_ERR_CUDA = -6      /* a CUDA runtime/driver call failed (see ts_last_cuda_error) */
} ts_status;

enum { TS_SESSION_CLOSED = 0, TS_SESSION_RESIDENT = 1, TS_SESSION_SUSPENDED = 2 };

/* ts_kv_append flags */
enum { TS_COMMIT = 1u }; /* advance P by chunk_frames and roll the window (R14: pass on the last layer of a step) */

typedef struct ts_pool_config {
  int32_t n_layers;      /* NL >= 1 */
  int32_t n_heads;       /* H >= 1 */
  int32_t head_dim;      /* D in {64, 128} */
  int32_t page_tokens;   /* B: power of two, 16 <= B <= 1024 */
  int32_t n_pages;       /* physical pages; one page holds B tokens of K and V for all heads and all layers */
  int32_t frame_tokens;  /* T >= 1 */
  int32_t window_frames; /* W; <= 0 means no rolling-window cap */
  int32_t max_sessions;  /* cap on live (resident + suspended) sessions and on the batch size ("bounded") */
  int32_t device;        /* CUDA device ordinal */
  int32_t reserved;
  /* Optional permutation of 0..n_pages-1 = initial FIFO free-list order (R8, R9). NULL = identity. Copied. */
  const int32_t* free_order; /* host */
  /* KV slab: device memory of at least ts_pool_slab_bytes() bytes, 1024-byte aligned.  NULL: the library
   * allocates it with cudaMalloc.  Caller-provided memory (e.g. a torch tensor) stays owned by the caller
   * and must outlive the pool.  The slab needs NO initialisation and is never cleared: no result depends on a
   * byte the library has not written itself ("isolated per-session state regions").  The
   * attention gathers only table entries that hold a cached token of the session; the slots of those pages
   * that hold no visible token (dead head slots, the tail behind the last token) are masked, and they are
   * the session's own older tokens or the append's zero fill. */
  void* kv_slab;          /* device */
  int64_t kv_slab_bytes;
  /* Pinned host arena for suspended sessions, in whole pages of ts_pool_page_bytes().  NULL with
   * host_bytes > 0: the library allocates it with cudaHostAlloc. */
  void* host_arena;       /* host, page-locked */
  int64_t host_bytes;
  /* Side stream (cudaStream_t) for suspend/resume copies.  NULL: the library creates a non-blocking one. */
  void* side_stream;
} ts_pool_config;

typedef struct ts_session_info_t {
  int32_t state;       /* TS_SESSION_* */
  int32_t frames;      /* P */
  int64_t len_tokens;  /* L = P*T */
  int32_t head_off;    /* o */
  int32_t n_pages;     /* |PT| (saved page count while suspended) */
} ts_session_info_t;

typedef struct ts_pool_stats_t {
  int32_t free_pages;
  int32_t resident;
  int32_t suspended;
  int32_t host_pages_used;
  int32_t host_pages_cap;
  int32_t reserved;
  int64_t page_bytes;
} ts_pool_stats_t;

/* Layout helpers (pure host arithmetic; usable without a GPU). Return < 0 on an invalid config. */
int64_t ts_pool_page_bytes(const ts_pool_config* cfg); /* NL * 2 * H * B * D * 2 */
int64_t ts_pool_slab_bytes(const ts_pool_config* cfg); /* n_pages * page bytes */

/* create the per-GPU pool: KV slab, free list, session table, offload arena, side stream. */
int ts_pool_create(const ts_pool_config* cfg, ts_pool** out);
int ts_pool_destroy(ts_pool* pool);

/* PAPER.md:74 "initialization": new session with the lowest free id (R13), P = o = 0, empty PT, RESIDENT. */
int ts_session_open(ts_pool* pool, int32_t* sid_out);
/* PAPER.md:74 "termination": releases every resource.  Legal from RESIDENT (pages pushed to the back of
 * the free list in logical order) or SUSPENDED (host copy dropped). */
int ts_session_close(ts_pool* pool, int32_t sid);

/*
 * PAPER.md:66 (i)-(iii), the attention contraction inside "invokes the model once for the batch".
 * For each session sids[b] (all RESIDENT, no duplicates), head h and chunk token i (frame f = i div T):
 *   out[i,h,:] = softmax_j( scale * <q[i,h,:], k_j> ) . v_j   over the visible keys j =
 *     the session's cached tokens of its last min(P, W - c) frames (whole cache if W <= 0)  (R6)
 *     U the chunk's own tokens of frames <= f  (frame-block-causal, R1).
 * bf16 operands, fp32 accumulation and fp32 online softmax, bf16 output (R3, R4).
 *   q, k, v, out : device bf16 [sum_b C_b][H][D], sessions concatenated in sids order, no padding (R15);
 *                  C_b = chunk_frames[b] * T.  q, k, v 16-byte aligned, out 32-byte aligned (it is written with 256-bit
 *                  stores, one full 32-byte sector per lane).
 *   lse          : device fp32 [sum_b C_b][H] natural-log logsumexp of the scaled logits, or NULL.
 *   scale        : softmax scale (R2).
 *   cuda_stream  : cudaStream_t of the caller (NULL = legacy default stream).
 * Does not change pool state (R5).  Waits (stream-side) for a pending resume of any session in the batch.
 * n == 0 is a no-op.
 */
int ts_chunk_attention(ts_pool* pool, int32_t layer, int32_t n, const int32_t* sids /*host*/,
                       const int32_t* chunk_frames /*host*/, const void* q, const void* k, const void* v,
                       void* out, float* lse, float scale, void* cuda_stream);

/*
 * ts_chunk_attention (PAPER.md:66 (i)-(iii), same arguments, same result) for callers that cannot allocate: a process with
 * a CUDA graph capture in progress (cudaMalloc is illegal then in the default capture mode), tight serving loops, harnesses
 * that forbid cudaMalloc.  The call makes no cudaMalloc, cudaFree,
 * cudaHostAlloc or event creation: the launch's schedule block (per-session tensor maps, session descriptors, packed page
 * tables, work items and the kernel's work-item cursor and feed rings) lives in ONE array of ts_static_scratch_bytes()
 * (256 KiB) bytes built into the library's device image - every GPU that loads the library holds it until the process
 * exits - and reaches it by one cudaMemcpyAsync from ordinary host memory on `cuda_stream`, followed by the one launch.
 * Limits and rules that ts_chunk_attention does not have:
 *   - TS_ERR_CAPACITY (ts_last_cuda_error() names both sizes) when the batch's block does not fit the array; nothing was
 *     enqueued.  53 KB for configs[2] (8 sessions x 12 heads), ~160 KB for 32 such sessions.
 *   - All calls on a device SHARE the array, which keeps the last call's contents: every call rewrites the whole block, the
 *     cursor and the rings as zeros, so nothing is inherited - but two calls whose GPU work can overlap (different streams,
 *     or different pools on one device, without an event between them) race on it.  One stream, or the caller's own
 *     event edges, is the rule; host threads are serialised by the library.
 *   - The call is not entered into the pool's event timelines: a session with a resume still copying in, or inside a step
 *     plan, is TS_ERR_STATE (no stream-side wait), and the caller must let the call's work complete (or order it by its
 *     own events) before it suspends, closes or migrates a session of the batch.
 *   - The host may wait for work already in `cuda_stream` (the block is copied from pageable memory).
 *   - Do not capture the call itself into a graph: the copy would become a node that re-reads, at every replay, a host image
 *     the next call overwrites.  ts_step_plan_run is the capturable launch.
 * Other errors as ts_chunk_attention.  Does not change pool state (R5).  n == 0 is a no-op.
 */
int ts_chunk_attention_static(ts_pool* pool, int32_t layer, int32_t n, const int32_t* sids /*host*/,
                              const int32_t* chunk_frames /*host*/, const void* q, const void* k, const void* v,
                              void* out, float* lse, float scale, void* cuda_stream);
/* Size in bytes of the static device scratch array behind ts_chunk_attention_static. */
int64_t ts_static_scratch_bytes(void);

/*
 * PAPER.md:66 (iii) "writes the generated chunks and updated states back to their corresponding sessions".
 * Sessions in sids order: grow PT by ceil((o+L+C)/B) - |PT| pages popped from the front of the free list
 * (idempotent across the layers of one step), scatter the chunk's K/V to logical positions [L, L+C) of
 * `layer` (byte-exact 128-bit copies).  With TS_COMMIT: P += c, then roll the window: evict e = max(0, P - W)
 * oldest whole frames, o += e*T, pages whose slots are all dead go to the back of the free list (R6, R10).
 *   k, v : device bf16 [sum_b C_b][H][D] as above.
 * Multi-layer protocol (R14): one step appends the SAME batch and chunk_frames to every layer and passes TS_COMMIT on the
 * last one; a table never shrinks on append (a session that already holds more pages than a call needs contributes no
 * demand), and the slots of the last page behind the appended tokens are zero-filled, so an uncommitted append must not be
 * followed by a shorter one to the same layer before the commit.
 */
int ts_kv_append(ts_pool* pool, int32_t layer, int32_t n, const int32_t* sids /*host*/,
                 const int32_t* chunk_frames /*host*/, const void* k, const void* v, uint32_t flags,
                 void* cuda_stream);

/*
 * One coalesced chunk step with DEVICE buffers: ts_chunk_attention followed by ts_kv_append(flags) as one call
 * (PAPER.md:66 (iii): "invokes the model once for the batch ... writes ... updated states back").  Results are those
 * of the two calls in sequence.  The append writes cache slots this step's attention does not read (R5) and is
 * HBM-bound while the attention is not, so it is carried out INSIDE the attention launch, by the two warps of every
 * CTA that have no other role: one kernel, and the step takes what the attention takes.
 * Arguments as in the two calls.  All-or-nothing: arguments and page demand are checked before anything changes.
 * PAPER.md:76 (iii): when some sessions of the batch still have a resume in flight on the side stream and others do not, the
 * call (like ts_chunk_attention) runs as TWO launches - the ready sessions first, the resuming ones behind their copy events -
 * so that the ready sessions' attention hides the copies instead of following them; results are those of one launch.  (A
 * CUDA failure between the two leaves the first group committed and the second group's tables grown, as after an
 * uncommitted append.)
 */
int ts_chunk_step(ts_pool* pool, int32_t layer, int32_t n, const int32_t* sids /*host*/,
                  const int32_t* chunk_frames /*host*/, const void* q, const void* k, const void* v, void* out,
                  float* lse, float scale, uint32_t flags, void* cuda_stream);

/*
 * One coalesced chunk step with HOST buffers (the end-to-end entry point): copies q,k,v from (pinned) host
 * memory to device staging owned by the pool, runs ts_chunk_attention and ts_kv_append(flags) on
 * `cuda_stream`, copies `out` back to out_host.  The call returns without waiting.
 *   q_host, k_host, v_host : host bf16 [sum_b C_b][H][D] (pinned for asynchronous copies).  They are read by a copy
 *       stream of the pool that does NOT wait for `cuda_stream`: the contents must be valid when the call is made
 *       and stay unchanged until `cuda_stream` has passed the call.  That is what lets the input copy of one call
 *       run under the attention and the output copy of the previous one (two staging sets).
 *   out_host : host bf16, same shape; complete once `cuda_stream` has passed the call (stream order).
 * Staging grows on demand (cudaMalloc; an outgrown buffer is kept until the pool is destroyed, nothing is waited for) and is
 * reused.  q_host, k_host, v_host packed behind one another ([3][sum C][H][D], tensor size a multiple of 1024 bytes) are copied
 * in ONE transfer.  Runs the fused ts_chunk_step (one launch).  All-or-nothing: arguments, states and the page demand are
 * checked before a single copy is enqueued (TS_ERR_NO_PAGES leaves out_host untouched).
 */
int ts_chunk_step_host(ts_pool* pool, int32_t layer, int32_t n, const int32_t* sids, const int32_t* chunk_frames,
                       const void* q_host, const void* k_host, const void* v_host, void* out_host,
                       float scale, uint32_t flags, void* cuda_stream);

/*
 * Capture-safe multi-layer chunk step.  PAPER.md:66 (iii): the worker "invokes the model once
 * for the batch" - NL layers x several denoising passes of attention over the SAME batch and the same caches - "and
 * writes the generated chunks and updated states back".  A plan splits ts_chunk_step into the part that depends on
 * the sessions' state (once per chunk step, host + one upload) and the part that is repeated per layer and pass (one
 * kernel launch and nothing else), so that the launches of a whole step can be captured into a CUDA graph once and
 * replayed for every later chunk step of the same batch:
 *
 *   ts_step_plan_create(pool, n, sids, chunk_frames, n_slots, &plan)   batch composition and buffers are fixed per plan
 *   ts_step_plan_bind(plan, slot, q, k, v, out, lse)                   n_slots sets of device tensors (e.g. one per layer,
 *                                                                      or one reused by all layers)
 *   per chunk step:
 *     ts_step_plan_prepare(plan, stream)      NOT capturable.  Validates as ts_chunk_step (TS_ERR_STATE, TS_ERR_NO_PAGES;
 *                                             all-or-nothing), grows the page tables for the step's append, builds the
 *                                             schedule (a1) and writes it into the plan's device block in stream order
 *                                             (one small copy kernel reading mapped pinned memory); enqueues the stream-side waits (pending
 *                                             resumes, copies out of recycled pages).  The block's address, the grid
 *                                             and every kernel argument are the same for every prepare of a plan.
 *     ts_step_plan_run(plan, layer, slot, scale, run_flags, stream)
 *                                             capturable: exactly one kernel launch, no copy, no event, no allocation.
 *                                             Attention of `layer` on the tensors of `slot`; with TS_RUN_APPEND the
 *                                             launch also appends the slot's K/V to `layer` (as ts_chunk_step does).
 *                                             Any number of runs per step, in stream order (layers x passes).
 *     ts_step_plan_commit(plan, flags, stream)  NOT capturable.  Ends the step: host bookkeeping of ts_kv_append(flags)
 *                                             (TS_COMMIT: P += c and the window roll; 0: the tables stay grown, nothing
 *                                             advances) and the event after which the step's launches count as done.
 *   ts_step_plan_destroy(plan)
 *
 * Between prepare and commit the batch's sessions belong to the plan: every other call that names one of them
 * (attention, append, step, suspend, close, migrate, another plan) returns TS_ERR_STATE.  Launches of one plan must not
 * overlap in time (one stream, or ordered streams): they share the plan's work-item cursor, which each launch rearms
 * for the next.  A graph captured between a prepare and a commit may be replayed after any later prepare of the same plan.
 * A plan points into its pool: destroy it before ts_pool_destroy.
 * Errors: create: as ts_chunk_attention's batch checks, TS_ERR_CUDA; bind: TS_ERR_INVALID (slot, null or misaligned
 * pointer), TS_ERR_STATE (plan prepared); run: TS_ERR_STATE (not prepared, slot not bound), TS_ERR_INVALID.
 */
typedef struct ts_step_plan ts_step_plan; /* opaque */
enum { TS_RUN_APPEND = 1u };              /* ts_step_plan_run flags */
int ts_step_plan_create(ts_pool* pool, int32_t n, const int32_t* sids /*host*/, const int32_t* chunk_frames /*host*/,
                        int32_t n_slots, ts_step_plan** out);
int ts_step_plan_bind(ts_step_plan* plan, int32_t slot, const void* q, const void* k, const void* v, void* out,
                      float* lse /*nullable*/); /* device bf16 [sum C][H][D] as ts_chunk_attention */
int ts_step_plan_prepare(ts_step_plan* plan, void* cuda_stream);
int ts_step_plan_run(ts_step_plan* plan, int32_t layer, int32_t slot, float scale, uint32_t run_flags, void* cuda_stream);
int ts_step_plan_commit(ts_step_plan* plan, uint32_t flags, void* cuda_stream);
int ts_step_plan_destroy(ts_step_plan* plan);
/* Size of the plan's device block (tensor maps, descriptors, page tables, work items), for reporting. */
int64_t ts_step_plan_block_bytes(ts_step_plan* plan);

/* PAPER.md:76 (i)-(ii): copy the session's pages (every layer, whole pages, logical order — R11) to the pinned
 * arena on the pool's suspend stream, after the compute-stream work already enqueued on that session; mark SUSPENDED;
 * push its page ids to the back of the free list in logical order.  A freed page is not handed to a later
 * writer before the copy out of it has completed (event-ordered).  Suspends (device -> host) and resumes (host -> device)
 * run on two streams of the pool, so that the two directions of the host link work at the same time; every dependency
 * between them (a resume into pages a suspend is still reading, a suspend into arena slots a resume is still reading, the
 * suspend and the resume of one session) is an event edge. */
int ts_session_suspend(ts_pool* pool, int32_t sid);
/* PAPER.md:76 (iii): pop the saved number of pages from the front of the free list, copy the host pages back
 * on the side stream, mark RESIDENT.  Later compute calls on the session wait (stream-side) for the copy. */
int ts_session_resume(ts_pool* pool, int32_t sid);
/* Host-blocks until all offload work (both streams) enqueued so far has completed. */
int ts_offload_sync(ts_pool* pool);

/*
 * PAPER.md:263 §6.1 "GPU-GPU state migration": move an active session from one worker (pool) to another by moving
 * only its per-session state region; "the target worker can then fetch the registered state buffers from the source
 * worker through ... one-sided GPU memory access and install them into its local session table".
 * PAPER.md:265 "migration consistency": only at chunk boundaries; (i) the source completes the current chunk update
 * and freezes the state, (ii) the target fetches it and verifies that the buffers are installed, (iii) ownership is
 * updated only after the transfer completes.
 * Reading R22 (the paper fixes neither ids nor page order): the target installs the session as a resume would -
 * lowest free id (returned in *sid_out), |PT| pages popped from the FRONT of its free list, whole pages of every
 * layer in logical order (R11), same (P, o), RESIDENT; the source releases it as a close would - page ids to the BACK
 * of its free list in logical order, id reusable.
 *   src, dst : two pools of identical geometry (NL, H, D, B, T, W), on the same device or on two devices of this
 *              process with peer access (the fetch is ONE kernel on the target's device and side stream that reads
 *              the source slab through the peer mapping: NVLink loads, no host staging, no copy-engine call per page).
 *   sid      : RESIDENT session of src (a SUSPENDED one is TS_ERR_STATE: resume it where it should live instead).
 * Ordering, all stream-side: the fetch starts after the compute work already enqueued on the session at the source
 * (i); compute calls on the new session wait for the fetch (ii); the source's pages are not handed to a later writer
 * before the fetch has completed (iii).  The host tables of both pools change at call time.
 * Errors (nothing changes): TS_ERR_STATE (sid closed or not RESIDENT), TS_ERR_INVALID (src == dst, geometry differs),
 * TS_ERR_CAPACITY (no free id on dst), TS_ERR_NO_PAGES (dst free list too short), TS_ERR_CUDA (no peer access).
 */
int ts_session_migrate(ts_pool* src, int32_t sid, ts_pool* dst, int32_t* sid_out);

/*
 * The same move between two WORKER PROCESSES (PAPER.md:66, :271: one worker per GPU; :263 "registers the corresponding
 * state buffers ... the target worker can then fetch the registered state buffers from the source worker through ...
 * one-sided GPU memory access"; :265 (i) freeze, (ii) fetch + verify, (iii) ownership flips after the transfer).  The two
 * pools live in two processes, on one GPU or on two GPUs of a node with peer access; CUDA IPC makes the source slab an
 * ordinary device pointer for the target's fetch kernel, and every GPU-side dependency is an interprocess event edge - no
 * host wait in either process.  What travels between the processes (the "control plane": a pipe, a socket - not this
 * library's business) is plain bytes, and must be delivered in order:
 *   registration, once per pair of workers:  ts_pool_export on each side -> the blob -> ts_peer_open on the other side
 *   per move:  source ts_session_freeze -> ticket + page ids -> target ts_session_import -> "enqueued" (any message)
 *              -> source ts_session_release.
 * Result and id / page-order rules exactly as ts_session_migrate (R22): the target installs the session under its lowest
 * free id with |PT| pages popped from the front of its free list; the source's page ids go to the back of its free list
 * in logical order when it releases.
 *
 * ts_pool_export  : fills `out` (opaque bytes: IPC handles of the slab's allocation and of two interprocess events,
 *                   geometry).  The slab must come from cudaMalloc (the pool's own, or a caller slab inside a cudaMalloc
 *                   allocation - not from a virtual-memory allocator).  Idempotent.  TS_ERR_CUDA if IPC is unavailable.
 * ts_peer_open    : maps the remote slab into `local`'s process; TS_ERR_INVALID if the blob is malformed or the geometry
 *                   (NL, H, D, B, T, W) differs from `local`'s.  A blob cannot be opened in the process that exported it.
 * ts_peer_close   : waits for `local`'s side stream, then unmaps.  Every peer opened on a blob must be closed before the pool
 *                   that exported it is destroyed (CUDA IPC: the exporter keeps the memory alive for its importers).
 * ts_session_freeze : (i).  sid RESIDENT and not held by a step plan (else TS_ERR_STATE).  Records "state frozen" on the
 *                   source's side stream behind the compute work already enqueued on the session; from here until
 *                   release / unfreeze every other call on the session is TS_ERR_STATE.  Writes the ticket and the
 *                   session's page ids in logical order (`cap` >= n_pages, else TS_ERR_INVALID and nothing changes).
 * ts_session_unfreeze : the move is called off (the target had no room): the session is RESIDENT again.
 * ts_session_import : (ii).  `source` = ts_peer_open of the source's blob on `dst`.  Verifies the ticket against the
 *                   geometry (o < B, P <= W, n_pages * B >= o + P * T, every page id inside the source slab:
 *                   TS_ERR_INVALID), then as the target half of ts_session_migrate: TS_ERR_CAPACITY, TS_ERR_NO_PAGES,
 *                   TS_ERR_CUDA leave `dst` unchanged.  The fetch (one kernel on dst's side stream) waits for the source's
 *                   "state frozen"; compute calls on the new session wait for the fetch; "installed" is recorded behind it.
 * ts_session_release : (iii).  `target` = ts_peer_open of the target's blob on `src` (NULL: the caller itself guarantees
 *                   that the fetch has completed).  The source's side stream waits for the target's "installed" before
 *                   the freed pages can be handed to a writer; the session id is free again.  Call it only after the
 *                   target has returned from ts_session_import.
 */
#define TS_POOL_EXPORT_BYTES 320
typedef struct ts_pool_export_t {
  unsigned char bytes[TS_POOL_EXPORT_BYTES];
} ts_pool_export_t;
typedef struct ts_migration_ticket_t {
  int32_t sid;       /* id at the source (for ts_session_release / ts_session_unfreeze) */
  int32_t frames;    /* P */
  int32_t head_off;  /* o */
  int32_t n_pages;   /* |PT| */
} ts_migration_ticket_t;
typedef struct ts_peer ts_peer;
int ts_pool_export(ts_pool* pool, ts_pool_export_t* out);
int ts_peer_open(ts_pool* local, const ts_pool_export_t* remote, ts_peer** out);
int ts_peer_close(ts_peer* peer);
int ts_session_freeze(ts_pool* src, int32_t sid, ts_migration_ticket_t* ticket, int32_t* pages_out /*host*/, int32_t cap);
int ts_session_unfreeze(ts_pool* src, int32_t sid);
int ts_session_import(ts_pool* dst, ts_peer* source, const ts_migration_ticket_t* ticket, const int32_t* pages /*host*/,
                      int32_t* sid_out);
int ts_session_release(ts_pool* src, int32_t sid, ts_peer* target /*nullable*/);

/* Introspection (parity is taken on these, never on raw slabs: the physical layout is private). */
int ts_session_info(ts_pool* pool, int32_t sid, ts_session_info_t* out);
/* Copies up to `cap` page ids (logical order) to `out` (host); *n_out = |PT|. */
int ts_session_page_table(ts_pool* pool, int32_t sid, int32_t* out, int32_t cap, int32_t* n_out);
/* Logical K and V of a RESIDENT session, device bf16 [L][H][D] each, gathered through the page table. */
int ts_gather_kv(ts_pool* pool, int32_t layer, int32_t sid, void* k_out, void* v_out, void* cuda_stream);
/* Copies up to `cap` ids of the free list, front first. */
int ts_pool_free_list(ts_pool* pool, int32_t* out, int32_t cap, int32_t* n_out);
int ts_pool_stats(ts_pool* pool, ts_pool_stats_t* out);
/* The offload streams in use (cudaStream_t), for timing offload with events: resumes and migration fetches run on the side
 * stream (ts_pool_config.side_stream, or the pool's own), suspends on the suspend stream (always the pool's own). */
void* ts_pool_side_stream(ts_pool* pool);
void* ts_pool_suspend_stream(ts_pool* pool);
/* Number of kernels the library has launched on this pool since creation, descriptor-upload kernels included
 * (bench.py's gpu_launches). */
int64_t ts_pool_launch_count(ts_pool* pool);

/* Number of times the ragged batch scheduler (a1) had to build a schedule (the rest were reuses of the cached one). */
int64_t ts_pool_sched_builds(ts_pool* pool);
/* Number of attention / step calls that ran as two launches because some of their sessions still had a resume in flight
 * (see ts_chunk_step). */
int64_t ts_pool_split_batches(ts_pool* pool);
/* Measurement aid: while `device_u64x2` (device, 8-byte aligned, caller-zeroed) is set, CTA 0 of every attention
 * launch (captured launches: those recorded while it was set) adds the SM cycles and the nanoseconds it ran for to
 * [0] and [1]; [0] / [1] is the SM clock in GHz under the kernel itself, which a host-side sampler cannot see.
 * NULL switches it off.  Launches must not overlap while it is on. */
int ts_pool_clock_probe(ts_pool* pool, void* device_u64x2);

const char* ts_strerror(int code);
/* Text of the last CUDA error seen by this pool's calls on this thread ("" if none). */
const char* ts_last_cuda_error(void);
/* Library version string. */
const char* ts_version(void);

#ifdef __cplusplus
}
#endif
#endif /* TURBOCHUNK_H_ */
