// Host side of the library: paged KV pool, deterministic FIFO free list, per-session page tables, lifecycle
// state machine, the ragged batch scheduler (step a1, PAPER.md:66 (i)-(ii)) and the
// C ABI of include/turbochunk.h.  Device work is launched from here; the kernels live in attention_sm100.cu
// and kv_copy.cu.
//
// Slab layout (private): [page][layer][K|V][H][B][D] bf16.  One page is one contiguous block of
// NL*2*H*B*D*2 bytes (one cudaMemcpyAsync unit for offload); one (page, layer, K|V, head) block is a dense
// [B][D] box that TMA loads with a 128-byte swizzle.
#include <cudaTypedefs.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <queue>
#include <string>

#include "internal.h"

namespace tc {

static thread_local std::string g_last_cuda_error;

static bool cuda_ok(cudaError_t e, const char* what) {
  if (e == cudaSuccess) return true;
  g_last_cuda_error = std::string(what) + ": " + cudaGetErrorString(e);
  cudaGetLastError();   // clear a non-sticky error
  return false;
}
#define TS_CUDA(call)                                  \
  do {                                                 \
    if (!tc::cuda_ok((call), #call)) return TS_ERR_CUDA; \
  } while (0)

static PFN_cuTensorMapEncodeTiled_v12000 get_encode() {
  static PFN_cuTensorMapEncodeTiled_v12000 fn = nullptr;
  if (fn == nullptr) {
    void* ptr = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<PFN_cuTensorMapEncodeTiled_v12000>(ptr);
  }
  return fn;
}

// Orders work between the caller's compute stream and the pool's side stream without host waits.
// Every recorded event gets a monotonically increasing sequence number; objects (sessions, pages) remember the
// sequence number after which they are safe to touch.
struct EventTimeline {
  std::deque<cudaEvent_t> live;      // events of the sequence numbers done + 1 .. next_seq - 1, oldest first
  std::vector<cudaEvent_t> spare;    // completed events, reused by record()
  uint64_t next_seq = 1;             // 0 means "nothing pending"
  uint64_t done = 0;                 // every seq <= done has completed
  bool init() { return true; }
  void destroy() {
    for (cudaEvent_t e : live) cudaEventDestroy(e);
    for (cudaEvent_t e : spare) cudaEventDestroy(e);
    live.clear();
    spare.clear();
  }
  void retire() {                    // never waits: events that have completed go back to the spare list
    while (!live.empty()) {
      if (cudaEventQuery(live.front()) != cudaSuccess) {
        cudaGetLastError();
        break;
      }
      spare.push_back(live.front());
      live.pop_front();
      ++done;
    }
  }
  bool is_done(uint64_t seq) {
    if (done < seq) retire();
    return done >= seq;
  }
  // The number of live events follows the work in flight (a few dozen); nothing here ever blocks the host.
  uint64_t record(cudaStream_t s) {
    if (live.size() >= 64) retire();
    cudaEvent_t e = nullptr;
    if (!spare.empty()) {
      e = spare.back();
      spare.pop_back();
    } else if (cudaEventCreateWithFlags(&e, cudaEventDisableTiming) != cudaSuccess) {
      cudaGetLastError();
      // out of events: fall back to draining the stream once, then this sequence number is trivially complete
      cudaStreamSynchronize(s);
      retire();
      return next_seq - 1;
    }
    cudaEventRecord(e, s);
    live.push_back(e);
    return next_seq++;
  }
  cudaError_t wait(cudaStream_t s, uint64_t seq) {
    if (seq == 0 || is_done(seq)) return cudaSuccess;
    return cudaStreamWaitEvent(s, live[(size_t)(seq - done - 1)], 0);
  }
  void sync_all() {                  // pool teardown only
    if (!live.empty()) cudaEventSynchronize(live.back());
    retire();
  }
};

struct Session {
  int state = TS_SESSION_CLOSED;
  int P = 0;                        // committed cached frames
  int o = 0;                        // dead slots at the head of the first page
  std::vector<int32_t> pt;          // physical page ids, logical order
  std::vector<int32_t> host_slots;  // arena slots holding the pages while SUSPENDED (logical order)
  uint64_t compute_seq = 0;         // last compute-stream call that touched the session
  uint64_t side_seq = 0;            // last side-stream copy that touched the session
  uint64_t ver = 0;                 // new value whenever P, o or pt change (keys the attention schedule cache)
  bool in_plan = false;             // between ts_step_plan_prepare and ts_step_plan_commit: no other call may touch it
  bool frozen = false;              // between ts_session_freeze and ts_session_release / _unfreeze (in_plan is set too, so
                                    // every other call refuses the session)
};

struct Staging {      // pinned (mapped) host + device buffer pair for per-call schedule records
  uint8_t* h = nullptr;
  uint8_t* h_dev = nullptr;      // the device-side address of `h` (what the upload kernel reads)
  uint8_t* d = nullptr;
  size_t cap = 0;
  cudaEvent_t ev = nullptr;      // recorded on the consumer's stream after the kernel that reads `d`
  cudaEvent_t ev_up = nullptr;   // recorded on the pool's upload stream after the upload kernel of the block
  bool in_flight = false;
};

}  // namespace tc

using namespace tc;

// The KV append of a fused chunk step, prepared on the host (pages already allocated) and carried out by the idle
// warps of the attention kernel.
struct FusedAppend {
  std::vector<CopySess> cs;            // pt_off is filled in from the attention schedule (same packed page tables)
  uint64_t wait_side = 0, wait_compute = 0;
  int total_rows = 0;
  std::vector<int32_t> popped;         // page ids taken from the free list, in pop order (rolled back on failure)
  void reset() {
    cs.clear();
    popped.clear();
    wait_side = wait_compute = 0;
    total_rows = 0;
  }
};

struct ts_pool {
  ts_pool_config cfg;
  int log2_B = 0;
  int64_t kv_bytes = 0;      // H*B*D*2 : one K (or V) block of one layer of one page
  int64_t layer_bytes = 0;   // 2*kv_bytes
  int64_t page_bytes = 0;    // NL*layer_bytes
  uint8_t* slab = nullptr;
  bool own_slab = false;
  uint8_t* host = nullptr;
  bool own_host = false;
  int host_pages_cap = 0;
  std::deque<int32_t> host_free;         // free arena slots, FIFO: a suspend takes the slots freed longest ago, not the ones a
                                         // resume on the other offload stream may still be reading
  std::deque<int32_t> free_q;            // FIFO free list (R8)
  std::vector<uint64_t> page_compute_seq, page_side_seq;
  std::vector<Session> sess;
  cudaStream_t side = nullptr;
  bool own_side = false;
  cudaStream_t side_out = nullptr;         // suspends (device -> host) run here, resumes (host -> device) on `side`: the host
                                           // link is full duplex, one stream would put the two directions behind one another
  std::vector<uint64_t> host_slot_seq;     // per arena slot: the resume (side timeline) that still reads it
  EventTimeline tl_compute, tl_side;
  std::vector<CUtensorMap> map_k, map_v;   // per layer
  int sm_count = 0;
  static constexpr int kRing = 8;
  Staging ring[kRing];
  int ring_next = 0;
  cudaStream_t up_s = nullptr;             // upload stream of the per-call schedule / descriptor blocks
  uint8_t* stage_dev = nullptr;            // ts_chunk_step_host: two device staging sets for q,k,v,out
  cudaStream_t h2d_s = nullptr, d2h_s = nullptr;   // ... its copy streams (input of step t+1 overlaps step t)
  cudaEvent_t ev_in = nullptr, ev_attn = nullptr, ev_out = nullptr, ev_free[2] = {nullptr, nullptr};
  uint64_t host_steps = 0;
  size_t stage_cap = 0;
  int64_t launches = 0;
  std::vector<int32_t> scratch_mark;       // duplicate detection
  std::vector<int32_t> scratch_need;       // per-session page demand of the call in progress
  std::vector<int64_t> scratch_key;        // schedule key of the call in progress
  std::vector<int32_t> scratch_pending, scratch_sub_sids, scratch_sub_cf, scratch_sub_off;   // run_batch(): groups of a split batch
  std::vector<tc::CopySess> scratch_sub_cs;
  int64_t split_batches = 0;               // batches run as two launches (ready sessions first, resuming ones behind their copies)
  std::vector<uint8_t*> retired;           // outgrown staging buffers, freed with the pool (never under running work)
  FusedAppend scratch_fused_obj;            // descriptors of the fused append of the call in progress
  FusedAppend* scratch_fused = &scratch_fused_obj;
  // attention schedule of the last batch (a1), reused while the batch and its sessions' page tables are unchanged:
  // every layer and denoising pass of one chunk step then pays the scheduler once
  uint64_t ver_seq = 0;                    // source of Session::ver values (never repeats, also across reopen)
  std::vector<int64_t> sched_key;
  std::vector<tc::SessDesc> sched_sess;
  std::vector<int32_t> sched_pt, sched_cta;
  std::vector<tc::WorkItem> sched_items;
  int64_t sched_builds = 0;
  unsigned long long* clock_probe = nullptr;   // ts_pool_clock_probe
  // migration between worker processes (ts_pool_export): interprocess events, recorded on the side stream
  cudaEvent_t ipc_frozen = nullptr;            // "state frozen": after the compute work of the last frozen session
  cudaEvent_t ipc_installed = nullptr;         // "installed": after the last fetch into this pool
  bool exported = false;
  ts_pool_export_t export_blob;
};

namespace tc {

static bool valid_config(const ts_pool_config* c) {
  if (c == nullptr) return false;
  if (c->n_layers < 1 || c->n_heads < 1 || c->n_pages < 1 || c->frame_tokens < 1 || c->max_sessions < 1) return false;
  if (c->head_dim != 64 && c->head_dim != 128) return false;
  const int B = c->page_tokens;
  if (B < 16 || B > 1024 || (B & (B - 1)) != 0) return false;
  return true;
}

static size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

static int acquire_staging(ts_pool* pool, size_t bytes, Staging** out) {
  Staging& s = pool->ring[pool->ring_next];
  pool->ring_next = (pool->ring_next + 1) % ts_pool::kRing;
  if (s.ev == nullptr) TS_CUDA(cudaEventCreateWithFlags(&s.ev, cudaEventDisableTiming));
  if (s.ev_up == nullptr) TS_CUDA(cudaEventCreateWithFlags(&s.ev_up, cudaEventDisableTiming));
  if (s.in_flight) {
    TS_CUDA(cudaEventSynchronize(s.ev));   // normally long done: the ring is 8 calls deep
    s.in_flight = false;
  }
  if (s.cap < bytes) {
    if (s.h) cudaFreeHost(s.h);
    if (s.d) cudaFree(s.d);
    s.h = s.d = nullptr;
    s.cap = 0;
    const size_t cap = align_up(std::max(bytes * 2, (size_t)65536), 4096);
    TS_CUDA(cudaHostAlloc((void**)&s.h, cap, cudaHostAllocMapped));
    TS_CUDA(cudaHostGetDevicePointer((void**)&s.h_dev, s.h, 0));
    TS_CUDA(cudaMalloc((void**)&s.d, cap));
    s.cap = cap;
  }
  *out = &s;
  return TS_OK;
}

// The per-call descriptor block does not depend on anything the caller's stream is doing: it is uploaded on the pool's
// own (high-priority) stream, so that the copy runs under / in the tail of the previous kernel instead of between two
// kernels of the caller's stream, which only waits for the (normally long complete) upload event.  The copy is a small
// kernel reading mapped pinned memory, never a DMA copy: those queue behind the offload traffic of the copy engines.
static int upload_staging(ts_pool* pool, Staging* st, size_t bytes, cudaStream_t consumer) {
  if (pool->up_s == nullptr) {
    int lo = 0, hi = 0;
    TS_CUDA(cudaDeviceGetStreamPriorityRange(&lo, &hi));
    TS_CUDA(cudaStreamCreateWithPriority(&pool->up_s, cudaStreamNonBlocking, hi));
  }
  TS_CUDA(launch_upload(st->h_dev, st->d, align_up(bytes, 16), pool->up_s));
  ++pool->launches;
  TS_CUDA(cudaEventRecord(st->ev_up, pool->up_s));
  TS_CUDA(cudaStreamWaitEvent(consumer, st->ev_up, 0));
  return TS_OK;
}

static int check_batch(ts_pool* pool, int32_t layer, int32_t n, const int32_t* sids, const int32_t* cf) {
  const ts_pool_config& c = pool->cfg;
  if (layer < 0 || layer >= c.n_layers || n < 0) return TS_ERR_INVALID;
  if (n == 0) return TS_OK;
  if (sids == nullptr || cf == nullptr) return TS_ERR_INVALID;
  if (n > c.max_sessions) return TS_ERR_CAPACITY;
  std::vector<int32_t>& mark = pool->scratch_mark;
  mark.assign(c.max_sessions, 0);
  int64_t total = 0;
  for (int b = 0; b < n; ++b) {
    if (cf[b] < 1 || (c.window_frames > 0 && cf[b] > c.window_frames)) return TS_ERR_INVALID;
    total += (int64_t)cf[b] * c.frame_tokens;
  }
  if (total > (int64_t)1 << 30) return TS_ERR_INVALID;
  // a malformed batch (the same id twice, R13) is TS_ERR_INVALID whatever the state of its sessions; states come second
  for (int b = 0; b < n; ++b) {
    const int sid = sids[b];
    if (sid < 0 || sid >= c.max_sessions) {
      for (int a = 0; a < b; ++a)
        if (sids[a] == sid) return TS_ERR_INVALID;
      continue;
    }
    if (mark[sid]) return TS_ERR_INVALID;
    mark[sid] = 1;
  }
  for (int b = 0; b < n; ++b) {
    const int sid = sids[b];
    if (sid < 0 || sid >= c.max_sessions) return TS_ERR_STATE;
    if (pool->sess[sid].state == TS_SESSION_CLOSED) return TS_ERR_STATE;
  }
  for (int b = 0; b < n; ++b)
    if (pool->sess[sids[b]].state != TS_SESSION_RESIDENT || pool->sess[sids[b]].in_plan) return TS_ERR_STATE;
  return TS_OK;
}

static bool encode_map(CUtensorMap* m, void* base, int rank, const cuuint64_t* dims, const cuuint64_t* strides,
                       const cuuint32_t* box) {
  PFN_cuTensorMapEncodeTiled_v12000 enc = get_encode();
  if (enc == nullptr) {
    g_last_cuda_error = "cuTensorMapEncodeTiled entry point not found";
    return false;
  }
  cuuint32_t es[5] = {1, 1, 1, 1, 1};
  CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, rank, base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                   CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    g_last_cuda_error = "cuTensorMapEncodeTiled failed with CUresult " + std::to_string((int)r);
    return false;
  }
  return true;
}

// ---- step a1: ragged batch scheduler ---------------------------------------------------------------------
// Builds, in one pinned staging block: per-session tensor maps, SessDesc, packed page tables, and the work
// items (session, head, query-tile pair) distributed over `grid` persistent CTAs by longest-processing-time
// first (cost = KV tiles x query tiles), so that ragged sessions finish together.
struct ScheduleLayout {
  size_t off_maps, off_sess, off_pt, off_cta, off_items, bytes;
  int n_items, grid;
};

static void item_geometry(const ts_pool_config& c, int C, int x_begin, int x_end, int q_tile, int max_tiles, int* n_q,
                          int* n_kv) {
  const int r0 = q_tile * 128;
  *n_q = (max_tiles >= 2 && r0 + 128 < C) ? 2 : 1;
  const int last_row = std::min(C, r0 + 128 * *n_q) - 1;
  const int kv_hi = std::min(C, (last_row / c.frame_tokens + 1) * c.frame_tokens);
  const int n_chunk = (kv_hi + 127) / 128;
  const int n_prior = x_end > x_begin ? ((x_end - 1) / 128 - x_begin / 128 + 1) : 0;
  *n_kv = n_prior + n_chunk;
}

}  // namespace tc

// =================================================================================================== C ABI
extern "C" {

const char* ts_version(void) { return "turbochunk 0.1 (sm_100a)"; }

const char* ts_strerror(int code) {
  switch (code) {
    case TS_OK: return "ok";
    case TS_ERR_INVALID: return "invalid argument";
    case TS_ERR_STATE: return "session is in the wrong state";
    case TS_ERR_NO_PAGES: return "not enough free device pages";
    case TS_ERR_NO_HOST: return "pinned host arena is full";
    case TS_ERR_CAPACITY: return "session capacity exceeded";
    case TS_ERR_CUDA: return "CUDA error";
    default: return "unknown status";
  }
}

const char* ts_last_cuda_error(void) { return tc::g_last_cuda_error.c_str(); }

int64_t ts_pool_page_bytes(const ts_pool_config* cfg) {
  if (!valid_config(cfg)) return TS_ERR_INVALID;
  return (int64_t)cfg->n_layers * 2 * cfg->n_heads * cfg->page_tokens * cfg->head_dim * 2;
}

int64_t ts_pool_slab_bytes(const ts_pool_config* cfg) {
  if (!valid_config(cfg)) return TS_ERR_INVALID;
  return ts_pool_page_bytes(cfg) * cfg->n_pages;
}

int ts_pool_destroy(ts_pool* pool) {
  if (pool == nullptr) return TS_ERR_INVALID;
  cudaSetDevice(pool->cfg.device);
  // wait for the pool's own work only (its streams and the last call recorded on each timeline), not for the device
  pool->tl_compute.sync_all();
  pool->tl_side.sync_all();
  if (pool->side) cudaStreamSynchronize(pool->side);
  if (pool->side_out) cudaStreamSynchronize(pool->side_out);
  for (cudaStream_t st : {pool->up_s, pool->h2d_s, pool->d2h_s})
    if (st) cudaStreamSynchronize(st);
  for (Staging& s : pool->ring)
    if (s.in_flight && s.ev) cudaEventSynchronize(s.ev);
  for (uint8_t* r : pool->retired) cudaFree(r);
  for (Staging& s : pool->ring) {
    if (s.h) cudaFreeHost(s.h);
    if (s.d) cudaFree(s.d);
    if (s.ev) cudaEventDestroy(s.ev);
    if (s.ev_up) cudaEventDestroy(s.ev_up);
  }
  if (pool->up_s) cudaStreamDestroy(pool->up_s);
  if (pool->stage_dev) cudaFree(pool->stage_dev);
  if (pool->h2d_s) cudaStreamDestroy(pool->h2d_s);
  if (pool->d2h_s) cudaStreamDestroy(pool->d2h_s);
  for (cudaEvent_t e : {pool->ev_in, pool->ev_attn, pool->ev_out, pool->ev_free[0], pool->ev_free[1]})
    if (e) cudaEventDestroy(e);
  pool->tl_compute.destroy();
  pool->tl_side.destroy();
  if (pool->ipc_frozen) cudaEventDestroy(pool->ipc_frozen);
  if (pool->ipc_installed) cudaEventDestroy(pool->ipc_installed);
  if (pool->own_side && pool->side) cudaStreamDestroy(pool->side);
  if (pool->side_out) cudaStreamDestroy(pool->side_out);
  if (pool->own_slab && pool->slab) cudaFree(pool->slab);
  if (pool->own_host && pool->host) cudaFreeHost(pool->host);
  cudaGetLastError();
  delete pool;
  return TS_OK;
}

int ts_pool_create(const ts_pool_config* cfg, ts_pool** out) {
  if (out == nullptr) return TS_ERR_INVALID;
  *out = nullptr;
  if (!valid_config(cfg)) return TS_ERR_INVALID;
  if (cfg->free_order != nullptr) {
    std::vector<char> seen(cfg->n_pages, 0);
    for (int i = 0; i < cfg->n_pages; ++i) {
      const int p = cfg->free_order[i];
      if (p < 0 || p >= cfg->n_pages || seen[p]) return TS_ERR_INVALID;
      seen[p] = 1;
    }
  }
  const int64_t page_bytes = ts_pool_page_bytes(cfg);
  const int64_t slab_bytes = page_bytes * cfg->n_pages;
  if (cfg->kv_slab != nullptr && (cfg->kv_slab_bytes < slab_bytes || ((uintptr_t)cfg->kv_slab & 1023) != 0)) return TS_ERR_INVALID;
  if (cfg->host_bytes < 0) return TS_ERR_INVALID;

  TS_CUDA(cudaSetDevice(cfg->device));
  cudaDeviceProp prop;
  TS_CUDA(cudaGetDeviceProperties(&prop, cfg->device));
  if (prop.major != 10) {
    g_last_cuda_error = "device is not sm_100-class (tcgen05/TMEM required); no fallback path exists";
    return TS_ERR_CUDA;
  }

  ts_pool* pool = new ts_pool();
  pool->cfg = *cfg;
  pool->cfg.free_order = nullptr;
  pool->sm_count = prop.multiProcessorCount;
  int l2 = 0;
  while ((1 << l2) < cfg->page_tokens) ++l2;
  pool->log2_B = l2;
  pool->kv_bytes = (int64_t)cfg->n_heads * cfg->page_tokens * cfg->head_dim * 2;
  pool->layer_bytes = 2 * pool->kv_bytes;
  pool->page_bytes = page_bytes;

  auto fail = [&](int code) {
    ts_pool_destroy(pool);
    return code;
  };
  if (!pool->tl_compute.init() || !pool->tl_side.init()) {
    g_last_cuda_error = "cudaEventCreate failed";
    return fail(TS_ERR_CUDA);
  }
  if (cfg->kv_slab != nullptr) {
    pool->slab = (uint8_t*)cfg->kv_slab;
  } else {
    if (!cuda_ok(cudaMalloc((void**)&pool->slab, slab_bytes), "cudaMalloc(kv slab)")) return fail(TS_ERR_CUDA);
    pool->own_slab = true;
  }
  pool->host_pages_cap = (int)(cfg->host_bytes / page_bytes);
  if (pool->host_pages_cap > 0) {
    if (cfg->host_arena != nullptr) {
      pool->host = (uint8_t*)cfg->host_arena;
    } else {
      if (!cuda_ok(cudaHostAlloc((void**)&pool->host, (size_t)pool->host_pages_cap * page_bytes, cudaHostAllocDefault),
                   "cudaHostAlloc(host arena)"))
        return fail(TS_ERR_CUDA);
      pool->own_host = true;
    }
  }
  for (int i = 0; i < pool->host_pages_cap; ++i) pool->host_free.push_back(i);
  if (cfg->side_stream != nullptr) {
    pool->side = (cudaStream_t)cfg->side_stream;
  } else {
    if (!cuda_ok(cudaStreamCreateWithFlags(&pool->side, cudaStreamNonBlocking), "cudaStreamCreate(side)")) return fail(TS_ERR_CUDA);
    pool->own_side = true;
  }
  if (!cuda_ok(cudaStreamCreateWithFlags(&pool->side_out, cudaStreamNonBlocking), "cudaStreamCreate(side_out)")) return fail(TS_ERR_CUDA);
  pool->host_slot_seq.assign(std::max(0, pool->host_pages_cap), 0);
  for (int i = 0; i < cfg->n_pages; ++i) pool->free_q.push_back(cfg->free_order ? cfg->free_order[i] : i);
  pool->page_compute_seq.assign(cfg->n_pages, 0);
  pool->page_side_seq.assign(cfg->n_pages, 0);
  pool->sess.resize(cfg->max_sessions);

  // per-layer TMA maps of the cached K and V: dims {D, B, H, n_pages}
  pool->map_k.resize(cfg->n_layers);
  pool->map_v.resize(cfg->n_layers);
  const cuuint64_t dims[4] = {(cuuint64_t)cfg->head_dim, (cuuint64_t)cfg->page_tokens, (cuuint64_t)cfg->n_heads,
                              (cuuint64_t)cfg->n_pages};
  const cuuint64_t strides[3] = {(cuuint64_t)cfg->head_dim * 2, (cuuint64_t)cfg->page_tokens * cfg->head_dim * 2,
                                 (cuuint64_t)page_bytes};
  const cuuint32_t box[4] = {64, (cuuint32_t)std::min(cfg->page_tokens, 64), 1, 1};   // half a 128-key tile at most
  for (int l = 0; l < cfg->n_layers; ++l) {
    uint8_t* base = pool->slab + (int64_t)l * pool->layer_bytes;
    if (!encode_map(&pool->map_k[l], base, 4, dims, strides, box)) return fail(TS_ERR_CUDA);
    if (!encode_map(&pool->map_v[l], base + pool->kv_bytes, 4, dims, strides, box)) return fail(TS_ERR_CUDA);
  }
  // load the attention kernel's module now (cudaFuncSetAttribute does): with lazy module loading the FIRST launch would do it,
  // and loading allocates device memory, which waits for every copy in flight - a resume on the side stream, for one
  if (!cuda_ok(attention_configure(cfg->head_dim), "cudaFuncSetAttribute(attention)")) return fail(TS_ERR_CUDA);
  *out = pool;
  return TS_OK;
}

int ts_session_open(ts_pool* pool, int32_t* sid_out) {
  if (pool == nullptr || sid_out == nullptr) return TS_ERR_INVALID;
  for (int i = 0; i < pool->cfg.max_sessions; ++i) {
    if (pool->sess[i].state == TS_SESSION_CLOSED) {
      Session& s = pool->sess[i];
      s = Session();
      s.state = TS_SESSION_RESIDENT;
      s.ver = ++pool->ver_seq;
      *sid_out = i;
      return TS_OK;
    }
  }
  return TS_ERR_CAPACITY;
}

int ts_session_close(ts_pool* pool, int32_t sid) {
  if (pool == nullptr) return TS_ERR_INVALID;
  if (sid < 0 || sid >= pool->cfg.max_sessions || pool->sess[sid].state == TS_SESSION_CLOSED) return TS_ERR_STATE;
  Session& s = pool->sess[sid];
  if (s.in_plan) return TS_ERR_STATE;   // a prepared step plan holds it until ts_step_plan_commit
  if (s.state == TS_SESSION_RESIDENT) {
    for (int32_t p : s.pt) {
      pool->page_compute_seq[p] = s.compute_seq;   // in-flight readers/writers of the page
      pool->page_side_seq[p] = s.side_seq;
      pool->free_q.push_back(p);
    }
  } else {
    for (int32_t slot : s.host_slots) {
      pool->host_slot_seq[slot] = s.side_seq;   // the copy out that fills the slot may still be running
      pool->host_free.push_back(slot);
    }
  }
  s = Session();
  return TS_OK;
}

int ts_session_info(ts_pool* pool, int32_t sid, ts_session_info_t* out) {
  if (pool == nullptr || out == nullptr) return TS_ERR_INVALID;
  if (sid < 0 || sid >= pool->cfg.max_sessions || pool->sess[sid].state == TS_SESSION_CLOSED) return TS_ERR_STATE;
  const Session& s = pool->sess[sid];
  out->state = s.state;
  out->frames = s.P;
  out->len_tokens = (int64_t)s.P * pool->cfg.frame_tokens;
  out->head_off = s.o;
  out->n_pages = s.state == TS_SESSION_RESIDENT ? (int32_t)s.pt.size() : (int32_t)s.host_slots.size();
  return TS_OK;
}

int ts_session_page_table(ts_pool* pool, int32_t sid, int32_t* out, int32_t cap, int32_t* n_out) {
  if (pool == nullptr || n_out == nullptr || cap < 0 || (cap > 0 && out == nullptr)) return TS_ERR_INVALID;
  if (sid < 0 || sid >= pool->cfg.max_sessions || pool->sess[sid].state == TS_SESSION_CLOSED) return TS_ERR_STATE;
  const Session& s = pool->sess[sid];
  *n_out = (int32_t)s.pt.size();
  for (int i = 0; i < std::min<int>(cap, (int)s.pt.size()); ++i) out[i] = s.pt[i];
  return TS_OK;
}

int ts_pool_free_list(ts_pool* pool, int32_t* out, int32_t cap, int32_t* n_out) {
  if (pool == nullptr || n_out == nullptr || cap < 0 || (cap > 0 && out == nullptr)) return TS_ERR_INVALID;
  *n_out = (int32_t)pool->free_q.size();
  for (int i = 0; i < std::min<int>(cap, (int)pool->free_q.size()); ++i) out[i] = pool->free_q[i];
  return TS_OK;
}

int ts_pool_stats(ts_pool* pool, ts_pool_stats_t* out) {
  if (pool == nullptr || out == nullptr) return TS_ERR_INVALID;
  int res = 0, sus = 0;
  for (const Session& s : pool->sess) {
    res += s.state == TS_SESSION_RESIDENT;
    sus += s.state == TS_SESSION_SUSPENDED;
  }
  out->free_pages = (int32_t)pool->free_q.size();
  out->resident = res;
  out->suspended = sus;
  out->host_pages_cap = pool->host_pages_cap;
  out->host_pages_used = pool->host_pages_cap - (int32_t)pool->host_free.size();
  out->reserved = 0;
  out->page_bytes = pool->page_bytes;
  return TS_OK;
}

void* ts_pool_side_stream(ts_pool* pool) { return pool ? (void*)pool->side : nullptr; }
void* ts_pool_suspend_stream(ts_pool* pool) { return pool ? (void*)pool->side_out : nullptr; }
int64_t ts_pool_sched_builds(ts_pool* pool) { return pool ? pool->sched_builds : 0; }
int64_t ts_pool_split_batches(ts_pool* pool) { return pool ? pool->split_batches : 0; }
int ts_pool_clock_probe(ts_pool* pool, void* device_u64x2) {
  if (pool == nullptr || ((uintptr_t)device_u64x2 & 7) != 0) return TS_ERR_INVALID;
  pool->clock_probe = (unsigned long long*)device_u64x2;
  return TS_OK;
}
int64_t ts_pool_launch_count(ts_pool* pool) { return pool ? pool->launches : 0; }

// --------------------------------------------------------------------------------------------- a1: schedule
// ---- a1: collect + coalesce.  The schedule (session descriptors, packed page tables, cluster work items) depends only
// on the batch and on its sessions' page-table state, so it is built once and reused by every later call with the same
// key - all layers and denoising passes of a chunk step.  Result in pool->sched_*.
// `q_offs` (optional): first token of every session in the packed call tensors, when the sessions are a SUBSET of the caller's
// batch (a batch split by resume readiness, run_batch()); otherwise the sessions are packed back to back.
static void build_schedule(ts_pool* pool, int32_t n, const int32_t* sids, const int32_t* chunk_frames,
                           const int32_t* q_offs = nullptr) {
  const ts_pool_config& c = pool->cfg;
  const int T = c.frame_tokens, H = c.n_heads, W = c.window_frames;
  std::vector<int64_t>& key = pool->scratch_key;
  key.clear();
  key.push_back(n);
  for (int b = 0; b < n; ++b) {
    key.push_back(sids[b]);
    key.push_back(chunk_frames[b]);
    key.push_back((int64_t)pool->sess[sids[b]].ver);
    key.push_back(q_offs ? q_offs[b] : -1);
  }
  if (key == pool->sched_key) return;
  const int grid_max = std::max(2, pool->sm_count & ~1);
  ++pool->sched_builds;
  std::vector<SessDesc>& sd = pool->sched_sess;
  std::vector<int32_t>& pt = pool->sched_pt;
  std::vector<int32_t>& cta_begin = pool->sched_cta;
  std::vector<WorkItem>& items = pool->sched_items;
  sd.assign(n, SessDesc());
  pt.clear();
  int q_off = 0;
  for (int b = 0; b < n; ++b) {
    const Session& s = pool->sess[sids[b]];
    const int cfr = chunk_frames[b];
    const int C = cfr * T;
    const int a = W > 0 ? std::max(0, s.P + cfr - W) : 0;     // window start in frames (R6 i)
    SessDesc& d = sd[b];
    d.q_off = q_offs ? q_offs[b] : q_off;
    d.C = C;
    d.x_begin = s.o + a * T;
    d.x_end = s.o + s.P * T;
    d.pt_off = (int32_t)pt.size();
    d.n_pt = (int32_t)s.pt.size();
    d.pad0 = d.pad1 = 0;
    pt.insert(pt.end(), s.pt.begin(), s.pt.end());
    q_off += C;
  }
  // Work items come in two granularities: pairs of 128-row query tiles (one K/V tile feeds 256 rows), or single
  // tiles whose KV tiles alternate between the two TMEM tile slots (half as long, same MMA work per step, twice the
  // K/V traffic per FLOP).  Pairs are the default; single tiles are taken when the batch is so small that pairs
  // leave clusters idle in the last wave (1-2 sessions), judged by the modelled makespan of both schedules.
  struct Cand {
    int cost, sess, head, q_tile, n_kv;
    bool single;
  };
  struct CItem {
    int cost;
    int64_t stream_cost;
    int stream;
    Cand a, b;       // b.q_tile < 0: no second item
    bool mc;
  };
  struct Plan {
    std::vector<CItem> citems;
    std::vector<std::vector<int>> per_cluster;
    int64_t makespan = 0;
  };
  auto make_plan = [&](int tiles_per_item) {
    Plan plan;
    std::vector<Cand> cands;
    for (int b = 0; b < n; ++b) {
      const SessDesc& d = sd[b];
      const int n_tiles = (d.C + 127) / 128;
      for (int t0 = 0; t0 < n_tiles; t0 += tiles_per_item) {
        int n_q, n_kv;
        item_geometry(c, d.C, d.x_begin, d.x_end, t0, tiles_per_item, &n_q, &n_kv);
        // time model in twentieths of a two-tile KV step, fitted to per-CTA cycle counts on configs[2]
        // (3184 clk per step + 14.7 k clk per item): 4.5 steps per item for the Q load, pipeline fill and epilogue.
        // A lone query tile alternates its KV tiles between the two TMEM tile slots (half the steps, plus the merge).
        const int cost = n_q == 2 ? 20 * n_kv + 90 : (n_kv >= 2 ? 10 * n_kv + 110 : 19 * n_kv + 90);
        for (int h = 0; h < H; ++h) cands.push_back({cost, b, h, t0, n_kv, tiles_per_item == 1});
      }
    }
    // ---- cluster items.  The items of one (session, head) stream read the same K/V pages: two of them at a time
    // go to the two CTAs of a cluster, which then load half of every K/V tile each and multicast it to both (mc).
    // A stream's odd item out is paired with another stream's (or with nothing): those two share a cluster without
    // sharing loads.  Both CTAs cycle max(n_kv) tiles through their smem rings to stay on the same ring position.
    std::vector<int64_t> stream_cost((size_t)n * H, 0);
    for (const Cand& x : cands) stream_cost[(size_t)x.sess * H + x.head] += x.cost;
    // within a stream: by KV length (longest first), two-tile items before a lone tile
    std::stable_sort(cands.begin(), cands.end(), [&](const Cand& x, const Cand& y) {
      const size_t sx = (size_t)x.sess * H + x.head, sy = (size_t)y.sess * H + y.head;
      if (sx != sy) return sx < sy;
      if (x.n_kv != y.n_kv) return x.n_kv > y.n_kv;
      return x.cost > y.cost;
    });
    std::vector<CItem>& citems = plan.citems;
    std::vector<Cand> odd;
    for (size_t i = 0; i < cands.size();) {
      size_t e = i;
      while (e < cands.size() && cands[e].sess == cands[i].sess && cands[e].head == cands[i].head) ++e;
      const int stream = cands[i].sess * H + cands[i].head;
      // pair items of EQUAL KV length first (neither CTA then waits for tiles only its partner needs); what is left
      // over (at most one item per length) is paired in length order, and the stream's last odd item goes to `odd`
      std::vector<Cand> rest;
      while (i < e) {
        if (i + 1 < e && cands[i].n_kv == cands[i + 1].n_kv) {
          citems.push_back({std::max(cands[i].cost, cands[i + 1].cost), stream_cost[stream], stream, cands[i], cands[i + 1], true});
          i += 2;
        } else {
          rest.push_back(cands[i++]);
        }
      }
      size_t r = 0;
      for (; r + 1 < rest.size(); r += 2)
        citems.push_back({std::max(rest[r].cost, rest[r + 1].cost), stream_cost[stream], stream, rest[r], rest[r + 1], true});
      if (r < rest.size()) odd.push_back(rest[r]);
    }
    std::stable_sort(odd.begin(), odd.end(), [](const Cand& x, const Cand& y) { return x.cost > y.cost; });
    for (size_t i = 0; i < odd.size(); i += 2) {
      Cand none = odd[i];
      none.q_tile = -1;
      none.n_kv = 0;
      none.cost = 0;
      const Cand& second = (i + 1 < odd.size()) ? odd[i + 1] : none;
      const int stream = odd[i].sess * H + odd[i].head;
      citems.push_back({std::max(odd[i].cost, second.cost), stream_cost[stream], stream, odd[i], second, false});
    }
    // List scheduling in stream order, heaviest streams first (LPT at stream granularity, so that the tail of the
    // schedule is made of short items): a stream's items are dealt out back to back, each to the least-loaded
    // cluster, and run at the same time - the stream's K/V then comes from DRAM once and from L2 afterwards.
    std::stable_sort(citems.begin(), citems.end(), [](const CItem& x, const CItem& y) {
      if (x.stream_cost != y.stream_cost) return x.stream_cost > y.stream_cost;
      if (x.stream != y.stream) return x.stream < y.stream;
      return x.cost > y.cost;
    });
    const int n_clusters = std::min(grid_max / 2, (int)citems.size());
    plan.per_cluster.assign(n_clusters, std::vector<int>());
    typedef std::pair<int64_t, int> Load;   // (load, cluster)
    std::priority_queue<Load, std::vector<Load>, std::greater<Load>> heap;
    for (int i = 0; i < n_clusters; ++i) heap.push({0, i});
    for (int i = 0; i < (int)citems.size(); ++i) {
      Load top = heap.top();
      heap.pop();
      plan.per_cluster[top.second].push_back(i);
      heap.push({top.first + citems[i].cost, top.second});
      plan.makespan = std::max(plan.makespan, top.first + citems[i].cost);
    }
    return plan;
  };
  Plan plan = make_plan(2);
  if (n * H * 2 <= grid_max) {               // small batch: fewer than two streams per cluster
    Plan fine = make_plan(1);
    if (fine.makespan * 108 < plan.makespan * 100) plan = std::move(fine);   // single tiles cost ~8 % more per FLOP
  }
  // The kernel hands cluster items out dynamically in THIS order (a global cursor): clusters that run a little
  // faster simply take more; the list-scheduling above only serves to compare the two plans.
  items.clear();
  for (const CItem& it : plan.citems) {
    for (int r = 0; r < 2; ++r) {
      const Cand& x = r ? it.b : it.a;
      WorkItem wi;
      wi.sess = x.sess;
      wi.head = x.head;
      wi.q_tile = x.q_tile;
      wi.pipe = (uint32_t)std::max(it.a.n_kv, it.b.n_kv) | (it.mc ? 0x80000000u : 0u) | (x.single ? 0x40000000u : 0u);
      items.push_back(wi);
    }
  }
  cta_begin.assign(1, 2 * (int)plan.per_cluster.size());   // [0] = grid
  pool->sched_key = key;
}

// One schedule block: everything a launch reads besides the caller's tensors and the slab, in one piece of (pinned host
// and, with the same layout, device) memory.  `n_slots` sets of per-session Q/Kn/Vn tensor maps come first.
struct BlockLayout {
  size_t off_maps, off_sess, off_pt, off_feed, off_items, off_copy, bytes, feed_bytes;
};

static BlockLayout block_layout(int n, int n_slots, size_t n_pt, size_t n_items, int grid, bool with_copy) {
  BlockLayout L;
  L.feed_bytes = 128 + (size_t)(grid / 2) * kFeedRing * 8;   // header (cursor, end count, n_citems) + per-cluster rings
  L.off_maps = 0;
  L.off_sess = align_up(L.off_maps + (size_t)n_slots * n * 3 * sizeof(CUtensorMap), 128);
  L.off_pt = align_up(L.off_sess + (size_t)n * sizeof(SessDesc), 128);
  L.off_feed = align_up(L.off_pt + n_pt * 4, 128);
  L.off_items = align_up(L.off_feed + L.feed_bytes, 128);
  L.off_copy = align_up(L.off_items + n_items * sizeof(WorkItem), 128);
  L.bytes = L.off_copy + (with_copy ? (size_t)n * sizeof(CopySess) : 0);
  return L;
}

// Everything of the block except the tensor maps, from the pool's current schedule.
static void fill_block(ts_pool* pool, uint8_t* h, const BlockLayout& L, int n, const CopySess* cs) {
  memcpy(h + L.off_sess, pool->sched_sess.data(), (size_t)n * sizeof(SessDesc));
  memcpy(h + L.off_pt, pool->sched_pt.data(), pool->sched_pt.size() * 4);
  memset(h + L.off_feed, 0, L.feed_bytes);
  reinterpret_cast<int32_t*>(h + L.off_feed)[2] = (int32_t)(pool->sched_items.size() / 2);
  memcpy(h + L.off_items, pool->sched_items.data(), pool->sched_items.size() * sizeof(WorkItem));
  if (cs != nullptr) {
    CopySess* dst = reinterpret_cast<CopySess*>(h + L.off_copy);
    for (int b = 0; b < n; ++b) {
      dst[b] = cs[b];
      dst[b].pt_off = pool->sched_sess[b].pt_off;   // the append shares the attention's packed page tables
    }
  }
}

// Per-session 3D maps {D, H, C} of the call's packed Q / Kn / Vn: rows past a session's chunk read as zeros, never as a
// neighbour's tokens.  `chunk_frames` fixes the geometry (q_off, C); nothing else of the schedule is needed.
static bool encode_session_maps(ts_pool* pool, CUtensorMap* maps, int n, const int32_t* chunk_frames, const void* q,
                                const void* k, const void* v, const int32_t* q_offs = nullptr) {
  const ts_pool_config& c = pool->cfg;
  const int H = c.n_heads, D = c.head_dim;
  size_t q_off = 0;
  for (int b = 0; b < n; ++b) {
    const size_t C = (size_t)chunk_frames[b] * c.frame_tokens;
    const cuuint64_t dims[3] = {(cuuint64_t)D, (cuuint64_t)H, (cuuint64_t)C};
    const cuuint64_t strides[2] = {(cuuint64_t)D * 2, (cuuint64_t)H * D * 2};
    const cuuint32_t box_q[3] = {64, 1, 128};
    const cuuint32_t box_kv[3] = {64, 1, (cuuint32_t)std::min(c.page_tokens, 64)};   // same box rows as the cache maps
    const size_t byte_off = (q_offs ? (size_t)q_offs[b] : q_off) * H * D * 2;
    if (!encode_map(&maps[b * 3 + 0], (uint8_t*)q + byte_off, 3, dims, strides, box_q)) return false;
    if (!encode_map(&maps[b * 3 + 1], (uint8_t*)k + byte_off, 3, dims, strides, box_kv)) return false;
    if (!encode_map(&maps[b * 3 + 2], (uint8_t*)v + byte_off, 3, dims, strides, box_kv)) return false;
    q_off += C;
  }
  return true;
}

// Kernel parameters of one launch on the block at device address `d` (tensor maps of set `slot`).
static AttnParams make_params(ts_pool* pool, const BlockLayout& L, uint8_t* d, int n, int slot, int32_t layer, const void* k,
                              const void* v, void* out, float* lse, float scale, bool with_copy, int total_rows) {
  const ts_pool_config& c = pool->cfg;
  AttnParams p;
  memset(&p.copy, 0, sizeof(p.copy));
  if (with_copy) {
    p.copy.sess = reinterpret_cast<const CopySess*>(d + L.off_copy);
    p.copy.page_tables = reinterpret_cast<const int32_t*>(d + L.off_pt);
    p.copy.n_sess = n;
    p.copy.total_rows = total_rows;
    p.copy.H = c.n_heads;
    p.copy.D = c.head_dim;
    p.copy.B = c.page_tokens;
    p.copy.log2_B = pool->log2_B;
    p.copy.page_stride = pool->page_bytes;
    p.copy.layer_k_off = (int64_t)layer * pool->layer_bytes;
    p.copy.layer_v_off = p.copy.layer_k_off + pool->kv_bytes;
    p.copy.slab = pool->slab;
    p.copy.src_k = (const uint8_t*)k;
    p.copy.src_v = (const uint8_t*)v;
  }
  p.map_k = pool->map_k[layer];
  p.map_v = pool->map_v[layer];
  p.sess_maps = reinterpret_cast<const CUtensorMap*>(d + L.off_maps) + (size_t)slot * n * 3;
  p.sess = reinterpret_cast<const SessDesc*>(d + L.off_sess);
  p.page_tables = reinterpret_cast<const int32_t*>(d + L.off_pt);
  p.clock_probe = pool->clock_probe;
  p.feed_hdr = reinterpret_cast<int32_t*>(d + L.off_feed);
  p.feed = reinterpret_cast<unsigned long long*>(d + L.off_feed + 128);
  p.items = reinterpret_cast<const WorkItem*>(d + L.off_items);
  p.out = (uint16_t*)out;
  p.lse = lse;
  p.H = c.n_heads;
  p.T = c.frame_tokens;
  p.B = c.page_tokens;
  p.log2_B = pool->log2_B;
  p.scale = scale;
  p.scale_log2 = scale * 1.4426950408889634f;
  return p;
}

// Page demand of appending the batch's chunks (O2: max(0, ceil((o + L + C) / B) - |PT|) per session, R14).
// Returns the total, the per-session demand in pool->scratch_need.
static int64_t page_demand(ts_pool* pool, int32_t n, const int32_t* sids, const int32_t* chunk_frames) {
  const int T = pool->cfg.frame_tokens, B = pool->cfg.page_tokens;
  pool->scratch_need.assign(n, 0);
  int64_t total = 0;
  for (int b = 0; b < n; ++b) {
    const Session& s = pool->sess[sids[b]];
    const int64_t end = (int64_t)s.o + (int64_t)s.P * T + (int64_t)chunk_frames[b] * T;
    pool->scratch_need[b] = (int)std::max<int64_t>(0, (end + B - 1) / B - (int64_t)s.pt.size());
    total += pool->scratch_need[b];
  }
  return total;
}

// Grows the page tables of the batch by pool->scratch_need (popping from the front of the free list, sessions in `sids`
// order) and describes the append of the chunks that follows.  The caller has checked the demand against the free list.
static void grow_for_append(ts_pool* pool, int32_t n, const int32_t* sids, const int32_t* chunk_frames, FusedAppend* fa) {
  const int T = pool->cfg.frame_tokens, B = pool->cfg.page_tokens;
  fa->cs.resize(n);
  int tok_off = 0, row_off = 0;
  for (int b = 0; b < n; ++b) {
    Session& s = pool->sess[sids[b]];
    const int need = pool->scratch_need[b];
    if (need > 0) s.ver = ++pool->ver_seq;
    for (int i = 0; i < need; ++i) {
      const int32_t pg = pool->free_q.front();
      pool->free_q.pop_front();
      fa->wait_side = std::max(fa->wait_side, pool->page_side_seq[pg]);        // a D2H copy out of the page may be pending
      fa->wait_compute = std::max(fa->wait_compute, pool->page_compute_seq[pg]);
      s.pt.push_back(pg);
      fa->popped.push_back(pg);
    }
    fa->wait_side = std::max(fa->wait_side, s.side_seq);
    const int C = chunk_frames[b] * T;
    const int x0 = s.o + s.P * T;
    CopySess& d = fa->cs[b];
    d.tok_off = tok_off;
    d.n_tok = C;
    d.n_zero = (B - ((x0 + C) & (B - 1))) & (B - 1);
    d.x0 = x0;
    d.pt_off = 0;
    d.row_off = row_off;
    d.pad0 = d.pad1 = 0;
    tok_off += C;
    row_off += d.n_tok + d.n_zero;
  }
  fa->total_rows = row_off;
}

// Undoes grow_for_append after a failure further down (all-or-nothing): the popped ids go back to the FRONT of the free
// list in their original order and leave the tables they were appended to.
static void ungrow(ts_pool* pool, int32_t n, const int32_t* sids, const FusedAppend& fa) {
  for (int b = n - 1; b >= 0; --b) {
    Session& s = pool->sess[sids[b]];
    for (int i = 0; i < pool->scratch_need[b]; ++i) s.pt.pop_back();
    if (pool->scratch_need[b] > 0) s.ver = ++pool->ver_seq;
  }
  for (auto it = fa.popped.rbegin(); it != fa.popped.rend(); ++it) pool->free_q.push_front(*it);
}

// --------------------------------------------------------------------------------------------- attention
// One launch for `n` sessions.  `cs` (optional): the append descriptors of a fused step, one per session; `q_offs` (optional):
// see build_schedule.
static int attention_impl(ts_pool* pool, int32_t layer, int32_t n, const int32_t* sids, const int32_t* chunk_frames,
                          const int32_t* q_offs, const void* q, const void* k, const void* v, void* out, float* lse,
                          float scale, void* cuda_stream, const CopySess* cs, uint64_t wait_side, uint64_t wait_compute,
                          uint64_t* seq_out) {
  if (pool == nullptr) return TS_ERR_INVALID;
  int rc = check_batch(pool, layer, n, sids, chunk_frames);
  if (rc != TS_OK) return rc;
  if (n == 0) return TS_OK;
  if (q == nullptr || k == nullptr || v == nullptr || out == nullptr) return TS_ERR_INVALID;
  if ((((uintptr_t)q | (uintptr_t)k | (uintptr_t)v) & 15) != 0 || ((uintptr_t)out & 31) != 0) return TS_ERR_INVALID;
  if (!(scale > 0.0f) || !std::isfinite(scale)) return TS_ERR_INVALID;
  const ts_pool_config& c = pool->cfg;
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  TS_CUDA(cudaSetDevice(c.device));

  build_schedule(pool, n, sids, chunk_frames, q_offs);
  const int grid = pool->sched_cta[0];
  const BlockLayout L = block_layout(n, 1, pool->sched_pt.size(), pool->sched_items.size(), grid, cs != nullptr);
  Staging* st = nullptr;
  rc = acquire_staging(pool, L.bytes, &st);
  if (rc != TS_OK) return rc;
  fill_block(pool, st->h, L, n, cs);
  if (!encode_session_maps(pool, reinterpret_cast<CUtensorMap*>(st->h + L.off_maps), n, chunk_frames, q, k, v, q_offs))
    return TS_ERR_CUDA;

  // ---- ordering: wait (stream-side) for pending resumes of the batch's sessions
  for (int b = 0; b < n; ++b) TS_CUDA(pool->tl_side.wait(stream, pool->sess[sids[b]].side_seq));
  if (cs != nullptr) {   // ... and for copies out of / readers of the pages the append is about to write
    TS_CUDA(pool->tl_side.wait(stream, wait_side));
    TS_CUDA(pool->tl_compute.wait(stream, wait_compute));
  }

  rc = upload_staging(pool, st, L.bytes, stream);
  if (rc != TS_OK) return rc;
  int total_rows = 0;
  if (cs != nullptr)
    for (int b = 0; b < n; ++b) total_rows += cs[b].n_tok + cs[b].n_zero;
  const AttnParams p = make_params(pool, L, st->d, n, 0, layer, k, v, out, lse, scale, cs != nullptr, total_rows);
  TS_CUDA(launch_attention(p, c.head_dim, grid, stream));
  ++pool->launches;
  TS_CUDA(cudaEventRecord(st->ev, stream));
  st->in_flight = true;
  const uint64_t seq = pool->tl_compute.record(stream);
  for (int b = 0; b < n; ++b) pool->sess[sids[b]].compute_seq = seq;
  if (seq_out) *seq_out = seq;
  return TS_OK;
}

static void append_commit(ts_pool* pool, int32_t n, const int32_t* sids, const int32_t* chunk_frames, uint32_t flags,
                          uint64_t seq);

// PAPER.md:76 (iii) "restored ... before chunk generation resumes", without making the rest of the batch wait: when some
// sessions of the batch still have a resume in flight on the side stream (and others do not), the batch runs as TWO launches -
// the sessions that are ready first, the resuming ones behind their copy events - so that the ready sessions' attention hides
// the copies instead of following them.  Results are those of one launch (sessions are independent); the packed
// tensors are addressed through per-session offsets, so a group need not be contiguous in them.  `fa`: the fused append of
// the whole batch (grown tables, descriptors in batch order) or null; with it, each group commits (`flags`) behind its own
// launch.
static int run_batch(ts_pool* pool, int32_t layer, int32_t n, const int32_t* sids, const int32_t* chunk_frames, const void* q,
                     const void* k, const void* v, void* out, float* lse, float scale, void* cuda_stream, const FusedAppend* fa,
                     uint32_t flags, int* groups_done) {
  *groups_done = 0;
  std::vector<int32_t>& pend = pool->scratch_pending;   // decided ONCE: a resume may complete while the groups are being built
  pend.assign(n, 0);
  int n_pending = 0;
  for (int b = 0; b < n; ++b) {
    pend[b] = !pool->tl_side.is_done(pool->sess[sids[b]].side_seq);
    n_pending += pend[b];
  }
  if (n_pending == 0 || n_pending == n) {
    uint64_t seq = 0;
    const int rc = attention_impl(pool, layer, n, sids, chunk_frames, nullptr, q, k, v, out, lse, scale, cuda_stream,
                                  fa ? fa->cs.data() : nullptr, fa ? fa->wait_side : 0, fa ? fa->wait_compute : 0, &seq);
    if (rc != TS_OK) return rc;
    if (fa) append_commit(pool, n, sids, chunk_frames, flags, seq);
    *groups_done = 1;
    return TS_OK;
  }
  ++pool->split_batches;
  std::vector<int32_t>& ss = pool->scratch_sub_sids;
  std::vector<int32_t>& sc = pool->scratch_sub_cf;
  std::vector<int32_t>& so = pool->scratch_sub_off;
  std::vector<CopySess>& scs = pool->scratch_sub_cs;
  for (int pass = 0; pass < 2; ++pass) {           // pass 0: the sessions that are ready; pass 1: the resuming ones
    ss.clear();
    sc.clear();
    so.clear();
    scs.clear();
    int q_off = 0;
    for (int b = 0; b < n; ++b) {
      if (pend[b] == pass) {
        ss.push_back(sids[b]);
        sc.push_back(chunk_frames[b]);
        so.push_back(q_off);
        if (fa) scs.push_back(fa->cs[b]);
      }
      q_off += chunk_frames[b] * pool->cfg.frame_tokens;
    }
    uint64_t seq = 0;
    const int rc = attention_impl(pool, layer, (int)ss.size(), ss.data(), sc.data(), so.data(), q, k, v, out, lse, scale,
                                  cuda_stream, fa ? scs.data() : nullptr, fa ? fa->wait_side : 0, fa ? fa->wait_compute : 0, &seq);
    if (rc != TS_OK) return rc;
    if (fa) append_commit(pool, (int)ss.size(), ss.data(), sc.data(), flags, seq);
    ++*groups_done;
  }
  return TS_OK;
}

int ts_chunk_attention(ts_pool* pool, int32_t layer, int32_t n, const int32_t* sids, const int32_t* chunk_frames,
                       const void* q, const void* k, const void* v, void* out, float* lse, float scale, void* cuda_stream) {
  if (pool == nullptr) return TS_ERR_INVALID;
  int rc = check_batch(pool, layer, n, sids, chunk_frames);
  if (rc != TS_OK) return rc;
  if (n == 0) return TS_OK;
  if (q == nullptr || k == nullptr || v == nullptr || out == nullptr) return TS_ERR_INVALID;
  if ((((uintptr_t)q | (uintptr_t)k | (uintptr_t)v) & 15) != 0 || ((uintptr_t)out & 31) != 0) return TS_ERR_INVALID;
  if (!(scale > 0.0f) || !std::isfinite(scale)) return TS_ERR_INVALID;
  int groups = 0;
  return run_batch(pool, layer, n, sids, chunk_frames, q, k, v, out, lse, scale, cuda_stream, nullptr, 0, &groups);
}

// --------------------------------------------------------------------------------------------- append
// Host bookkeeping after an append has been enqueued (its completion is `seq` on the compute timeline): with
// TS_COMMIT the sessions grow by their chunk and the window rolls (a4).
static void append_commit(ts_pool* pool, int32_t n, const int32_t* sids, const int32_t* chunk_frames, uint32_t flags,
                          uint64_t seq) {
  const int T = pool->cfg.frame_tokens, B = pool->cfg.page_tokens, W = pool->cfg.window_frames;
  for (int b = 0; b < n; ++b) {
    Session& s = pool->sess[sids[b]];
    s.compute_seq = seq;
    if (flags & TS_COMMIT) {
      s.ver = ++pool->ver_seq;
      s.P += chunk_frames[b];
      const int e = W > 0 ? std::max(0, s.P - W) : 0;   // a4: evict oldest whole frames (R6 ii, R10)
      s.P -= e;
      s.o += e * T;
      while (s.o >= B) {
        const int32_t pg = s.pt.front();
        s.pt.erase(s.pt.begin());
        pool->page_compute_seq[pg] = seq;
        pool->page_side_seq[pg] = s.side_seq;
        pool->free_q.push_back(pg);
        s.o -= B;
      }
    }
  }
}

int ts_kv_append(ts_pool* pool, int32_t layer, int32_t n, const int32_t* sids, const int32_t* chunk_frames, const void* k,
                 const void* v, uint32_t flags, void* cuda_stream) {
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  if (pool == nullptr) return TS_ERR_INVALID;
  int rc = check_batch(pool, layer, n, sids, chunk_frames);
  if (rc != TS_OK) return rc;
  if (n == 0) return TS_OK;
  if (k == nullptr || v == nullptr || (((uintptr_t)k | (uintptr_t)v) & 15) != 0) return TS_ERR_INVALID;
  if ((flags & ~(uint32_t)TS_COMMIT) != 0) return TS_ERR_INVALID;
  const ts_pool_config& c = pool->cfg;
  TS_CUDA(cudaSetDevice(c.device));
  const int T = c.frame_tokens, B = c.page_tokens;

  // demand check first: all-or-nothing (O2)
  const int64_t need_total = page_demand(pool, n, sids, chunk_frames);
  const std::vector<int32_t>& need = pool->scratch_need;
  size_t n_pt_total = 0;
  for (int b = 0; b < n; ++b) n_pt_total += pool->sess[sids[b]].pt.size() + need[b];
  if (need_total > (int64_t)pool->free_q.size()) return TS_ERR_NO_PAGES;

  const size_t off_sess = 0;
  const size_t off_pt = align_up((size_t)n * sizeof(CopySess), 128);
  const size_t bytes = off_pt + n_pt_total * 4;
  Staging* st = nullptr;
  rc = acquire_staging(pool, bytes, &st);
  if (rc != TS_OK) return rc;
  CopySess* cs = reinterpret_cast<CopySess*>(st->h + off_sess);
  int32_t* pt = reinterpret_cast<int32_t*>(st->h + off_pt);

  uint64_t wait_side = 0, wait_compute = 0;
  int tok_off = 0, pt_off = 0, row_off = 0;
  for (int b = 0; b < n; ++b) {
    Session& s = pool->sess[sids[b]];
    if (need[b] > 0) s.ver = ++pool->ver_seq;
    for (int i = 0; i < need[b]; ++i) {
      const int32_t pg = pool->free_q.front();
      pool->free_q.pop_front();
      wait_side = std::max(wait_side, pool->page_side_seq[pg]);        // a D2H copy out of the page may be pending
      wait_compute = std::max(wait_compute, pool->page_compute_seq[pg]);
      s.pt.push_back(pg);
    }
    wait_side = std::max(wait_side, s.side_seq);
    const int C = chunk_frames[b] * T;
    const int x0 = s.o + s.P * T;
    CopySess& d = cs[b];
    d.tok_off = tok_off;
    d.n_tok = C;
    d.n_zero = (B - ((x0 + C) & (B - 1))) & (B - 1);
    d.x0 = x0;
    d.pt_off = pt_off;
    d.row_off = row_off;
    d.pad0 = d.pad1 = 0;
    std::copy(s.pt.begin(), s.pt.end(), pt + pt_off);
    tok_off += C;
    pt_off += (int)s.pt.size();
    row_off += d.n_tok + d.n_zero;
  }
  TS_CUDA(pool->tl_side.wait(stream, wait_side));
  TS_CUDA(pool->tl_compute.wait(stream, wait_compute));
  rc = upload_staging(pool, st, bytes, stream);
  if (rc != TS_OK) return rc;
  CopyParams p;
  memset(&p, 0, sizeof(p));
  p.sess = reinterpret_cast<const CopySess*>(st->d + off_sess);
  p.page_tables = reinterpret_cast<const int32_t*>(st->d + off_pt);
  p.n_sess = n;
  p.total_rows = row_off;
  p.H = c.n_heads;
  p.D = c.head_dim;
  p.B = B;
  p.log2_B = pool->log2_B;
  p.page_stride = pool->page_bytes;
  p.layer_k_off = (int64_t)layer * pool->layer_bytes;
  p.layer_v_off = p.layer_k_off + pool->kv_bytes;
  p.slab = pool->slab;
  p.src_k = (const uint8_t*)k;
  p.src_v = (const uint8_t*)v;
  TS_CUDA(launch_append(p, pool->sm_count, stream));
  ++pool->launches;
  TS_CUDA(cudaEventRecord(st->ev, stream));
  st->in_flight = true;
  const uint64_t seq = pool->tl_compute.record(stream);

  append_commit(pool, n, sids, chunk_frames, flags, seq);
  return TS_OK;
}

// --------------------------------------------------------------------------------------------- fused device step
int ts_chunk_step(ts_pool* pool, int32_t layer, int32_t n, const int32_t* sids, const int32_t* chunk_frames, const void* q,
                  const void* k, const void* v, void* out, float* lse, float scale, uint32_t flags, void* cuda_stream) {
  if (pool == nullptr) return TS_ERR_INVALID;
  int rc = check_batch(pool, layer, n, sids, chunk_frames);
  if (rc != TS_OK) return rc;
  if (n == 0) return TS_OK;
  if (q == nullptr || k == nullptr || v == nullptr || out == nullptr) return TS_ERR_INVALID;
  if ((((uintptr_t)q | (uintptr_t)k | (uintptr_t)v) & 15) != 0 || ((uintptr_t)out & 31) != 0) return TS_ERR_INVALID;
  if (!(scale > 0.0f) || !std::isfinite(scale)) return TS_ERR_INVALID;
  if ((flags & ~(uint32_t)TS_COMMIT) != 0) return TS_ERR_INVALID;
  // page demand of the append, before anything changes or is enqueued (all-or-nothing, O2)
  if (page_demand(pool, n, sids, chunk_frames) > (int64_t)pool->free_q.size()) return TS_ERR_NO_PAGES;
  // grow the page tables first: the attention schedule is then built from the grown tables (the attention itself only
  // reads [x_begin, x_end), R5) and its packed page-table array also serves the append, which the idle warps of the
  // attention kernel carry out - it is HBM-bound, the attention is not, so it costs the step nothing there
  FusedAppend& fa = *pool->scratch_fused;   // (the vectors keep their capacity from call to call)
  fa.reset();
  grow_for_append(pool, n, sids, chunk_frames, &fa);
  int groups = 0;
  rc = run_batch(pool, layer, n, sids, chunk_frames, q, k, v, out, lse, scale, cuda_stream, &fa, flags, &groups);
  if (rc != TS_OK) {
    // a CUDA failure on the way.  Nothing enqueued yet: the tables and the free list are as before the call.  The first of
    // two groups already running (a batch split by resume readiness): it stays committed, the tables of the second stay
    // grown as after an uncommitted append.
    if (groups == 0) ungrow(pool, n, sids, fa);
    return rc;
  }
  return TS_OK;
}

// --------------------------------------------------------------------------------------------- step plan (capture-safe)
}  // extern "C"

struct ts_step_plan {
  ts_pool* pool = nullptr;
  int n = 0, n_slots = 0, grid = 0;
  std::vector<int32_t> sids, cf;
  struct Slot {
    const void *q = nullptr, *k = nullptr, *v = nullptr;
    void* out = nullptr;
    float* lse = nullptr;
    bool bound = false;
  };
  std::vector<Slot> slots;
  std::vector<CUtensorMap> maps;     // [n_slots][n][3], encoded at bind time
  BlockLayout L;                     // fixed at creation for the largest page tables / item lists the batch can have
  size_t max_pt = 0, max_items = 0;
  uint8_t* d = nullptr;              // device block: its address never changes, so captured launches stay valid
  uint8_t* h[2] = {nullptr, nullptr};
  uint8_t* h_dev[2] = {nullptr, nullptr};   // device-side addresses of the mapped pinned buffers
  cudaEvent_t h_ev[2] = {nullptr, nullptr};
  bool h_busy[2] = {false, false};
  int h_next = 0;
  bool prepared = false;
  int total_rows = 0;
  int64_t prepares = 0;
};

extern "C" {

int ts_step_plan_destroy(ts_step_plan* plan) {
  if (plan == nullptr) return TS_ERR_INVALID;
  ts_pool* pool = plan->pool;
  cudaSetDevice(pool->cfg.device);
  if (plan->prepared)
    for (int32_t sid : plan->sids) pool->sess[sid].in_plan = false;
  for (int i = 0; i < 2; ++i) {
    if (plan->h_ev[i]) {
      if (plan->h_busy[i]) cudaEventSynchronize(plan->h_ev[i]);
      cudaEventDestroy(plan->h_ev[i]);
    }
    if (plan->h[i]) cudaFreeHost(plan->h[i]);
  }
  if (plan->d) cudaFree(plan->d);   // (synchronises with launches still reading the block)
  cudaGetLastError();
  delete plan;
  return TS_OK;
}

int ts_step_plan_create(ts_pool* pool, int32_t n, const int32_t* sids, const int32_t* chunk_frames, int32_t n_slots,
                        ts_step_plan** out) {
  if (pool == nullptr || out == nullptr) return TS_ERR_INVALID;
  *out = nullptr;
  if (n < 1 || n_slots < 1 || n_slots > 4096) return TS_ERR_INVALID;
  int rc = check_batch(pool, 0, n, sids, chunk_frames);
  if (rc != TS_OK) return rc;
  const ts_pool_config& c = pool->cfg;
  TS_CUDA(cudaSetDevice(c.device));
  ts_step_plan* plan = new ts_step_plan();
  plan->pool = pool;
  plan->n = n;
  plan->n_slots = n_slots;
  plan->sids.assign(sids, sids + n);
  plan->cf.assign(chunk_frames, chunk_frames + n);
  plan->slots.resize(n_slots);
  plan->maps.resize((size_t)n_slots * n * 3);
  plan->grid = std::max(2, pool->sm_count & ~1);   // always the full grid: the launch configuration never changes
  // upper bounds that hold for every state the batch's sessions can be in: a table holds at most o + (W + c) T tokens
  // (all of the pool without a window), and a stream of t query tiles makes at most t cluster items (2 t work items)
  const int64_t T = c.frame_tokens, B = c.page_tokens;
  for (int b = 0; b < n; ++b) {
    int64_t pages = c.n_pages;
    if (c.window_frames > 0)
      pages = std::min<int64_t>(pages, (B - 1 + ((int64_t)c.window_frames + chunk_frames[b]) * T + B - 1) / B + 1);
    plan->max_pt += (size_t)pages;
    const int64_t tiles = ((int64_t)chunk_frames[b] * T + 127) / 128;
    plan->max_items += (size_t)(2 * tiles * c.n_heads);
  }
  plan->L = block_layout(n, n_slots, plan->max_pt, plan->max_items, plan->grid, true);
  auto fail = [&](int code) {
    ts_step_plan_destroy(plan);
    return code;
  };
  if (!cuda_ok(cudaMalloc((void**)&plan->d, align_up(plan->L.bytes, 16)), "cudaMalloc(step plan)")) return fail(TS_ERR_CUDA);
  if (!cuda_ok(cudaMemset(plan->d, 0, plan->L.bytes), "cudaMemset(step plan)")) return fail(TS_ERR_CUDA);
  for (int i = 0; i < 2; ++i) {
    if (!cuda_ok(cudaHostAlloc((void**)&plan->h[i], align_up(plan->L.bytes, 16), cudaHostAllocMapped), "cudaHostAlloc(step plan)"))
      return fail(TS_ERR_CUDA);
    if (!cuda_ok(cudaHostGetDevicePointer((void**)&plan->h_dev[i], plan->h[i], 0), "cudaHostGetDevicePointer")) return fail(TS_ERR_CUDA);
    if (!cuda_ok(cudaEventCreateWithFlags(&plan->h_ev[i], cudaEventDisableTiming), "cudaEventCreate")) return fail(TS_ERR_CUDA);
  }
  if (!cuda_ok(attention_configure(c.head_dim), "cudaFuncSetAttribute(attention)")) return fail(TS_ERR_CUDA);
  *out = plan;
  return TS_OK;
}

int ts_step_plan_bind(ts_step_plan* plan, int32_t slot, const void* q, const void* k, const void* v, void* out, float* lse) {
  if (plan == nullptr || slot < 0 || slot >= plan->n_slots) return TS_ERR_INVALID;
  if (q == nullptr || k == nullptr || v == nullptr || out == nullptr) return TS_ERR_INVALID;
  if ((((uintptr_t)q | (uintptr_t)k | (uintptr_t)v) & 15) != 0 || ((uintptr_t)out & 31) != 0) return TS_ERR_INVALID;
  if (plan->prepared) return TS_ERR_STATE;   // the maps travel with the prepare upload
  if (!encode_session_maps(plan->pool, plan->maps.data() + (size_t)slot * plan->n * 3, plan->n, plan->cf.data(), q, k, v))
    return TS_ERR_CUDA;
  ts_step_plan::Slot& s = plan->slots[slot];
  s.q = q;
  s.k = k;
  s.v = v;
  s.out = out;
  s.lse = lse;
  s.bound = true;
  return TS_OK;
}

int ts_step_plan_prepare(ts_step_plan* plan, void* cuda_stream) {
  if (plan == nullptr) return TS_ERR_INVALID;
  if (plan->prepared) return TS_ERR_STATE;
  ts_pool* pool = plan->pool;
  const int n = plan->n;
  const int32_t* sids = plan->sids.data();
  const int32_t* cf = plan->cf.data();
  int rc = check_batch(pool, 0, n, sids, cf);
  if (rc != TS_OK) return rc;
  if (page_demand(pool, n, sids, cf) > (int64_t)pool->free_q.size()) return TS_ERR_NO_PAGES;
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  TS_CUDA(cudaSetDevice(pool->cfg.device));
  const int slot = plan->h_next;
  if (plan->h_busy[slot]) {           // the upload two prepares ago: long done
    TS_CUDA(cudaEventSynchronize(plan->h_ev[slot]));
    plan->h_busy[slot] = false;
  }
  FusedAppend& fa = *pool->scratch_fused;
  fa.reset();
  grow_for_append(pool, n, sids, cf, &fa);
  build_schedule(pool, n, sids, cf);
  if (pool->sched_pt.size() > plan->max_pt || pool->sched_items.size() > plan->max_items) {   // cannot happen: bounds above
    ungrow(pool, n, sids, fa);
    return TS_ERR_INVALID;
  }
  uint8_t* h = plan->h[slot];
  fill_block(pool, h, plan->L, n, fa.cs.data());
  memcpy(h + plan->L.off_maps, plan->maps.data(), plan->maps.size() * sizeof(CUtensorMap));
  // ordering, all stream-side: pending resumes of the batch, copies out of / readers of the pages the append will write
  cudaError_t e = cudaSuccess;
  for (int b = 0; b < n && e == cudaSuccess; ++b) e = pool->tl_side.wait(stream, pool->sess[sids[b]].side_seq);
  if (e == cudaSuccess) e = pool->tl_side.wait(stream, fa.wait_side);
  if (e == cudaSuccess) e = pool->tl_compute.wait(stream, fa.wait_compute);
  // the block is rewritten in stream order: after the previous step's launches, before this step's
  if (e == cudaSuccess) {
    e = launch_upload(plan->h_dev[slot], plan->d, align_up(plan->L.bytes, 16), stream);
    ++pool->launches;
  }
  if (e == cudaSuccess) e = cudaEventRecord(plan->h_ev[slot], stream);
  if (!cuda_ok(e, "ts_step_plan_prepare")) {
    ungrow(pool, n, sids, fa);
    return TS_ERR_CUDA;
  }
  plan->h_busy[slot] = true;
  plan->h_next ^= 1;
  plan->total_rows = fa.total_rows;
  plan->prepared = true;
  ++plan->prepares;
  for (int b = 0; b < n; ++b) pool->sess[sids[b]].in_plan = true;
  return TS_OK;
}

int ts_step_plan_run(ts_step_plan* plan, int32_t layer, int32_t slot, float scale, uint32_t run_flags, void* cuda_stream) {
  if (plan == nullptr) return TS_ERR_INVALID;
  ts_pool* pool = plan->pool;
  if (layer < 0 || layer >= pool->cfg.n_layers || slot < 0 || slot >= plan->n_slots) return TS_ERR_INVALID;
  if ((run_flags & ~(uint32_t)TS_RUN_APPEND) != 0 || !(scale > 0.0f) || !std::isfinite(scale)) return TS_ERR_INVALID;
  if (!plan->prepared || !plan->slots[slot].bound) return TS_ERR_STATE;
  const ts_step_plan::Slot& s = plan->slots[slot];
  const bool with_copy = (run_flags & TS_RUN_APPEND) != 0;
  const AttnParams p = make_params(pool, plan->L, plan->d, plan->n, slot, layer, s.k, s.v, s.out, s.lse, scale, with_copy,
                                   plan->total_rows);
  TS_CUDA(launch_attention(p, pool->cfg.head_dim, plan->grid, (cudaStream_t)cuda_stream));   // the only stream operation
  ++pool->launches;
  return TS_OK;
}

int ts_step_plan_commit(ts_step_plan* plan, uint32_t flags, void* cuda_stream) {
  if (plan == nullptr || (flags & ~(uint32_t)TS_COMMIT) != 0) return TS_ERR_INVALID;
  if (!plan->prepared) return TS_ERR_STATE;
  ts_pool* pool = plan->pool;
  TS_CUDA(cudaSetDevice(pool->cfg.device));
  const uint64_t seq = pool->tl_compute.record((cudaStream_t)cuda_stream);   // after every launch of the step
  for (int32_t sid : plan->sids) pool->sess[sid].in_plan = false;
  append_commit(pool, plan->n, plan->sids.data(), plan->cf.data(), flags, seq);
  plan->prepared = false;
  return TS_OK;
}

int64_t ts_step_plan_block_bytes(ts_step_plan* plan) { return plan ? (int64_t)plan->L.bytes : 0; }

// --------------------------------------------------------------------------------------------- gather
int ts_gather_kv(ts_pool* pool, int32_t layer, int32_t sid, void* k_out, void* v_out, void* cuda_stream) {
  if (pool == nullptr) return TS_ERR_INVALID;
  const ts_pool_config& c = pool->cfg;
  if (layer < 0 || layer >= c.n_layers) return TS_ERR_INVALID;
  if (sid < 0 || sid >= c.max_sessions || pool->sess[sid].state != TS_SESSION_RESIDENT) return TS_ERR_STATE;
  Session& s = pool->sess[sid];
  const int L = s.P * c.frame_tokens;
  if (L == 0) return TS_OK;
  if (k_out == nullptr || v_out == nullptr || (((uintptr_t)k_out | (uintptr_t)v_out) & 15) != 0) return TS_ERR_INVALID;
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  TS_CUDA(cudaSetDevice(c.device));
  const size_t off_pt = 128;
  const size_t bytes = off_pt + s.pt.size() * 4;
  Staging* st = nullptr;
  int rc = acquire_staging(pool, bytes, &st);
  if (rc != TS_OK) return rc;
  CopySess* cs = reinterpret_cast<CopySess*>(st->h);
  cs->tok_off = 0;
  cs->n_tok = L;
  cs->n_zero = 0;
  cs->x0 = s.o;
  cs->pt_off = 0;
  cs->row_off = 0;
  cs->pad0 = cs->pad1 = 0;
  std::copy(s.pt.begin(), s.pt.end(), reinterpret_cast<int32_t*>(st->h + off_pt));
  TS_CUDA(pool->tl_side.wait(stream, s.side_seq));
  rc = upload_staging(pool, st, bytes, stream);
  if (rc != TS_OK) return rc;
  CopyParams p;
  memset(&p, 0, sizeof(p));
  p.sess = reinterpret_cast<const CopySess*>(st->d);
  p.page_tables = reinterpret_cast<const int32_t*>(st->d + off_pt);
  p.n_sess = 1;
  p.total_rows = L;
  p.H = c.n_heads;
  p.D = c.head_dim;
  p.B = c.page_tokens;
  p.log2_B = pool->log2_B;
  p.page_stride = pool->page_bytes;
  p.layer_k_off = (int64_t)layer * pool->layer_bytes;
  p.layer_v_off = p.layer_k_off + pool->kv_bytes;
  p.slab = pool->slab;
  p.dst_k = (uint8_t*)k_out;
  p.dst_v = (uint8_t*)v_out;
  TS_CUDA(launch_gather(p, pool->sm_count, stream));
  ++pool->launches;
  TS_CUDA(cudaEventRecord(st->ev, stream));
  st->in_flight = true;
  s.compute_seq = pool->tl_compute.record(stream);
  return TS_OK;
}

// Page copies of a suspend (to_host) or resume on the side stream: one copy per run of pages that are adjacent both in the
// slab and in the arena (FIFO allocation keeps a session's pages largely contiguous: a full window then moves at the
// rate of one large copy; a permuted pool degenerates to one copy per page, 0.87 of it at 1.57 MB per page - alternating
// the pages between two copy streams was measured and does not help: the copy engine serialises them).
static int copy_session_pages(ts_pool* pool, const Session& s, bool to_host) {
  const cudaMemcpyKind kind = to_host ? cudaMemcpyDeviceToHost : cudaMemcpyHostToDevice;
  for (size_t i = 0; i < s.pt.size();) {
    size_t e = i + 1;
    while (e < s.pt.size() && s.pt[e] == s.pt[e - 1] + 1 && s.host_slots[e] == s.host_slots[e - 1] + 1) ++e;
    uint8_t* dev_ptr = pool->slab + (int64_t)s.pt[i] * pool->page_bytes;
    uint8_t* host_ptr = pool->host + (int64_t)s.host_slots[i] * pool->page_bytes;
    TS_CUDA(cudaMemcpyAsync(to_host ? host_ptr : dev_ptr, to_host ? dev_ptr : host_ptr, (size_t)(e - i) * pool->page_bytes, kind,
                            to_host ? pool->side_out : pool->side));
    i = e;
  }
  return TS_OK;
}

// --------------------------------------------------------------------------------------------- offload
int ts_session_suspend(ts_pool* pool, int32_t sid) {
  if (pool == nullptr) return TS_ERR_INVALID;
  const ts_pool_config& c = pool->cfg;
  if (sid < 0 || sid >= c.max_sessions || pool->sess[sid].state != TS_SESSION_RESIDENT) return TS_ERR_STATE;
  Session& s = pool->sess[sid];
  if (s.in_plan) return TS_ERR_STATE;   // chunk-boundary rule (R12): not inside a prepared step
  if (s.pt.size() > pool->host_free.size()) return TS_ERR_NO_HOST;
  TS_CUDA(cudaSetDevice(c.device));
  // chunk-boundary rule (R12): the copy out starts after the compute work already enqueued on the session - and after a
  // resume of it that may still be copying in (resumes run on the other offload stream)
  TS_CUDA(pool->tl_compute.wait(pool->side_out, s.compute_seq));
  TS_CUDA(pool->tl_side.wait(pool->side_out, s.side_seq));
  s.host_slots.clear();
  uint64_t wait_slots = 0;
  for (size_t i = 0; i < s.pt.size(); ++i) {
    const int32_t slot = pool->host_free.front();
    pool->host_free.pop_front();
    wait_slots = std::max(wait_slots, pool->host_slot_seq[slot]);   // a resume may still be reading the slot
    s.host_slots.push_back(slot);
  }
  TS_CUDA(pool->tl_side.wait(pool->side_out, wait_slots));
  {
    const int rc = copy_session_pages(pool, s, true);
    if (rc != TS_OK) return rc;
  }
  const uint64_t seq = pool->tl_side.record(pool->side_out);
  for (int32_t pg : s.pt) {
    pool->page_side_seq[pg] = seq;
    pool->page_compute_seq[pg] = s.compute_seq;
    pool->free_q.push_back(pg);
  }
  s.pt.clear();
  s.side_seq = seq;
  s.state = TS_SESSION_SUSPENDED;
  return TS_OK;
}

int ts_session_resume(ts_pool* pool, int32_t sid) {
  if (pool == nullptr) return TS_ERR_INVALID;
  const ts_pool_config& c = pool->cfg;
  if (sid < 0 || sid >= c.max_sessions || pool->sess[sid].state != TS_SESSION_SUSPENDED) return TS_ERR_STATE;
  Session& s = pool->sess[sid];
  if (s.host_slots.size() > pool->free_q.size()) return TS_ERR_NO_PAGES;
  TS_CUDA(cudaSetDevice(c.device));
  uint64_t wait_compute = 0, wait_side = s.side_seq;                     // its own copy out comes first
  for (size_t i = 0; i < s.host_slots.size(); ++i) {
    const int32_t pg = pool->free_q.front();
    pool->free_q.pop_front();
    wait_compute = std::max(wait_compute, pool->page_compute_seq[pg]);   // readers of the page's previous owner
    wait_side = std::max(wait_side, pool->page_side_seq[pg]);            // ... and a copy out of it still in flight
    s.pt.push_back(pg);
  }
  TS_CUDA(pool->tl_compute.wait(pool->side, wait_compute));
  TS_CUDA(pool->tl_side.wait(pool->side, wait_side));
  {
    const int rc = copy_session_pages(pool, s, false);
    if (rc != TS_OK) return rc;
  }
  s.side_seq = pool->tl_side.record(pool->side);
  for (int32_t slot : s.host_slots) {
    pool->host_slot_seq[slot] = s.side_seq;                              // the slot may be overwritten after this copy
    pool->host_free.push_back(slot);
  }
  s.host_slots.clear();
  s.ver = ++pool->ver_seq;
  s.state = TS_SESSION_RESIDENT;
  return TS_OK;
}

// --------------------------------------------------------------------------------------------- migration
int ts_session_migrate(ts_pool* src, int32_t sid, ts_pool* dst, int32_t* sid_out) {
  if (src == nullptr || dst == nullptr || sid_out == nullptr) return TS_ERR_INVALID;
  if (sid < 0 || sid >= src->cfg.max_sessions || src->sess[sid].state == TS_SESSION_CLOSED) return TS_ERR_STATE;
  const ts_pool_config &a = src->cfg, &b = dst->cfg;
  if (src == dst) return TS_ERR_INVALID;
  if (a.n_layers != b.n_layers || a.n_heads != b.n_heads || a.head_dim != b.head_dim || a.page_tokens != b.page_tokens ||
      a.frame_tokens != b.frame_tokens || a.window_frames != b.window_frames)
    return TS_ERR_INVALID;
  Session& s = src->sess[sid];
  if (s.state != TS_SESSION_RESIDENT || s.in_plan) return TS_ERR_STATE;   // (i): only a live, frozen state moves
  int new_sid = -1;
  for (int i = 0; i < b.max_sessions && new_sid < 0; ++i)
    if (dst->sess[i].state == TS_SESSION_CLOSED) new_sid = i;
  if (new_sid < 0) return TS_ERR_CAPACITY;
  const size_t n = s.pt.size();
  if (n > dst->free_q.size()) return TS_ERR_NO_PAGES;
  TS_CUDA(cudaSetDevice(b.device));
  if (a.device != b.device) {   // one-sided access: the target maps the source's memory ("registers")
    int can = 0;
    TS_CUDA(cudaDeviceCanAccessPeer(&can, b.device, a.device));
    if (!can) {
      g_last_cuda_error = "no peer access from the target device to the source device";
      return TS_ERR_CUDA;
    }
    const cudaError_t e = cudaDeviceEnablePeerAccess(a.device, 0);
    if (e == cudaErrorPeerAccessAlreadyEnabled) cudaGetLastError();
    else TS_CUDA(e);
  }
  Staging* st = nullptr;
  if (n > 0) {
    const int rc = acquire_staging(dst, n * 8, &st);
    if (rc != TS_OK) return rc;
  }
  // ---- install on the target (as a resume would); a CUDA failure below puts the popped ids back (nothing changes)
  Session& t = dst->sess[new_sid];
  t = Session();
  t.P = s.P;
  t.o = s.o;
  uint64_t wait_compute = 0, wait_dst_side = 0;
  for (size_t i = 0; i < n; ++i) {
    const int32_t pg = dst->free_q.front();
    dst->free_q.pop_front();
    wait_compute = std::max(wait_compute, dst->page_compute_seq[pg]);   // readers of the page's previous owner
    wait_dst_side = std::max(wait_dst_side, dst->page_side_seq[pg]);    // ... and a copy out of it still in flight
    t.pt.push_back(pg);
  }
  auto undo = [&]() {
    for (auto it = t.pt.rbegin(); it != t.pt.rend(); ++it) dst->free_q.push_front(*it);
    t = Session();
    return TS_ERR_CUDA;
  };
#define TS_CUDA_UNDO(call)                    \
  do {                                        \
    if (!tc::cuda_ok((call), #call)) return undo(); \
  } while (0)
  uint64_t seq_src = s.side_seq;
  if (n > 0) {
    int32_t* pairs = reinterpret_cast<int32_t*>(st->h);
    for (size_t i = 0; i < n; ++i) {
      pairs[2 * i] = s.pt[i];
      pairs[2 * i + 1] = t.pt[i];
    }
    // (i) chunk boundary: after the compute work already enqueued on the session at the source, and after a resume
    // of it that may still be copying in
    TS_CUDA_UNDO(src->tl_compute.wait(dst->side, s.compute_seq));
    TS_CUDA_UNDO(src->tl_side.wait(dst->side, s.side_seq));
    TS_CUDA_UNDO(dst->tl_compute.wait(dst->side, wait_compute));
    TS_CUDA_UNDO(dst->tl_side.wait(dst->side, wait_dst_side));
    TS_CUDA_UNDO(launch_upload(st->h_dev, st->d, align_up(n * 8, 16), dst->side));   // not a DMA copy: see upload_staging
    ++dst->launches;
    PullParams p;
    p.src_slab = src->slab;
    p.dst_slab = dst->slab;
    p.pairs = reinterpret_cast<const int32_t*>(st->d);
    p.n_pages = (int32_t)n;
    p.vec_per_page = (int32_t)(dst->page_bytes / 16);
    p.page_stride = dst->page_bytes;
    TS_CUDA_UNDO(launch_page_pull(p, dst->sm_count, dst->side));   // (ii) the target fetches
    // ---- the fetch is enqueued: from here on the move is carried through (the remaining calls only order streams)
    ++dst->launches;
    cuda_ok(cudaEventRecord(st->ev, dst->side), "cudaEventRecord");
    st->in_flight = true;
    t.side_seq = dst->tl_side.record(dst->side);              // compute calls on the new session wait for this
    // (iii) the source's pages may be rewritten only after the fetch: mark that point on the source's side timeline
    cuda_ok(cudaSetDevice(a.device), "cudaSetDevice");
    cuda_ok(dst->tl_side.wait(src->side, t.side_seq), "cudaStreamWaitEvent");
    seq_src = src->tl_side.record(src->side);
  }
#undef TS_CUDA_UNDO
  t.ver = ++dst->ver_seq;
  t.state = TS_SESSION_RESIDENT;
  for (int32_t pg : s.pt) {                                   // release on the source (as a close would)
    src->page_side_seq[pg] = seq_src;
    src->page_compute_seq[pg] = s.compute_seq;
    src->free_q.push_back(pg);
  }
  s = Session();
  *sid_out = new_sid;
  return TS_OK;
}

int ts_offload_sync(ts_pool* pool) {
  if (pool == nullptr) return TS_ERR_INVALID;
  TS_CUDA(cudaSetDevice(pool->cfg.device));
  TS_CUDA(cudaStreamSynchronize(pool->side));
  TS_CUDA(cudaStreamSynchronize(pool->side_out));
  return TS_OK;
}

// --------------------------------------------------------------------------------------------- host-buffer step
int ts_chunk_step_host(ts_pool* pool, int32_t layer, int32_t n, const int32_t* sids, const int32_t* chunk_frames,
                       const void* q_host, const void* k_host, const void* v_host, void* out_host, float scale, uint32_t flags,
                       void* cuda_stream) {
  if (pool == nullptr) return TS_ERR_INVALID;
  int rc = check_batch(pool, layer, n, sids, chunk_frames);
  if (rc != TS_OK) return rc;
  if (n == 0) return TS_OK;
  if (q_host == nullptr || k_host == nullptr || v_host == nullptr || out_host == nullptr) return TS_ERR_INVALID;
  if (!(scale > 0.0f) || !std::isfinite(scale)) return TS_ERR_INVALID;
  if ((flags & ~(uint32_t)TS_COMMIT) != 0) return TS_ERR_INVALID;
  // all-or-nothing: the page demand of the step is checked before a single copy is enqueued
  if (page_demand(pool, n, sids, chunk_frames) > (int64_t)pool->free_q.size()) return TS_ERR_NO_PAGES;
  const ts_pool_config& c = pool->cfg;
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  TS_CUDA(cudaSetDevice(c.device));
  int64_t tokens = 0;
  for (int b = 0; b < n; ++b) tokens += (int64_t)chunk_frames[b] * c.frame_tokens;
  const size_t nbytes = (size_t)tokens * c.n_heads * c.head_dim * 2;
  const size_t tensor_bytes = align_up(nbytes, 1024);
  if (pool->h2d_s == nullptr) {
    TS_CUDA(cudaStreamCreateWithFlags(&pool->h2d_s, cudaStreamNonBlocking));
    TS_CUDA(cudaStreamCreateWithFlags(&pool->d2h_s, cudaStreamNonBlocking));
    for (cudaEvent_t* e : {&pool->ev_in, &pool->ev_attn, &pool->ev_out, &pool->ev_free[0], &pool->ev_free[1]})
      TS_CUDA(cudaEventCreateWithFlags(e, cudaEventDisableTiming));
  }
  if (pool->stage_cap < 8 * tensor_bytes) {
    // Staging grows without waiting for anything: the outgrown buffer may still be read by launches in flight, so it is
    // kept until the pool is destroyed (sizes double, so what is kept is less than what is in use).
    uint8_t* fresh = nullptr;
    const size_t cap = std::max(8 * tensor_bytes, 2 * pool->stage_cap);
    TS_CUDA(cudaMalloc((void**)&fresh, cap));
    if (pool->stage_dev) pool->retired.push_back(pool->stage_dev);
    pool->stage_dev = fresh;
    pool->stage_cap = cap;
    pool->host_steps = 0;
  }
  // Two staging sets and two copy streams: the H2D of this call does not wait for the caller's stream (host buffers
  // are read like any pinned cudaMemcpyAsync source: valid from the call until the stream reaches the end of the
  // call), only for the staging set to be free, so it runs under the attention and the D2H of the previous call.
  const int slot = (int)(pool->host_steps & 1);
  const bool slot_used = pool->host_steps >= 2;
  ++pool->host_steps;
  uint8_t* dq = pool->stage_dev + (size_t)slot * (pool->stage_cap / 2);
  uint8_t* dk = dq + tensor_bytes;
  uint8_t* dv = dk + tensor_bytes;
  uint8_t* dout = dv + tensor_bytes;
  if (slot_used) TS_CUDA(cudaStreamWaitEvent(pool->h2d_s, pool->ev_free[slot], 0));
  const uint8_t *hq = (const uint8_t*)q_host, *hk = (const uint8_t*)k_host, *hv = (const uint8_t*)v_host;
  if (hk == hq + tensor_bytes && hv == hk + tensor_bytes) {   // one packed host buffer: one copy
    TS_CUDA(cudaMemcpyAsync(dq, hq, 2 * tensor_bytes + nbytes, cudaMemcpyHostToDevice, pool->h2d_s));
  } else {
    TS_CUDA(cudaMemcpyAsync(dq, hq, nbytes, cudaMemcpyHostToDevice, pool->h2d_s));
    TS_CUDA(cudaMemcpyAsync(dk, hk, nbytes, cudaMemcpyHostToDevice, pool->h2d_s));
    TS_CUDA(cudaMemcpyAsync(dv, hv, nbytes, cudaMemcpyHostToDevice, pool->h2d_s));
  }
  TS_CUDA(cudaEventRecord(pool->ev_in, pool->h2d_s));
  TS_CUDA(cudaStreamWaitEvent(stream, pool->ev_in, 0));
  // the product's best path: attention and append in ONE launch
  rc = ts_chunk_step(pool, layer, n, sids, chunk_frames, dq, dk, dv, dout, nullptr, scale, flags, cuda_stream);
  if (rc != TS_OK) {                                          // only a CUDA failure can get here (everything else was checked)
    cudaEventRecord(pool->ev_free[slot], stream);             // the set's next user still waits for what was enqueued
    return rc;
  }
  TS_CUDA(cudaEventRecord(pool->ev_attn, stream));
  TS_CUDA(cudaStreamWaitEvent(pool->d2h_s, pool->ev_attn, 0));
  TS_CUDA(cudaMemcpyAsync(out_host, dout, nbytes, cudaMemcpyDeviceToHost, pool->d2h_s));
  TS_CUDA(cudaEventRecord(pool->ev_out, pool->d2h_s));
  TS_CUDA(cudaStreamWaitEvent(stream, pool->ev_out, 0));   // stream order: out_host is complete when the call is
  TS_CUDA(cudaEventRecord(pool->ev_free[slot], stream));   // ... and the staging set is free again
  return TS_OK;
}

}  // extern "C"

// --------------------------------------------------------------------------------------------- allocation-free attention
// ts_chunk_attention_static: ts_chunk_attention for callers that cannot allocate (CUDA graph capture around the call,
// tight serving loops, harnesses that forbid cudaMalloc).  The launch's schedule block - per-session tensor maps, session
// descriptors, packed page tables, the work-item list and the kernel's work-item cursor and per-cluster feed rings (the only
// part the kernel WRITES: scratch that has to be zero at launch) - does not go through the pool's staging ring (whose
// buffers are cudaMalloc'ed and grow on demand) but into ONE file-scope device array of a fixed size.  Every GPU that loads
// the library holds these kStaticScratchBytes until the process exits.
//
// In host code `g_static_scratch` is a host-side stand-in for the symbol, not a device address: the address the kernel
// gets is looked up per device with cudaGetSymbolAddress, once, with that device current (static_scratch_ptr()).
constexpr size_t kStaticScratchBytes = 256 * 1024;   // 32 Wan-1.3B-shaped sessions need ~160 KB, configs[2] 53 KB
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

namespace {

std::mutex g_static_mu;                               // the host image below and the per-device addresses
unsigned char* g_static_dev[64] = {};                 // device address of g_static_scratch on device i (null: not looked up yet)
alignas(256) unsigned char g_static_host[kStaticScratchBytes];   // the block is assembled here (ordinary host memory)

// Set-up, once per device, with that device current.  Allocates nothing: the array exists from the moment the library's
// module is loaded on the device.
int static_scratch_ptr(int device, unsigned char** out) {
  if (device < 0 || device >= 64) return TS_ERR_INVALID;
  if (g_static_dev[device] == nullptr) {
    void* ptr = nullptr;
    if (!tc::cuda_ok(cudaSetDevice(device), "cudaSetDevice(static scratch)")) return TS_ERR_CUDA;
    if (!tc::cuda_ok(cudaGetSymbolAddress(&ptr, g_static_scratch), "cudaGetSymbolAddress(g_static_scratch)")) return TS_ERR_CUDA;
    if (ptr == nullptr || ((uintptr_t)ptr & 255) != 0) {
      tc::g_last_cuda_error = "cudaGetSymbolAddress(g_static_scratch): null or misaligned device address";
      return TS_ERR_CUDA;
    }
    g_static_dev[device] = (unsigned char*)ptr;
  }
  *out = g_static_dev[device];
  return TS_OK;
}

}  // namespace

extern "C" {

int64_t ts_static_scratch_bytes(void) { return (int64_t)kStaticScratchBytes; }

int ts_chunk_attention_static(ts_pool* pool, int32_t layer, int32_t n, const int32_t* sids, const int32_t* chunk_frames,
                              const void* q, const void* k, const void* v, void* out, float* lse, float scale,
                              void* cuda_stream) {
  if (pool == nullptr) return TS_ERR_INVALID;
  int rc = check_batch(pool, layer, n, sids, chunk_frames);
  if (rc != TS_OK) return rc;
  if (n == 0) return TS_OK;
  if (q == nullptr || k == nullptr || v == nullptr || out == nullptr) return TS_ERR_INVALID;
  if ((((uintptr_t)q | (uintptr_t)k | (uintptr_t)v) & 15) != 0 || ((uintptr_t)out & 31) != 0) return TS_ERR_INVALID;
  if (!(scale > 0.0f) || !std::isfinite(scale)) return TS_ERR_INVALID;
  const ts_pool_config& c = pool->cfg;
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  // This call stays outside the pool's event timelines (recording into them creates events on demand, and an event recorded
  // under stream capture cannot be waited for outside the graph): a session with a resume still copying in is refused.
  for (int b = 0; b < n; ++b) {
    const Session& s = pool->sess[sids[b]];
    if (s.in_plan || !pool->tl_side.is_done(s.side_seq)) return TS_ERR_STATE;
  }
  TS_CUDA(cudaSetDevice(c.device));
  std::lock_guard<std::mutex> lock(g_static_mu);
  unsigned char* d = nullptr;
  rc = static_scratch_ptr(c.device, &d);
  if (rc != TS_OK) return rc;

  build_schedule(pool, n, sids, chunk_frames);
  const int grid = pool->sched_cta[0];
  const BlockLayout L = block_layout(n, 1, pool->sched_pt.size(), pool->sched_items.size(), grid, false);
  if (L.bytes > kStaticScratchBytes) {
    char msg[200];
    snprintf(msg, sizeof msg, "ts_chunk_attention_static: the batch's schedule block needs %zu bytes, the static scratch array holds %zu",
             L.bytes, kStaticScratchBytes);
    tc::g_last_cuda_error = msg;
    return TS_ERR_CAPACITY;
  }
  // The whole block is rewritten by every call, the cursor and the feed rings as zeros (fill_block): nothing of the previous
  // call's contents is relied on.  The source is ordinary host memory: the copy has left it when cudaMemcpyAsync returns.
  fill_block(pool, g_static_host, L, n, nullptr);
  if (!encode_session_maps(pool, reinterpret_cast<CUtensorMap*>(g_static_host + L.off_maps), n, chunk_frames, q, k, v))
    return TS_ERR_CUDA;
  TS_CUDA(cudaMemcpyAsync(d, g_static_host, align_up(L.bytes, 16), cudaMemcpyHostToDevice, stream));
  const AttnParams p = make_params(pool, L, d, n, 0, layer, k, v, out, lse, scale, false, 0);
  TS_CUDA(launch_attention(p, c.head_dim, grid, stream));
  ++pool->launches;
  return TS_OK;
}

}  // extern "C"

// --------------------------------------------------------------------------------------------- migration between processes
// one worker process per GPU; :263: "registers the corresponding state buffers ... the target worker can
// then fetch the registered state buffers from the source worker through ... one-sided GPU memory access"; :265: freeze at a
// chunk boundary, fetch + verify, ownership flips after the transfer.  ts_session_migrate does this between two pools of one
// process; here the two pools live in two processes (on one GPU, or on two GPUs of a node with peer access):
//   registration  ts_pool_export  -> blob over the control plane ->  ts_peer_open   (CUDA IPC: the source slab becomes an
//                                                                     ordinary device pointer for page_pull_kernel)
//   (i)   freeze  ts_session_freeze  on the source  -> ticket (P, o, page ids) over the control plane
//   (ii)  fetch   ts_session_import  on the target  -> "enqueued" over the control plane
//   (iii) flip    ts_session_release on the source
// Every GPU-side dependency is an interprocess event edge (no host wait in either process): the fetch waits for the source's
// "state frozen" event, the source's side stream waits for the target's "installed" event before its freed pages can be
// handed to a writer.  The control-plane messages only have to be delivered in order: a wait is enqueued after the record
// it is meant for has been enqueued in the other process.
namespace {

struct ExportBlob {
  uint32_t magic, version;
  cudaIpcMemHandle_t mem;             // the allocation that holds the slab
  cudaIpcEventHandle_t frozen, installed;
  int64_t slab_offset;                // slab start inside that allocation
  int64_t page_bytes;
  int32_t n_layers, n_heads, head_dim, page_tokens, frame_tokens, window_frames, n_pages, pad;
};
static_assert(sizeof(ExportBlob) <= sizeof(ts_pool_export_t), "ts_pool_export_t too small");
constexpr uint32_t kExportMagic = 0x54534950u;   // "TSIP"

typedef CUresult (*PFN_addr_range)(CUdeviceptr*, size_t*, CUdeviceptr);
PFN_addr_range get_addr_range() {
  static PFN_addr_range fn = nullptr;
  if (fn == nullptr) {
    void* ptr = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuMemGetAddressRange", &ptr, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<PFN_addr_range>(ptr);
  }
  return fn;
}

int ensure_export(ts_pool* pool) {
  if (pool->exported) return TS_OK;
  TS_CUDA(cudaSetDevice(pool->cfg.device));
  PFN_addr_range range = get_addr_range();
  CUdeviceptr base = 0;
  size_t size = 0;
  if (range == nullptr || range(&base, &size, (CUdeviceptr)pool->slab) != CUDA_SUCCESS) {
    tc::g_last_cuda_error = "cuMemGetAddressRange(kv slab) failed";
    return TS_ERR_CUDA;
  }
  ExportBlob b;
  memset(&b, 0, sizeof(b));
  b.magic = kExportMagic;
  b.version = 1;
  TS_CUDA(cudaIpcGetMemHandle(&b.mem, (void*)base));
  if (pool->ipc_frozen == nullptr)
    TS_CUDA(cudaEventCreateWithFlags(&pool->ipc_frozen, cudaEventDisableTiming | cudaEventInterprocess));
  if (pool->ipc_installed == nullptr)
    TS_CUDA(cudaEventCreateWithFlags(&pool->ipc_installed, cudaEventDisableTiming | cudaEventInterprocess));
  TS_CUDA(cudaIpcGetEventHandle(&b.frozen, pool->ipc_frozen));
  TS_CUDA(cudaIpcGetEventHandle(&b.installed, pool->ipc_installed));
  // an event that was never recorded counts as complete: a waiter that comes first does not block
  b.slab_offset = (int64_t)((CUdeviceptr)pool->slab - base);
  b.page_bytes = pool->page_bytes;
  const ts_pool_config& c = pool->cfg;
  b.n_layers = c.n_layers;
  b.n_heads = c.n_heads;
  b.head_dim = c.head_dim;
  b.page_tokens = c.page_tokens;
  b.frame_tokens = c.frame_tokens;
  b.window_frames = c.window_frames;
  b.n_pages = c.n_pages;
  memset(&pool->export_blob, 0, sizeof(pool->export_blob));
  memcpy(&pool->export_blob, &b, sizeof(b));
  pool->exported = true;
  return TS_OK;
}

}  // namespace

struct ts_peer {
  ts_pool* local = nullptr;
  uint8_t* base = nullptr;       // cudaIpcOpenMemHandle mapping of the remote allocation
  uint8_t* slab = nullptr;       // the remote pool's slab inside it
  cudaEvent_t frozen = nullptr, installed = nullptr;
  int32_t n_pages = 0;
};

extern "C" {

int ts_pool_export(ts_pool* pool, ts_pool_export_t* out) {
  if (pool == nullptr || out == nullptr) return TS_ERR_INVALID;
  const int rc = ensure_export(pool);
  if (rc != TS_OK) return rc;
  *out = pool->export_blob;
  return TS_OK;
}

int ts_peer_open(ts_pool* local, const ts_pool_export_t* remote, ts_peer** out) {
  if (local == nullptr || remote == nullptr || out == nullptr) return TS_ERR_INVALID;
  ExportBlob b;
  memcpy(&b, remote, sizeof(b));
  const ts_pool_config& c = local->cfg;
  if (b.magic != kExportMagic || b.version != 1) return TS_ERR_INVALID;
  if (b.n_layers != c.n_layers || b.n_heads != c.n_heads || b.head_dim != c.head_dim || b.page_tokens != c.page_tokens ||
      b.frame_tokens != c.frame_tokens || b.window_frames != c.window_frames || b.page_bytes != local->page_bytes ||
      b.n_pages < 1 || b.slab_offset < 0)
    return TS_ERR_INVALID;
  int rc = ensure_export(local);   // the local pool's own events are needed on both ends of a move
  if (rc != TS_OK) return rc;
  TS_CUDA(cudaSetDevice(c.device));
  ts_peer* peer = new ts_peer();
  peer->local = local;
  peer->n_pages = b.n_pages;
  void* base = nullptr;
  if (!tc::cuda_ok(cudaIpcOpenMemHandle(&base, b.mem, cudaIpcMemLazyEnablePeerAccess), "cudaIpcOpenMemHandle(remote kv slab)") ||
      !tc::cuda_ok(cudaIpcOpenEventHandle(&peer->frozen, b.frozen), "cudaIpcOpenEventHandle(frozen)") ||
      !tc::cuda_ok(cudaIpcOpenEventHandle(&peer->installed, b.installed), "cudaIpcOpenEventHandle(installed)")) {
    if (base) cudaIpcCloseMemHandle(base);
    if (peer->frozen) cudaEventDestroy(peer->frozen);
    delete peer;
    return TS_ERR_CUDA;
  }
  peer->base = (uint8_t*)base;
  peer->slab = peer->base + b.slab_offset;
  *out = peer;
  return TS_OK;
}

int ts_peer_close(ts_peer* peer) {
  if (peer == nullptr) return TS_ERR_INVALID;
  cudaSetDevice(peer->local->cfg.device);
  cudaStreamSynchronize(peer->local->side);     // no fetch of ours still reads the mapping
  if (peer->frozen) cudaEventDestroy(peer->frozen);
  if (peer->installed) cudaEventDestroy(peer->installed);
  if (peer->base) cudaIpcCloseMemHandle(peer->base);
  cudaGetLastError();
  delete peer;
  return TS_OK;
}

int ts_session_freeze(ts_pool* src, int32_t sid, ts_migration_ticket_t* ticket, int32_t* pages_out, int32_t cap) {
  if (src == nullptr || ticket == nullptr || (pages_out == nullptr && cap > 0) || cap < 0) return TS_ERR_INVALID;
  if (sid < 0 || sid >= src->cfg.max_sessions) return TS_ERR_STATE;
  Session& s = src->sess[sid];
  if (s.state != TS_SESSION_RESIDENT || s.in_plan) return TS_ERR_STATE;
  if ((size_t)cap < s.pt.size()) return TS_ERR_INVALID;
  int rc = ensure_export(src);
  if (rc != TS_OK) return rc;
  TS_CUDA(cudaSetDevice(src->cfg.device));
  // (i) chunk boundary: "state frozen" = after the compute work already enqueued on the session and after a resume of it
  // that may still be copying in
  TS_CUDA(src->tl_compute.wait(src->side, s.compute_seq));
  TS_CUDA(src->tl_side.wait(src->side, s.side_seq));
  TS_CUDA(cudaEventRecord(src->ipc_frozen, src->side));
  s.in_plan = s.frozen = true;
  ticket->sid = sid;
  ticket->frames = s.P;
  ticket->head_off = s.o;
  ticket->n_pages = (int32_t)s.pt.size();
  std::copy(s.pt.begin(), s.pt.end(), pages_out);
  return TS_OK;
}

int ts_session_unfreeze(ts_pool* src, int32_t sid) {
  if (src == nullptr) return TS_ERR_INVALID;
  if (sid < 0 || sid >= src->cfg.max_sessions || !src->sess[sid].frozen) return TS_ERR_STATE;
  src->sess[sid].in_plan = src->sess[sid].frozen = false;
  return TS_OK;
}

int ts_session_import(ts_pool* dst, ts_peer* source, const ts_migration_ticket_t* ticket, const int32_t* pages,
                      int32_t* sid_out) {
  if (dst == nullptr || source == nullptr || ticket == nullptr || sid_out == nullptr || source->local != dst)
    return TS_ERR_INVALID;
  const ts_pool_config& c = dst->cfg;
  const int64_t n = ticket->n_pages;
  // (ii) "verifies": the ticket describes a state this geometry can hold, and every page id lies inside the source slab
  if (n < 0 || (n > 0 && pages == nullptr) || ticket->frames < 0 || ticket->head_off < 0 || ticket->head_off >= c.page_tokens ||
      n * c.page_tokens < (int64_t)ticket->head_off + (int64_t)ticket->frames * c.frame_tokens ||
      (c.window_frames > 0 && ticket->frames > c.window_frames))
    return TS_ERR_INVALID;
  for (int64_t i = 0; i < n; ++i)
    if (pages[i] < 0 || pages[i] >= source->n_pages) return TS_ERR_INVALID;
  int new_sid = -1;
  for (int i = 0; i < c.max_sessions && new_sid < 0; ++i)
    if (dst->sess[i].state == TS_SESSION_CLOSED) new_sid = i;
  if (new_sid < 0) return TS_ERR_CAPACITY;
  if ((size_t)n > dst->free_q.size()) return TS_ERR_NO_PAGES;
  TS_CUDA(cudaSetDevice(c.device));
  Staging* st = nullptr;
  if (n > 0) {
    const int rc = acquire_staging(dst, (size_t)n * 8, &st);
    if (rc != TS_OK) return rc;
  }
  Session& t = dst->sess[new_sid];
  t = Session();
  t.P = ticket->frames;
  t.o = ticket->head_off;
  uint64_t wait_compute = 0, wait_dst_side = 0;
  for (int64_t i = 0; i < n; ++i) {
    const int32_t pg = dst->free_q.front();
    dst->free_q.pop_front();
    wait_compute = std::max(wait_compute, dst->page_compute_seq[pg]);
    wait_dst_side = std::max(wait_dst_side, dst->page_side_seq[pg]);
    t.pt.push_back(pg);
  }
  auto undo = [&]() {
    for (auto it = t.pt.rbegin(); it != t.pt.rend(); ++it) dst->free_q.push_front(*it);
    t = Session();
    return TS_ERR_CUDA;
  };
#define TS_CUDA_UNDO(call)                    \
  do {                                        \
    if (!tc::cuda_ok((call), #call)) return undo(); \
  } while (0)
  if (n > 0) {
    int32_t* pairs = reinterpret_cast<int32_t*>(st->h);
    for (int64_t i = 0; i < n; ++i) {
      pairs[2 * i] = pages[i];
      pairs[2 * i + 1] = t.pt[(size_t)i];
    }
    TS_CUDA_UNDO(cudaStreamWaitEvent(dst->side, source->frozen, 0));   // the source's "state frozen"
    TS_CUDA_UNDO(dst->tl_compute.wait(dst->side, wait_compute));
    TS_CUDA_UNDO(dst->tl_side.wait(dst->side, wait_dst_side));
    TS_CUDA_UNDO(launch_upload(st->h_dev, st->d, align_up((size_t)n * 8, 16), dst->side));
    ++dst->launches;
    PullParams p;
    p.src_slab = source->slab;
    p.dst_slab = dst->slab;
    p.pairs = reinterpret_cast<const int32_t*>(st->d);
    p.n_pages = (int32_t)n;
    p.vec_per_page = (int32_t)(dst->page_bytes / 16);
    p.page_stride = dst->page_bytes;
    TS_CUDA_UNDO(launch_page_pull(p, dst->sm_count, dst->side));
    ++dst->launches;
    cuda_ok(cudaEventRecord(st->ev, dst->side), "cudaEventRecord");
    st->in_flight = true;
    t.side_seq = dst->tl_side.record(dst->side);   // compute calls on the new session wait for the fetch
  }
#undef TS_CUDA_UNDO
  // "installed": what the source's side stream waits for before its pages can be rewritten (also for an empty session, so
  // that a release always has a record to wait for)
  cuda_ok(cudaEventRecord(dst->ipc_installed, dst->side), "cudaEventRecord(installed)");
  t.ver = ++dst->ver_seq;
  t.state = TS_SESSION_RESIDENT;
  *sid_out = new_sid;
  return TS_OK;
}

int ts_session_release(ts_pool* src, int32_t sid, ts_peer* target) {
  if (src == nullptr || (target != nullptr && target->local != src)) return TS_ERR_INVALID;
  if (sid < 0 || sid >= src->cfg.max_sessions || !src->sess[sid].frozen) return TS_ERR_STATE;
  Session& s = src->sess[sid];
  TS_CUDA(cudaSetDevice(src->cfg.device));
  // (iii) ownership flips; the freed pages may be handed to a writer only after the target's fetch has completed
  uint64_t seq_src = s.side_seq;
  if (target != nullptr) {
    TS_CUDA(cudaStreamWaitEvent(src->side, target->installed, 0));
    seq_src = src->tl_side.record(src->side);
  }
  for (int32_t pg : s.pt) {
    src->page_side_seq[pg] = seq_src;
    src->page_compute_seq[pg] = s.compute_seq;
    src->free_q.push_back(pg);
  }
  s = Session();
  return TS_OK;
}

}  // extern "C"
