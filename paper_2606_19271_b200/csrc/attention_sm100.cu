// Coalesced chunk attention for sm_100a (step a2 of SURVEY.md §8(a); PAPER.md:66 (iii)).
//
// Persistent CTAs, one per SM, in 2-CTA clusters.  Each CTA walks a host-built list of work items (session, head,
// pair of 128-row query tiles).  Per item the KV sequence is: the session's visible cached tokens in PHYSICAL page
// order (softmax is order-invariant over keys), gathered page by page through the page table with TMA, then the
// chunk's own K/V tiles from the packed call tensors.  Only the first/last cache tile and the chunk tiles that
// cross a frame boundary take the masked path.
//
// Warp roles (384 threads):
//   warp 0      TMA producer   Q tiles once per item, K/V tiles into a ring of kSlots smem slots
//   warp 1      MMA issuer     tcgen05.mma, one elected thread; S = Q K^T (SS), O += P V (TS, P in TMEM)
//   warps 2-3   idle, or (fused chunk step) the KV append of the batch: 128-bit streaming copies into the pages
//   warps 4-7   softmax for query tile 0 (one thread per row): online softmax in fp32, lazy rescale of O,
//   warps 8-11  softmax for query tile 1                        P written back to TMEM as bf16, epilogue
// TMEM (512 columns): S0 [0,128) / P0 aliases [0,64); S1 [128,256) / P1; O0 [256,256+D); O1 [256+D,256+2D).
// Issue order  S0(0) S1(0) | PV0(j) S0(j+1) PV1(j) S1(j+1) | ...  keeps the tensor pipe busy while the other
// tile's softmax runs (two-tile ping-pong); P is handed over in two 64-key halves so that the first half of
// O += P V runs under the second half of the exponentials.
//
// Cluster: the host gives the two CTAs of a cluster two items of the SAME (session, head) wherever it can.  Each
// CTA then loads half of every K/V tile and multicasts it to both (one L2 read per pair of CTAs); both CTAs cycle
// the same number of tiles through their rings so that a tile sits at the same smem offset in both.  Every slot
// release goes to the kv_empty barriers of both CTAs (count 2), also when the two CTAs work on unrelated items.
#include <mutex>

#include "internal.h"
#include "kv_copy.cuh"
#include "ptx.cuh"

namespace tc {

constexpr int kThreads = 384;
constexpr int kTmemCols = 512;
constexpr float kRescaleThresholdLog2 = 8.0f;   // lazy rescale: tolerate p up to 2^8 before touching O
// Register file split (setmaxnreg): the CTA is launched with 384 x 168 registers; warps 0-3 (TMA, MMA, two idle)
// drop to kRegsProducer so that the 8 softmax warps can hold a full 128-wide fp32 score row without spilling.
constexpr int kRegsProducer = 72;
constexpr int kRegsSoftmax = 216;
static_assert(128 * kRegsProducer + 256 * kRegsSoftmax <= 384 * 168, "register pool");

// One MUFU.EX2 per score costs exactly as many SM cycles as the score's two MMAs at D = 128 (16/clk/SM against 8192
// FLOP/clk/SM), and the exp phase of a tile sits on the S -> softmax -> PV -> S chain.  kPolyPairs of every 16 score
// pairs are therefore evaluated on the FMA pipe instead.  One warp owns a tile's rows, so the instructions this adds
// (11 per pair against 2 MUFU) soon make the phase issue-bound: measured on configs[2], 4 of 16 is the optimum (+1.3 %),
// 6 of 16 already loses.
constexpr int kPolyPairs = 4;

// 2^x for a pair on the FMA pipe (Cody-Waite): x = n + f with n = round(x), f in [-0.5, 0.5]; 2^f by a degree-3 minimax
// polynomial (max relative error 7.5e-5, far below the 2^-9 of the bf16 rounding of P); 2^n as the fp32 whose bits are
// (n + 127) << 23 - n + 127 sits in the low mantissa bits of x + (1.5 * 2^23 + 127).  x is clamped at -127 (masked
// scores are -inf): n + 127 = 0 there, the scale factor is +0.0 and p is exactly 0, as on the MUFU path.
__device__ __forceinline__ void exp2_poly_pair(float x0, float x1, float& p0, float& p1) {
  x0 = fmaxf(x0, -127.f);
  x1 = fmaxf(x1, -127.f);
  float f0, f1, n0, n1, r0, r1, q0, q1;
  addc2(f0, f1, x0, x1, 12583039.f);
  addc2(n0, n1, f0, f1, -12583039.f);
  sub2(r0, r1, x0, x1, n0, n1);
  fma2_bcast(q0, q1, r0, r1, 0.05517083778977394f, 0.24260935187339783f);
  fma2_pc(q0, q1, q0, q1, r0, r1, 0.6932609677314758f);
  fma2_pc(q0, q1, q0, q1, r0, r1, 0.9999281764030457f);
  p0 = q0 * __uint_as_float(shl_alu(__float_as_uint(f0), 23));
  p1 = q1 * __uint_as_float(shl_alu(__float_as_uint(f1), 23));
}

template <int D>
struct Cfg {
  static constexpr int kTileBytes = 128 * D * 2;        // one [128 x D] bf16 tile
  static constexpr int kDBlocks = D / 64;               // 64-column (128-byte) swizzle blocks per tile
  static constexpr int kBlockBytes = 128 * 128;         // one [128 rows x 128 B] swizzle block
  static constexpr int kSlots = (D == 128) ? 5 : 8;
  static constexpr int kSmemQ = 2 * kTileBytes;
  static constexpr int kSmemKV = kSlots * kTileBytes;
  static constexpr int kNumBars = 2 * kSlots + 2 + 10;
  static constexpr int kXchgBytes = 2 * 128 * 2 * 4;    // (m, l) of a row from each softmax warpgroup (lone-tile merge)
  static constexpr int kSmemBytes = kSmemQ + kSmemKV + kXchgBytes + kNumBars * 8 + 16 + 16;   // + TMEM base, clock-probe stamps
};

struct ItemGeom {
  int sess, head, r0, n_q, C, q_off, pt_off, n_pt;
  int x_begin, x_end, t0, n_prior, n_chunk, n_kv;
  int n_pipe;   // KV tiles flowing through the smem ring for this item (>= n_kv: the cluster partner may see more)
  bool mc;      // K/V tiles are loaded half by this CTA, half by the cluster partner, multicast to both
  bool split;   // lone query tile: its KV tiles alternate between the two TMEM tile slots (even / odd), merged at the end
};

// Cluster items are handed out dynamically, in the host's (session, head) stream order: the TMA thread of CTA rank 0
// takes the next one from a global cursor when it gets there (it runs ahead of every other role) and publishes it as
// the k-th item of its cluster; every other role of both CTAs reads entry k of the cluster's ring.  An entry carries
// its sequence number, so a stale value of the ring slot's previous use is never mistaken for it.  -1: no more items.
// A fetcher sees the end of the list exactly once; the last cluster to see it sets the cursor back to zero (no fetcher
// touches it again in this launch), and every cluster clears its own ring on exit: the block is rearmed for the next
// launch by the kernel itself.
__device__ __forceinline__ int next_cluster_item(const AttnParams& p, uint32_t k, bool fetcher) {
  unsigned long long* slot = p.feed + (size_t)(blockIdx.x >> 1) * kFeedRing + (k % kFeedRing);
  if (fetcher) {
    int idx = atomicAdd(p.feed_hdr, 1);
    if (idx >= __ldg(p.feed_hdr + 2)) idx = -1;
    const unsigned long long v = ((unsigned long long)(k + 1) << 32) | (uint32_t)(idx + 1);
    // relaxed: the 64-bit word IS the message (sequence number and item index); the records it points to were written by the
    // host before the launch.  An acquire on the reading side would invalidate L1 at every poll for nothing.
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(slot), "l"(v) : "memory");
    if (idx < 0 && atomicAdd(p.feed_hdr + 1, 1) == (int)(gridDim.x >> 1) - 1) {
      p.feed_hdr[1] = 0;
      p.feed_hdr[0] = 0;
    }
    return idx;
  }
  unsigned long long v;
  do {
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(slot) : "memory");
  } while ((uint32_t)(v >> 32) != k + 1);
  return (int)(uint32_t)v - 1;
}

__device__ __forceinline__ ItemGeom decode_item(const AttnParams& p, int citem, uint32_t cta_rank) {
  const WorkItem w = p.items[2 * citem + cta_rank];
  const SessDesc s = p.sess[w.sess];
  ItemGeom g;
  g.sess = w.sess;
  g.head = w.head;
  g.r0 = w.q_tile * 128;
  g.C = s.C;
  g.q_off = s.q_off;
  g.pt_off = s.pt_off;
  g.n_pt = s.n_pt;
  g.x_begin = s.x_begin;
  g.x_end = s.x_end;
  g.n_pipe = (int)(w.pipe & 0xffffffu);
  g.mc = (w.pipe >> 31) != 0;
  if (s.x_end > s.x_begin) {
    g.t0 = s.x_begin >> 7;
    g.n_prior = ((s.x_end - 1) >> 7) - g.t0 + 1;
  } else {
    g.t0 = 0;
    g.n_prior = 0;
  }
  if (w.q_tile < 0) {   // no query rows: only the loader and the slot releases run
    g.r0 = 0;
    g.n_q = 0;
    g.n_chunk = 0;
    g.n_kv = 0;
  } else {
    g.n_q = (!(w.pipe & 0x40000000u) && g.r0 + 128 < s.C) ? 2 : 1;
    const int last_row = min(s.C, g.r0 + 128 * g.n_q) - 1;
    const int kv_hi = min(s.C, (last_row / p.T + 1) * p.T);   // chunk keys visible to the item's last row
    g.n_chunk = (kv_hi + 127) >> 7;
    g.n_kv = g.n_prior + g.n_chunk;
  }
  g.split = (g.n_q == 1) && (g.n_kv >= 2);
  return g;
}

template <int D>
__global__ void __launch_bounds__(kThreads, 1) chunk_attention_kernel(const __grid_constant__ AttnParams p) {
  using C = Cfg<D>;
  extern __shared__ __align__(1024) uint8_t smem[];   // swizzle-128B operands need 1024-byte alignment
  uint8_t* sQ = smem;
  uint8_t* sKV = smem + C::kSmemQ;
  float2* xchg = reinterpret_cast<float2*>(sKV + C::kSmemKV);   // [warpgroup][row]
  uint64_t* bars = reinterpret_cast<uint64_t*>(sKV + C::kSmemKV + C::kXchgBytes);
  uint64_t* kv_full = bars;
  uint64_t* kv_empty = bars + C::kSlots;
  uint64_t* q_full = bars + 2 * C::kSlots;
  uint64_t* q_empty = q_full + 1;
  uint64_t* s_full = q_full + 2;    // [2]
  uint64_t* p_half = q_full + 4;    // [2][2] P tile i, keys [64h, 64h+64) written by softmax
  uint64_t* o_done = q_full + 8;    // [2]
  uint64_t* o_free = q_full + 10;   // [2]
  uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(bars + C::kNumBars);

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;

  if (warp == 0 && lane == 0) {
    if (smem_u32(smem) & 1023u) __trap();
    for (int i = 0; i < C::kSlots; ++i) {
      mbar_init(&kv_full[i], 1);
      mbar_init(&kv_empty[i], 2);   // released by the MMA warps of both CTAs of the cluster
    }
    mbar_init(q_full, 1);
    mbar_init(q_empty, 1);
    for (int i = 0; i < 2; ++i) {
      mbar_init(&s_full[i], 1);
      mbar_init(&p_half[2 * i], 128);
      mbar_init(&p_half[2 * i + 1], 128);
      mbar_init(&o_done[i], 1);
      mbar_init(&o_free[i], 256);   // two arrivals per thread of the tile's warpgroup, or one from each of both
    }
    fence_mbar_init();
    tma_prefetch_desc(&p.map_k);
    tma_prefetch_desc(&p.map_v);
  }
  if (warp == 1) tmem_alloc(tmem_ptr, kTmemCols);
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();   // the partner's barriers are initialised before any multicast load or commit reaches them
  tc_fence_after();
  const uint32_t cta_rank = cluster_ctarank();
  const uint32_t tmem_base = *tmem_ptr;
  // optional in-kernel clock probe (one thread of CTA 0, a warp without a role on the critical path)
  // (the start stamps wait in shared memory: no register lives across the kernel for it)
  unsigned long long* probe_smem = reinterpret_cast<unsigned long long*>(tmem_ptr + 4);
  if (p.clock_probe != nullptr && blockIdx.x == 0 && threadIdx.x == 96) {
    unsigned long long ns0;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(ns0));
    probe_smem[0] = (unsigned long long)clock64();
    probe_smem[1] = ns0;
  }


  if (warp < 4) {
    setmaxnreg_dec<kRegsProducer>();
  if (warp == 0) {
    // ===================================================================== TMA producer
    if (elect_one()) {
      uint32_t kv_it = 0;
      uint32_t q_cnt = 0;
      const int sb = min(p.B, 64);            // tokens per TMA box of K/V (the maps are encoded with this box)
      const int n_sub = 128 / sb;             // boxes per 128-key tile
      for (uint32_t k_item = 0;; ++k_item) {
        const int idx = next_cluster_item(p, k_item, cta_rank == 0);
        if (idx < 0) break;
        const ItemGeom g = decode_item(p, idx, cta_rank);
        const CUtensorMap* mq = p.sess_maps + g.sess * 3;
        const CUtensorMap* mkn = mq + 1;
        const CUtensorMap* mvn = mq + 2;
        const int32_t* pt = p.page_tables + g.pt_off;
        if (g.n_q > 0) {
          // the Q tiles cannot land before the previous item's last S = Q K^T has read the buffer: pull them into L2 now
          for (int i = 0; i < g.n_q; ++i)
            for (int b = 0; b < C::kDBlocks; ++b) tma_prefetch_3d(mq, 64 * b, g.head, g.r0 + 128 * i);
          mbar_wait_long(q_empty, (q_cnt & 1) ^ 1);
          ++q_cnt;
          mbar_arrive_expect_tx(q_full, g.n_q * C::kTileBytes);
          for (int i = 0; i < g.n_q; ++i)
            for (int b = 0; b < C::kDBlocks; ++b)
              tma_load_3d(sQ + i * C::kTileBytes + b * C::kBlockBytes, mq, 64 * b, g.head, g.r0 + 128 * i, q_full);
        }
        for (int j = 0; j < g.n_pipe; ++j) {
          for (int kv = 0; kv < 2; ++kv, ++kv_it) {
            const uint32_t slot = kv_it % C::kSlots;
            const uint32_t ph = (kv_it / C::kSlots) & 1;
            mbar_wait_long(&kv_empty[slot], ph ^ 1);
            if (!g.mc && j >= g.n_kv) {
              // a tile of the partner's unrelated item: nothing to load, but the slot is cycled so that both CTAs
              // of the cluster stay on the same ring position (multicast needs equal smem offsets)
              mbar_arrive(&kv_full[slot]);
              continue;
            }
            mbar_arrive_expect_tx(&kv_full[slot], C::kTileBytes);   // own boxes + (multicast) the partner's
            uint8_t* dst = sKV + slot * C::kTileBytes;
            for (int sx = 0; sx < n_sub; ++sx) {
              if (g.mc && (uint32_t)(sx & 1) != cta_rank) continue;   // the partner loads and multicasts this box
              uint8_t* d = dst + sx * sb * 128;
              if (j < g.n_prior) {
                const CUtensorMap* mc = kv ? &p.map_v : &p.map_k;
                const int x = ((g.t0 + j) << 7) + sx * sb;            // page-table coordinate of the box
                // Boxes past the last cached token re-read the last page that HOLDS a cached token (masked): its tail is
                // real data or the append's zero fill.  Never a later table entry: a fused step and layers > 0 of a
                // multi-layer step see tables already grown by pages whose bytes in this layer are not written yet
                // (stale memory of a previous owner: P = 0 times a NaN there would be NaN inside the MMA).
                const int page = pt[min(x >> p.log2_B, (g.x_end - 1) >> p.log2_B)];
                const int tok = x & (p.B - 1);
                for (int b = 0; b < C::kDBlocks; ++b) {
                  if (g.mc) tma_load_4d_mc(d + b * C::kBlockBytes, mc, 64 * b, tok, g.head, page, &kv_full[slot], 3);
                  else tma_load_4d(d + b * C::kBlockBytes, mc, 64 * b, tok, g.head, page, &kv_full[slot]);
                }
              } else {
                const CUtensorMap* mc = kv ? mvn : mkn;
                const int row = ((j - g.n_prior) << 7) + sx * sb;
                for (int b = 0; b < C::kDBlocks; ++b) {
                  if (g.mc) tma_load_3d_mc(d + b * C::kBlockBytes, mc, 64 * b, g.head, row, &kv_full[slot], 3);
                  else tma_load_3d(d + b * C::kBlockBytes, mc, 64 * b, g.head, row, &kv_full[slot]);
                }
              }
            }
          }
        }
      }
    }
  } else if (warp == 1) {
    // ===================================================================== MMA issuer
    if (elect_one()) {
      constexpr uint32_t idesc_s = make_idesc_bf16(128, 128, 0, 0);
      constexpr uint32_t idesc_pv = make_idesc_bf16(128, D, 0, 1);
      // operand addresses in 16-byte units, reduced ONCE to the descriptor's 14-bit field (a shared-memory address carries the
      // CTA's rank within the cluster above bit 18): from here on descriptor arithmetic is plain addition
      const uint32_t sQ16 = (smem_u32(sQ) >> 4) & 0x3FFFu;
      const uint32_t sKV16 = (smem_u32(sKV) >> 4) & 0x3FFFu;
      // S of TMEM tile slot `i` = (query tile `qi` in smem) x (K tile in ring slot `slot`)^T
      auto issue_s_q = [&](int qi, int i, uint32_t slot) {
        const uint32_t a = sQ16 + qi * (C::kTileBytes >> 4);
        const uint32_t b = sKV16 + slot * (C::kTileBytes >> 4);
#pragma unroll
        for (int kk = 0; kk < D / 16; ++kk) {
          const uint32_t off = (kk >> 2) * (C::kBlockBytes >> 4) + (kk & 3) * 2;
          mma_ss(tmem_base + i * 128, make_smem_desc_sw128_a16(a + off, 16, 1024), make_smem_desc_sw128_a16(b + off, 16, 1024),
                 idesc_s, kk > 0);
        }
      };
      auto issue_s = [&](int i, uint32_t slot) { issue_s_q(i, i, slot); };
      // half h of O_i += P_i V: the 16-key steps 4h .. 4h+3 (keys [64h, 64h+64))
      auto issue_pv_half = [&](int i, uint32_t slot, int h, bool acc) {
        const uint32_t b = sKV16 + slot * (C::kTileBytes >> 4);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const int kk = 4 * h + q;
          mma_ts(tmem_base + 256 + i * D, tmem_base + i * 128 + kk * 8,
                 make_smem_desc_sw128_a16(b + kk * 128, C::kBlockBytes, 1024), idesc_pv, (acc || q > 0) ? 1u : 0u);
        }
      };
      uint32_t kv_it = 0, q_cnt = 0;
      // per tile slot: P hand-offs and items so far (scalars with selects: a runtime-indexed array would live in local memory)
      uint32_t cnt_p0 = 0, cnt_p1 = 0, cnt_it0 = 0, cnt_it1 = 0;
      for (uint32_t k_item = 0;; ++k_item) {
        const int idx = next_cluster_item(p, k_item, false);
        if (idx < 0) break;
        const ItemGeom g = decode_item(p, idx, cta_rank);
        // hand a K/V slot back once every MMA issued so far has read it - always to BOTH CTAs of the cluster, also
        // when the two work on unrelated items: a slot is refilled (possibly by the partner's multicast) only after
        // both CTAs are done with their tile at that ring position
        auto release = [&](uint32_t slot) { mma_commit_mc(&kv_empty[slot], 3); };
        if (g.split) {
          // lone query tile: K/V tile j goes to TMEM tile slot j & 1, so two tiles are in flight as for a pair.
          // Ring positions relative to the item: K_j at 2j, V_j at 2j + 1.
          const uint32_t base = kv_it;
          mbar_wait(q_full, q_cnt & 1);
          ++q_cnt;
          for (int i = 0; i < 2; ++i) {
            const uint32_t it = base + 2 * i, slot = it % C::kSlots, ph = (it / C::kSlots) & 1;
            mbar_wait(&kv_full[slot], ph);
            tc_fence_after();
            issue_s_q(0, i, slot);
            mma_commit(&s_full[i]);
            release(slot);
          }
          if (g.n_kv == 2) mma_commit(q_empty);
          for (int j = 0; j < g.n_kv; ++j) {
            const int i = j & 1;
            const uint32_t it_v = base + 2 * j + 1, slot_v = it_v % C::kSlots, ph_v = (it_v / C::kSlots) & 1;
            const uint32_t par = (i ? cnt_p1 : cnt_p0) & 1;
            cnt_p0 += (i == 0);
            cnt_p1 += (i != 0);
            mbar_wait(&p_half[2 * i], par);
            mbar_wait(&kv_full[slot_v], ph_v);
            if (j < 2) mbar_wait(&o_free[i], ((i ? cnt_it1 : cnt_it0) & 1) ^ 1);
            tc_fence_after();
            issue_pv_half(i, slot_v, 0, j >= 2);
            mbar_poll(&p_half[2 * i + 1], par);   // short and on the critical path: poll
            tc_fence_after();
            issue_pv_half(i, slot_v, 1, true);
            mma_commit(&o_done[i]);
            release(slot_v);
            if (j + 2 < g.n_kv) {
              const uint32_t it_k = base + 2 * (j + 2), slot_k = it_k % C::kSlots, ph_k = (it_k / C::kSlots) & 1;
              mbar_wait(&kv_full[slot_k], ph_k);
              tc_fence_after();
              issue_s_q(0, i, slot_k);
              mma_commit(&s_full[i]);
              release(slot_k);
              if (j + 3 == g.n_kv) mma_commit(q_empty);
            }
          }
          kv_it = base + 2 * g.n_kv;
          ++cnt_it0;
          ++cnt_it1;
        } else {
        if (g.n_q > 0) {
          mbar_wait(q_full, q_cnt & 1);
          ++q_cnt;
          const uint32_t slot = kv_it % C::kSlots, ph = (kv_it / C::kSlots) & 1;
          ++kv_it;
          mbar_wait(&kv_full[slot], ph);
          tc_fence_after();
          for (int i = 0; i < g.n_q; ++i) {
            issue_s(i, slot);
            mma_commit(&s_full[i]);
          }
          release(slot);
          if (g.n_kv == 1) mma_commit(q_empty);
        }
        for (int j = 0; j < g.n_kv; ++j) {
          const uint32_t slot_v = kv_it % C::kSlots, ph_v = (kv_it / C::kSlots) & 1;
          ++kv_it;
          const bool has_next = (j + 1 < g.n_kv);
          uint32_t slot_k = 0, ph_k = 0;
          if (has_next) {
            slot_k = kv_it % C::kSlots;
            ph_k = (kv_it / C::kSlots) & 1;
            ++kv_it;
          }
          for (int i = 0; i < g.n_q; ++i) {
            const uint32_t par = (i ? cnt_p1 : cnt_p0) & 1;
            cnt_p0 += (i == 0);
            cnt_p1 += (i != 0);
            mbar_wait(&p_half[2 * i], par);
            if (i == 0) mbar_wait(&kv_full[slot_v], ph_v);
            if (j == 0) mbar_wait(&o_free[i], ((i ? cnt_it1 : cnt_it0) & 1) ^ 1);
            tc_fence_after();
            issue_pv_half(i, slot_v, 0, j > 0);
            mbar_poll(&p_half[2 * i + 1], par);   // short and on the critical path: poll
            tc_fence_after();
            issue_pv_half(i, slot_v, 1, true);
            mma_commit(&o_done[i]);
            if (i == g.n_q - 1) release(slot_v);
            if (has_next) {
              if (i == 0) {
                mbar_wait(&kv_full[slot_k], ph_k);
                tc_fence_after();
              }
              issue_s(i, slot_k);
              mma_commit(&s_full[i]);
              if (i == g.n_q - 1) {
                release(slot_k);
                if (j + 2 == g.n_kv) mma_commit(q_empty);
              }
            }
          }
        }
        cnt_it0 += (g.n_q >= 1);
        cnt_it1 += (g.n_q >= 2);
        }
        // K/V tiles only the cluster partner needs (it sees more chunk frames, or this CTA has no query rows)
        for (int e = 2 * g.n_kv; e < 2 * g.n_pipe; ++e) {
          const uint32_t slot = kv_it % C::kSlots, ph = (kv_it / C::kSlots) & 1;
          ++kv_it;
          mbar_wait(&kv_full[slot], ph);
          release(slot);
        }
      }
    }
  } else if (p.copy.n_sess > 0) {
    // ===================================================================== warps 2-3: KV append of a fused chunk step
    // The append writes cache slots this launch's attention never reads (R5); it is HBM-bound and the attention is not,
    // so it costs the step nothing when it runs here, under the attention.
    append_by_workers(p.copy, (int64_t)blockIdx.x * 64 + (threadIdx.x - 64), (int64_t)gridDim.x * 64);
  }
  } else {
    setmaxnreg_inc<kRegsSoftmax>();
    // ===================================================================== softmax + epilogue, one thread per query row
    const int wg = (warp - 4) >> 2;                       // query tile handled by this warpgroup
    const int row_in_tile = (warp & 3) * 32 + lane;
    const uint32_t lane_sel = (uint32_t)((warp & 3) * 32) << 16;
    const uint32_t taddr_s = tmem_base + lane_sel + wg * 128;
    const uint32_t taddr_o = tmem_base + lane_sel + 256 + wg * D;
    const float c = p.scale_log2;
    const float thr = kRescaleThresholdLog2 / c;
    uint32_t cnt_s = 0, cnt_pv = 0;
    uint32_t cnt_pv_other = 0;                            // PV groups committed so far on the OTHER tile slot
    for (uint32_t k_item = 0;; ++k_item) {
      const int idx = next_cluster_item(p, k_item, false);
      if (idx < 0) break;
      const ItemGeom g = decode_item(p, idx, cta_rank);
      if (!g.split && wg >= g.n_q) {
        if (g.n_q == 1) cnt_pv_other += g.n_kv;           // warpgroup 1 sits out a lone tile that runs on slot 0 alone
        continue;
      }
      // a split lone tile: both warpgroups work on the SAME 128 query rows, this one on KV tiles wg, wg+2, ...
      const int j0 = g.split ? wg : 0, dj = g.split ? 2 : 1;
      const int first_row = g.r0 + (g.split ? 0 : 128 * wg);
      const int row = first_row + row_in_tile;
      const int lim_row = min(g.C, (min(row, g.C - 1) / p.T + 1) * p.T);   // chunk keys visible to this row
      const int lim_min = min(g.C, (first_row / p.T + 1) * p.T);           // ... to the tile's first row
      // -1e30 rather than -inf: a split tile's first KV tile may hold no visible key for a row (all scores -inf);
      // (-inf) - (-1e30) = -inf gives p = 0 where (-inf) - (-inf) would give NaN
      float m = -1e30f, l = 0.f;
      for (int j = j0; j < g.n_kv; j += dj) {
        mbar_wait(&s_full[wg], cnt_s & 1);
        ++cnt_s;
        tc_fence_after();
        uint32_t s[128];
        tmem_ld32(taddr_s + 0, s + 0);
        tmem_ld32(taddr_s + 32, s + 32);
        tmem_ld32(taddr_s + 64, s + 64);
        tmem_ld32(taddr_s + 96, s + 96);
        tmem_ld_wait();
        // ---- mask (rare path)
        int lo = 0, hi = 128;
        bool need_mask;
        if (j < g.n_prior) {
          if (j == 0) lo = g.x_begin - (g.t0 << 7);
          if (j == g.n_prior - 1) hi = g.x_end - ((g.t0 + j) << 7);
          need_mask = (lo > 0) || (hi < 128);
        } else {
          const int base = (j - g.n_prior) << 7;
          need_mask = base + 128 > lim_min;
          hi = max(0, min(128, lim_row - base));
        }
        if (need_mask) {
#pragma unroll
          for (int k = 0; k < 128; ++k)
            if (k < lo || k >= hi) s[k] = 0xff800000u;   // -inf
        }
        // ---- row max (3-input FMNMX: two new values per instruction)
        float mx0 = __uint_as_float(s[0]), mx1 = __uint_as_float(s[1]), mx2 = __uint_as_float(s[2]), mx3 = __uint_as_float(s[3]);
#pragma unroll
        for (int k = 4; k < 124; k += 8) {
          mx0 = max3(mx0, __uint_as_float(s[k + 0]), __uint_as_float(s[k + 1]));
          mx1 = max3(mx1, __uint_as_float(s[k + 2]), __uint_as_float(s[k + 3]));
          mx2 = max3(mx2, __uint_as_float(s[k + 4]), __uint_as_float(s[k + 5]));
          mx3 = max3(mx3, __uint_as_float(s[k + 6]), __uint_as_float(s[k + 7]));
        }
        mx0 = max3(mx0, __uint_as_float(s[124]), __uint_as_float(s[125]));
        mx1 = max3(mx1, __uint_as_float(s[126]), __uint_as_float(s[127]));
        const float mx = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3));
        if (j == j0) {
          m = fmaxf(mx, m);   // first tile of the row: nothing accumulated yet, no rescale
        } else {
          const bool need = mx > m + thr;
          if (__any_sync(0xffffffffu, need)) {
            // rescale this warp's rows of O in TMEM: needs PV(j-1) of this tile complete
            const float m_new = fmaxf(m, mx);
            const float f = ex2_approx((m - m_new) * c);
            l *= f;
            m = m_new;
            mbar_wait(&o_done[wg], (cnt_pv - 1) & 1);
            tc_fence_after();
#pragma unroll
            for (int cc = 0; cc < D; cc += 32) {
              uint32_t o[32];
              tmem_ld32(taddr_o + cc, o);
              tmem_ld_wait();
#pragma unroll
              for (int k = 0; k < 32; k += 2) {
                float a0, a1;
                mul2_bcast(a0, a1, __uint_as_float(o[k]), __uint_as_float(o[k + 1]), f);
                o[k] = __float_as_uint(a0);
                o[k + 1] = __float_as_uint(a1);
              }
              tmem_st32(taddr_o + cc, o);
            }
          }
        }
        // ---- p = exp2(s*c - m*c); row sum; bf16 P back into TMEM (aliases the first 64 columns of S)
        const float neg_mc = -m * c;
        float l0 = 0.f, l1 = 0.f, l2 = 0.f, l3 = 0.f;
#pragma unroll
        for (int cc = 0; cc < 128; cc += 32) {
          uint32_t pk[16];
#pragma unroll
          for (int k = 0; k < 32; k += 4) {
            float x0, x1, x2, x3;
            fma2_bcast(x0, x1, __uint_as_float(s[cc + k]), __uint_as_float(s[cc + k + 1]), c, neg_mc);
            fma2_bcast(x2, x3, __uint_as_float(s[cc + k + 2]), __uint_as_float(s[cc + k + 3]), c, neg_mc);
            float p0, p1, p2, p3;
            {
              const int pj = k >> 1;   // index of (x0, x1) among the 16 pairs of this 32-column chunk
              if (((pj + 1) * kPolyPairs) / 16 != (pj * kPolyPairs) / 16) exp2_poly_pair(x0, x1, p0, p1);
              else { p0 = ex2_approx(x0); p1 = ex2_approx(x1); }
              if (((pj + 2) * kPolyPairs) / 16 != ((pj + 1) * kPolyPairs) / 16) exp2_poly_pair(x2, x3, p2, p3);
              else { p2 = ex2_approx(x2); p3 = ex2_approx(x3); }
            }
            add2(l0, l1, p0, p1);
            add2(l2, l3, p2, p3);
            pk[k >> 1] = pack_bf16x2(p0, p1);
            pk[(k >> 1) + 1] = pack_bf16x2(p2, p3);
          }
          tmem_st16(taddr_s + (cc >> 1), pk);
          if (cc & 32) {   // a 64-key half of P is stored: hand it to the MMA warp
            tmem_st_wait();
            tc_fence_before();
            mbar_arrive(&p_half[2 * wg + (cc >> 6)]);
          }
        }
        l += (l0 + l1) + (l2 + l3);
        ++cnt_pv;
      }
      const bool store = row < g.C;
      uint16_t* orow = p.out + ((size_t)(g.q_off + row) * p.H + g.head) * D;
      if (!g.split) {
        // ---- epilogue: O / l -> bf16 -> global
        if (g.n_q == 2) cnt_pv_other += g.n_kv;
        mbar_wait(&o_done[wg], (cnt_pv - 1) & 1);
        tc_fence_after();
        const float inv_l = 1.0f / l;
#pragma unroll
        for (int cc = 0; cc < D; cc += 32) {
          uint32_t o[32];
          tmem_ld32(taddr_o + cc, o);
          tmem_ld_wait();
          if (store) {
#pragma unroll
            for (int k = 0; k < 32; k += 16) {   // 16 bf16 = one full 32-byte sector per lane and store (st.global.v8:
              uint32_t w[8];                     // -1 % SM cycles per launch against 128-bit stores of half sectors)
#pragma unroll
              for (int t = 0; t < 8; ++t)
                w[t] = pack_bf16x2(__uint_as_float(o[k + 2 * t]) * inv_l, __uint_as_float(o[k + 2 * t + 1]) * inv_l);
              st_global_v8(orow + cc + k, w[0], w[1], w[2], w[3], w[4], w[5], w[6], w[7]);
            }
          }
        }
        tc_fence_before();
        mbar_arrive_n(&o_free[wg], 2);
        if (p.lse != nullptr && store)
          p.lse[(size_t)(g.q_off + row) * p.H + g.head] = (m * c + log2f(l)) * 0.6931471805599453f;
      } else {
        // ---- epilogue of a split lone tile: merge the two partial softmax states of every row.  The two threads of
        //      a row swap (m, l) through smem; each then reads BOTH partial O rows from TMEM (same lanes) for its half
        //      of the D columns:  O = (a_own O_own + a_oth O_oth) / (a_own l_own + a_oth l_oth),  a = 2^((m - m_tot) c)
        cnt_pv_other += (uint32_t)((g.n_kv - (wg ^ 1) + 1) >> 1);
        const int bar_id = 1 + (warp & 3);
        xchg[wg * 128 + row_in_tile] = make_float2(m, l);
        named_bar_sync(bar_id, 64);
        const float2 oth = xchg[(wg ^ 1) * 128 + row_in_tile];
        named_bar_sync(bar_id, 64);                       // both reads are done before the next split item writes
        const float m_tot = fmaxf(m, oth.x);
        const float a_own = ex2_approx((m - m_tot) * c), a_oth = ex2_approx((oth.x - m_tot) * c);
        const float l_tot = a_own * l + a_oth * oth.y;
        const float inv_l = 1.0f / l_tot;
        const float w_own = a_own * inv_l, w_oth = a_oth * inv_l;
        mbar_wait(&o_done[wg], (cnt_pv - 1) & 1);
        mbar_wait(&o_done[wg ^ 1], (cnt_pv_other - 1) & 1);
        tc_fence_after();
        const int col0 = wg * (D / 2);
        const uint32_t taddr_o_other = tmem_base + lane_sel + 256 + (wg ^ 1) * D;
#pragma unroll
        for (int cc = 0; cc < D / 2; cc += 32) {
          uint32_t o[32], q[32];
          tmem_ld32(taddr_o + col0 + cc, o);
          tmem_ld32(taddr_o_other + col0 + cc, q);
          tmem_ld_wait();
          if (store) {
#pragma unroll
            for (int k = 0; k < 32; k += 16) {
              uint32_t r[8];
#pragma unroll
              for (int t = 0; t < 8; ++t)
                r[t] = pack_bf16x2(__uint_as_float(o[k + 2 * t]) * w_own + __uint_as_float(q[k + 2 * t]) * w_oth,
                                   __uint_as_float(o[k + 2 * t + 1]) * w_own + __uint_as_float(q[k + 2 * t + 1]) * w_oth);
              st_global_v8(orow + col0 + cc + k, r[0], r[1], r[2], r[3], r[4], r[5], r[6], r[7]);
            }
          }
        }
        tc_fence_before();
        mbar_arrive(&o_free[0]);
        mbar_arrive(&o_free[1]);
        if (p.lse != nullptr && store && wg == 0)
          p.lse[(size_t)(g.q_off + row) * p.H + g.head] = (m_tot * c + log2f(l_tot)) * 0.6931471805599453f;
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  cluster_sync_all();   // no CTA exits while its partner may still multicast into it or arrive on its barriers
  if (warp == 1) tmem_dealloc(tmem_base, kTmemCols);
  if (p.clock_probe != nullptr && blockIdx.x == 0 && threadIdx.x == 96) {
    unsigned long long ns1;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(ns1));
    const unsigned long long* probe_smem = reinterpret_cast<const unsigned long long*>(tmem_ptr + 4);
    p.clock_probe[0] += (unsigned long long)clock64() - probe_smem[0];
    p.clock_probe[1] += ns1 - probe_smem[1];
  }
  // every role of both CTAs has read the ring's last entry: clear it for the next launch on this block
  if (cta_rank == 0 && threadIdx.x >= 64 && threadIdx.x < 64 + kFeedRing)
    p.feed[(size_t)(blockIdx.x >> 1) * kFeedRing + (threadIdx.x - 64)] = 0ull;
}

int attention_smem_bytes(int head_dim) { return head_dim == 128 ? Cfg<128>::kSmemBytes : Cfg<64>::kSmemBytes; }

// The dynamic shared memory limit is an attribute of the function on the CURRENT device: set once per device.
template <int D>
static cudaError_t configure_once() {
  static std::mutex mu;
  static bool configured[64] = {};
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  std::lock_guard<std::mutex> lock(mu);
  if (dev < 0 || dev >= 64 || !configured[dev]) {
    e = cudaFuncSetAttribute(chunk_attention_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg<D>::kSmemBytes);
    if (e != cudaSuccess) return e;
    if (dev >= 0 && dev < 64) configured[dev] = true;
  }
  return cudaSuccess;
}

cudaError_t attention_configure(int head_dim) { return head_dim == 128 ? configure_once<128>() : configure_once<64>(); }

template <int D>
static cudaError_t launch_clustered(const AttnParams& p, int grid, cudaStream_t stream) {
  cudaError_t e = configure_once<D>();
  if (e != cudaSuccess) return e;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)grid, 1, 1);
  cfg.blockDim = dim3(kThreads, 1, 1);
  cfg.dynamicSmemBytes = Cfg<D>::kSmemBytes;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = 2;   // CTA pairs: K/V tiles of a shared (session, head) are loaded once per pair
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, chunk_attention_kernel<D>, p);
}

// grid must be even: CTAs 2c and 2c+1 form cluster c and walk item lists of equal length.
cudaError_t launch_attention(const AttnParams& p, int head_dim, int grid, cudaStream_t stream) {
  if (grid <= 0 || (grid & 1)) return cudaErrorInvalidValue;
  return head_dim == 128 ? launch_clustered<128>(p, grid, stream) : launch_clustered<64>(p, grid, stream);
}

}  // namespace tc
