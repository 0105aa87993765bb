// Coalesced chunk attention for sm_100a, "Q in TMEM" variant (step a2 of SURVEY.md §8(a); PAPER.md:66 (iii)).
//
// Same boundary, work list and K/V page gather as attention_sm100.cu; what differs is the pipeline inside a CTA.  There a
// CTA holds TWO query tiles, each with one score buffer and one accumulator in TMEM (2 x (S 128 + O 128) = 512 columns):
// S = Q K^T reads both operands from shared memory (8 KB per instruction = the SM's whole 128 B/clk: 86 clk instead of 64),
// and S(j+1) of a tile cannot be issued before P(j) V has read P(j) out of the buffer S(j+1) lands in, so every KV step
// walks the closed chain S -> softmax -> P -> P V -> S.
// Here a CTA holds ONE query tile, resident IN TMEM as the A operand of S = Q K^T (64 columns of packed bf16 pairs: the
// instruction then reads only the K tile from shared memory, 4 KB, at the tensor rate), TWO score buffers and one
// accumulator: S0 [0,128) | S1 [128,256) | Q [256,320) | O [384,512).
//   MMA issue order   S(0) S(1) | PV(0) S(2) | PV(1) S(3) | ...          (S(j+2) lands in the buffer PV(j) has read)
//   softmax           warpgroup 0 takes the even KV tiles (buffer 0), warpgroup 1 the odd ones (buffer 1), same 128 rows
// so a score tile is being exponentiated while the next one is being computed: the chain is open by one tile.  Shared
// memory traffic per 128 x 128 tile and KV step: K + V written by TMA 64 KB, K read 32 KB, V read 32 KB = 128 KB - what the
// two-tile kernel moves (a single-tile kernel with Q in shared memory moves 160 KB and was measured slower).
//
// Q reaches TMEM through the softmax threads: TMA brings the tile into a staging buffer (128-byte swizzle), each thread
// reads half of its own row (the A operand layout in TMEM is lane = row, column c = elements 2c, 2c+1: the row's own 32-bit
// words) and stores it with tcgen05.st; the staging buffer is free for the next item's tile right away.
//
// One accumulator for both warpgroups means ONE running maximum per row, in KV-tile order.  The owner of tile j takes
// m(j-1) from a shared-memory word the owner of tile j-1 published right after its row maximum, decides m(j) = m(j-1)
// unless its own maximum exceeds it by more than the lazy threshold, publishes m(j), and - in that rare case only -
// rescales the row of O in TMEM between PV(j-1) and PV(j) (PV(j) cannot start: it needs this thread's P).  Each warpgroup
// keeps the row sum of its own tiles with the reference maximum it is expressed in; the two partial sums meet in the
// epilogue.  This is the sequential online softmax over tiles 0, 1, 2, ... exactly, for any input.
//
// K/V tiles travel through the smem ring in CONSUMPTION order (K0 K1 V0 K2 V1 K3 ...); the order is a function of the
// cluster item's tile count alone, so that the two CTAs of a cluster (multicast halves, attention_sm100.cu) stay on the same
// ring position.
#include <mutex>

#include "attention_common.cuh"
#include "internal.h"
#include "kv_copy.cuh"
#include "ptx.cuh"

namespace tc {
namespace qt {

template <int D>
struct Cfg {
  static constexpr int kTileBytes = 128 * D * 2;        // one [128 x D] bf16 tile
  static constexpr int kDBlocks = D / 64;               // 64-column (128-byte) swizzle blocks per tile
  static constexpr int kBlockBytes = 128 * 128;         // one [128 rows x 128 B] swizzle block
  static constexpr int kSlots = (D == 128) ? 6 : 10;
  static constexpr int kSmemQ = kTileBytes;             // staging only: the operand lives in TMEM
  static constexpr int kSmemKV = kSlots * kTileBytes;
  static constexpr int kPubBytes = 128 * 8;             // per row: (m of the latest KV tile, its sequence number)
  static constexpr int kSumBytes = 2 * 128 * 4;         // per warpgroup and row: partial row sum (epilogue)
  static constexpr int kNumBars = 2 * kSlots + 16;
  static constexpr int kSmemBytes = kSmemQ + kSmemKV + kPubBytes + kSumBytes + kNumBars * 8 + 16 + 16;
  static constexpr int kTmemQ = 256;                    // first TMEM column of the Q operand (D / 2 columns)
  static constexpr int kTmemO = 384;                    // first TMEM column of the accumulator (D columns)
};
static_assert(Cfg<128>::kSmemBytes <= 232448, "shared memory per CTA");

struct ItemGeom {
  int sess, head, r0, C, q_off, pt_off;
  int x_begin, x_end, t0, n_prior, n_kv;
  int n_pipe;   // KV tiles flowing through the smem ring for this item (>= n_kv: the cluster partner may see more)
  bool mc;      // K/V tiles are loaded half by this CTA, half by the cluster partner, multicast to both
};

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
    g.n_kv = 0;
  } else {
    const int last_row = min(s.C, g.r0 + 128) - 1;
    const int kv_hi = min(s.C, (last_row / p.T + 1) * p.T);   // chunk keys visible to the item's last row
    g.n_kv = g.n_prior + ((kv_hi + 127) >> 7);
  }
  return g;
}

template <int D>
__global__ void __launch_bounds__(kThreads, 1) chunk_attention_qt_kernel(const __grid_constant__ AttnParams p) {
  using C = Cfg<D>;
  extern __shared__ __align__(1024) uint8_t smem[];   // swizzle-128B operands need 1024-byte alignment
  uint8_t* sQ = smem;
  uint8_t* sKV = smem + C::kSmemQ;
  unsigned long long* pub = reinterpret_cast<unsigned long long*>(sKV + C::kSmemKV);   // [row]: (seq << 32) | bits of m
  float* lsum = reinterpret_cast<float*>(sKV + C::kSmemKV + C::kPubBytes);             // [warpgroup][row]
  uint64_t* bars = reinterpret_cast<uint64_t*>(sKV + C::kSmemKV + C::kPubBytes + C::kSumBytes);
  uint64_t* kv_full = bars;
  uint64_t* kv_empty = bars + C::kSlots;
  uint64_t* q_full = bars + 2 * C::kSlots;   // TMA -> softmax threads: the Q tile is in the staging buffer
  uint64_t* q_read = q_full + 1;             // softmax threads -> TMA: the staging buffer has been read (256 arrivals)
  uint64_t* qt_full = q_full + 2;            // softmax threads -> MMA: Q is in TMEM (256 arrivals)
  uint64_t* qt_free = q_full + 3;            // MMA -> softmax threads: the item's last S = Q K^T has completed
  uint64_t* s_full = q_full + 4;             // [2]    score buffer b holds S of its current tile
  uint64_t* p_half = q_full + 6;             // [2][2] P in buffer b, keys [64h, 64h+64), written by warpgroup b
  uint64_t* pv_done = q_full + 10;           // [2]    O += P V of the tile in buffer b has completed
  uint64_t* o_final = q_full + 12;           //        the item's last P V has completed
  uint64_t* o_free = q_full + 13;            //        both warpgroups have read O
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
    mbar_init(q_read, 256);
    mbar_init(qt_full, 256);
    mbar_init(qt_free, 1);
    for (int i = 0; i < 2; ++i) {
      mbar_init(&s_full[i], 1);
      mbar_init(&p_half[2 * i], 128);
      mbar_init(&p_half[2 * i + 1], 128);
      mbar_init(&pv_done[i], 1);
    }
    mbar_init(o_final, 1);
    mbar_init(o_free, 256);
    fence_mbar_init();
    tma_prefetch_desc(&p.map_k);
    tma_prefetch_desc(&p.map_v);
  }
  if (threadIdx.x >= 128 && threadIdx.x < 256) pub[threadIdx.x - 128] = 0ull;   // sequence numbers start at 1
  if (warp == 1) tmem_alloc(tmem_ptr, kTmemCols);
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();   // the partner's barriers are initialised before any multicast load or commit reaches them
  tc_fence_after();
  const uint32_t cta_rank = cluster_ctarank();
  const uint32_t tmem_base = *tmem_ptr;
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
          if (g.n_kv > 0) {
            // the staging buffer is free as soon as the previous item's tile has been copied to TMEM
            mbar_wait_long(q_read, (q_cnt & 1) ^ 1);
            ++q_cnt;
            mbar_arrive_expect_tx(q_full, C::kTileBytes);
            for (int b = 0; b < C::kDBlocks; ++b) tma_load_3d(sQ + b * C::kBlockBytes, mq, 64 * b, g.head, g.r0, q_full);
          }
          // tile t of the item (kv = 0: K, 1: V) into the next ring slot
          auto load_tile = [&](int t, int kv) {
            const uint32_t slot = kv_it % C::kSlots;
            const uint32_t ph = (kv_it / C::kSlots) & 1;
            ++kv_it;
            mbar_wait_long(&kv_empty[slot], ph ^ 1);
            if (!g.mc && t >= g.n_kv) {
              // a tile of the partner's unrelated item: nothing to load, but the slot is cycled so that both CTAs
              // of the cluster stay on the same ring position (multicast needs equal smem offsets)
              mbar_arrive(&kv_full[slot]);
              return;
            }
            mbar_arrive_expect_tx(&kv_full[slot], C::kTileBytes);   // own boxes + (multicast) the partner's
            uint8_t* dst = sKV + slot * C::kTileBytes;
            for (int sx = 0; sx < n_sub; ++sx) {
              if (g.mc && (uint32_t)(sx & 1) != cta_rank) continue;   // the partner loads and multicasts this box
              uint8_t* d = dst + sx * sb * 128;
              if (t < g.n_prior) {
                const CUtensorMap* mc = kv ? &p.map_v : &p.map_k;
                const int x = ((g.t0 + t) << 7) + sx * sb;            // page-table coordinate of the box
                // Boxes past the last cached token re-read the last page that HOLDS a cached token (masked): its tail is
                // real data or the append's zero fill, never a page whose bytes in this layer are not written yet.
                const int page = pt[min(x >> p.log2_B, (g.x_end - 1) >> p.log2_B)];
                const int tok = x & (p.B - 1);
                for (int b = 0; b < C::kDBlocks; ++b) {
                  if (g.mc) tma_load_4d_mc(d + b * C::kBlockBytes, mc, 64 * b, tok, g.head, page, &kv_full[slot], 3);
                  else tma_load_4d(d + b * C::kBlockBytes, mc, 64 * b, tok, g.head, page, &kv_full[slot]);
                }
              } else {
                const CUtensorMap* mc = kv ? mvn : mkn;
                const int row = ((t - g.n_prior) << 7) + sx * sb;
                for (int b = 0; b < C::kDBlocks; ++b) {
                  if (g.mc) tma_load_3d_mc(d + b * C::kBlockBytes, mc, 64 * b, g.head, row, &kv_full[slot], 3);
                  else tma_load_3d(d + b * C::kBlockBytes, mc, 64 * b, g.head, row, &kv_full[slot]);
                }
              }
            }
          };
          for (int t = 0; t < min(2, g.n_pipe); ++t) load_tile(t, 0);
          for (int j = 0; j < g.n_pipe; ++j) {
            load_tile(j, 1);
            if (j + 2 < g.n_pipe) load_tile(j + 2, 0);
          }
        }
      }
    } else if (warp == 1) {
      // ===================================================================== MMA issuer
      if (elect_one()) {
        constexpr uint32_t idesc_s = make_idesc_bf16(128, 128, 0, 0);
        constexpr uint32_t idesc_pv = make_idesc_bf16(128, D, 0, 1);
        const uint32_t sKV_addr = smem_u32(sKV);
        const uint32_t tmem_q = tmem_base + C::kTmemQ;
        const uint32_t tmem_o = tmem_base + C::kTmemO;
        uint32_t kv_it = 0, n_items = 0;
        uint32_t use0 = 0, use1 = 0;   // tiles that have gone through score buffer 0 / 1 so far (phases of p_half)
        auto next_slot = [&](uint32_t& slot) {
          slot = kv_it % C::kSlots;
          const uint32_t ph = (kv_it / C::kSlots) & 1;
          ++kv_it;
          mbar_wait(&kv_full[slot], ph);
        };
        // hand a K/V slot back once every MMA issued so far has read it - always to BOTH CTAs of the cluster
        auto release = [&](uint32_t slot) { mma_commit_mc(&kv_empty[slot], 3); };
        // S of buffer `buf` = Q (TMEM, lane = row, 8 columns per 16-element K step) x (K tile in ring slot `slot`)^T
        auto issue_s = [&](uint32_t buf, uint32_t slot) {
          const uint32_t b = sKV_addr + slot * C::kTileBytes;
#pragma unroll
          for (int kk = 0; kk < D / 16; ++kk) {
            const uint32_t off = (kk >> 2) * C::kBlockBytes + (kk & 3) * 32;
            mma_ts(tmem_base + buf * 128, tmem_q + kk * 8, make_smem_desc_sw128(b + off, 16, 1024), idesc_s, kk > 0);
          }
        };
        // half h of O += P V: the 16-key steps 4h .. 4h+3 (keys [64h, 64h+64))
        auto issue_pv_half = [&](uint32_t buf, uint32_t slot, int h, bool acc) {
          const uint32_t b = sKV_addr + slot * C::kTileBytes;
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            const int kk = 4 * h + q;
            mma_ts(tmem_o, tmem_base + buf * 128 + kk * 8, make_smem_desc_sw128(b + kk * 2048, C::kBlockBytes, 1024), idesc_pv,
                   (acc || q > 0) ? 1u : 0u);
          }
        };
        for (uint32_t k_item = 0;; ++k_item) {
          const int idx = next_cluster_item(p, k_item, false);
          if (idx < 0) break;
          const ItemGeom g = decode_item(p, idx, cta_rank);
          if (g.n_kv > 0) mbar_wait(qt_full, n_items & 1);
          for (int t = 0; t < min(2, g.n_pipe); ++t) {
            uint32_t slot;
            next_slot(slot);
            if (t < g.n_kv) {
              tc_fence_after();
              issue_s((uint32_t)t, slot);
              mma_commit(&s_full[t]);
              if (t == g.n_kv - 1) mma_commit(qt_free);
            }
            release(slot);
          }
          for (int j = 0; j < g.n_pipe; ++j) {
            const uint32_t buf = (uint32_t)(j & 1);
            uint32_t slot;
            next_slot(slot);
            if (j < g.n_kv) {
              const uint32_t par = (buf ? use1 : use0) & 1;
              use0 += (buf == 0);
              use1 += (buf != 0);
              mbar_wait(&p_half[2 * buf], par);
              if (j == 0) mbar_wait(o_free, (n_items & 1) ^ 1);
              tc_fence_after();
              issue_pv_half(buf, slot, 0, j > 0);
              mbar_wait(&p_half[2 * buf + 1], par);
              tc_fence_after();
              issue_pv_half(buf, slot, 1, true);
              mma_commit(&pv_done[buf]);
              if (j == g.n_kv - 1) mma_commit(o_final);
            }
            release(slot);
            if (j + 2 < g.n_pipe) {
              next_slot(slot);
              if (j + 2 < g.n_kv) {
                tc_fence_after();
                issue_s(buf, slot);           // tile j + 2 lands in the buffer P V(j) has just read
                mma_commit(&s_full[buf]);
                if (j + 2 == g.n_kv - 1) mma_commit(qt_free);
              }
              release(slot);
            }
          }
          n_items += (g.n_kv > 0);
        }
      }
    } else if (p.copy.n_sess > 0) {
      // ===================================================================== warps 2-3: KV append of a fused chunk step
      append_by_workers(p.copy, (int64_t)blockIdx.x * 64 + (threadIdx.x - 64), (int64_t)gridDim.x * 64);
    }
  } else {
    setmaxnreg_inc<kRegsSoftmax>();
    // ===================================================================== softmax + epilogue, one thread per query row
    const int wg = (warp - 4) >> 2;                       // this warpgroup takes the item's KV tiles j = wg, wg + 2, ... (buffer wg)
    const int row_in_tile = (warp & 3) * 32 + lane;
    const uint32_t lane_sel = (uint32_t)((warp & 3) * 32) << 16;
    const uint32_t taddr_s = tmem_base + lane_sel + wg * 128;
    const uint32_t taddr_q = tmem_base + lane_sel + C::kTmemQ;
    const uint32_t taddr_o = tmem_base + lane_sel + C::kTmemO;
    const float c = p.scale_log2;
    const float thr = kRescaleThresholdLog2 / c;
    volatile unsigned long long* pub_row = pub + row_in_tile;
    const int bar_id = 1 + (warp & 3);
    uint32_t n_items = 0;
    uint32_t G0 = 0;                      // KV tiles of this CTA's earlier items (sequence numbers of the published maxima)
    uint32_t use_own = 0, use_oth = 0;    // tiles that have gone through this warpgroup's / the other score buffer so far
    for (uint32_t k_item = 0;; ++k_item) {
      const int idx = next_cluster_item(p, k_item, false);
      if (idx < 0) break;
      const ItemGeom g = decode_item(p, idx, cta_rank);
      if (g.n_kv == 0) continue;
      // ---- Q: staging buffer -> registers -> TMEM.  This warpgroup copies elements [64 wg, 64 wg + 64) of every row (with
      //      D = 64: [32 wg, 32 wg + 32)): D / 4 32-bit words per thread, 16-byte chunks un-swizzled (chunk ^ (row & 7)).
      mbar_wait(q_full, n_items & 1);
      {
        constexpr int kWords = D / 4;                                   // per thread
        uint32_t qw[kWords];
        const int e0 = wg * (D / 2);                                    // first element of this thread's part of the row
        const uint8_t* blk = sQ + (e0 >> 6) * C::kBlockBytes + row_in_tile * 128;
        const int chunk0 = (e0 & 63) >> 3;                              // first 16-byte chunk inside the 128-byte row segment
#pragma unroll
        for (int i = 0; i < kWords / 4; ++i) {
          const uint4 v = *reinterpret_cast<const uint4*>(blk + (((chunk0 + i) ^ (row_in_tile & 7)) << 4));
          qw[4 * i + 0] = v.x;
          qw[4 * i + 1] = v.y;
          qw[4 * i + 2] = v.z;
          qw[4 * i + 3] = v.w;
        }
        mbar_arrive(q_read);                                            // the staging buffer may be refilled
        mbar_wait(qt_free, (n_items & 1) ^ 1);                          // the previous item's last S has read the old Q
        tc_fence_after();
        if constexpr (D == 128) {
          tmem_st32(taddr_q + wg * 32, qw);
        } else {
          tmem_st16(taddr_q + wg * 16, qw);
        }
        tmem_st_wait();
        tc_fence_before();
        mbar_arrive(qt_full);
      }
      const int row = g.r0 + row_in_tile;
      const int lim_row = min(g.C, (min(row, g.C - 1) / p.T + 1) * p.T);   // chunk keys visible to this row
      const int lim_min = min(g.C, (g.r0 / p.T + 1) * p.T);                // ... to the tile's first row
      // l: sum of this warpgroup's p, expressed with reference maximum m_l.  -1e30 rather than -inf: a row's first tile
      // may hold no visible key (all scores -inf); (-inf) - (-1e30) = -inf gives p = 0 where (-inf) - (-inf) is NaN
      float l = 0.f, m_l = -1e30f, m = -1e30f;
      for (int j = wg; j < g.n_kv; j += 2) {
        mbar_wait(&s_full[wg], use_own & 1);
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
        // ---- the row's running maximum, in KV-tile order across both warpgroups
        const uint32_t seq = G0 + (uint32_t)j + 1;
        if (j == 0) {
          m = fmaxf(mx, -1e30f);   // first tile of the row: nothing accumulated yet, no rescale
          *pub_row = ((unsigned long long)seq << 32) | __float_as_uint(m);
        } else {
          unsigned long long w;
          do {
            w = *pub_row;
          } while ((uint32_t)(w >> 32) != seq - 1);
          const float m_prev = __uint_as_float((uint32_t)w);
          const bool need = mx > m_prev + thr;
          const bool any = __any_sync(0xffffffffu, need);
          m = any ? fmaxf(m_prev, mx) : m_prev;
          *pub_row = ((unsigned long long)seq << 32) | __float_as_uint(m);
          if (any) {
            // rescale this warp's rows of O in TMEM, between P V(j-1) (the other buffer's latest tile) and P V(j), which
            // waits for this thread's P
            const float f = ex2_approx((m_prev - m) * c);
            mbar_wait(&pv_done[wg ^ 1], (use_oth + (uint32_t)((j - 1) >> 1)) & 1);
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
        if (__any_sync(0xffffffffu, m != m_l)) {   // the reference maximum moved since this warpgroup's previous tile
          l *= ex2_approx((m_l - m) * c);
          m_l = m;
        }
        // ---- p = exp2(s*c - m*c); row sum; bf16 P back into TMEM (aliases the first 64 columns of the score buffer)
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
        ++use_own;
      }
      // ---- epilogue: the two partial row sums meet; each warpgroup writes half of the row's D columns
      const uint32_t seq_last = G0 + (uint32_t)g.n_kv;
      if (((g.n_kv - 1) & 1) != wg) {   // the other warpgroup owned the last tile: take the final maximum from it
        unsigned long long w;
        do {
          w = *pub_row;
        } while ((uint32_t)(w >> 32) != seq_last);
        m = __uint_as_float((uint32_t)w);
      }
      const float l_own = l * ex2_approx((m_l - m) * c);
      lsum[wg * 128 + row_in_tile] = l_own;
      named_bar_sync(bar_id, 64);
      const float l_tot = l_own + lsum[(wg ^ 1) * 128 + row_in_tile];
      named_bar_sync(bar_id, 64);                       // both reads are done before the next item writes
      const float inv_l = 1.0f / l_tot;
      const bool store = row < g.C;
      const int col0 = wg * (D / 2);
      uint16_t* orow = p.out + ((size_t)(g.q_off + row) * p.H + g.head) * D + col0;
      mbar_wait(o_final, n_items & 1);
      tc_fence_after();
#pragma unroll
      for (int cc = 0; cc < D / 2; cc += 32) {
        uint32_t o[32];
        tmem_ld32(taddr_o + col0 + cc, o);
        tmem_ld_wait();
        if (store) {
#pragma unroll
          for (int k = 0; k < 32; k += 16) {   // 16 bf16 = one full 32-byte sector per lane and store
            uint32_t w[8];
#pragma unroll
            for (int t = 0; t < 8; ++t)
              w[t] = pack_bf16x2(__uint_as_float(o[k + 2 * t]) * inv_l, __uint_as_float(o[k + 2 * t + 1]) * inv_l);
            st_global_v8(orow + cc + k, w[0], w[1], w[2], w[3], w[4], w[5], w[6], w[7]);
          }
        }
      }
      tc_fence_before();
      mbar_arrive(o_free);
      if (p.lse != nullptr && store && wg == 0)
        p.lse[(size_t)(g.q_off + row) * p.H + g.head] = (m * c + log2f(l_tot)) * 0.6931471805599453f;
      ++n_items;
      G0 += (uint32_t)g.n_kv;
      use_oth += (uint32_t)((g.n_kv + wg) >> 1);   // tiles of this item that went through the other buffer
    }
  }

  tc_fence_before();
  __syncthreads();
  cluster_sync_all();   // no CTA exits while its partner may still multicast into it or arrive on its barriers
  if (warp == 1) tmem_dealloc(tmem_base, kTmemCols);
  if (p.clock_probe != nullptr && blockIdx.x == 0 && threadIdx.x == 96) {
    unsigned long long ns1;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(ns1));
    p.clock_probe[0] += (unsigned long long)clock64() - probe_smem[0];
    p.clock_probe[1] += ns1 - probe_smem[1];
  }
  // every role of both CTAs has read the ring's last entry: clear it for the next launch on this block
  if (cta_rank == 0 && threadIdx.x >= 64 && threadIdx.x < 64 + kFeedRing)
    p.feed[(size_t)(blockIdx.x >> 1) * kFeedRing + (threadIdx.x - 64)] = 0ull;
}

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
    e = cudaFuncSetAttribute(chunk_attention_qt_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg<D>::kSmemBytes);
    if (e != cudaSuccess) return e;
    if (dev >= 0 && dev < 64) configured[dev] = true;
  }
  return cudaSuccess;
}

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
  return cudaLaunchKernelEx(&cfg, chunk_attention_qt_kernel<D>, p);
}

}  // namespace qt

cudaError_t attention_qt_configure(int head_dim) {
  return head_dim == 128 ? qt::configure_once<128>() : qt::configure_once<64>();
}

// grid must be even: CTAs 2c and 2c+1 form cluster c.
cudaError_t launch_attention_qt(const AttnParams& p, int head_dim, int grid, cudaStream_t stream) {
  if (grid <= 0 || (grid & 1)) return cudaErrorInvalidValue;
  return head_dim == 128 ? qt::launch_clustered<128>(p, grid, stream) : qt::launch_clustered<64>(p, grid, stream);
}

}  // namespace tc
