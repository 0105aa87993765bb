// Pieces shared by the attention kernels: thread / register budget, software exp2, the dynamic work-item feed.
#pragma once
#include "internal.h"
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
    asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(slot), "l"(v) : "memory");
    if (idx < 0 && atomicAdd(p.feed_hdr + 1, 1) == (int)(gridDim.x >> 1) - 1) {
      p.feed_hdr[1] = 0;
      p.feed_hdr[0] = 0;
    }
    return idx;
  }
  unsigned long long v;
  do {
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(slot) : "memory");
  } while ((uint32_t)(v >> 32) != k + 1);
  return (int)(uint32_t)v - 1;
}

}  // namespace tc
