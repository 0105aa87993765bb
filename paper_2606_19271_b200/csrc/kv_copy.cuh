// Device helpers shared by the stand-alone KV append / gather kernels (kv_copy.cu) and by the idle warps of the
// attention kernel, which perform the append of a fused chunk step (attention_sm100.cu).
#pragma once
#include "internal.h"

namespace tc {

__device__ __forceinline__ uint4 ld_stream(const void* p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}

// Byte offset inside the slab (relative to the layer's K or V block of the page) of 16-byte element `e`
// of a session, where e indexes [row][H][D/8] and row is relative to x0.
__device__ __forceinline__ int64_t paged_offset(const CopyParams& p, const CopySess& s, const int32_t* pt, int64_t e,
                                                int vec_per_head, int vec_per_row) {
  const int row = (int)(e / vec_per_row);
  const int rem = (int)(e - (int64_t)row * vec_per_row);
  const int h = rem / vec_per_head;
  const int v = rem - h * vec_per_head;
  const int x = s.x0 + row;
  const int page = pt[x >> p.log2_B];
  const int slot = x & (p.B - 1);
  return (int64_t)page * p.page_stride + ((int64_t)h * p.B + slot) * (p.D * 2) + v * 16;
}

// The whole append of a batch done by `n_workers` threads that are otherwise idle (worker = this thread's index):
// consecutive workers take consecutive 16-byte elements, so a warp moves 512 contiguous source bytes per step.
__device__ __forceinline__ void append_by_workers(const CopyParams& p, int64_t worker, int64_t n_workers) {
  const int vec_per_head = p.D / 8;
  const int vec_per_row = p.H * vec_per_head;
  uint8_t* dst_k = p.slab + p.layer_k_off;
  uint8_t* dst_v = p.slab + p.layer_v_off;
  for (int si = 0; si < p.n_sess; ++si) {
    const CopySess s = p.sess[si];
    const int32_t* pt = p.page_tables + s.pt_off;
    const int64_t n_copy = (int64_t)s.n_tok * vec_per_row;
    const int64_t n_all = (int64_t)(s.n_tok + s.n_zero) * vec_per_row;
    const uint8_t* src_k = p.src_k + (int64_t)s.tok_off * vec_per_row * 16;
    const uint8_t* src_v = p.src_v + (int64_t)s.tok_off * vec_per_row * 16;
    for (int64_t e0 = worker; e0 < n_all; e0 += 2 * n_workers) {
      const int64_t e1 = e0 + n_workers;
      uint4 k0 = make_uint4(0, 0, 0, 0), v0 = k0, k1 = k0, v1 = k0;   // zero-fill of the dead tail of the last page
      if (e0 < n_copy) {
        k0 = ld_stream(src_k + e0 * 16);
        v0 = ld_stream(src_v + e0 * 16);
      }
      if (e1 < n_copy) {
        k1 = ld_stream(src_k + e1 * 16);
        v1 = ld_stream(src_v + e1 * 16);
      }
      const int64_t off0 = paged_offset(p, s, pt, e0, vec_per_head, vec_per_row);
      *reinterpret_cast<uint4*>(dst_k + off0) = k0;
      *reinterpret_cast<uint4*>(dst_v + off0) = v0;
      if (e1 < n_all) {
        const int64_t off1 = paged_offset(p, s, pt, e1, vec_per_head, vec_per_row);
        *reinterpret_cast<uint4*>(dst_k + off1) = k1;
        *reinterpret_cast<uint4*>(dst_v + off1) = v1;
      }
    }
  }
}

}  // namespace tc
