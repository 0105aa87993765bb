// KV append (step a3, PAPER.md:66 (iii) "writes ... updated states back") and logical gather (parity
// introspection).  Both are pure byte movers: 128-bit vectorised, coalesced on the packed side
// (contiguous [tokens][H][D]) and in 2*D-byte runs on the paged side ([page][layer][K|V][H][B][D]).
// HBM-bound: algorithmic bytes = read + write of K and V = 4 * tokens * H * D * 2.
#include "internal.h"
#include "kv_copy.cuh"

namespace tc {

constexpr int kCopyThreads = 256;
constexpr int kCopyUnroll = 4;

__global__ void __launch_bounds__(kCopyThreads) kv_append_kernel(const CopyParams p) {
  const CopySess s = p.sess[blockIdx.y];
  const int32_t* pt = p.page_tables + s.pt_off;
  const int vec_per_head = p.D / 8;
  const int vec_per_row = p.H * vec_per_head;
  const int64_t n_copy = (int64_t)s.n_tok * vec_per_row;
  const int64_t n_all = (int64_t)(s.n_tok + s.n_zero) * vec_per_row;
  const uint8_t* src_k = p.src_k + (int64_t)s.tok_off * vec_per_row * 16;
  const uint8_t* src_v = p.src_v + (int64_t)s.tok_off * vec_per_row * 16;
  uint8_t* dst_k = p.slab + p.layer_k_off;
  uint8_t* dst_v = p.slab + p.layer_v_off;
  const int64_t stride = (int64_t)gridDim.x * kCopyThreads;
  for (int64_t e0 = (int64_t)blockIdx.x * kCopyThreads + threadIdx.x; e0 < n_all; e0 += stride * kCopyUnroll) {
    uint4 k[kCopyUnroll], v[kCopyUnroll];
#pragma unroll
    for (int u = 0; u < kCopyUnroll; ++u) {
      const int64_t e = e0 + u * stride;
      if (e < n_copy) {
        k[u] = ld_stream(src_k + e * 16);
        v[u] = ld_stream(src_v + e * 16);
      } else {
        k[u] = make_uint4(0, 0, 0, 0);   // zero-fill of the dead tail of the session's last page
        v[u] = make_uint4(0, 0, 0, 0);
      }
    }
#pragma unroll
    for (int u = 0; u < kCopyUnroll; ++u) {
      const int64_t e = e0 + u * stride;
      if (e < n_all) {
        const int64_t off = paged_offset(p, s, pt, e, vec_per_head, vec_per_row);
        *reinterpret_cast<uint4*>(dst_k + off) = k[u];
        *reinterpret_cast<uint4*>(dst_v + off) = v[u];
      }
    }
  }
}

__global__ void __launch_bounds__(kCopyThreads) kv_gather_kernel(const CopyParams p) {
  const CopySess s = p.sess[blockIdx.y];
  const int32_t* pt = p.page_tables + s.pt_off;
  const int vec_per_head = p.D / 8;
  const int vec_per_row = p.H * vec_per_head;
  const int64_t n_copy = (int64_t)s.n_tok * vec_per_row;
  const uint8_t* src_k = p.slab + p.layer_k_off;
  const uint8_t* src_v = p.slab + p.layer_v_off;
  uint8_t* dst_k = p.dst_k + (int64_t)s.tok_off * vec_per_row * 16;
  uint8_t* dst_v = p.dst_v + (int64_t)s.tok_off * vec_per_row * 16;
  const int64_t stride = (int64_t)gridDim.x * kCopyThreads;
  for (int64_t e = (int64_t)blockIdx.x * kCopyThreads + threadIdx.x; e < n_copy; e += stride) {
    const int64_t off = paged_offset(p, s, pt, e, vec_per_head, vec_per_row);
    const uint4 k = *reinterpret_cast<const uint4*>(src_k + off);
    const uint4 v = *reinterpret_cast<const uint4*>(src_v + off);
    *reinterpret_cast<uint4*>(dst_k + e * 16) = k;
    *reinterpret_cast<uint4*>(dst_v + e * 16) = v;
  }
}

// Migration fetch (the TARGET worker fetches the state buffers from the source through one-sided GPU
// memory access).  blockIdx.y = page of the session (logical order), blockIdx.x strides over the page's 16-byte
// vectors; kPullUnroll independent 128-bit loads in flight per thread (the source may sit behind NVLink).  On one
// device it is HBM-bound: algorithmic bytes = 2 * n_pages * page bytes.
constexpr int kPullUnroll = 8;

__global__ void __launch_bounds__(kCopyThreads) page_pull_kernel(const PullParams p) {
  const int32_t sp = p.pairs[2 * blockIdx.y], dp = p.pairs[2 * blockIdx.y + 1];
  const uint8_t* src = p.src_slab + (int64_t)sp * p.page_stride;
  uint8_t* dst = p.dst_slab + (int64_t)dp * p.page_stride;
  const int stride = gridDim.x * kCopyThreads;
  for (int e0 = blockIdx.x * kCopyThreads + threadIdx.x; e0 < p.vec_per_page; e0 += stride * kPullUnroll) {
    uint4 r[kPullUnroll];
#pragma unroll
    for (int u = 0; u < kPullUnroll; ++u) {
      const int e = e0 + u * stride;
      if (e < p.vec_per_page) r[u] = ld_stream(src + (int64_t)e * 16);
    }
#pragma unroll
    for (int u = 0; u < kPullUnroll; ++u) {
      const int e = e0 + u * stride;
      if (e < p.vec_per_page) *reinterpret_cast<uint4*>(dst + (int64_t)e * 16) = r[u];
    }
  }
}

cudaError_t launch_page_pull(const PullParams& p, int sm_count, cudaStream_t stream) {
  const int want = (p.vec_per_page + kCopyThreads * kPullUnroll - 1) / (kCopyThreads * kPullUnroll);
  const int cap = (sm_count * 8 + p.n_pages - 1) / p.n_pages;   // 8 resident CTAs of 256 threads per SM
  const int gx = want < cap ? want : cap;
  page_pull_kernel<<<dim3((unsigned)(gx < 1 ? 1 : gx), (unsigned)p.n_pages, 1), kCopyThreads, 0, stream>>>(p);
  return cudaGetLastError();
}

// Descriptor upload without a copy engine.  Per-call schedule / descriptor blocks (tens of KB) are pulled from mapped
// pinned host memory by a few warps instead of a cudaMemcpyAsync: a DMA copy queues behind whatever the copy engine is
// already moving - a 201 MB resume on the side stream delayed a 2.45 ms step by 4.2 ms that way (bench.py `overlap`).
// ld.cv: system-memory lines are never served from a stale cache line (the host rewrites the staging ring).
constexpr int kUploadThreads = 64;
constexpr int kUploadUnroll = 4;

__global__ void __launch_bounds__(kUploadThreads) upload_kernel(const uint4* __restrict__ src, uint4* __restrict__ dst, int n_vec) {
  const int stride = gridDim.x * kUploadThreads;
  for (int e0 = blockIdx.x * kUploadThreads + threadIdx.x; e0 < n_vec; e0 += stride * kUploadUnroll) {
    uint4 r[kUploadUnroll];
#pragma unroll
    for (int u = 0; u < kUploadUnroll; ++u) {
      const int e = e0 + u * stride;
      if (e < n_vec)
        asm volatile("ld.global.cv.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r[u].x), "=r"(r[u].y), "=r"(r[u].z), "=r"(r[u].w) : "l"(src + e));
    }
#pragma unroll
    for (int u = 0; u < kUploadUnroll; ++u) {
      const int e = e0 + u * stride;
      if (e < n_vec) dst[e] = r[u];
    }
  }
}

// bytes: a multiple of 16; src_mapped: the device-side address of mapped pinned host memory
cudaError_t launch_upload(const void* src_mapped, void* dst, size_t bytes, cudaStream_t stream) {
  const int n_vec = (int)(bytes / 16);
  int grid = (n_vec + kUploadThreads * kUploadUnroll - 1) / (kUploadThreads * kUploadUnroll);
  grid = grid < 1 ? 1 : (grid > 32 ? 32 : grid);
  upload_kernel<<<grid, kUploadThreads, 0, stream>>>(reinterpret_cast<const uint4*>(src_mapped), reinterpret_cast<uint4*>(dst), n_vec);
  return cudaGetLastError();
}

static dim3 copy_grid(const CopyParams& p, int sm_count, int64_t max_vecs_per_sess) {
  // enough CTAs to fill the machine (8 resident CTAs of 256 threads per SM), split evenly over sessions
  int64_t want = (max_vecs_per_sess + (int64_t)kCopyThreads * kCopyUnroll - 1) / ((int64_t)kCopyThreads * kCopyUnroll);
  int64_t per_sess_cap = ((int64_t)sm_count * 8 + p.n_sess - 1) / p.n_sess;
  int64_t gx = want < per_sess_cap ? want : per_sess_cap;
  if (gx < 1) gx = 1;
  return dim3((unsigned)gx, (unsigned)p.n_sess, 1);
}

cudaError_t launch_append(const CopyParams& p, int sm_count, cudaStream_t stream) {
  // largest per-session element count bounds grid.x; sessions are descriptors on the device, so use the mean
  const int64_t vec_per_row = (int64_t)p.H * (p.D / 8);
  const int64_t mean_rows = (p.total_rows + p.n_sess - 1) / p.n_sess;
  kv_append_kernel<<<copy_grid(p, sm_count, mean_rows * vec_per_row), kCopyThreads, 0, stream>>>(p);
  return cudaGetLastError();
}

cudaError_t launch_gather(const CopyParams& p, int sm_count, cudaStream_t stream) {
  const int64_t vec_per_row = (int64_t)p.H * (p.D / 8);
  const int64_t mean_rows = (p.total_rows + p.n_sess - 1) / p.n_sess;
  kv_gather_kernel<<<copy_grid(p, sm_count, mean_rows * vec_per_row), kCopyThreads, 0, stream>>>(p);
  return cudaGetLastError();
}

}  // namespace tc
