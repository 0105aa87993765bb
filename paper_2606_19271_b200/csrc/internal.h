// Internal declarations shared by the host-side pool / scheduler and the kernel launchers.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <deque>
#include <vector>

#include "../../include/turbochunk.h"

namespace tc {

// ---- device-visible schedule records (built per call by the ragged batch scheduler, step a1) ----
struct SessDesc {      // one per session of the batch
  int32_t q_off;       // first token of the session in the packed [sum C][H][D] tensors
  int32_t C;           // chunk tokens
  int32_t x_begin;     // o + a*T : first visible prior token, in page-table coordinates
  int32_t x_end;       // o + L   : end of the cached tokens, in page-table coordinates
  int32_t pt_off;      // offset of this session's page table in the packed page-table array
  int32_t n_pt;        // pages in the table
  int32_t pad0, pad1;
};
static_assert(sizeof(SessDesc) == 32, "SessDesc layout");

struct WorkItem {      // one (session, head, one or two 128-row query tiles) for one CTA of a 2-CTA cluster
  int32_t sess;        // index into the batch
  int32_t head;
  int32_t q_tile;      // first query tile: rows [128*q_tile, ...) of the session's chunk; -1: no query rows (the CTA
                       // only loads its half of the partner's K/V tiles)
  uint32_t pipe;       // bits 0-23: KV tiles that flow through this CTA's smem ring for the item (>= the item's own
                       // KV tiles); bit 31: the two CTAs of the cluster work on the same (session, head) and each
                       // loads half of every K/V tile, multicast to both; bit 30: one query tile only, also when
                       // the chunk has rows left for a second one
};
static_assert(sizeof(WorkItem) == 16, "WorkItem layout");

struct CopySess {      // append / gather descriptor
  int32_t tok_off;     // first token in the packed source (append) / 0 (gather)
  int32_t n_tok;       // tokens to copy
  int32_t n_zero;      // append: trailing slots of the last page to zero-fill after the copied tokens
  int32_t x0;          // page-table coordinate of the first copied token (o + L for append, o for gather)
  int32_t pt_off;
  int32_t row_off;     // cumulative (n_tok + n_zero) rows before this session
  int32_t pad0, pad1;
};
static_assert(sizeof(CopySess) == 32, "CopySess layout");

struct CopyParams {
  const CopySess* sess;
  const int32_t* page_tables;
  int32_t n_sess;
  int32_t total_rows;       // sum over sessions of (n_tok + n_zero)
  int32_t H, D, B, log2_B;
  int64_t page_stride;      // bytes between pages in the slab
  int64_t layer_k_off;      // byte offset of this layer's K block inside a page
  int64_t layer_v_off;
  uint8_t* slab;
  const uint8_t* src_k;     // append: packed chunk K ; gather: unused
  const uint8_t* src_v;
  uint8_t* dst_k;           // gather: logical [L][H][D] output
  uint8_t* dst_v;
};

struct PullParams {          // migration fetch: whole pages, source slab -> target slab
  const uint8_t* src_slab;   // may be peer memory (another device of this process)
  uint8_t* dst_slab;
  const int32_t* pairs;      // device [n_pages][2]: (source page id, target page id), logical order
  int32_t n_pages;
  int32_t vec_per_page;      // page bytes / 16
  int64_t page_stride;       // bytes per page, same in both slabs (identical geometry)
};

constexpr int kFeedRing = 16;   // entries of a cluster's item-feed ring

struct AttnParams {
  CUtensorMap map_k;             // this layer's cached K: 4D {D, B, H, n_pages}
  CUtensorMap map_v;             // this layer's cached V
  const CUtensorMap* sess_maps;  // device [n][3]: per-session Q, Kn, Vn maps (3D {D, H, C_s}); OOB rows zero-fill
  const SessDesc* sess;
  const int32_t* page_tables;
  const WorkItem* items;
  unsigned long long* feed;      // [grid/2][kFeedRing] per-cluster ring of (sequence number, cluster item) pairs
  int32_t* feed_hdr;             // [0] the global cursor into the cluster-item list, [1] clusters that have seen its end,
                                 // [2] n_citems (items[2*i + r] is the work of CTA rank r for cluster item i).  [0], [1] and
                                 // the rings are zero at launch and zero again at exit (the kernel rearms them itself, so a
                                 // captured launch can be replayed without a memset): see next_cluster_item()
  uint16_t* out;                 // bf16 [sum C][H][D]
  float* lse;                    // fp32 [sum C][H] or null
  int32_t H, T, B, log2_B;
  float scale_log2;              // scale * log2(e)
  float scale;
  unsigned long long* clock_probe;  // null, or device uint64[2]: CTA 0 adds the SM cycles (clock64) and the nanoseconds
                                 // (globaltimer) it ran for, so that sum cycles / sum ns is the SM clock under THIS kernel
  CopyParams copy;               // fused chunk step: the KV append, done by the two idle warps of every CTA
                                 // (copy.n_sess == 0: none)
};

// kernel launchers (return cudaGetLastError())
cudaError_t launch_attention(const AttnParams& p, int head_dim, int grid, cudaStream_t stream);
cudaError_t launch_append(const CopyParams& p, int sm_count, cudaStream_t stream);
cudaError_t launch_gather(const CopyParams& p, int sm_count, cudaStream_t stream);
cudaError_t launch_page_pull(const PullParams& p, int sm_count, cudaStream_t stream);
cudaError_t launch_upload(const void* src_mapped, void* dst, size_t bytes, cudaStream_t stream);
int attention_smem_bytes(int head_dim);
cudaError_t attention_configure(int head_dim);   // sets the kernel's dynamic shared memory limit on the current device (idempotent)

}  // namespace tc
