// Shared parameter block of the bounded-attention kernels (SIMT and tcgen05).
#pragma once
#include "common.cuh"

namespace vcs {

struct AttnParams {
  const void* q;
  long long q_stride;      // elements between query rows
  const int32_t* q_pos3;
  const int32_t* nq_d;
  int nq_cap;
  const int32_t* page_table;
  const int32_t* n_vis_d;
  int n_vis_cap;
  int self_page, self_offset;
  float scale;
  void* out;
  long long out_stride;
  float* lse;
  int32_t* status;
  const void* k_pages;
  const void* v_pages;
  const int32_t* page_len;
  int n_pages, page_cap, Hkv, Hq, d;
  RopeParams rope;
  // split-KV (tcgen05 kernel only): grid.z = n_split CTAs share one (q tile, head) item; each writes an
  // unnormalised partial (O fp32 [128][128], m[128], l[128]) and the last one to arrive merges them
  int n_split;
  int tail_split;   // 1: items of an under-filled LAST wave are split over the CTAs that would exit early (device choice)
  int sm_count;
  float* part;
  unsigned int* part_counter;
#ifdef VCS_ATTN_TRACE
  void* trace;   // debug builds only: clock64 stamps of one CTA's pipeline (see attn_tc.cu)
#endif
};

int launch_attn_simt(const AttnParams& p, int dtype, cudaStream_t st);
// tcgen05 / TMA kernel (bf16, head_dim 128)
bool attn_tc_supported(const vcs_kv_pool* pool);
size_t attn_tc_workspace_bytes(const vcs_kv_pool* pool, int nq_cap, int n_vis_cap);
int attn_tc_splits(const vcs_kv_pool* pool, int nq_cap, int n_vis_cap);
int launch_attn_tc(const AttnParams& p, const vcs_kv_pool* pool, void* workspace, size_t workspace_bytes,
                   cudaStream_t st);

}  // namespace vcs
