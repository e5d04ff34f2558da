// vcs_bounded_prefill_attn{,_batched} entry points: argument validation and kernel selection.
#include "attn.cuh"

#include <cmath>

using namespace vcs;

extern "C" size_t vcs_bounded_prefill_attn_workspace_bytes(const vcs_kv_pool* pool, int nq_cap, int n_vis_cap) {
  if (!pool || nq_cap < 0 || n_vis_cap < 0) return 0;
  size_t tc = attn_tc_supported(pool) ? attn_tc_workspace_bytes(pool) : 0;
  return tc < 256 ? 256 : tc;
}

static int attn_common(const vcs_kv_pool* pool, const void* q, int64_t q_batch_stride, int64_t q_row_stride,
                       const int32_t* q_pos3, const int32_t* nq_d, int nq_cap, const int32_t* page_table_d,
                       const int32_t* n_vis_d, int n_vis_cap, int32_t self_page, const int32_t* self_pages_d,
                       int32_t self_offset, float softmax_scale, void* out, int64_t out_batch_stride,
                       int64_t out_row_stride, float* lse, int B, int flags, int32_t* status_d, void* workspace,
                       size_t workspace_bytes, void* stream) {
  int rc = validate_pool(pool, true);
  if (rc != VCS_OK) return rc;
  if (nq_cap < 0 || n_vis_cap < 0) VCS_FAIL(VCS_EINVAL, "attention: negative capacity");
  if (B < 0 || B > kAttnMaxStreams) VCS_FAIL(VCS_ECAP, "attention: B = %d streams per launch (at most %d)", B, kAttnMaxStreams);
  if (nq_cap == 0 || B == 0) return VCS_OK;
  if (!q || !q_pos3 || !out) VCS_FAIL(VCS_EINVAL, "attention: NULL q / q_pos3 / out");
  if (n_vis_cap > 0 && !page_table_d) VCS_FAIL(VCS_EINVAL, "attention: NULL page table");
  if (self_page >= pool->n_pages) VCS_FAIL(VCS_ECAP, "attention: self_page %d out of range", self_page);
  if ((self_page >= 0 || self_pages_d) && (self_offset < 0 || self_offset > pool->page_cap))
    VCS_FAIL(VCS_EINVAL, "attention: self_offset %d outside [0, page_cap]", self_offset);
  if (!(softmax_scale >= 0.f) || std::isinf(softmax_scale)) VCS_FAIL(VCS_EINVAL, "attention: bad softmax_scale");
  const size_t eb = elem_bytes(pool->dtype);
  const int64_t min_stride = (int64_t)pool->Hq * pool->d;
  if (q_row_stride < min_stride || out_row_stride < min_stride) VCS_FAIL(VCS_EINVAL, "attention: row stride smaller than Hq*d");
  if (!aligned16(q) || !aligned16(out) || (q_row_stride * eb) % 16 || (out_row_stride * eb) % 16 ||
      (q_batch_stride * eb) % 16 || (out_batch_stride * eb) % 16)
    VCS_FAIL(VCS_EALIGN, "attention: q / out and their strides must be 16-byte aligned");
  if (flags != VCS_ATTN_AUTO && flags != VCS_ATTN_SIMT && flags != VCS_ATTN_TC) VCS_FAIL(VCS_EINVAL, "attention: flags %d", flags);

  AttnParams p;
  p.q = q; p.q_stride = q_row_stride; p.q_bstride = q_batch_stride; p.q_pos3 = q_pos3; p.nq_d = nq_d; p.nq_cap = nq_cap;
  p.page_table = page_table_d; p.n_vis_d = n_vis_d; p.n_vis_cap = n_vis_cap;
  p.self_page = self_page < 0 ? -1 : self_page; p.self_pages_d = self_pages_d; p.self_offset = self_offset;
  p.scale = softmax_scale > 0.f ? softmax_scale : 1.0f / sqrtf((float)pool->d);
  p.out = out; p.out_stride = out_row_stride; p.out_bstride = out_batch_stride; p.lse = lse; p.status = status_d;
  p.k_pages = pool->k_pages; p.v_pages = pool->v_pages; p.page_len = pool->page_len;
  p.n_pages = pool->n_pages; p.page_cap = pool->page_cap; p.Hkv = pool->Hkv; p.Hq = pool->Hq; p.d = pool->d;
  p.B = B;
  p.rope = rope_params(pool);
  p.grid = 0; p.desc = nullptr; p.part = nullptr;

  const bool tc_ok = attn_tc_supported(pool);
  if (flags == VCS_ATTN_TC && !tc_ok) VCS_FAIL(VCS_EUNSUPPORTED, "attention: tcgen05 kernel needs bf16, head_dim 128 and TMA maps");
  if (flags == VCS_ATTN_TC || (flags == VCS_ATTN_AUTO && tc_ok)) {
    if (!workspace || workspace_bytes < attn_tc_workspace_bytes(pool)) VCS_FAIL(VCS_ECAP, "attention: workspace too small");
    if (!aligned16(workspace)) VCS_FAIL(VCS_EALIGN, "attention: workspace must be 16-byte aligned");
    return launch_attn_tc(p, pool, workspace, workspace_bytes, (cudaStream_t)stream);
  }
  return launch_attn_simt(p, pool->dtype, (cudaStream_t)stream);
}

extern "C" int vcs_bounded_prefill_attn(const vcs_kv_pool* pool, const void* q, int64_t q_row_stride,
                                        const int32_t* q_pos3, const int32_t* nq_d, int nq_cap,
                                        const int32_t* page_table_d, const int32_t* n_vis_d, int n_vis_cap,
                                        int32_t self_page, int32_t self_offset, float softmax_scale, void* out,
                                        int64_t out_row_stride, float* lse, int flags, int32_t* status_d,
                                        void* workspace, size_t workspace_bytes, void* stream) {
  return attn_common(pool, q, 0, q_row_stride, q_pos3, nq_d, nq_cap, page_table_d, n_vis_d, n_vis_cap, self_page, nullptr,
                     self_offset, softmax_scale, out, 0, out_row_stride, lse, 1, flags, status_d, workspace, workspace_bytes,
                     stream);
}

extern "C" int vcs_bounded_prefill_attn_batched(const vcs_kv_pool* pool, const void* q, int64_t q_batch_stride,
                                                int64_t q_row_stride, const int32_t* q_pos3, const int32_t* nq_d,
                                                int nq_cap, const int32_t* page_tables_d, const int32_t* n_vis_d,
                                                int n_vis_cap, const int32_t* self_pages_d, int32_t self_offset,
                                                float softmax_scale, void* out, int64_t out_batch_stride,
                                                int64_t out_row_stride, float* lse, int B, int flags, int32_t* status_d,
                                                void* workspace, size_t workspace_bytes, void* stream) {
  return attn_common(pool, q, q_batch_stride, q_row_stride, q_pos3, nq_d, nq_cap, page_tables_d, n_vis_d, n_vis_cap, -1,
                     self_pages_d, self_offset, softmax_scale, out, out_batch_stride, out_row_stride, lse, B, flags, status_d,
                     workspace, workspace_bytes, stream);
}
