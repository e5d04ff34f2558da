// vcs_chunk_ingest{,_host}: the whole per-chunk hot path as one C call (drop -> append -> prefill),
// optionally with host buffers (H2D of the chunk's inputs, D2H of its results on the same stream).
#include "common.cuh"

using namespace vcs;

static int check_call(const vcs_kv_pool* pool, const vcs_chunk_call* c) {
  int rc = validate_pool(pool, true);
  if (rc != VCS_OK) return rc;
  if (!c) VCS_FAIL(VCS_EINVAL, "chunk_ingest: NULL call");
  if (!c->z_d || !c->q_d || !c->k_d || !c->v_d || !c->out_d || !c->kept_idx_d || !c->kept_count_d || !c->pos3_d ||
      !c->ws_drop || !c->ws_append || !c->ws_attn)
    VCS_FAIL(VCS_EINVAL, "chunk_ingest: NULL member in vcs_chunk_call");
  if (c->G <= 0 || c->P <= 0 || c->D <= 0) VCS_FAIL(VCS_EINVAL, "chunk_ingest: bad sizes");
  return VCS_OK;
}

extern "C" int vcs_chunk_ingest(const vcs_kv_pool* pool, const vcs_chunk_call* c, void* stream) {
  int rc = check_call(pool, c);
  if (rc != VCS_OK) return rc;
  const int T = c->G * c->P;
  rc = vcs_temporal_drop(c->z_d, c->mode == VCS_DROP_CONSECUTIVE ? c->prev_last_group_d : nullptr, 1, c->G, c->P, c->D, c->z_dtype, c->tau, c->mode, c->kept_idx_d,
                         c->kept_count_d, nullptr, c->pos3_d, c->Hg, c->Wg, c->t_stride, c->pos_base_d, c->ws_drop,
                         c->ws_drop_bytes, stream);
  if (rc != VCS_OK) return rc;
  const int64_t kv_stride = (int64_t)pool->Hkv * pool->d, q_stride = (int64_t)pool->Hq * pool->d;
  rc = vcs_kv_append_pages(pool, c->k_d, c->v_d, kv_stride, kv_stride, c->pos3_d, c->kept_count_d, T, c->page_id, 0,
                           c->status_d, c->ws_append, c->ws_append_bytes, stream);
  if (rc != VCS_OK) return rc;
  return vcs_bounded_prefill_attn(pool, c->q_d, q_stride, c->pos3_d, c->kept_count_d, T, c->page_table_d, c->n_vis_d,
                                  c->n_vis_cap, c->page_id, 0, 0.f, c->out_d, q_stride, nullptr, c->attn_flags,
                                  c->status_d, c->ws_attn, c->ws_attn_bytes, stream);
}

extern "C" int vcs_chunk_upload(const vcs_kv_pool* pool, const vcs_chunk_call* c, const void* z_h, const void* q_h,
                                const void* k_h, const void* v_h, void* stream) {
  int rc = check_call(pool, c);
  if (rc != VCS_OK) return rc;
  if (!z_h || !q_h || !k_h || !v_h) VCS_FAIL(VCS_EINVAL, "chunk_upload: NULL host buffer");
  cudaStream_t st = (cudaStream_t)stream;
  const size_t T = (size_t)c->G * c->P, eb = elem_bytes(pool->dtype);
  VCS_CUDA_OK(cudaMemcpyAsync(c->z_d, z_h, T * c->D * elem_bytes(c->z_dtype), cudaMemcpyHostToDevice, st));
  VCS_CUDA_OK(cudaMemcpyAsync(c->q_d, q_h, T * pool->Hq * pool->d * eb, cudaMemcpyHostToDevice, st));
  VCS_CUDA_OK(cudaMemcpyAsync(c->k_d, k_h, T * pool->Hkv * pool->d * eb, cudaMemcpyHostToDevice, st));
  VCS_CUDA_OK(cudaMemcpyAsync(c->v_d, v_h, T * pool->Hkv * pool->d * eb, cudaMemcpyHostToDevice, st));
  return VCS_OK;
}

extern "C" int vcs_chunk_download(const vcs_kv_pool* pool, const vcs_chunk_call* c, void* out_h, int32_t* kept_idx_h,
                                  int32_t* kept_count_h, void* stream) {
  int rc = check_call(pool, c);
  if (rc != VCS_OK) return rc;
  if (!out_h || !kept_idx_h || !kept_count_h) VCS_FAIL(VCS_EINVAL, "chunk_download: NULL host buffer");
  cudaStream_t st = (cudaStream_t)stream;
  const size_t T = (size_t)c->G * c->P, eb = elem_bytes(pool->dtype);
  VCS_CUDA_OK(cudaMemcpyAsync(out_h, c->out_d, T * pool->Hq * pool->d * eb, cudaMemcpyDeviceToHost, st));
  VCS_CUDA_OK(cudaMemcpyAsync(kept_idx_h, c->kept_idx_d, T * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  VCS_CUDA_OK(cudaMemcpyAsync(kept_count_h, c->kept_count_d, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  return VCS_OK;
}

extern "C" int vcs_chunk_ingest_host(const vcs_kv_pool* pool, const vcs_chunk_call* c, const void* z_h, const void* q_h,
                                     const void* k_h, const void* v_h, void* out_h, int32_t* kept_idx_h,
                                     int32_t* kept_count_h, void* stream) {
  int rc = vcs_chunk_upload(pool, c, z_h, q_h, k_h, v_h, stream);
  if (rc != VCS_OK) return rc;
  rc = vcs_chunk_ingest(pool, c, stream);
  if (rc != VCS_OK) return rc;
  return vcs_chunk_download(pool, c, out_h, kept_idx_h, kept_count_h, stream);
}
