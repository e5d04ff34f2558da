// vcs_chunk_ingest{,_host}: the whole per-chunk hot path as one C call (drop -> append -> prefill),
// optionally with host buffers (H2D of the chunk's inputs, D2H of its results on the same stream).
#include "attn.cuh"

#include <vector>

using namespace vcs;

// Workspace checks shared by the one-call forms: everything is looked at before the first enqueue, so that an
// error cannot leave a chunk half ingested.
static int check_workspaces(const char* who, const void* ws_drop, size_t drop_bytes, size_t drop_need, const void* ws_append,
                            size_t append_bytes, size_t append_need, const void* ws_attn, size_t attn_bytes, size_t attn_need) {
  if (!aligned16(ws_drop) || !aligned16(ws_append) || !aligned16(ws_attn))
    VCS_FAIL(VCS_EALIGN, "%s: ws_drop / ws_append / ws_attn must be 16-byte aligned", who);
  if (drop_bytes < drop_need) VCS_FAIL(VCS_ECAP, "%s: ws_drop too small (%zu < %zu)", who, drop_bytes, drop_need);
  if (append_bytes < append_need) VCS_FAIL(VCS_ECAP, "%s: ws_append too small (%zu < %zu)", who, append_bytes, append_need);
  if (attn_bytes < attn_need) VCS_FAIL(VCS_ECAP, "%s: ws_attn too small (%zu < %zu)", who, attn_bytes, attn_need);
  return VCS_OK;
}

static int check_call(const vcs_kv_pool* pool, const vcs_chunk_call* c) {
  int rc = validate_pool(pool, true);
  if (rc != VCS_OK) return rc;
  if (!c) VCS_FAIL(VCS_EINVAL, "chunk_ingest: NULL call");
  if (!c->z_d || !c->q_d || !c->k_d || !c->v_d || !c->out_d || !c->kept_idx_d || !c->kept_count_d || !c->pos3_d ||
      !c->ws_drop || !c->ws_append || !c->ws_attn)
    VCS_FAIL(VCS_EINVAL, "chunk_ingest: NULL member in vcs_chunk_call");
  if (c->G <= 0 || c->P <= 0 || c->D <= 0) VCS_FAIL(VCS_EINVAL, "chunk_ingest: bad sizes");
  if (c->n_vis_cap < 0 || (c->n_vis_cap > 0 && !c->page_table_d)) VCS_FAIL(VCS_EINVAL, "chunk_ingest: NULL page table");
  const int T = c->G * c->P;
  return check_workspaces("chunk_ingest", c->ws_drop, c->ws_drop_bytes, vcs_temporal_drop_workspace_bytes(1, c->G, c->P),
                          c->ws_append, c->ws_append_bytes, vcs_kv_append_workspace_bytes(pool, T), c->ws_attn,
                          c->ws_attn_bytes, vcs_bounded_prefill_attn_workspace_bytes(pool, T, c->n_vis_cap));
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
  const size_t rows = c->host_rows > 0 && (size_t)c->host_rows < T ? (size_t)c->host_rows : T;   // live q / k / v rows
  VCS_CUDA_OK(cudaMemcpyAsync(c->z_d, z_h, T * c->D * elem_bytes(c->z_dtype), cudaMemcpyHostToDevice, st));
  VCS_CUDA_OK(cudaMemcpyAsync(c->q_d, q_h, rows * pool->Hq * pool->d * eb, cudaMemcpyHostToDevice, st));
  VCS_CUDA_OK(cudaMemcpyAsync(c->k_d, k_h, rows * pool->Hkv * pool->d * eb, cudaMemcpyHostToDevice, st));
  VCS_CUDA_OK(cudaMemcpyAsync(c->v_d, v_h, rows * pool->Hkv * pool->d * eb, cudaMemcpyHostToDevice, st));
  return VCS_OK;
}

extern "C" int vcs_chunk_download(const vcs_kv_pool* pool, const vcs_chunk_call* c, void* out_h, int32_t* kept_idx_h,
                                  int32_t* kept_count_h, void* stream) {
  int rc = check_call(pool, c);
  if (rc != VCS_OK) return rc;
  if (!out_h || !kept_idx_h || !kept_count_h) VCS_FAIL(VCS_EINVAL, "chunk_download: NULL host buffer");
  cudaStream_t st = (cudaStream_t)stream;
  const size_t T = (size_t)c->G * c->P, eb = elem_bytes(pool->dtype);
  const size_t rows = c->host_rows > 0 && (size_t)c->host_rows < T ? (size_t)c->host_rows : T;
  VCS_CUDA_OK(cudaMemcpyAsync(out_h, c->out_d, rows * pool->Hq * pool->d * eb, cudaMemcpyDeviceToHost, st));
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

// ---- L layers x B streams: one token drop per stream (the drop sits before the LLM), then for
// every layer one batched KV append and one batched bounded prefill over the B streams (PAPER.md:73, :95:
// several chunks in flight; here they share launches instead of threads) -------------------------------
extern "C" int vcs_ingest_layers(const vcs_kv_pool* const* pools_h, const vcs_multi_call* c, void* stream) {
  if (!pools_h || !c) VCS_FAIL(VCS_EINVAL, "ingest_layers: NULL pools / call");
  if (c->L <= 0 || c->B <= 0 || c->G <= 0 || c->P <= 0 || c->D <= 0) VCS_FAIL(VCS_EINVAL, "ingest_layers: bad sizes");
  if (c->B > kAttnMaxStreams) VCS_FAIL(VCS_ECAP, "ingest_layers: B = %d streams per launch (at most %d)", c->B, kAttnMaxStreams);
  if (c->n_vis_cap < 0 || (c->n_vis_cap > 0 && !c->page_tables_d)) VCS_FAIL(VCS_EINVAL, "ingest_layers: NULL page tables");
  if (!c->z_d || !c->q_d || !c->k_d || !c->v_d || !c->out_d || !c->kept_idx_d || !c->kept_count_d || !c->pos3_d ||
      !c->page_ids_d || !c->ws_drop || !c->ws_append || !c->ws_attn)
    VCS_FAIL(VCS_EINVAL, "ingest_layers: NULL member in vcs_multi_call");
  for (int l = 0; l < c->L; ++l) {
    int rc = validate_pool(pools_h[l], true);
    if (rc != VCS_OK) return rc;
    if (pools_h[l]->Hq != pools_h[0]->Hq || pools_h[l]->Hkv != pools_h[0]->Hkv || pools_h[l]->d != pools_h[0]->d ||
        pools_h[l]->dtype != pools_h[0]->dtype || pools_h[l]->n_pages != pools_h[0]->n_pages ||
        pools_h[l]->page_cap != pools_h[0]->page_cap || pools_h[l]->rope_theta != pools_h[0]->rope_theta ||
        pools_h[l]->rope_sections[0] != pools_h[0]->rope_sections[0] || pools_h[l]->rope_sections[1] != pools_h[0]->rope_sections[1] ||
        pools_h[l]->rope_sections[2] != pools_h[0]->rope_sections[2])
      VCS_FAIL(VCS_EINVAL, "ingest_layers: the layers' pools must have the same geometry (heads, d, dtype, pages, page_cap, rope)");
  }
  const vcs_kv_pool* p0 = pools_h[0];
  const int T = c->G * c->P;
  int rc = check_workspaces("ingest_layers", c->ws_drop, c->ws_drop_bytes, vcs_temporal_drop_workspace_bytes(c->B, c->G, c->P),
                            c->ws_append, c->ws_append_bytes, vcs_kv_append_batched_workspace_bytes(p0, T, c->B), c->ws_attn,
                            c->ws_attn_bytes, vcs_bounded_prefill_attn_workspace_bytes(p0, T, c->n_vis_cap));
  if (rc != VCS_OK) return rc;
  rc = vcs_temporal_drop(c->z_d, c->mode == VCS_DROP_CONSECUTIVE ? c->prev_last_group_d : nullptr, c->B, c->G, c->P, c->D,
                             c->z_dtype, c->tau, c->mode, c->kept_idx_d, c->kept_count_d, nullptr, c->pos3_d, c->Hg, c->Wg,
                             c->t_stride, c->pos_base_d, c->ws_drop, c->ws_drop_bytes, stream);
  if (rc != VCS_OK) return rc;
  const int64_t kv_row = (int64_t)p0->Hkv * p0->d, q_row = (int64_t)p0->Hq * p0->d;
  const int64_t kv_stream = kv_row * T, q_stream = q_row * T;
  const size_t eb = elem_bytes(p0->dtype);
  for (int l = 0; l < c->L; ++l) {
    const char* kl = static_cast<const char*>(c->k_d) + (size_t)l * c->kv_layer_stride * eb;
    const char* vl = static_cast<const char*>(c->v_d) + (size_t)l * c->kv_layer_stride * eb;
    const char* ql = static_cast<const char*>(c->q_d) + (size_t)l * c->q_layer_stride * eb;
    char* ol = static_cast<char*>(c->out_d) + (size_t)l * c->out_layer_stride * eb;
    rc = vcs_kv_append_pages_batched(pools_h[l], kl, vl, kv_stream, kv_stream, kv_row, kv_row, c->pos3_d, c->kept_count_d, T,
                                     c->page_ids_d, c->B, c->status_d, c->ws_append, c->ws_append_bytes, stream);
    if (rc != VCS_OK) return rc;
    rc = vcs_bounded_prefill_attn_batched(pools_h[l], ql, q_stream, q_row, c->pos3_d, c->kept_count_d, T, c->page_tables_d,
                                          c->n_vis_d, c->n_vis_cap, c->page_ids_d, 0, 0.f, ol, q_stream, q_row, nullptr, c->B,
                                          c->attn_flags, c->status_d, c->ws_attn, c->ws_attn_bytes, stream);
    if (rc != VCS_OK) return rc;
  }
  return VCS_OK;
}

// ---- CUDA graphs: record whatever vcs calls (and other stream work) the caller enqueues between begin and end
// into a graph, replay it with one launch.  The programmatic-dependent-launch edges between consecutive vcs
// kernels are kept by the capture. ------------------------------------------------------------------------
struct VcsGraph {
  cudaGraph_t graph;
  cudaGraphExec_t exec;
};

// Destroying a graph while this thread records another one would invalidate the capture (the CUDA calls involved
// are not allowed inside a thread-local capture): such a destroy is parked here and carried out by vcs_graph_end.
static thread_local int t_capturing = 0;
static thread_local std::vector<VcsGraph*> t_parked;

static void graph_free(VcsGraph* h) {
  cudaGraphExecDestroy(h->exec);
  cudaGraphDestroy(h->graph);
  delete h;
}

extern "C" int vcs_graph_begin(void* stream) {
  VCS_CUDA_OK(cudaStreamBeginCapture((cudaStream_t)stream, cudaStreamCaptureModeThreadLocal));
  ++t_capturing;
  return VCS_OK;
}

extern "C" int vcs_graph_end(void* stream, void** graph_out) {
  if (!graph_out) VCS_FAIL(VCS_EINVAL, "graph_end: NULL output");
  *graph_out = nullptr;
  cudaGraph_t g = nullptr;
  const cudaError_t end_err = cudaStreamEndCapture((cudaStream_t)stream, &g);
  if (t_capturing > 0) --t_capturing;
  if (t_capturing == 0) {
    for (VcsGraph* parked : t_parked) graph_free(parked);
    t_parked.clear();
  }
  VCS_CUDA_OK(end_err);
  cudaGraphExec_t e = nullptr;
  cudaError_t err = cudaGraphInstantiate(&e, g, 0);
  if (err != cudaSuccess) {
    cudaGraphDestroy(g);
    VCS_FAIL(VCS_ECUDA, "cudaGraphInstantiate: %s", cudaGetErrorString(err));
  }
  VcsGraph* h = new VcsGraph{g, e};
  *graph_out = h;
  return VCS_OK;
}

extern "C" int vcs_graph_launch(void* graph, void* stream) {
  if (!graph) VCS_FAIL(VCS_EINVAL, "graph_launch: NULL graph");
  VCS_CUDA_OK(cudaGraphLaunch(static_cast<VcsGraph*>(graph)->exec, (cudaStream_t)stream));
  return VCS_OK;
}

extern "C" int vcs_graph_destroy(void* graph) {
  if (!graph) return VCS_OK;
  VcsGraph* h = static_cast<VcsGraph*>(graph);
  if (t_capturing > 0) {
    t_parked.push_back(h);       // any number of them: a free inside the capture would invalidate the recording
    return VCS_OK;
  }
  graph_free(h);
  return VCS_OK;
}
