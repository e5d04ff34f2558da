// vcs_retrieval_score: query-chunk similarity (Eq. 3) against the per-page mean
// pre-RoPE key summaries kept by vcs_kv_append_pages, and device-side top-k.
// Latency-bound (0.5 MB of summaries for a 256-page bank): two small launches, no host sync.
#include "common.cuh"

namespace vcs {

constexpr int kRetThreads = 256;

struct RetParams {
  const void* q;
  long long q_stride;
  const int32_t* nq_d;
  int nq_cap;
  const int32_t* cand;
  int n_cand;
  const int32_t* excl;
  int n_excl;
  int normalize;
  float* scores;
  int k;
  int32_t* topk;
  const float* k_sum;
  const int32_t* page_len;
  int n_pages, Hkv, Hq, d;
  float* qbar;             // workspace [kQbarSplit][Hkv*d]: row-slice sums of the query
  uint8_t* eligible;       // workspace [n_cand]
  unsigned int* counter;   // workspace [1]
};

// q_bar[kv][:] = mean over rows i < nq and the Hq/Hkv heads of group kv (reading D19).
constexpr int kQbarThreads = 1024;
constexpr int kQbarSplit = 8;     // row slices per kv head; the scorer adds the slices' sums in slice order
// One block per (kv head, row slice); thread = (row group, column).  The rows of a thread are independent loads, issued
// eight at a time (the kernel is a handful of L2 / HBM round trips long, not bandwidth), then a fixed-order
// reduction over the row groups through shared memory.
template <typename E>
__global__ void __launch_bounds__(kQbarThreads) qbar_kernel(const RetParams p) {
  pdl_wait();
  pdl_launch_dependents();
  __shared__ float s_part[kQbarThreads];
  const int kv = blockIdx.x, g = p.Hq / p.Hkv;
  int nq = p.nq_d ? *p.nq_d : p.nq_cap;
  nq = max(0, min(nq, p.nq_cap));
  const int col = threadIdx.x % p.d, lane_grp = threadIdx.x / p.d, n_grp = kQbarThreads / p.d;
  const int rows_all = nq * g;
  const int r_lo = (int)((long long)blockIdx.y * rows_all / kQbarSplit), rows = (int)((long long)(blockIdx.y + 1) * rows_all / kQbarSplit);
  auto at = [&](int r) {
    const int i = r / g, hh = r - i * g;
    const E* qp = static_cast<const E*>(p.q) + (size_t)i * p.q_stride + (size_t)(kv * g + hh) * p.d + col;
    if constexpr (sizeof(E) == 2) return __bfloat162float(*reinterpret_cast<const __nv_bfloat16*>(qp));
    else return *reinterpret_cast<const float*>(qp);
  };
  float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  if (lane_grp < n_grp) {
    int r = r_lo + lane_grp;
    for (; r + 7 * n_grp < rows; r += 8 * n_grp) {
#pragma unroll
      for (int u = 0; u < 8; ++u) acc[u] += at(r + u * n_grp);
    }
    for (; r < rows; r += n_grp) acc[0] += at(r);
  }
  s_part[threadIdx.x] = ((acc[0] + acc[1]) + (acc[2] + acc[3])) + ((acc[4] + acc[5]) + (acc[6] + acc[7]));
  __syncthreads();
  if (threadIdx.x < p.d) {
    float t = 0.f;
    for (int gi = 0; gi < n_grp; ++gi) t += s_part[gi * p.d + threadIdx.x];
    p.qbar[(size_t)blockIdx.y * p.Hkv * p.d + kv * p.d + threadIdx.x] = t;   // slice SUM; the scorer divides by the row count
  }
}

__global__ void __launch_bounds__(kRetThreads) score_topk_kernel(const RetParams p) {
  pdl_wait();
  pdl_launch_dependents();
  __shared__ int s_last;
  __shared__ float s_best[kRetThreads / 32];
  __shared__ int s_page[kRetThreads / 32];
  __shared__ int s_idx[kRetThreads / 32];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int HD = p.Hkv * p.d;
  // q_bar = (sum of the row slices, in slice order) / rows, rebuilt by every block in shared memory
  extern __shared__ __align__(16) float s_qbar[];   // [Hkv*d]
  {
    int nq = p.nq_d ? *p.nq_d : p.nq_cap;
    nq = max(0, min(nq, p.nq_cap));
    const int rows = nq * (p.Hq / p.Hkv);
    for (int e = threadIdx.x; e < HD; e += kRetThreads) {
      float t = 0.f;
#pragma unroll
      for (int sp = 0; sp < kQbarSplit; ++sp) t += __ldcg(p.qbar + (size_t)sp * HD + e);
      s_qbar[e] = rows > 0 ? t / (float)rows : 0.f;
    }
    __syncthreads();
  }
  const int c = blockIdx.x * (kRetThreads / 32) + warp;
  if (c < p.n_cand) {
    const int page = p.cand[c];
    const bool valid = page >= 0 && page < p.n_pages;
    const int len = valid ? p.page_len[page] : 0;
    float dot = 0.f, nx = 0.f, nqv = 0.f;
    if (len > 0) {
      const float inv = 1.f / (float)len;
      const float* ks = p.k_sum + (size_t)page * HD;
      const float4* ks4 = reinterpret_cast<const float4*>(ks);      // HD is a multiple of 8; both bases are 16-byte aligned
      const float4* qb4 = reinterpret_cast<const float4*>(s_qbar);
#pragma unroll 4
      for (int e = lane; e < HD / 4; e += 32) {
        const float4 k4 = ks4[e], q4 = qb4[e];
        const float xs[4] = {k4.x * inv, k4.y * inv, k4.z * inv, k4.w * inv}, qs[4] = {q4.x, q4.y, q4.z, q4.w};
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          dot = fmaf(qs[u], xs[u], dot);
          nx = fmaf(xs[u], xs[u], nx);
          nqv = fmaf(qs[u], qs[u], nqv);
        }
      }
    }
    dot = warp_sum(dot); nx = warp_sum(nx); nqv = warp_sum(nqv);
    float s = dot;
    if (p.normalize) s = (nx == 0.f || nqv == 0.f) ? 0.f : dot / (sqrtf(nx) * sqrtf(nqv));
    bool elig = valid && s == s;          // a NaN score never wins
    for (int e = lane; e < p.n_excl; e += 32) elig = elig && (p.excl[e] != page);
    elig = __all_sync(0xffffffffu, elig);
    if (lane == 0) {
      p.scores[c] = s;
      p.eligible[c] = elig ? 1 : 0;
    }
  }
  if (!p.topk || p.k <= 0) return;
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    const unsigned int t = atomicAdd(p.counter, 1u);
    s_last = (t == gridDim.x - 1);
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  // top-k by k rounds of block arg-max over (score desc, page id asc)
  // the thread's first candidate lives in registers (all of them when n_cand <= kRetThreads); the rest are re-read
  __shared__ int s_win;
  const int i0 = threadIdx.x;
  bool e0 = false;
  float sc0 = 0.f;
  int pg0 = 0;
  if (i0 < p.n_cand) { e0 = __ldcg(p.eligible + i0) != 0; sc0 = __ldcg(p.scores + i0); pg0 = p.cand[i0]; }
  if (p.n_cand <= kRetThreads) {
    // every candidate has its own thread: its output slot is its rank in (score desc, page id asc, index asc)
    // among the eligible ones.  Branch-free compare: the short-circuit form diverges per lane and was 4x slower.
    __shared__ float s_sc[kRetThreads];
    __shared__ int s_pg[kRetThreads];
    __shared__ int s_el[kRetThreads];
    s_sc[i0] = sc0; s_pg[i0] = pg0; s_el[i0] = e0 ? 1 : 0;
    const int n_elig = __syncthreads_count(e0 ? 1 : 0);
    int rank = 0;
#pragma unroll 8
    for (int j = 0; j < p.n_cand; ++j) {
      const float sj = s_sc[j];
      const int pj = s_pg[j];
      const bool beats = (sj > sc0) | ((sj == sc0) & ((pj < pg0) | ((pj == pg0) & (j < i0))));
      rank += (beats & (s_el[j] != 0)) ? 1 : 0;
    }
    if (e0 && rank < p.k) p.topk[rank] = pg0;
    if (i0 < p.k && i0 >= n_elig) p.topk[i0] = -1;
    if (threadIdx.x == 0) *p.counter = 0u;
    return;
  }
  for (int r = 0; r < p.k; ++r) {
    float best = -INFINITY;
    int bpage = 0x7fffffff, bidx = -1;
    if (e0) { best = sc0; bpage = pg0; bidx = i0; }
    for (int i = threadIdx.x + kRetThreads; i < p.n_cand; i += kRetThreads) {
      if (!__ldcg(p.eligible + i)) continue;
      const float s = __ldcg(p.scores + i);
      const int pg = p.cand[i];
      if (bidx < 0 || s > best || (s == best && pg < bpage)) { best = s; bpage = pg; bidx = i; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const float ob = __shfl_xor_sync(0xffffffffu, best, o);
      const int op = __shfl_xor_sync(0xffffffffu, bpage, o);
      const int oi = __shfl_xor_sync(0xffffffffu, bidx, o);
      if (oi >= 0 && (bidx < 0 || ob > best || (ob == best && op < bpage))) { best = ob; bpage = op; bidx = oi; }
    }
    if (lane == 0) { s_best[warp] = best; s_page[warp] = bpage; s_idx[warp] = bidx; }
    __syncthreads();
    if (threadIdx.x == 0) {
      for (int w = 1; w < kRetThreads / 32; ++w) {
        if (s_idx[w] >= 0 && (s_idx[0] < 0 || s_best[w] > s_best[0] || (s_best[w] == s_best[0] && s_page[w] < s_page[0]))) {
          s_best[0] = s_best[w]; s_page[0] = s_page[w]; s_idx[0] = s_idx[w];
        }
      }
      p.topk[r] = s_idx[0] >= 0 ? s_page[0] : -1;
      if (s_idx[0] >= kRetThreads) p.eligible[s_idx[0]] = 0;
      s_win = s_idx[0];
      __threadfence_block();
    }
    __syncthreads();
    if (s_win == i0) e0 = false;
  }
  if (threadIdx.x == 0) *p.counter = 0u;
}

// Threshold form of the query visibility, V_qry = { j : s_j >= tau_q }: one block
// compacts the candidates whose score reaches tau_q (and that are not excluded) in candidate order.
__global__ void __launch_bounds__(kRetThreads) threshold_kernel(const float* scores, const int32_t* cand, int n_cand,
                                                                 const int32_t* excl, int n_excl, float tau_q,
                                                                 int32_t* out_pages, int out_cap, int32_t* out_count,
                                                                 int n_pages) {
  pdl_wait();
  pdl_launch_dependents();
  __shared__ int s_warp[kRetThreads / 32];
  __shared__ int s_base;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (threadIdx.x == 0) s_base = 0;
  __syncthreads();
  for (int c0 = 0; c0 < n_cand; c0 += kRetThreads) {
    const int c = c0 + threadIdx.x;
    bool keep = false;
    int page = -1;
    if (c < n_cand) {
      page = cand[c];
      keep = page >= 0 && page < n_pages && scores[c] >= tau_q;
      for (int e = 0; e < n_excl && keep; ++e) keep = excl[e] != page;
    }
    const unsigned bal = __ballot_sync(0xffffffffu, keep);
    if (lane == 0) s_warp[warp] = __popc(bal);
    __syncthreads();
    int off = s_base;
    for (int w = 0; w < warp; ++w) off += s_warp[w];
    off += __popc(bal & ((1u << lane) - 1u));
    if (keep && off < out_cap) out_pages[off] = page;
    __syncthreads();
    if (threadIdx.x == 0) {
      int t = s_base;
      for (int w = 0; w < kRetThreads / 32; ++w) t += s_warp[w];
      s_base = t;
    }
    __syncthreads();
  }
  const int total = s_base;
  for (int i = total + threadIdx.x; i < out_cap; i += kRetThreads) out_pages[i] = -1;
  if (threadIdx.x == 0) *out_count = min(total, out_cap);
}

}  // namespace vcs

using namespace vcs;

extern "C" size_t vcs_retrieval_score_workspace_bytes(const vcs_kv_pool* pool, int n_cand) {
  if (!pool || n_cand < 0) return 0;
  return 256 + round_up((size_t)kQbarSplit * pool->Hkv * pool->d * sizeof(float), 256) + round_up((size_t)n_cand, 256);
}

extern "C" int vcs_retrieval_score(const vcs_kv_pool* pool, const void* q, int64_t q_row_stride, const int32_t* nq_d,
                                   int nq_cap, const int32_t* cand_pages_d, int n_cand,
                                   const int32_t* exclude_pages_d, int n_excl, int normalize, float* scores, int k,
                                   int32_t* topk_pages, void* workspace, size_t workspace_bytes, void* stream) {
  int rc = validate_pool(pool, true);
  if (rc != VCS_OK) return rc;
  if (nq_cap < 0 || n_cand < 0 || n_excl < 0 || k < 0) VCS_FAIL(VCS_EINVAL, "retrieval: negative size");
  if (k > kRetThreads) VCS_FAIL(VCS_ECAP, "retrieval: k = %d (at most %d)", k, kRetThreads);
  if (!workspace) VCS_FAIL(VCS_EINVAL, "retrieval: NULL workspace");
  if (workspace_bytes < vcs_retrieval_score_workspace_bytes(pool, n_cand)) VCS_FAIL(VCS_ECAP, "retrieval: workspace too small");
  if (n_cand > 0 && (!cand_pages_d || !scores)) VCS_FAIL(VCS_EINVAL, "retrieval: NULL candidates / scores");
  if (nq_cap > 0 && !q) VCS_FAIL(VCS_EINVAL, "retrieval: NULL q");
  if (n_excl > 0 && !exclude_pages_d) VCS_FAIL(VCS_EINVAL, "retrieval: NULL exclude list");
  if (q_row_stride < (int64_t)pool->Hq * pool->d && nq_cap > 0) VCS_FAIL(VCS_EINVAL, "retrieval: row stride smaller than Hq*d");
  cudaStream_t st = (cudaStream_t)stream;
  if (n_cand == 0) {
    if (topk_pages && k > 0) VCS_CUDA_OK(cudaMemsetAsync(topk_pages, 0xff, sizeof(int32_t) * k, st));
    return VCS_OK;
  }
  RetParams p;
  p.q = q; p.q_stride = q_row_stride; p.nq_d = nq_d; p.nq_cap = nq_cap; p.cand = cand_pages_d; p.n_cand = n_cand;
  p.excl = exclude_pages_d; p.n_excl = n_excl; p.normalize = normalize; p.scores = scores; p.k = k; p.topk = topk_pages;
  p.k_sum = pool->k_sum; p.page_len = pool->page_len; p.n_pages = pool->n_pages; p.Hkv = pool->Hkv; p.Hq = pool->Hq;
  p.d = pool->d;
  char* ws = static_cast<char*>(workspace);
  p.counter = reinterpret_cast<unsigned int*>(ws);
  p.qbar = reinterpret_cast<float*>(ws + 256);
  p.eligible = reinterpret_cast<uint8_t*>(ws + 256 + round_up((size_t)kQbarSplit * pool->Hkv * pool->d * sizeof(float), 256));
  if (pool->dtype == VCS_BF16) qbar_kernel<__nv_bfloat16><<<dim3(pool->Hkv, kQbarSplit), kQbarThreads, 0, st>>>(p);
  else qbar_kernel<float><<<dim3(pool->Hkv, kQbarSplit), kQbarThreads, 0, st>>>(p);
  const int wpb = kRetThreads / 32;
  launch_pdl(score_topk_kernel, dim3((n_cand + wpb - 1) / wpb), dim3(kRetThreads), (size_t)pool->Hkv * pool->d * sizeof(float), st, p);
  cudaError_t err = cudaGetLastError();
  if (err != cudaSuccess) VCS_FAIL(VCS_ECUDA, "retrieval launch: %s", cudaGetErrorString(err));
  return VCS_OK;
}

extern "C" int vcs_retrieval_threshold(const vcs_kv_pool* pool, const float* scores, const int32_t* cand_pages_d, int n_cand,
                                       const int32_t* exclude_pages_d, int n_excl, float tau_q, int32_t* vis_pages,
                                       int vis_cap, int32_t* vis_count_d, void* stream) {
  int rc = validate_pool(pool, false);
  if (rc != VCS_OK) return rc;
  if (n_cand < 0 || n_excl < 0 || vis_cap < 0) VCS_FAIL(VCS_EINVAL, "retrieval_threshold: negative size");
  if (!vis_count_d || (vis_cap > 0 && !vis_pages)) VCS_FAIL(VCS_EINVAL, "retrieval_threshold: NULL output");
  if (n_cand > 0 && (!scores || !cand_pages_d)) VCS_FAIL(VCS_EINVAL, "retrieval_threshold: NULL scores / candidates");
  if (n_excl > 0 && !exclude_pages_d) VCS_FAIL(VCS_EINVAL, "retrieval_threshold: NULL exclude list");
  if (!(tau_q == tau_q)) VCS_FAIL(VCS_EINVAL, "retrieval_threshold: tau_q is NaN");
  cudaError_t err = launch_pdl(threshold_kernel, dim3(1), dim3(kRetThreads), 0, (cudaStream_t)stream, scores, cand_pages_d,
                               n_cand, exclude_pages_d, n_excl, tau_q, vis_pages, vis_cap, vis_count_d, pool->n_pages);
  if (err == cudaSuccess) err = cudaGetLastError();
  if (err != cudaSuccess) VCS_FAIL(VCS_ECUDA, "retrieval_threshold launch: %s", cudaGetErrorString(err));
  return VCS_OK;
}
