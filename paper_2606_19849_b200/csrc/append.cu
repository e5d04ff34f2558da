// vcs_kv_append_pages: write the retained tokens' K (M-RoPE rotated) and V into one page of the
// chunk-granular paged KV cache ("historical visual cache"; step a5), keep the
// page's pre-RoPE key sum (retrieval summary of Eq. 3, reading D19) and its length.
//
// HBM-bound: each thread moves the (m..m+7, m+d/2..m+d/2+7) pair of 16-byte vectors of one
// (token, kv head) for K and V -- 128-bit coalesced loads and stores, sin/cos in registers.
// Per-block key sums go to the workspace; the last block (ticket) adds them in block order, so
// k_sum is deterministic.
#include "common.cuh"

namespace vcs {

constexpr int kAppendThreads = 256;

struct AppendParams {
  const void* k;
  const void* v;
  long long k_stride, v_stride;  // elements between tokens
  const int32_t* pos3;
  const int32_t* n_d;
  int n_cap;
  int page_id, page_offset;
  void* k_pages;
  void* v_pages;
  int32_t* page_len;
  float* k_sum;
  int page_cap, Hkv, d;
  int32_t* status;
  float* partial;          // [gridDim.x][Hkv*d]
  unsigned int* counter;   // two-level ticket counters
  int tok_per_block;
  RopeParams rope;
};

template <typename E>
struct KV;
template <>
struct KV<__nv_bfloat16> {
  static constexpr int kElems = 8;
  static __device__ __forceinline__ void unpack(const uint4& v, float* f) {
    f[0] = bf16_lo(v.x); f[1] = bf16_hi(v.x); f[2] = bf16_lo(v.y); f[3] = bf16_hi(v.y);
    f[4] = bf16_lo(v.z); f[5] = bf16_hi(v.z); f[6] = bf16_lo(v.w); f[7] = bf16_hi(v.w);
  }
  static __device__ __forceinline__ uint4 pack(const float* f) {
    return make_uint4(pack_bf16(f[0], f[1]), pack_bf16(f[2], f[3]), pack_bf16(f[4], f[5]), pack_bf16(f[6], f[7]));
  }
};
template <>
struct KV<float> {
  static constexpr int kElems = 4;
  static __device__ __forceinline__ void unpack(const uint4& v, float* f) {
    f[0] = __uint_as_float(v.x); f[1] = __uint_as_float(v.y); f[2] = __uint_as_float(v.z); f[3] = __uint_as_float(v.w);
  }
  static __device__ __forceinline__ uint4 pack(const float* f) {
    return make_uint4(__float_as_uint(f[0]), __float_as_uint(f[1]), __float_as_uint(f[2]), __float_as_uint(f[3]));
  }
};

template <typename E>
__global__ void __launch_bounds__(kAppendThreads) append_kernel(const AppendParams p) {
  pdl_wait();
  pdl_launch_dependents();
  constexpr int VE = KV<E>::kElems;
  extern __shared__ float s_sum[];  // [tok_per_block][Hkv*d]
  __shared__ int s_last;

  const int HD = p.Hkv * p.d;
  const int half = p.d / 2;
  const int vec_per_head = half / VE;             // vector pairs per (token, head)
  const int vec_per_tok = p.Hkv * vec_per_head;
  int n = p.n_d ? *p.n_d : p.n_cap;
  bool clamped = false, overflow = false;
  if (n > p.n_cap) { n = p.n_cap; clamped = true; }
  if (n < 0) n = 0;
  int n_fit = n;
  if (p.page_offset + n_fit > p.page_cap) { n_fit = p.page_cap - p.page_offset; overflow = true; }

  const int tid = threadIdx.x;
  const int tl = tid / vec_per_tok;               // token slot within the block
  const int rem = tid - tl * vec_per_tok;
  const int h = rem / vec_per_head;
  const int m0 = (rem - h * vec_per_head) * VE;   // first rotary pair of this thread
  const int tok = blockIdx.x * p.tok_per_block + tl;
  const bool active = tl < p.tok_per_block && tok < n_fit;

  float klo[VE], khi[VE];
#pragma unroll
  for (int e = 0; e < VE; ++e) klo[e] = khi[e] = 0.f;
  if (active) {
    const E* kp = static_cast<const E*>(p.k) + (size_t)tok * p.k_stride + h * p.d;
    const E* vp = static_cast<const E*>(p.v) + (size_t)tok * p.v_stride + h * p.d;
    const uint4 k0 = ldg_nc_v4(kp + m0), k1 = ldg_nc_v4(kp + m0 + half);
    const uint4 v0 = ldg_nc_v4(vp + m0), v1 = ldg_nc_v4(vp + m0 + half);
    const int pt = p.pos3[3 * tok + 0], ph = p.pos3[3 * tok + 1], pw = p.pos3[3 * tok + 2];
    KV<E>::unpack(k0, klo);
    KV<E>::unpack(k1, khi);
    float rlo[VE], rhi[VE];
#pragma unroll
    for (int e = 0; e < VE; ++e) {
      const int m = m0 + e;
      const int ax = p.rope.axis_of[m];
      const int pos = ax == 0 ? pt : (ax == 1 ? ph : pw);
      float s, c;
      rope_sincos(pos, p.rope.inv_freq[m], &s, &c);
      rlo[e] = klo[e] * c - khi[e] * s;   // (x_m, x_{m+d/2}) <- (x_m c - x_{m+d/2} s, x_{m+d/2} c + x_m s)
      rhi[e] = khi[e] * c + klo[e] * s;
    }
    const size_t row = ((size_t)p.page_id * p.Hkv + h) * p.page_cap + (p.page_offset + tok);
    E* ko = static_cast<E*>(p.k_pages) + row * p.d;
    E* vo = static_cast<E*>(p.v_pages) + row * p.d;
    stg_v4(ko + m0, KV<E>::pack(rlo));
    stg_v4(ko + m0 + half, KV<E>::pack(rhi));
    stg_v4(vo + m0, v0);
    stg_v4(vo + m0 + half, v1);
  }

  // per-block sum of the PRE-RoPE keys, tokens added in order
  if (tl < p.tok_per_block) {
    float* row = s_sum + (size_t)tl * HD + h * p.d;
#pragma unroll
    for (int e = 0; e < VE; ++e) { row[m0 + e] = klo[e]; row[m0 + half + e] = khi[e]; }
  }
  __syncthreads();
  for (int c = tid; c < HD; c += kAppendThreads) {
    float s = 0.f;
    for (int t = 0; t < p.tok_per_block; ++t) s += s_sum[(size_t)t * HD + c];
    p.partial[(size_t)blockIdx.x * HD + c] = s;
  }
  __syncthreads();
  if (tid == 0) s_last = last_block_ticket(p.counter, blockIdx.x, gridDim.x) ? 1 : 0;
  __syncthreads();
  if (!s_last) return;
  // last block: add the per-block partial sums in a fixed order (=> deterministic k_sum).  One
  // float4 column per thread, `groups` thread groups striding over the blocks with all their loads
  // in flight at once (the loads are L2 round trips and this block is the kernel's critical path),
  // then the group sums are combined in group order through shared memory.
  const int nblk_used = (n_fit + p.tok_per_block - 1) / p.tok_per_block;
  float* ks = p.k_sum + (size_t)p.page_id * HD;
  const int nq4 = HD / 4;
  const int cols = min(nq4, kAppendThreads), groups = kAppendThreads / cols;
  const int grp = tid / cols, cl = tid - grp * cols;
  float4* s4 = reinterpret_cast<float4*>(s_sum);
  for (int q0 = 0; q0 < nq4; q0 += cols) {
    const int q = q0 + cl;
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    if (q < nq4 && grp < groups) {
      const float4* src = reinterpret_cast<const float4*>(p.partial) + q;
#pragma unroll 16
      for (int bb = grp; bb < nblk_used; bb += groups) {
        const float4 v = __ldcg(src + (size_t)bb * nq4);
        acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
      }
    }
    __syncthreads();
    if (grp < groups) s4[grp * cols + cl] = acc;
    __syncthreads();
    if (grp == 0 && q < nq4) {
      float4 t = p.page_offset > 0 ? reinterpret_cast<const float4*>(ks)[q] : make_float4(0.f, 0.f, 0.f, 0.f);
      for (int g2 = 0; g2 < groups; ++g2) {
        const float4 v = s4[g2 * cols + cl];
        t.x += v.x; t.y += v.y; t.z += v.z; t.w += v.w;
      }
      reinterpret_cast<float4*>(ks)[q] = t;
    }
  }
  if (tid == 0) {
    p.page_len[p.page_id] = p.page_offset + n_fit;
    if (p.status && (clamped || overflow))
      atomicOr(p.status, (clamped ? VCS_FLAG_COUNT_CLAMPED : 0) | (overflow ? VCS_FLAG_PAGE_OVERFLOW : 0));
  }
}

static int append_tok_per_block(const vcs_kv_pool* pool) {
  const int ve = pool->dtype == VCS_BF16 ? 8 : 4;
  const int vec_per_tok = pool->Hkv * (pool->d / 2 / ve);
  int t = kAppendThreads / vec_per_tok;
  return t < 1 ? 0 : t;
}

}  // namespace vcs

using namespace vcs;

extern "C" size_t vcs_kv_append_workspace_bytes(const vcs_kv_pool* pool, int n_cap) {
  if (!pool || n_cap < 0) return 0;
  const int tpb = append_tok_per_block(pool);
  if (tpb == 0) return 0;
  const size_t nblk = (size_t)(n_cap + tpb - 1) / tpb + 1;
  return kTicketBytes + nblk * pool->Hkv * pool->d * sizeof(float);
}

extern "C" int vcs_kv_append_pages(const vcs_kv_pool* pool, const void* k, const void* v, int64_t k_row_stride,
                                   int64_t v_row_stride, const int32_t* pos3, const int32_t* n_d, int n_cap,
                                   int32_t page_id, int32_t page_offset, int32_t* status_d, void* workspace,
                                   size_t workspace_bytes, void* stream) {
  int rc = validate_pool(pool, true);
  if (rc != VCS_OK) return rc;
  if (n_cap < 0) VCS_FAIL(VCS_EINVAL, "kv_append: n_cap < 0");
  if (page_id < 0 || page_id >= pool->n_pages) VCS_FAIL(VCS_ECAP, "kv_append: page_id %d out of range [0,%d)", page_id, pool->n_pages);
  if (page_offset < 0 || page_offset > pool->page_cap) VCS_FAIL(VCS_ECAP, "kv_append: page_offset %d out of range", page_offset);
  if (!workspace) VCS_FAIL(VCS_EINVAL, "kv_append: NULL workspace");
  if (n_cap > 0 && (!k || !v || !pos3)) VCS_FAIL(VCS_EINVAL, "kv_append: NULL k / v / pos3");
  const size_t eb = elem_bytes(pool->dtype);
  const int64_t min_stride = (int64_t)pool->Hkv * pool->d;
  if (n_cap > 0 && (k_row_stride < min_stride || v_row_stride < min_stride))
    VCS_FAIL(VCS_EINVAL, "kv_append: row stride smaller than Hkv*d");
  if (n_cap > 0 && (!aligned16(k) || !aligned16(v) || (k_row_stride * eb) % 16 || (v_row_stride * eb) % 16))
    VCS_FAIL(VCS_EALIGN, "kv_append: k / v and their row strides must be 16-byte aligned");
  const int tpb = append_tok_per_block(pool);
  if (tpb == 0) VCS_FAIL(VCS_EUNSUPPORTED, "kv_append: Hkv*d too large for one block");
  if (workspace_bytes < vcs_kv_append_workspace_bytes(pool, n_cap)) VCS_FAIL(VCS_ECAP, "kv_append: workspace too small");

  AppendParams p;
  p.k = k; p.v = v; p.k_stride = k_row_stride; p.v_stride = v_row_stride;
  p.pos3 = pos3; p.n_d = n_d; p.n_cap = n_cap; p.page_id = page_id; p.page_offset = page_offset;
  p.k_pages = pool->k_pages; p.v_pages = pool->v_pages; p.page_len = pool->page_len; p.k_sum = pool->k_sum;
  p.page_cap = pool->page_cap; p.Hkv = pool->Hkv; p.d = pool->d; p.status = status_d;
  p.counter = reinterpret_cast<unsigned int*>(workspace);
  p.partial = reinterpret_cast<float*>(static_cast<char*>(workspace) + kTicketBytes);
  p.tok_per_block = tpb;
  p.rope = rope_params(pool);

  const int nblk = n_cap > 0 ? (n_cap + tpb - 1) / tpb : 1;
  const size_t smem = (size_t)tpb * pool->Hkv * pool->d * sizeof(float);
  cudaStream_t st = (cudaStream_t)stream;
  if (pool->dtype == VCS_BF16) launch_pdl(append_kernel<__nv_bfloat16>, dim3(nblk), dim3(kAppendThreads), smem, st, p);
  else launch_pdl(append_kernel<float>, dim3(nblk), dim3(kAppendThreads), smem, st, p);
  cudaError_t err = cudaGetLastError();
  if (err != cudaSuccess) VCS_FAIL(VCS_ECUDA, "kv_append launch: %s", cudaGetErrorString(err));
  return VCS_OK;
}
