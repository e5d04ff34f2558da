// SIMT bounded-attention kernel (fp32 arithmetic end to end): the production path for the fp32
// Tiny configuration and for shapes the tcgen05 kernel does not take (head_dim 64), and a second,
// structurally different GPU implementation that the tests run against the tensor-core kernel.
// One warp per (query row, q head); lanes own keys for Q.K^T and d-slices for P.V; online softmax.
// Computes PAPER.md:129 / :138 over the page-table visible set with the causal self page.
#include "common.cuh"
#include "attn.cuh"

namespace vcs {

constexpr int kSimtRows = 4;  // warps (query rows) per block

template <typename E>
struct Ld;
template <>
struct Ld<__nv_bfloat16> {
  static constexpr int kElems = 8;
  static __device__ __forceinline__ void unpack(const uint4& v, float* f) {
    f[0] = bf16_lo(v.x); f[1] = bf16_hi(v.x); f[2] = bf16_lo(v.y); f[3] = bf16_hi(v.y);
    f[4] = bf16_lo(v.z); f[5] = bf16_hi(v.z); f[6] = bf16_lo(v.w); f[7] = bf16_hi(v.w);
  }
  static __device__ __forceinline__ float load1(const __nv_bfloat16* p) { return __bfloat162float(*p); }
  static __device__ __forceinline__ void store1(__nv_bfloat16* p, float v) { *p = __float2bfloat16_rn(v); }
};
template <>
struct Ld<float> {
  static constexpr int kElems = 4;
  static __device__ __forceinline__ void unpack(const uint4& v, float* f) {
    f[0] = __uint_as_float(v.x); f[1] = __uint_as_float(v.y); f[2] = __uint_as_float(v.z); f[3] = __uint_as_float(v.w);
  }
  static __device__ __forceinline__ float load1(const float* p) { return *p; }
  static __device__ __forceinline__ void store1(float* p, float v) { *p = v; }
};

template <typename E, int HD>
__global__ void __launch_bounds__(kSimtRows * 32) attn_simt_kernel(const AttnParams p) {
  pdl_wait();
  pdl_launch_dependents();
  constexpr int VE = Ld<E>::kElems;
  constexpr int PER = HD / 32;  // output elements per lane
  __shared__ float s_q[kSimtRows][HD];

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int h = blockIdx.y, kvh = h / (p.Hq / p.Hkv), b = blockIdx.z;
  const int i = blockIdx.x * kSimtRows + warp;  // query row
  int nq = p.nq_d ? p.nq_d[b] : p.nq_cap;
  if (nq > p.nq_cap) {
    nq = p.nq_cap;
    if (p.status && threadIdx.x == 0 && blockIdx.x == 0 && h == 0) atomicOr(p.status, VCS_FLAG_COUNT_CLAMPED);
  }
  if (i >= nq) return;
  const int32_t* q_pos3 = p.q_pos3 + (size_t)b * p.nq_cap * 3;
  const int32_t* page_table = p.page_table + (size_t)b * p.n_vis_cap;
  int self_page = p.self_pages_d ? p.self_pages_d[b] : p.self_page;
  if (self_page >= p.n_pages) self_page = -1;

  // rotate the query row (M-RoPE, pairs (m, m + d/2)) and fold in the softmax scale
  {
    const E* q = static_cast<const E*>(p.q) + (size_t)b * p.q_bstride + (size_t)i * p.q_stride + (size_t)h * HD;
    const int pt = q_pos3[3 * i + 0], ph = q_pos3[3 * i + 1], pw = q_pos3[3 * i + 2];
    for (int m = lane; m < HD / 2; m += 32) {
      const int ax = p.rope.axis_of[m];
      const int pos = ax == 0 ? pt : (ax == 1 ? ph : pw);
      float s, c;
      rope_sincos(pos, p.rope.inv_freq[m], &s, &c);
      const float lo = Ld<E>::load1(q + m), hi = Ld<E>::load1(q + m + HD / 2);
      s_q[warp][m] = (lo * c - hi * s) * p.scale;
      s_q[warp][m + HD / 2] = (hi * c + lo * s) * p.scale;
    }
  }
  __syncwarp();

  float m_run = -INFINITY, l_run = 0.f;
  float acc[PER];
#pragma unroll
  for (int e = 0; e < PER; ++e) acc[e] = 0.f;

  int n_vis = p.n_vis_d ? p.n_vis_d[b] : p.n_vis_cap;
  n_vis = max(0, min(n_vis, p.n_vis_cap));
  const int n_pages_iter = n_vis + (self_page >= 0 ? 1 : 0);

  for (int pi = 0; pi < n_pages_iter; ++pi) {
    const bool is_self = pi == n_vis;
    const int page = is_self ? self_page : page_table[pi];
    if (page < 0 || page >= p.n_pages) {
      if (page != -1 && p.status && lane == 0) atomicOr(p.status, VCS_FLAG_BAD_PAGE);   // -1 is padding
      continue;
    }
    int len = min(p.page_len[page], p.page_cap);
    if (is_self) len = min(len, p.self_offset + i + 1);  // causal inside the current chunk
    const E* Kp = static_cast<const E*>(p.k_pages) + ((size_t)page * p.Hkv + kvh) * p.page_cap * HD;
    const E* Vp = static_cast<const E*>(p.v_pages) + ((size_t)page * p.Hkv + kvh) * p.page_cap * HD;
    for (int t0 = 0; t0 < len; t0 += 32) {
      const int tok = t0 + lane;
      float s = -INFINITY;
      if (tok < len) {
        const uint4* kr = reinterpret_cast<const uint4*>(Kp + (size_t)tok * HD);
        float dot = 0.f;
#pragma unroll 4
        for (int v = 0; v < HD / VE; ++v) {
          float f[VE];
          Ld<E>::unpack(__ldg(kr + v), f);
#pragma unroll
          for (int e = 0; e < VE; ++e) dot = fmaf(s_q[warp][v * VE + e], f[e], dot);
        }
        s = dot;
      }
      const float m_new = fmaxf(m_run, warp_max(s));   // finite: tile has >= 1 valid key
      const float pj = tok < len ? expf(s - m_new) : 0.f;
      const float corr = expf(m_run - m_new);           // 0 on the first tile (m_run = -inf)
      l_run = l_run * corr + warp_sum(pj);
#pragma unroll
      for (int e = 0; e < PER; ++e) acc[e] *= corr;
      const int cnt = min(32, len - t0);
      for (int j = 0; j < cnt; ++j) {
        const float w = __shfl_sync(0xffffffffu, pj, j);
        const E* vr = Vp + (size_t)(t0 + j) * HD + lane * PER;
#pragma unroll
        for (int e = 0; e < PER; ++e) acc[e] = fmaf(w, Ld<E>::load1(vr + e), acc[e]);
      }
      m_run = m_new;
    }
  }

  E* o = static_cast<E*>(p.out) + (size_t)b * p.out_bstride + (size_t)i * p.out_stride + (size_t)h * HD + lane * PER;
  const float inv = l_run > 0.f ? 1.f / l_run : 0.f;
#pragma unroll
  for (int e = 0; e < PER; ++e) Ld<E>::store1(o + e, acc[e] * inv);
  if (p.lse && lane == 0) p.lse[((size_t)b * p.Hq + h) * p.nq_cap + i] = l_run > 0.f ? m_run + logf(l_run) : -INFINITY;
}

int launch_attn_simt(const AttnParams& p, int dtype, cudaStream_t st) {
  dim3 grid((p.nq_cap + kSimtRows - 1) / kSimtRows, p.Hq, p.B);
  dim3 block(kSimtRows * 32);
  if (dtype == VCS_BF16 && p.d == 128) launch_pdl(attn_simt_kernel<__nv_bfloat16, 128>, dim3(grid), dim3(block), 0, st, p);
  else if (dtype == VCS_BF16 && p.d == 64) launch_pdl(attn_simt_kernel<__nv_bfloat16, 64>, dim3(grid), dim3(block), 0, st, p);
  else if (dtype == VCS_F32 && p.d == 128) launch_pdl(attn_simt_kernel<float, 128>, dim3(grid), dim3(block), 0, st, p);
  else if (dtype == VCS_F32 && p.d == 64) launch_pdl(attn_simt_kernel<float, 64>, dim3(grid), dim3(block), 0, st, p);
  else VCS_FAIL(VCS_EUNSUPPORTED, "attention: dtype %d / head_dim %d", dtype, p.d);
  cudaError_t err = cudaGetLastError();
  if (err != cudaSuccess) VCS_FAIL(VCS_ECUDA, "attention (SIMT) launch: %s", cudaGetErrorString(err));
  return VCS_OK;
}

}  // namespace vcs
