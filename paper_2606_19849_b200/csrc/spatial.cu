// vcs_spatial_entropy_topk: entropy-based spatial token selection (Table 8-middle
// PAPER.md:335-336).  Per token I(x) = -sum_m p_m log p_m with p = softmax(x) over the D feature
// dimensions (reading D30); per frame (temporal group) the K tokens with the highest
// entropy are retained, ties -> lower index, output in ascending sequence order.
//
// HBM-bound like the temporal drop: one warp per token, 128-bit loads; the second sweep over the
// token (sums after the max) hits L1.  One block per (stream, frame) then ranks the P entropies in
// shared memory (P^2 comparisons, P ~ 1e3) and compacts the winners with warp ballots.
#include "common.cuh"

namespace vcs {

constexpr int kEntThreads = 256;

template <typename E>
__device__ __forceinline__ void unpack_vec(const uint4& v, float* f);
template <>
__device__ __forceinline__ void unpack_vec<__nv_bfloat16>(const uint4& v, float* f) {
  f[0] = bf16_lo(v.x); f[1] = bf16_hi(v.x); f[2] = bf16_lo(v.y); f[3] = bf16_hi(v.y);
  f[4] = bf16_lo(v.z); f[5] = bf16_hi(v.z); f[6] = bf16_lo(v.w); f[7] = bf16_hi(v.w);
}
template <>
__device__ __forceinline__ void unpack_vec<float>(const uint4& v, float* f) {
  f[0] = __uint_as_float(v.x); f[1] = __uint_as_float(v.y); f[2] = __uint_as_float(v.z); f[3] = __uint_as_float(v.w);
}

// entropy[token] for n_tok tokens of D features
template <typename E>
__global__ void __launch_bounds__(kEntThreads) entropy_kernel(const E* z, long long n_tok, int D, float* entropy) {
  pdl_wait();
  pdl_launch_dependents();
  constexpr int VE = 16 / sizeof(E);
  const int lane = threadIdx.x & 31;
  const long long tok = (long long)blockIdx.x * (kEntThreads / 32) + (threadIdx.x >> 5);
  if (tok >= n_tok) return;
  const uint4* row = reinterpret_cast<const uint4*>(z + tok * D);
  const int nvec = D / VE;
  float m = -INFINITY;
  for (int v = lane; v < nvec; v += 32) {
    float f[VE];
    unpack_vec<E>(__ldg(row + v), f);
#pragma unroll
    for (int e = 0; e < VE; ++e) m = fmaxf(m, f[e]);
  }
  m = warp_max(m);
  // H = log(S) - T / S with S = sum e^(x-m), T = sum (x-m) e^(x-m)
  float S = 0.f, T = 0.f;
  for (int v = lane; v < nvec; v += 32) {
    float f[VE];
    unpack_vec<E>(__ldg(row + v), f);
#pragma unroll
    for (int e = 0; e < VE; ++e) {
      const float x = f[e] - m, w = expf(x);
      S += w;
      T = fmaf(x, w, T);
    }
  }
  S = warp_sum(S);
  T = warp_sum(T);
  if (lane == 0) entropy[tok] = logf(S) - T / S;
}

struct SelectParams {
  const float* entropy;   // [B][G][P]
  int G, P, K;
  int32_t* kept_idx;      // [B][G*K]
  int32_t* kept_count;    // [B]
  int32_t* pos3;          // [B][G*K][3] or null
  int Hg, Wg, t_stride;
  const int32_t* pos_base;
};

// one block per (frame g = blockIdx.x, stream b = blockIdx.y)
__global__ void __launch_bounds__(kEntThreads) entropy_select_kernel(const SelectParams p) {
  pdl_wait();
  pdl_launch_dependents();
  extern __shared__ float s_h[];   // [P]
  __shared__ int s_warp[kEntThreads / 32];
  __shared__ int s_base;
  const int g = blockIdx.x, b = blockIdx.y;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const float* h = p.entropy + ((size_t)b * p.G + g) * p.P;
  for (int i = threadIdx.x; i < p.P; i += kEntThreads) s_h[i] = h[i];
  if (threadIdx.x == 0) s_base = 0;
  __syncthreads();
  const int K = min(p.K, p.P);
  int32_t* idx = p.kept_idx + (size_t)b * p.G * K + (size_t)g * K;
  int32_t* pos = p.pos3 ? p.pos3 + ((size_t)b * p.G * K + (size_t)g * K) * 3 : nullptr;
  const int base = p.pos_base ? p.pos_base[b] : 0;
  for (int i0 = 0; i0 < p.P; i0 += kEntThreads) {
    const int i = i0 + threadIdx.x;
    bool keep = false;
    if (i < p.P) {
      const float hi = s_h[i];
      int rank = 0;   // tokens that beat token i: higher entropy, or equal entropy and lower index
      for (int j = 0; j < p.P; ++j) {
        const float hj = s_h[j];
        rank += (hj > hi || (hj == hi && j < i)) ? 1 : 0;
      }
      keep = rank < K;
    }
    const unsigned bal = __ballot_sync(0xffffffffu, keep);
    if (lane == 0) s_warp[warp] = __popc(bal);
    __syncthreads();
    int off = s_base;
    for (int w = 0; w < warp; ++w) off += s_warp[w];
    off += __popc(bal & ((1u << lane) - 1u));
    if (keep) {
      idx[off] = g * p.P + i;
      if (pos) {
        const int r = i / p.Wg, c = i - r * p.Wg;
        pos[3 * off + 0] = base + g * p.t_stride;
        pos[3 * off + 1] = base + r;
        pos[3 * off + 2] = base + c;
      }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
      int t = s_base;
      for (int w = 0; w < kEntThreads / 32; ++w) t += s_warp[w];
      s_base = t;
    }
    __syncthreads();
  }
  if (g == 0 && threadIdx.x == 0) p.kept_count[b] = p.G * K;
}

}  // namespace vcs

using namespace vcs;

extern "C" size_t vcs_spatial_entropy_topk_workspace_bytes(int B, int G, int P) {
  if (B <= 0 || G <= 0 || P <= 0) return 0;
  return round_up((size_t)B * G * P * sizeof(float), 256);
}

extern "C" int vcs_spatial_entropy_topk(const void* z, int B, int G, int P, int D, int dtype, int K, int32_t* kept_idx,
                                        int32_t* kept_count, float* entropy, int32_t* pos3, int Hg, int Wg, int t_stride,
                                        const int32_t* pos_base_d, void* workspace, size_t workspace_bytes, void* stream) {
  if (B < 0 || G <= 0 || P < 0 || D <= 0 || K < 0) VCS_FAIL(VCS_EINVAL, "spatial_entropy_topk: bad sizes B=%d G=%d P=%d D=%d K=%d", B, G, P, D, K);
  if (dtype != VCS_F32 && dtype != VCS_BF16) VCS_FAIL(VCS_EUNSUPPORTED, "spatial_entropy_topk: dtype %d", dtype);
  cudaStream_t st = (cudaStream_t)stream;
  if (B == 0 || P == 0) {
    if (B > 0 && kept_count) VCS_CUDA_OK(cudaMemsetAsync(kept_count, 0, sizeof(int32_t) * B, st));
    return VCS_OK;
  }
  if (!z || !kept_idx || !kept_count) VCS_FAIL(VCS_EINVAL, "spatial_entropy_topk: NULL z / kept_idx / kept_count");
  if (!entropy && (!workspace || workspace_bytes < vcs_spatial_entropy_topk_workspace_bytes(B, G, P)))
    VCS_FAIL(VCS_ECAP, "spatial_entropy_topk: workspace too small");
  if (pos3 && ((long long)Hg * Wg != P || Hg <= 0 || Wg <= 0)) VCS_FAIL(VCS_EINVAL, "spatial_entropy_topk: pos3 needs Hg*Wg == P");
  if (!aligned16(z) || ((size_t)D * elem_bytes(dtype)) % 16 != 0)
    VCS_FAIL(VCS_EALIGN, "spatial_entropy_topk: z must be 16-byte aligned and D*elem_size a multiple of 16");
  if ((size_t)P * sizeof(float) > 200 * 1024) VCS_FAIL(VCS_ECAP, "spatial_entropy_topk: P too large for one block");
  float* h = entropy ? entropy : static_cast<float*>(workspace);
  const long long n_tok = (long long)B * G * P;
  const unsigned nblk = (unsigned)((n_tok + kEntThreads / 32 - 1) / (kEntThreads / 32));
  cudaError_t err;
  if (dtype == VCS_BF16) err = launch_pdl(entropy_kernel<__nv_bfloat16>, dim3(nblk), dim3(kEntThreads), 0, st,
                                          static_cast<const __nv_bfloat16*>(z), n_tok, D, h);
  else err = launch_pdl(entropy_kernel<float>, dim3(nblk), dim3(kEntThreads), 0, st, static_cast<const float*>(z), n_tok, D, h);
  if (err != cudaSuccess) VCS_FAIL(VCS_ECUDA, "spatial_entropy_topk launch: %s", cudaGetErrorString(err));
  SelectParams p;
  p.entropy = h; p.G = G; p.P = P; p.K = K; p.kept_idx = kept_idx; p.kept_count = kept_count; p.pos3 = pos3;
  p.Hg = Hg; p.Wg = Wg > 0 ? Wg : 1; p.t_stride = t_stride; p.pos_base = pos_base_d;
  const size_t smem = (size_t)P * sizeof(float);
  if (smem > 48 * 1024) VCS_CUDA_OK(cudaFuncSetAttribute(entropy_select_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  err = launch_pdl(entropy_select_kernel, dim3(G, B), dim3(kEntThreads), smem, st, p);
  if (err == cudaSuccess) err = cudaGetLastError();
  if (err != cudaSuccess) VCS_FAIL(VCS_ECUDA, "spatial_entropy_topk launch: %s", cudaGetErrorString(err));
  return VCS_OK;
}
