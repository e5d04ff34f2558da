// vcs_temporal_drop: chunk-level temporal token dropping (Eq. 1-2) fused
// with stream compaction into a kept-index list.
//
// HBM-bound: every token is read exactly once with 128-bit coalesced loads; the G norms and
// G(G-1)/2 dot products of a position live in registers (fp32 FMA of exact bf16 products).
// One position is owned by `split` warps (each a contiguous D-slice) so that a single small
// chunk still puts all of its bytes in flight at once; B independent streams batch in grid.y.
// The last block of a stream to finish (ticket counter) scans that stream's T keep flags and
// writes kept_idx / pos3 / kept_count -- no second launch, no host round trip.
#include "common.cuh"

namespace vcs {

constexpr int kDropWarps = 8;
constexpr int kDropThreads = kDropWarps * 32;
constexpr int kMaxNT = 9;  // templated token counts: G <= 8 (+1 for the previous chunk's last group)

struct DropParams {
  const void* z;
  const void* prev;
  int B, G, P, D;
  float tau;
  int mode, has_prev;
  int split, pos_per_block;
  uint8_t* mask;        // [B][T]
  int32_t* kept_idx;    // [B][T]
  int32_t* kept_count;  // [B]
  int32_t* pos3;        // [B][T][3] or null
  int Hg, Wg, t_stride;
  const int32_t* pos_base;
  unsigned int* counters;  // [B] two-level tickets, counter_stride ints apart
  int counter_stride;
};

template <typename E>
struct Vec;
template <>
struct Vec<__nv_bfloat16> {
  static constexpr int kElems = 8;
  static __device__ __forceinline__ void unpack(const uint4& v, float* f) {
    f[0] = bf16_lo(v.x); f[1] = bf16_hi(v.x); f[2] = bf16_lo(v.y); f[3] = bf16_hi(v.y);
    f[4] = bf16_lo(v.z); f[5] = bf16_hi(v.z); f[6] = bf16_lo(v.w); f[7] = bf16_hi(v.w);
  }
};
template <>
struct Vec<float> {
  static constexpr int kElems = 4;
  static __device__ __forceinline__ void unpack(const uint4& v, float* f) {
    f[0] = __uint_as_float(v.x); f[1] = __uint_as_float(v.y);
    f[2] = __uint_as_float(v.z); f[3] = __uint_as_float(v.w);
  }
};

// index of pair (i<j) in the packed upper triangle, NT tokens
template <int NT>
__device__ __forceinline__ constexpr int pair_idx(int i, int j) {
  return i * NT - i * (i + 1) / 2 + (j - i - 1);
}

// Eq. 1-2 without sqrt / divide: S = dot / sqrt(ni nj) > tau, decided on squared quantities (the
// decide step runs in one lane per position, so its instruction count is latency, not throughput).
// Reading D6: S := 0 when a norm is 0.  fp32 throughout; the generators keep |S - tau| >= 1e-4.
__device__ __forceinline__ bool sim_gt(float dot, float ni, float nj, float tau) {
  if (ni == 0.f || nj == 0.f) return 0.f > tau;
  const float rhs = tau * tau * (ni * nj);
  const float d2 = dot * dot;
  return tau >= 0.f ? (dot > 0.f && d2 > rhs) : (dot >= 0.f || d2 < rhs);
}

#ifdef VCS_DROP_TRACE
__device__ long long g_drop_trace[8192 * 4];
__device__ __forceinline__ long long gtime() { unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return (long long)t; }
#define DTRACE(slot) do { if (threadIdx.x == 0 && blockIdx.y == 0 && blockIdx.x < 8192) g_drop_trace[blockIdx.x * 4 + (slot)] = gtime(); } while (0)
#define TTRACE(slot) do { if (threadIdx.x == 0) { g_drop_trace[8192 * 4 - 16 + (slot)] = gtime(); g_drop_trace[8192 * 4 - 8 + (slot)] = clock64(); } } while (0)
#else
#define DTRACE(slot) do { } while (0)
#define TTRACE(slot) do { } while (0)
#endif

// Block-wide tail: scan the T keep flags of stream b (g-major order) and emit the compacted list.
// Warp w owns the contiguous token range [w*C, (w+1)*C); a step handles 32 consecutive tokens
// (one flag per lane, __ballot_sync), so kept tokens of a step land in consecutive output slots
// and every store of idx / pos3 is coalesced.  Pass 1 counts, a tiny scan over the 8 warps gives
// each warp its base, pass 2 re-reads the flags (L2/L1 hits) and writes.
__device__ void drop_compact_tail(const DropParams& p, int b) {
  __shared__ int s_warp[kDropWarps];
  const int T = p.G * p.P;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint8_t* mask = p.mask + (size_t)b * T;
  int32_t* idx = p.kept_idx + (size_t)b * T;
  int32_t* pos = p.pos3 ? p.pos3 + (size_t)b * T * 3 : nullptr;
  const int base = p.pos_base ? p.pos_base[b] : 0;
  const int C = ((T + kDropWarps * 32 - 1) / (kDropWarps * 32)) * 32;
  const int lo = min(T, warp * C), hi = min(T, lo + C);
  const unsigned lt = (1u << lane) - 1u;
  TTRACE(0);
  // The flag loads are L2 round trips: issue them all before the first ballot (bit s of `mine` =
  // this lane's flag in step s), 32 steps = 1024 tokens per warp per super-step.
  int running = 0;   // kept tokens of all warps in the super-steps done so far
  const float inv_P = 1.0f / (float)p.P, inv_W = 1.0f / (float)p.Wg;
  for (int s0 = 0; s0 < C; s0 += 1024) {
    const int nsteps = min(32, (C - s0) / 32);
    unsigned mine = 0u;
#pragma unroll 8
    for (int s = 0; s < nsteps; ++s) {
      const int i = lo + s0 + 32 * s + lane;
      if (i < hi) mine |= (__ldcg(mask + i) != 0 ? 1u : 0u) << s;
    }
    int cnt = 0;
#pragma unroll 1
    for (int s = 0; s < nsteps; ++s) cnt += __popc(__ballot_sync(0xffffffffu, (mine >> s) & 1u));
    __syncthreads();
    if (lane == 0) s_warp[warp] = cnt;
    __syncthreads();
    int off = running, total = 0;
#pragma unroll
    for (int k = 0; k < kDropWarps; ++k) {
      const int c = s_warp[k];
      off += k < warp ? c : 0;
      total += c;
    }
    running += total;
#pragma unroll 1
    for (int s = 0; s < nsteps; ++s) {
      const bool keep = (mine >> s) & 1u;
      const unsigned bal = __ballot_sync(0xffffffffu, keep);
      if (keep) {
        const int i = lo + s0 + 32 * s + lane;
        const int o = off + __popc(bal & lt);
        idx[o] = i;
        if (pos) {
          // exact floor divisions by reciprocal + one correction step (i < 2^24 * ... is not assumed)
          int g = __float2int_rz(__int2float_rz(i) * inv_P);
          g += (g + 1) * p.P <= i ? 1 : 0;  g -= g * p.P > i ? 1 : 0;
          const int pp = i - g * p.P;
          int r = __float2int_rz(__int2float_rz(pp) * inv_W);
          r += (r + 1) * p.Wg <= pp ? 1 : 0;  r -= r * p.Wg > pp ? 1 : 0;
          pos[3 * o + 0] = base + g * p.t_stride;
          pos[3 * o + 1] = base + r;
          pos[3 * o + 2] = base + (pp - r * p.Wg);
        }
      }
      off += __popc(bal);
    }
  }
  const int total = running;
  TTRACE(3);
  for (int i = total + tid; i < T; i += kDropThreads) idx[i] = -1;
  if (tid == 0) p.kept_count[b] = total;
  TTRACE(4);
}

template <int NT>
__device__ __forceinline__ void drop_decide(const DropParams& p, int b, int pos, const float* acc) {
  // acc: [0,NT) squared norms, then packed upper-triangle dots
  const int T = p.G * p.P;
  uint8_t* mask = p.mask + (size_t)b * T;
  if (p.mode == VCS_DROP_CHUNK_ALLPAIRS) {
    bool drop = NT > 1;
#pragma unroll
    for (int i = 0; i < NT; ++i)
#pragma unroll
      for (int j = i + 1; j < NT; ++j)
        drop = drop && sim_gt(acc[NT + pair_idx<NT>(i, j)], acc[i], acc[j], p.tau);
    mask[pos] = 1;  // first group = anchor
    for (int g = 1; g < p.G; ++g) mask[g * p.P + pos] = drop ? 0 : 1;
  } else {
    // token list: [prev,] group 0 .. G-1; group g is dropped iff S(previous token, it) > tau
    const int first = p.has_prev ? 1 : 0;  // list index of group 0
    if (!p.has_prev) mask[pos] = 1;
#pragma unroll
    for (int t = 1; t < NT; ++t) {
      const bool drop = sim_gt(acc[NT + pair_idx<NT>(t - 1, t)], acc[t - 1], acc[t], p.tau);
      mask[(t - first) * p.P + pos] = drop ? 0 : 1;
    }
  }
}

template <int NT, typename E>
__global__ void __launch_bounds__(kDropThreads) drop_kernel(const DropParams p) {
  pdl_wait();
  pdl_launch_dependents();
  constexpr int NACC = NT + NT * (NT - 1) / 2;
  constexpr int VE = Vec<E>::kElems;
  constexpr bool kLaneReduce = NACC <= 14;   // NT <= 4: 8 x 14 x 32 floats = 14 KB of shared memory
  __shared__ float s_part[kLaneReduce ? 1 : kDropWarps][kLaneReduce ? 1 : NACC];
  __shared__ float s_lane[kLaneReduce ? kDropWarps : 1][kLaneReduce ? NACC : 1][kLaneReduce ? 32 : 1];
  __shared__ int s_last;

  const int b = blockIdx.y;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int slot = warp / p.split, sub = warp - slot * p.split;
  const int pos = blockIdx.x * p.pos_per_block + slot;
  const bool active = slot < p.pos_per_block && pos < p.P;

  float acc[NACC];
#pragma unroll
  for (int i = 0; i < NACC; ++i) acc[i] = 0.f;
  DTRACE(0);

#if defined(VCS_DROP_EXP) && (VCS_DROP_EXP & 1)
  if (false) {
#else
  if (active && NT > 1) {
#endif
    const int nvec = p.D / VE;
    const int per = (nvec + p.split - 1) / p.split;
    const int v0 = sub * per, v1 = min(nvec, v0 + per);
    const uint4* tok[NT];
    {
      const int first = (p.mode == VCS_DROP_CONSECUTIVE && p.has_prev) ? 1 : 0;
      if (first) tok[0] = reinterpret_cast<const uint4*>(static_cast<const E*>(p.prev) + ((size_t)b * p.P + pos) * p.D);
#pragma unroll
      for (int t = first; t < NT; ++t)
        tok[t] = reinterpret_cast<const uint4*>(static_cast<const E*>(p.z) +
                                                (((size_t)b * p.G + (t - first)) * p.P + pos) * p.D);
    }
    auto accumulate = [&](const uint4 (&x)[NT]) {
      float f[NT][VE];
#pragma unroll
      for (int t = 0; t < NT; ++t) Vec<E>::unpack(x[t], f[t]);
#pragma unroll
      for (int e = 0; e < VE; ++e) {
#pragma unroll
        for (int i = 0; i < NT; ++i) {
          acc[i] = fmaf(f[i][e], f[i][e], acc[i]);
#pragma unroll
          for (int j = i + 1; j < NT; ++j)
            acc[NT + pair_idx<NT>(i, j)] = fmaf(f[i][e], f[j][e], acc[NT + pair_idx<NT>(i, j)]);
        }
      }
    };
    // two 16-byte vectors per token in flight per lane (NT x 1 KB per warp), then a one-vector tail
    int v = v0 + lane;
#pragma unroll 1
    for (; v + 32 < v1; v += 64) {
      uint4 x0[NT], x1[NT];
#pragma unroll
      for (int t = 0; t < NT; ++t) x0[t] = ldg_nc_v4(tok[t] + v);
#pragma unroll
      for (int t = 0; t < NT; ++t) x1[t] = ldg_nc_v4(tok[t] + v + 32);
      accumulate(x0);
      accumulate(x1);
    }
    if (v < v1) {
      uint4 x0[NT];
#pragma unroll
      for (int t = 0; t < NT; ++t) x0[t] = ldg_nc_v4(tok[t] + v);
      accumulate(x0);
    }
  }

  // Cross-lane / cross-warp reduction.  With split > 1 and few accumulators the `split` warps of a
  // position first add their per-lane partials through shared memory, so only ONE warp per
  // position pays the NACC x 5 shuffle butterflies (they dominate a small chunk otherwise).
  if constexpr (kLaneReduce) {
    if (p.split > 1) {
#pragma unroll
      for (int i = 0; i < NACC; ++i) s_lane[warp][i][lane] = acc[i];
      __syncthreads();
      if (sub == 0) {
        for (int s = 1; s < p.split; ++s)
#pragma unroll
          for (int i = 0; i < NACC; ++i) acc[i] += s_lane[warp + s][i][lane];
      }
    }
    if (sub == 0) {
#pragma unroll
      for (int i = 0; i < NACC; ++i) acc[i] = warp_sum(acc[i]);
    }
  } else {
#pragma unroll
    for (int i = 0; i < NACC; ++i) acc[i] = warp_sum(acc[i]);
    if (p.split > 1) {
      if (lane == 0) {
#pragma unroll
        for (int i = 0; i < NACC; ++i) s_part[warp][i] = acc[i];
      }
      __syncthreads();
      if (active && sub == 0 && lane == 0) {
        for (int s = 1; s < p.split; ++s)
#pragma unroll
          for (int i = 0; i < NACC; ++i) acc[i] += s_part[warp + s][i];
      }
    }
  }
#if defined(VCS_DROP_EXP) && (VCS_DROP_EXP & 2)
  if (active && sub == 0 && lane == 0) { for (int g = 0; g < p.G; ++g) p.mask[(size_t)b * p.G * p.P + g * p.P + pos] = acc[0] > 1e30f ? 0 : 1; }
#else
  if (active && sub == 0 && lane == 0) drop_decide<NT>(p, b, pos, acc);
#endif

  // ticket: the last block of stream b compacts it
  __syncthreads();
  DTRACE(1);
  if (threadIdx.x == 0)
    s_last = last_block_ticket(p.counters + (size_t)b * p.counter_stride, blockIdx.x, gridDim.x) ? 1 : 0;
  __syncthreads();
  DTRACE(2);
  if (s_last) drop_compact_tail(p, b);
#ifdef VCS_DROP_TRACE
  __syncthreads();
  DTRACE(3);
#ifdef VCS_DROP_TWICE
  if (s_last) {
    long long t0 = gtime();
    drop_compact_tail(p, b);
    __syncthreads();
    if (threadIdx.x == 0) g_drop_trace[8192 * 4 - 1] = gtime() - t0;
  }
#endif
#endif
}

// Generic path for G > 8: one warp per position, every needed pair re-streams its two tokens
// (correct for any G; not tuned -- the paper's configurations use c <= 32 frames = G <= 16).
template <typename E>
__global__ void __launch_bounds__(kDropThreads) drop_kernel_generic(const DropParams p) {
  pdl_wait();
  pdl_launch_dependents();
  constexpr int VE = Vec<E>::kElems;
  __shared__ int s_last;
  const int b = blockIdx.y;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int pos = blockIdx.x * kDropWarps + warp;
  const int T = p.G * p.P;
  if (pos < p.P) {
    uint8_t* mask = p.mask + (size_t)b * T;
    const int nvec = p.D / VE;
    auto token = [&](int g) -> const uint4* {
      if (g < 0) return reinterpret_cast<const uint4*>(static_cast<const E*>(p.prev) + ((size_t)b * p.P + pos) * p.D);
      return reinterpret_cast<const uint4*>(static_cast<const E*>(p.z) + (((size_t)b * p.G + g) * p.P + pos) * p.D);
    };
    auto sim_above = [&](int gi, int gj) -> bool {
      const uint4 *a = token(gi), *c = token(gj);
      float dot = 0.f, na = 0.f, nc = 0.f;
      for (int v = lane; v < nvec; v += 32) {
        float fa[VE], fc[VE];
        Vec<E>::unpack(__ldg(a + v), fa);
        Vec<E>::unpack(__ldg(c + v), fc);
#pragma unroll
        for (int e = 0; e < VE; ++e) {
          dot = fmaf(fa[e], fc[e], dot);
          na = fmaf(fa[e], fa[e], na);
          nc = fmaf(fc[e], fc[e], nc);
        }
      }
      return sim_gt(warp_sum(dot), warp_sum(na), warp_sum(nc), p.tau);
    };
    if (p.mode == VCS_DROP_CHUNK_ALLPAIRS) {
      bool drop = p.G > 1;
      for (int i = 0; i < p.G && drop; ++i)
        for (int j = i + 1; j < p.G && drop; ++j) drop = sim_above(i, j);
      if (lane == 0) {
        mask[pos] = 1;
        for (int g = 1; g < p.G; ++g) mask[g * p.P + pos] = drop ? 0 : 1;
      }
    } else {
      for (int g = 0; g < p.G; ++g) {
        bool keep = true;
        if (g > 0 || p.has_prev) keep = !sim_above(g - 1, g);
        if (lane == 0) mask[g * p.P + pos] = keep ? 1 : 0;
      }
    }
  }
  __syncthreads();
  if (threadIdx.x == 0)
    s_last = last_block_ticket(p.counters + (size_t)b * p.counter_stride, blockIdx.x, gridDim.x) ? 1 : 0;
  __syncthreads();
  if (s_last) drop_compact_tail(p, b);
}

template <typename E>
static cudaError_t launch_drop(const DropParams& p, int NT, dim3 grid, cudaStream_t st) {
  switch (NT) {
#define VCS_CASE(n) \
  case n: launch_pdl(drop_kernel<n, E>, dim3(grid), dim3(kDropThreads), 0, st, p); break;
    VCS_CASE(1) VCS_CASE(2) VCS_CASE(3) VCS_CASE(4) VCS_CASE(5) VCS_CASE(6) VCS_CASE(7) VCS_CASE(8) VCS_CASE(9)
#undef VCS_CASE
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

static size_t drop_counter_stride_bytes(int) { return kTicketBytes; }
static size_t drop_counter_bytes(int B, int P) { return (size_t)B * drop_counter_stride_bytes(P); }

}  // namespace vcs

using namespace vcs;

#ifdef VCS_DROP_TRACE
extern "C" VCS_API int vcs_debug_drop_trace(long long* host, int n) {
  return (int)cudaMemcpyFromSymbol(host, g_drop_trace, sizeof(long long) * n);
}
#endif

extern "C" size_t vcs_temporal_drop_workspace_bytes(int B, int G, int P) {
  if (B <= 0 || G <= 0 || P <= 0) return 0;
  return drop_counter_bytes(B, P) + round_up((size_t)B * G * P, 256);
}

extern "C" int vcs_temporal_drop(const void* z, const void* prev_last_group, int B, int G, int P, int D,
                                 int dtype, float tau, int mode, int32_t* kept_idx, int32_t* kept_count,
                                 uint8_t* keep_mask, int32_t* pos3, int Hg, int Wg, int t_stride,
                                 const int32_t* pos_base_d, void* workspace, size_t workspace_bytes,
                                 void* stream) {
  if (B < 0 || G <= 0 || P < 0 || D <= 0) VCS_FAIL(VCS_EINVAL, "temporal_drop: bad sizes B=%d G=%d P=%d D=%d", B, G, P, D);
  if (dtype != VCS_F32 && dtype != VCS_BF16) VCS_FAIL(VCS_EUNSUPPORTED, "temporal_drop: dtype %d", dtype);
  if (mode != VCS_DROP_CHUNK_ALLPAIRS && mode != VCS_DROP_CONSECUTIVE) VCS_FAIL(VCS_EINVAL, "temporal_drop: mode %d", mode);
  if (B == 0 || P == 0) {
    if (B > 0 && kept_count) VCS_CUDA_OK(cudaMemsetAsync(kept_count, 0, sizeof(int32_t) * B, (cudaStream_t)stream));
    return VCS_OK;  // empty input: nothing kept
  }
  if (!z || !kept_idx || !kept_count || !workspace) VCS_FAIL(VCS_EINVAL, "temporal_drop: NULL z / kept_idx / kept_count / workspace");
  if (!(tau == tau)) VCS_FAIL(VCS_EINVAL, "temporal_drop: tau is NaN");
  if ((size_t)G * P > 0x7fffffffu / 4) VCS_FAIL(VCS_ECAP, "temporal_drop: G*P too large");
  if (B > 65535) VCS_FAIL(VCS_ECAP, "temporal_drop: B > 65535");
  if (pos3 && ((long long)Hg * Wg != P || Hg <= 0 || Wg <= 0)) VCS_FAIL(VCS_EINVAL, "temporal_drop: pos3 needs Hg*Wg == P");
  if (!aligned16(z) || (prev_last_group && !aligned16(prev_last_group)) ||
      ((size_t)D * elem_bytes(dtype)) % 16 != 0)
    VCS_FAIL(VCS_EALIGN, "temporal_drop: z must be 16-byte aligned and D*elem_size a multiple of 16");
  if (workspace_bytes < vcs_temporal_drop_workspace_bytes(B, G, P))
    VCS_FAIL(VCS_ECAP, "temporal_drop: workspace too small (%zu < %zu)", workspace_bytes,
             vcs_temporal_drop_workspace_bytes(B, G, P));

  DropParams p;
  p.z = z; p.prev = prev_last_group; p.B = B; p.G = G; p.P = P; p.D = D; p.tau = tau; p.mode = mode;
  p.has_prev = (mode == VCS_DROP_CONSECUTIVE && prev_last_group) ? 1 : 0;
  p.counters = reinterpret_cast<unsigned int*>(workspace);
  p.counter_stride = (int)(drop_counter_stride_bytes(P) / sizeof(unsigned int));
  p.mask = keep_mask ? keep_mask : reinterpret_cast<uint8_t*>(workspace) + drop_counter_bytes(B, P);
  p.kept_idx = kept_idx; p.kept_count = kept_count; p.pos3 = pos3;
  p.Hg = Hg; p.Wg = Wg > 0 ? Wg : 1; p.t_stride = t_stride; p.pos_base = pos_base_d;

  cudaStream_t st = (cudaStream_t)stream;
  const int NT = G + p.has_prev;
  cudaError_t err;
  if (NT <= kMaxNT) {
    // warps per position: enough to put ~2 blocks on every SM, but at least one vector per lane
    const int nvec = (int)((size_t)D * elem_bytes(dtype) / 16);
    int split = 1;
    while (split < kDropWarps && (long long)B * P * split < 148LL * 12 && nvec / (split * 2) >= 32) split *= 2;
    p.split = split;
    p.pos_per_block = kDropWarps / split;
    dim3 grid((P + p.pos_per_block - 1) / p.pos_per_block, B);
    err = dtype == VCS_BF16 ? launch_drop<__nv_bfloat16>(p, NT, grid, st) : launch_drop<float>(p, NT, grid, st);
  } else {
    p.split = 1; p.pos_per_block = kDropWarps;
    dim3 grid((P + kDropWarps - 1) / kDropWarps, B);
    if (dtype == VCS_BF16) launch_pdl(drop_kernel_generic<__nv_bfloat16>, dim3(grid), dim3(kDropThreads), 0, st, p);
    else launch_pdl(drop_kernel_generic<float>, dim3(grid), dim3(kDropThreads), 0, st, p);
    err = cudaGetLastError();
  }
  if (err != cudaSuccess) VCS_FAIL(VCS_ECUDA, "temporal_drop launch: %s", cudaGetErrorString(err));
  return VCS_OK;
}
