// vcs_temporal_drop: chunk-level temporal token dropping (Eq. 1-2) fused
// with stream compaction into a kept-index list.
//
// HBM-bound: every token is read exactly once with 128-bit coalesced loads; the G norms and
// G(G-1)/2 dot products of a position live in registers (fp32 FMA of exact bf16 products).
// One position is owned by `split` warps (each a contiguous D-slice) so that a single small
// chunk still puts all of its bytes in flight at once; B independent streams batch in grid.y.
// The last block of a stream to finish (ticket counter) scans that stream's T keep flags (16 per
// thread, one 128-bit load each) and writes kept_idx / pos3 / kept_count in ascending order -- no
// second launch, no host round trip.
#include "common.cuh"

namespace vcs {

constexpr int kDropFill = 12;   // position-warps per SM below which a position is split over more warps

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
  uint8_t* mask;        // internal flags [B][mask_stride] in the workspace, rows 16-byte aligned, padding zero
  int mask_stride;
  uint8_t* user_mask;   // optional caller output [B][T]
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
// Reading D6: S := 0 when a norm is 0.  Reading D31: |S| <= 1 (Cauchy-Schwarz), so nothing exceeds
// tau >= 1 and everything exceeds tau < -1 whatever the rounding of dot^2 against ni * nj (identical
// tokens, the static-pixel case, give dot^2 == ni * nj up to one ulp either way).  fp32 throughout;
// the generators keep |S - tau| >= 1e-4.
__device__ __forceinline__ bool sim_gt(float dot, float ni, float nj, float tau) {
  if (ni == 0.f || nj == 0.f) return 0.f > tau;
  if (tau >= 1.f) return false;
  if (tau < -1.f) return true;
  const float rhs = tau * tau * (ni * nj);
  const float d2 = dot * dot;
  return tau >= 0.f ? (dot > 0.f && d2 > rhs) : (dot >= 0.f || d2 < rhs);
}

// Block-wide tail: scan the T keep flags of stream b (g-major order) and emit the compacted list.
// A pass covers kDropThreads * 16 consecutive tokens: thread t owns tokens [16 t, 16 t + 16) of the pass
// (one 128-bit load of its flags), a block-wide exclusive scan of the per-thread counts gives its first
// slot, the kept indices of the pass are staged in shared memory in output order, and the block then
// writes idx / pos3 with consecutive lanes on consecutive output slots (coalesced; per-thread scattered
// stores cost 32 LSU wavefronts per instruction and made this tail 8 us for a 7B-shaped chunk).  Passes run
// in sequence with a running base, so the list is ascending for ANY T.
__device__ void drop_compact_tail(const DropParams& p, int b) {
  __shared__ int s_warp[kDropWarps];
  __shared__ int s_total;
  __shared__ int s_idx[kDropThreads * 16];
  const int T = p.G * p.P;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint8_t* mask = p.mask + (size_t)b * p.mask_stride;       // rows are 16-byte aligned
  int32_t* idx = p.kept_idx + (size_t)b * T;
  int32_t* pos = p.pos3 ? p.pos3 + (size_t)b * T * 3 : nullptr;
  const int base = p.pos_base ? p.pos_base[b] : 0;
  const float inv_P = 1.0f / (float)p.P, inv_W = 1.0f / (float)p.Wg;
  int running = 0;
  for (int i0 = 0; i0 < T; i0 += kDropThreads * 16) {
    const int first = i0 + tid * 16;
    uint4 f = make_uint4(0u, 0u, 0u, 0u);
    if (first < T) f = __ldcg(reinterpret_cast<const uint4*>(mask + first));
    uint32_t w[4] = {f.x & 0x01010101u, f.y & 0x01010101u, f.z & 0x01010101u, f.w & 0x01010101u};
    if (first < T && first + 16 > T) {   // row padding may hold stale flags of an earlier call with another shape
#pragma unroll
      for (int e = 0; e < 16; ++e)
        if (first + e >= T) w[e >> 2] &= ~(1u << (8 * (e & 3)));
    }
    const int cnt = __popc(w[0]) + __popc(w[1]) + __popc(w[2]) + __popc(w[3]);
    int incl = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int v = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += v;
    }
    __syncthreads();                     // previous pass has read s_warp / s_total / s_idx
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    int off = incl - cnt;                // slot inside this pass
#pragma unroll
    for (int k = 0; k < kDropWarps; ++k) off += k < warp ? s_warp[k] : 0;
    if (tid == kDropThreads - 1) s_total = off + cnt;
#pragma unroll
    for (int e = 0; e < 16; ++e)
      if ((w[e >> 2] >> (8 * (e & 3))) & 1u) s_idx[off++] = first + e;
    __syncthreads();
    const int n_pass = s_total;
    for (int o = tid; o < n_pass; o += kDropThreads) {
      const int i = s_idx[o], dst = running + o;
      idx[dst] = i;
      if (pos) {
        // exact floor divisions by reciprocal + one correction step
        int g = __float2int_rz(__int2float_rz(i) * inv_P);
        g += (g + 1) * p.P <= i ? 1 : 0;  g -= g * p.P > i ? 1 : 0;
        const int pp = i - g * p.P;
        int r = __float2int_rz(__int2float_rz(pp) * inv_W);
        r += (r + 1) * p.Wg <= pp ? 1 : 0;  r -= r * p.Wg > pp ? 1 : 0;
        pos[3 * dst + 0] = base + g * p.t_stride;
        pos[3 * dst + 1] = base + r;
        pos[3 * dst + 2] = base + (pp - r * p.Wg);
      }
    }
    running += n_pass;
  }
  const int total = running;
  for (int i = total + tid; i < T; i += kDropThreads) idx[i] = -1;
  if (tid == 0) p.kept_count[b] = total;
}

template <int NT>
__device__ __forceinline__ void drop_decide(const DropParams& p, int b, int pos, const float* acc) {
  // acc: [0,NT) squared norms, then packed upper-triangle dots
  const int T = p.G * p.P;
  uint8_t* mask = p.mask + (size_t)b * p.mask_stride;
  uint8_t* umask = p.user_mask ? p.user_mask + (size_t)b * T : nullptr;
  auto put = [&](int i, bool keep) {
    mask[i] = keep ? 1 : 0;
    if (umask) umask[i] = keep ? 1 : 0;
  };
  if (p.mode == VCS_DROP_CHUNK_ALLPAIRS) {
    bool drop = NT > 1;
#pragma unroll
    for (int i = 0; i < NT; ++i)
#pragma unroll
      for (int j = i + 1; j < NT; ++j)
        drop = drop && sim_gt(acc[NT + pair_idx<NT>(i, j)], acc[i], acc[j], p.tau);
    put(pos, true);  // first group = anchor
    for (int g = 1; g < p.G; ++g) put(g * p.P + pos, !drop);
  } else {
    // token list: [prev,] group 0 .. G-1; group g is dropped iff S(previous token, it) > tau
    const int first = p.has_prev ? 1 : 0;  // list index of group 0
    if (!p.has_prev) put(pos, true);
#pragma unroll
    for (int t = 1; t < NT; ++t) {
      const bool drop = sim_gt(acc[NT + pair_idx<NT>(t - 1, t)], acc[t - 1], acc[t], p.tau);
      put((t - first) * p.P + pos, !drop);
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

  if (active && NT > 1) {
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
  if (active && sub == 0 && lane == 0) drop_decide<NT>(p, b, pos, acc);

  // ticket: the last block of stream b compacts it
  __syncthreads();
  if (threadIdx.x == 0)
    s_last = last_block_ticket(p.counters + (size_t)b * p.counter_stride, blockIdx.x, gridDim.x) ? 1 : 0;
  __syncthreads();
  if (s_last) drop_compact_tail(p, b);
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
    uint8_t* mask = p.mask + (size_t)b * p.mask_stride;
    uint8_t* umask = p.user_mask ? p.user_mask + (size_t)b * T : nullptr;
    auto put = [&](int i, bool keep) {
      mask[i] = keep ? 1 : 0;
      if (umask) umask[i] = keep ? 1 : 0;
    };
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
        put(pos, true);
        for (int g = 1; g < p.G; ++g) put(g * p.P + pos, !drop);
      }
    } else {
      for (int g = 0; g < p.G; ++g) {
        bool keep = true;
        if (g > 0 || p.has_prev) keep = !sim_above(g - 1, g);
        if (lane == 0) put(g * p.P + pos, keep);
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

extern "C" size_t vcs_temporal_drop_workspace_bytes(int B, int G, int P) {
  if (B <= 0 || G <= 0 || P <= 0) return 0;
  return drop_counter_bytes(B, P) + round_up((size_t)B * round_up((size_t)G * P, 16), 256);
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
  if (!aligned16(workspace)) VCS_FAIL(VCS_EALIGN, "temporal_drop: workspace must be 16-byte aligned (128-bit flag loads)");

  DropParams p;
  p.z = z; p.prev = prev_last_group; p.B = B; p.G = G; p.P = P; p.D = D; p.tau = tau; p.mode = mode;
  p.has_prev = (mode == VCS_DROP_CONSECUTIVE && prev_last_group) ? 1 : 0;
  p.counters = reinterpret_cast<unsigned int*>(workspace);
  p.counter_stride = (int)(drop_counter_stride_bytes(P) / sizeof(unsigned int));
  // the flags live in the workspace (rows padded to 16 bytes);
  // the caller's keep_mask, if any, is written beside them
  p.mask = reinterpret_cast<uint8_t*>(workspace) + drop_counter_bytes(B, P);
  p.mask_stride = (int)round_up((size_t)G * P, 16);
  p.user_mask = keep_mask;
  p.kept_idx = kept_idx; p.kept_count = kept_count; p.pos3 = pos3;
  p.Hg = Hg; p.Wg = Wg > 0 ? Wg : 1; p.t_stride = t_stride; p.pos_base = pos_base_d;

  cudaStream_t st = (cudaStream_t)stream;
  const int NT = G + p.has_prev;
  cudaError_t err;
  if (NT <= kMaxNT) {
    // warps per position: enough to put ~2 blocks on every SM, but at least one vector per lane
    const int nvec = (int)((size_t)D * elem_bytes(dtype) / 16);
    int split = 1;
    const long long sms = device_sm_count();
    if (sms <= 0) VCS_FAIL(VCS_ECUDA, "temporal_drop: cannot query the SM count of the current device");
    while (split < kDropWarps && (long long)B * P * split < sms * kDropFill && nvec / (split * 2) >= 32) split *= 2;
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

// ---- vcs_temporal_drop_static: the same launch with the library's own fixed scratch -----------------------
// Some callers cannot obtain device memory for the workspace above: an inference server that gave the whole
// HBM to its own pool at start-up (cudaMalloc then fails), a per-frame loop that must not pay cudaMalloc's
// device-wide synchronisation, a plug-in that is handed tensors but no allocator.  For them the ticket
// counters and keep flags live in the array below.  It is part of the library image: every GPU that loads
// libvcs.so holds these VCS_DROP_STATIC_SCRATCH_BYTES until the process exits, whether or not it is used.
namespace vcs {

static __device__ __align__(256) unsigned char g_drop_static_scratch[VCS_DROP_STATIC_SCRATCH_BYTES];

// Device address of the array on each device (0 = not looked up yet).  In host code the symbol
// `g_drop_static_scratch` is only a handle of the runtime: its host address is NOT device memory, so the
// address a kernel may use has to come from cudaGetSymbolAddress, with the owning device current.
static std::atomic<void*> g_drop_static_addr[kMaxDevices];

static int drop_static_scratch(void** out) {
  int dev = -1;
  VCS_CUDA_OK(cudaGetDevice(&dev));
  const bool cached = dev >= 0 && dev < kMaxDevices;
  void* ptr = cached ? g_drop_static_addr[dev].load(std::memory_order_acquire) : nullptr;
  if (!ptr) {
    const cudaError_t e = cudaGetSymbolAddress(&ptr, g_drop_static_scratch);
    if (e != cudaSuccess || !ptr)
      VCS_FAIL(VCS_ECUDA, "temporal_drop_static: cudaGetSymbolAddress on device %d: %s", dev, cudaGetErrorString(e));
    if (cached) g_drop_static_addr[dev].store(ptr, std::memory_order_release);   // same value from any thread
  }
  *out = ptr;
  return VCS_OK;
}

}  // namespace vcs

extern "C" int vcs_temporal_drop_static(const void* z, const void* prev_last_group, int B, int G, int P, int D,
                                        int dtype, float tau, int mode, int32_t* kept_idx, int32_t* kept_count,
                                        uint8_t* keep_mask, int32_t* pos3, int Hg, int Wg, int t_stride,
                                        const int32_t* pos_base_d, void* stream) {
  // the size test needs no device, so it answers first (and on a machine without a GPU)
  const size_t need = (B > 0 && G > 0 && P > 0 && (size_t)G * P <= 0x7fffffffu / 4 && B <= 65535)
                          ? vcs_temporal_drop_workspace_bytes(B, G, P) : 0;
  if (need > (size_t)VCS_DROP_STATIC_SCRATCH_BYTES)
    VCS_FAIL(VCS_ECAP, "temporal_drop_static: B=%d G=%d P=%d needs %zu bytes of scratch, the built-in array holds %zu; "
                       "use vcs_temporal_drop with a caller workspace", B, G, P, need, (size_t)VCS_DROP_STATIC_SCRATCH_BYTES);
  void* scratch = nullptr;
  if (need > 0) {
    const int rc = drop_static_scratch(&scratch);
    if (rc != VCS_OK) return rc;
    // The array keeps whatever the previous call (of any shape, from any thread) left in it.  The ticket
    // counters must read zero when the kernel starts; stale keep flags are harmless (every flag of the T tokens is
    // rewritten before the compaction reads it, and the row padding is masked off there).
    VCS_CUDA_OK(cudaMemsetAsync(scratch, 0, drop_counter_bytes(B, P), (cudaStream_t)stream));
  }
  return vcs_temporal_drop(z, prev_last_group, B, G, P, D, dtype, tau, mode, kept_idx, kept_count, keep_mask, pos3,
                           Hg, Wg, t_stride, pos_base_d, need > 0 ? scratch : (void*)&need, VCS_DROP_STATIC_SCRATCH_BYTES,
                           stream);
}
