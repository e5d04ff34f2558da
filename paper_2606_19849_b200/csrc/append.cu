// vcs_kv_append_pages: write the retained tokens' K (M-RoPE rotated) and V into one page of the
// chunk-granular paged KV cache ("historical visual cache"; step a5), keep the
// page's pre-RoPE key sum (retrieval summary of Eq. 3, reading D19) and its length.
//
// HBM-bound: each thread of the 8 K warps moves the (m..m+7, m+d/2..m+d/2+7) pair of 16-byte
// vectors of one (token, kv head) of K -- 128-bit coalesced loads and stores, sin/cos in registers.
// V needs no arithmetic, so it never enters a register: a ninth warp moves the block's V rows with
// the bulk-copy engine (cp.async.bulk global -> shared ring -> one row store per (token, kv head)),
// which keeps V's bytes in flight without a warp stalled on them and leaves the K warps' registers
// to K.
// The page's key sum: small launches let every block add its own 16-byte columns of the key rows over all
// tokens (second pass over rows that sit in L2; no cross-block reduction, no tail); large batched launches
// keep one pass over the keys, write per-block sums to the workspace and let the last block (ticket) add
// them in block order.  Either way the order is fixed: k_sum is deterministic for a given launch shape.
#include "common.cuh"

namespace vcs {

constexpr int kAppendThreads = 256;

constexpr int kVStages = 3;   // ring of V token groups in shared memory (moved by the extra warp)

__device__ __forceinline__ uint32_t app_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void app_mbar_init(uint32_t bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void app_mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void app_mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t done = 0;
  while (!done)
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(bar), "r"(parity)
        : "memory");
}
__device__ __forceinline__ void app_bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(bar)
               : "memory");
}
__device__ __forceinline__ void app_bulk_s2g(void* dst, uint32_t src, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src), "r"(bytes) : "memory");
}

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
  int tok_per_block, iters;
  int column_sums;         // 1: every block adds its own columns of the key rows (latency path); 0: per-block partial sums + ticket
  RopeParams rope;
  // batched form (grid.y = stream b): per-stream strides; page id from page_ids[b]
  long long k_bstride, v_bstride;   // elements between streams
  const int32_t* page_ids;          // device [B] or null (use page_id)
  int n_pages;
  long long ws_bstride;             // bytes between the streams' workspaces
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
__global__ void __launch_bounds__(kAppendThreads + 32, 3) append_kernel(const AppendParams p) {
  pdl_wait();
  pdl_launch_dependents();
  // ---- batched form: rebase the per-stream pointers on stream b = blockIdx.y (p stays in the
  // constant bank: its inv_freq / axis tables are indexed dynamically) ----
  const int b = blockIdx.y;
  const E* kbase = static_cast<const E*>(p.k) + (size_t)b * p.k_bstride;
  const E* vbase = static_cast<const E*>(p.v) + (size_t)b * p.v_bstride;
  const int32_t* pos3 = p.pos3 + (size_t)b * p.n_cap * 3;
  const int32_t* n_d = p.n_d ? p.n_d + b : nullptr;
  unsigned int* counter = reinterpret_cast<unsigned int*>(reinterpret_cast<char*>(p.counter) + (size_t)b * p.ws_bstride);
  float* partial = reinterpret_cast<float*>(reinterpret_cast<char*>(p.partial) + (size_t)b * p.ws_bstride);
  int page_id = p.page_ids ? p.page_ids[b] : p.page_id;
  bool bad_page = false;
  if (page_id < 0 || page_id >= p.n_pages) { bad_page = true; page_id = 0; }
  constexpr int VE = KV<E>::kElems;
  extern __shared__ __align__(128) float s_sum[];  // [tok_per_block][Hkv*d] floats, then the V ring: kVStages x [tok_per_block][Hkv*d] of E
  __shared__ int s_last;
  __shared__ __align__(8) unsigned long long v_bar[kVStages];

  const int HD = p.Hkv * p.d;
  const int half = p.d / 2;
  const int vec_per_head = half / VE;             // vector pairs per (token, head)
  const int vec_per_tok = p.Hkv * vec_per_head;
  int n = n_d ? *n_d : p.n_cap;
  if (bad_page) n = 0;               // nothing is written; the ticket below still runs
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
  // a block handles `iters` groups of tok_per_block tokens (iters > 1 only for large batched
  // launches: fewer blocks, tickets and partial sums); the thread's pre-RoPE keys add up in registers
  float klo[VE], khi[VE];
#pragma unroll
  for (int e = 0; e < VE; ++e) klo[e] = khi[e] = 0.f;
  // software pipeline of depth 2: the loads of token group it+1 are in flight while group it is rotated
  // and stored (the kernel is bound by bytes in flight per SM, not by arithmetic)
  auto tok_of = [&](int it) { return (blockIdx.x * p.iters + it) * p.tok_per_block + tl; };
  auto live = [&](int it) { return it < p.iters && tl < p.tok_per_block && tok_of(it) < n_fit; };
  uint4 k0, k1;
  int pt = 0, ph = 0, pw = 0;
  auto load = [&](int it, uint4& a0, uint4& a1, int& t0, int& t1, int& t2) {
    const int tok = tok_of(it);
    const E* kp = kbase + (size_t)tok * p.k_stride + h * p.d;
    a0 = ldg_nc_v4(kp + m0); a1 = ldg_nc_v4(kp + m0 + half);
    t0 = pos3[3 * tok + 0]; t1 = pos3[3 * tok + 1]; t2 = pos3[3 * tok + 2];
  };
  // this thread's rotary pairs are the same for every token group: fetch their table entries once
  // (constant-bank loads with a thread-dependent index are slow: they showed up as the top stall)
  unsigned long long tfrac[VE];
  double ifreq[VE];
  unsigned axbits = 0u;
#pragma unroll
  for (int e = 0; e < VE; ++e) {
    tfrac[e] = p.rope.turn_frac[m0 + e];
    if constexpr (sizeof(E) != 2) ifreq[e] = p.rope.inv_freq[m0 + e];
    axbits |= (unsigned)p.rope.axis_of[m0 + e] << (2 * e);
  }
  if (tid >= kAppendThreads) {
    // ---- V warp: V needs no arithmetic, so it never enters a register.  This warp runs the block's
    // token groups through a ring in shared memory with the bulk-copy engine: one load per group when
    // the rows are contiguous, one row store per (token, kv head) out ----
    const int lane = tid & 31;
    const uint32_t row_bytes = (uint32_t)p.d * sizeof(E), tok_bytes = (uint32_t)HD * sizeof(E);
    const uint32_t stage_bytes = (uint32_t)p.tok_per_block * tok_bytes;
    const uint32_t ring = app_smem_u32(s_sum) + (uint32_t)p.tok_per_block * HD * sizeof(float);
    auto group = [&](int it, int& g0) {   // live tokens of token group `it` of this block
      g0 = (blockIdx.x * p.iters + it) * p.tok_per_block;
      return it < p.iters ? max(0, min(p.tok_per_block, n_fit - g0)) : 0;
    };
    auto issue = [&](int it) {
      int g0;
      const int cnt = group(it, g0);
      if (cnt <= 0) return;
      const uint32_t bar = app_smem_u32(&v_bar[it % kVStages]), dst = ring + (it % kVStages) * stage_bytes;
      app_mbar_expect_tx(bar, cnt * tok_bytes);
      if (p.v_stride == HD) app_bulk_g2s(dst, vbase + (size_t)g0 * HD, cnt * tok_bytes, bar);
      else
        for (int t = 0; t < cnt; ++t) app_bulk_g2s(dst + t * tok_bytes, vbase + (size_t)(g0 + t) * p.v_stride, tok_bytes, bar);
    };
    if (lane == 0) {
      for (int s = 0; s < kVStages; ++s) app_mbar_init(app_smem_u32(&v_bar[s]), 1);
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
      for (int it = 0; it < kVStages - 1; ++it) issue(it);
    }
    __syncwarp();
#pragma unroll 1
    for (int it = 0; it < p.iters; ++it) {
      int g0;
      const int cnt = group(it, g0);
      if (cnt <= 0) break;
      app_mbar_wait(app_smem_u32(&v_bar[it % kVStages]), (it / kVStages) & 1);
      const uint32_t src = ring + (it % kVStages) * stage_bytes;
      for (int r = lane; r < cnt * p.Hkv; r += 32) {
        const int hh = r / cnt, t = r - hh * cnt;
        const size_t prow = ((size_t)page_id * p.Hkv + hh) * p.page_cap + (p.page_offset + g0 + t);
        app_bulk_s2g(static_cast<E*>(p.v_pages) + prow * p.d, src + t * tok_bytes + hh * row_bytes, row_bytes);
      }
      asm volatile("cp.async.bulk.commit_group;" ::: "memory");
      asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");   // group it - 1 has left its slot
      __syncwarp();
      if (lane == 0) issue(it + kVStages - 1);
    }
    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // the ring is free; the writes land before the grid completes
  }
  if (live(0)) load(0, k0, k1, pt, ph, pw);
#pragma unroll 1
  for (int it = 0; it < p.iters; ++it) {
    const bool cur = live(it);
    uint4 nk0, nk1;
    int npt = 0, nph = 0, npw = 0;
    if (live(it + 1)) load(it + 1, nk0, nk1, npt, nph, npw);
    if (cur) {
      const int tok = tok_of(it);
      float xlo[VE], xhi[VE];
      KV<E>::unpack(k0, xlo);
      KV<E>::unpack(k1, xhi);
      float rlo[VE], rhi[VE];
#pragma unroll
      for (int e = 0; e < VE; ++e) {
        const unsigned ax = (axbits >> (2 * e)) & 3u;
        const int pos = ax == 0u ? pt : (ax == 1u ? ph : pw);
        float sn, cs;
        if constexpr (sizeof(E) == 2) rope_sincos_fast(pos, tfrac[e], &sn, &cs);
        else rope_sincos(pos, ifreq[e], &sn, &cs);
        rlo[e] = xlo[e] * cs - xhi[e] * sn;   // (x_m, x_{m+d/2}) <- (x_m c - x_{m+d/2} s, x_{m+d/2} c + x_m s)
        rhi[e] = xhi[e] * cs + xlo[e] * sn;
        klo[e] += xlo[e];
        khi[e] += xhi[e];
      }
      const size_t row = ((size_t)page_id * p.Hkv + h) * p.page_cap + (p.page_offset + tok);
      E* ko = static_cast<E*>(p.k_pages) + row * p.d;
      stg_v4(ko + m0, KV<E>::pack(rlo));
      stg_v4(ko + m0 + half, KV<E>::pack(rhi));
    }
    k0 = nk0; k1 = nk1; pt = npt; ph = nph; pw = npw;
  }

  // The tcgen05 attention kernel reads whole 128-token tiles of V and multiplies the rows beyond
  // page_len by P = 0: they must be finite (0 x NaN = NaN), whatever the pool held before.  Zero the rows
  // [page_offset + n_fit, next multiple of 128) of every kv head; the blocks share them row by row.
  if (!bad_page && tid < kAppendThreads) {
    const int end = p.page_offset + n_fit;
    const int pad_end = min(p.page_cap, (end + 127) & ~127);
    const int vec_per_row = p.d / VE;                       // 16-byte vectors per (token, head) row
    for (int r = end + blockIdx.x; r < pad_end; r += gridDim.x)
      for (int e = tid; e < p.Hkv * vec_per_row; e += kAppendThreads) {
        const int hh = e / vec_per_row, ve = e - hh * vec_per_row;
        const size_t prow = ((size_t)page_id * p.Hkv + hh) * p.page_cap + r;
        stg_v4(static_cast<E*>(p.v_pages) + prow * p.d + ve * VE, make_uint4(0u, 0u, 0u, 0u));
      }
  }

  if (p.column_sums) {
    // k_sum without a cross-block reduction (launches of a wave or two, where the kernel is a chain of latencies):
    // the Hkv * d / VE 16-byte columns of the key rows are dealt to the blocks, and a block adds ITS columns over
    // all n tokens itself -- the rows were just read by the copy path, so this second pass hits L2 -- in a
    // fixed order (thread t: tokens t, t + 256, ...; then the threads in order): deterministic, no tickets, no
    // partial sums in global memory, no last-block tail (which was half of this kernel's duration).
    float* red = s_sum;                                         // [kAppendThreads][VE] floats of scratch
    const int ncol = HD / VE;
    float* ksum = p.k_sum + (size_t)page_id * HD;
    // dealt from the last block down: with a device count below n_cap the last blocks hold no tokens
    for (int vc = (int)gridDim.x - 1 - (int)blockIdx.x; vc < ncol; vc += gridDim.x) {
      float acc[VE];
#pragma unroll
      for (int e = 0; e < VE; ++e) acc[e] = 0.f;
      if (tid < kAppendThreads) {
        const E* col = kbase + (size_t)vc * VE;
#pragma unroll 4
        for (int tok = tid; tok < n_fit; tok += kAppendThreads) {
          float x[VE];
          KV<E>::unpack(ldg_nc_v4(col + (size_t)tok * p.k_stride), x);
#pragma unroll
          for (int e = 0; e < VE; ++e) acc[e] += x[e];
        }
#pragma unroll
        for (int e = 0; e < VE; ++e) red[tid * VE + e] = acc[e];
      }
      __syncthreads();
      if (tid < VE && !bad_page) {
        float t = p.page_offset > 0 ? ksum[vc * VE + tid] : 0.f;
        for (int k = 0; k < kAppendThreads; ++k) t += red[k * VE + tid];
        ksum[vc * VE + tid] = t;
      }
      __syncthreads();
    }
    if (tid == 0 && blockIdx.x == 0) {
      if (!bad_page) p.page_len[page_id] = p.page_offset + n_fit;
      if (p.status && (clamped || overflow || bad_page))
        atomicOr(p.status, (clamped ? VCS_FLAG_COUNT_CLAMPED : 0) | (overflow ? VCS_FLAG_PAGE_OVERFLOW : 0) |
                               (bad_page ? VCS_FLAG_BAD_PAGE : 0));
    }
    return;
  }
  // per-block sum of the PRE-RoPE keys, tokens added in order (large batched launches: bandwidth path)
  if (tl < p.tok_per_block) {
    float* row = s_sum + (size_t)tl * HD + h * p.d;
#pragma unroll
    for (int e = 0; e < VE; ++e) { row[m0 + e] = klo[e]; row[m0 + half + e] = khi[e]; }
  }
  __syncthreads();
  for (int c = tid; c < HD && tid < kAppendThreads; c += kAppendThreads) {
    float s = 0.f;
    for (int t = 0; t < p.tok_per_block; ++t) s += s_sum[(size_t)t * HD + c];
    partial[(size_t)blockIdx.x * HD + c] = s;
  }
  __syncthreads();
  if (tid == 0) s_last = last_block_ticket(counter, blockIdx.x, gridDim.x) ? 1 : 0;
  __syncthreads();
  if (!s_last) return;
  // last block: add the per-block partial sums in a fixed order (=> deterministic k_sum).  One
  // float4 column per thread, `groups` thread groups striding over the blocks with all their loads
  // in flight at once (the loads are L2 round trips and this block is the kernel's critical path),
  // then the group sums are combined in group order through shared memory.
  const int nblk_used = (n_fit + p.tok_per_block * p.iters - 1) / (p.tok_per_block * p.iters);
  float* ks = p.k_sum + (size_t)page_id * HD;
  const int nq4 = HD / 4;
  const int cols = min(nq4, kAppendThreads), groups = kAppendThreads / cols;
  const int grp = tid / cols, cl = tid - grp * cols;
  float4* s4 = reinterpret_cast<float4*>(s_sum);
  for (int q0 = 0; q0 < nq4; q0 += cols) {
    const int q = q0 + cl;
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    if (q < nq4 && grp < groups) {
      const float4* src = reinterpret_cast<const float4*>(partial) + q;
#pragma unroll 16
      for (int bb = grp; bb < nblk_used; bb += groups) {
        const float4 v = __ldcg(src + (size_t)bb * nq4);
        acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
      }
    }
    __syncthreads();
    if (grp < groups) s4[grp * cols + cl] = acc;
    __syncthreads();
    if (grp == 0 && q < nq4 && !bad_page) {
      float4 t = p.page_offset > 0 ? reinterpret_cast<const float4*>(ks)[q] : make_float4(0.f, 0.f, 0.f, 0.f);
      for (int g2 = 0; g2 < groups; ++g2) {
        const float4 v = s4[g2 * cols + cl];
        t.x += v.x; t.y += v.y; t.z += v.z; t.w += v.w;
      }
      reinterpret_cast<float4*>(ks)[q] = t;
    }
  }
  if (tid == 0) {
    if (!bad_page) p.page_len[page_id] = p.page_offset + n_fit;
    if (p.status && (clamped || overflow || bad_page))
      atomicOr(p.status, (clamped ? VCS_FLAG_COUNT_CLAMPED : 0) | (overflow ? VCS_FLAG_PAGE_OVERFLOW : 0) |
                             (bad_page ? VCS_FLAG_BAD_PAGE : 0));
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
  return round_up(kTicketBytes + ((size_t)(n_cap + tpb - 1) / tpb + 1) * pool->Hkv * pool->d * sizeof(float), 256);
}

static size_t append_ws_stream_bytes(const vcs_kv_pool* pool, int n_cap, int tpb) {
  const size_t nblk = (size_t)(n_cap + tpb - 1) / tpb + 1;
  return round_up(kTicketBytes + nblk * pool->Hkv * pool->d * sizeof(float), 256);
}

// shared by the single-page and the batched entry points (B streams = grid.y)
static int append_launch(const vcs_kv_pool* pool, const void* k, const void* v, int64_t k_bstride, int64_t v_bstride,
                         int64_t k_row_stride, int64_t v_row_stride, const int32_t* pos3, const int32_t* n_d, int n_cap,
                         int32_t page_id, const int32_t* page_ids_d, int B, int32_t page_offset, int32_t* status_d,
                         void* workspace, size_t workspace_bytes, void* stream) {
  if (n_cap < 0) VCS_FAIL(VCS_EINVAL, "kv_append: n_cap < 0");
  if (page_offset < 0 || page_offset > pool->page_cap) VCS_FAIL(VCS_ECAP, "kv_append: page_offset %d out of range", page_offset);
  if (!workspace) VCS_FAIL(VCS_EINVAL, "kv_append: NULL workspace");
  if (n_cap > 0 && (!k || !v || !pos3)) VCS_FAIL(VCS_EINVAL, "kv_append: NULL k / v / pos3");
  const size_t eb = elem_bytes(pool->dtype);
  const int64_t min_stride = (int64_t)pool->Hkv * pool->d;
  if (n_cap > 0 && (k_row_stride < min_stride || v_row_stride < min_stride))
    VCS_FAIL(VCS_EINVAL, "kv_append: row stride smaller than Hkv*d");
  if (n_cap > 0 && (!aligned16(k) || !aligned16(v) || (k_row_stride * eb) % 16 || (v_row_stride * eb) % 16 ||
                    (k_bstride * eb) % 16 || (v_bstride * eb) % 16))
    VCS_FAIL(VCS_EALIGN, "kv_append: k / v and their strides must be 16-byte aligned");
  const int tpb = append_tok_per_block(pool);
  if (tpb == 0) VCS_FAIL(VCS_EUNSUPPORTED, "kv_append: Hkv*d too large for one block");
  const size_t per_stream = append_ws_stream_bytes(pool, n_cap, tpb);
  if (workspace_bytes < per_stream * B) VCS_FAIL(VCS_ECAP, "kv_append: workspace too small");

  AppendParams p;
  p.k = k; p.v = v; p.k_stride = k_row_stride; p.v_stride = v_row_stride;
  p.pos3 = pos3; p.n_d = n_d; p.n_cap = n_cap; p.page_id = page_id; p.page_offset = page_offset;
  p.k_pages = pool->k_pages; p.v_pages = pool->v_pages; p.page_len = pool->page_len; p.k_sum = pool->k_sum;
  p.page_cap = pool->page_cap; p.Hkv = pool->Hkv; p.d = pool->d; p.status = status_d;
  p.counter = reinterpret_cast<unsigned int*>(workspace);
  p.partial = reinterpret_cast<float*>(static_cast<char*>(workspace) + kTicketBytes);
  p.tok_per_block = tpb;
  p.rope = rope_params(pool);
  p.k_bstride = k_bstride; p.v_bstride = v_bstride; p.page_ids = page_ids_d; p.n_pages = pool->n_pages;
  p.ws_bstride = (long long)per_stream;

  // token groups per block: 1 until the launch would no longer be resident in ONE wave (3 blocks per
  // SM by registers), then grow: a second, partly filled wave costs a whole wave time
  const long long groups = n_cap > 0 ? (n_cap + tpb - 1) / tpb : 1;
  long long iters = (groups * B + 399) / 400;
  iters = iters < 1 ? 1 : (iters > 64 ? 64 : iters);
  p.iters = (int)iters;
  // a launch whose keys stay in L2 (<= 16 MB) is a chain of latencies: let the blocks add their own key columns in
  // a second pass (no ticket, no last-block tail); a large batched launch is bound by HBM bytes: keep the keys'
  // single pass and the ticket
  p.column_sums = (long long)n_cap * B * pool->Hkv * pool->d * (long long)eb <= (16LL << 20) ? 1 : 0;
  const int nblk = (int)((groups + iters - 1) / iters);
  const size_t smem = (size_t)tpb * pool->Hkv * pool->d * (sizeof(float) + kVStages * eb);
  cudaStream_t st = (cudaStream_t)stream;
  static PerDeviceOnce attr_once;   // dynamic + static shared memory can pass the 48 KB default by a few bytes
  int arc = attr_once.run([&]() {
    cudaError_t e = cudaFuncSetAttribute(append_kernel<__nv_bfloat16>, cudaFuncAttributeMaxDynamicSharedMemorySize, 72 * 1024);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(append_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, 72 * 1024);
    return e;
  });
  if (arc != VCS_OK) return arc;
  cudaError_t err = pool->dtype == VCS_BF16
                        ? launch_pdl(append_kernel<__nv_bfloat16>, dim3(nblk, B), dim3(kAppendThreads + 32), smem, st, p)
                        : launch_pdl(append_kernel<float>, dim3(nblk, B), dim3(kAppendThreads + 32), smem, st, p);
  if (err == cudaSuccess) err = cudaGetLastError();
  if (err != cudaSuccess) VCS_FAIL(VCS_ECUDA, "kv_append launch: %s", cudaGetErrorString(err));
  return VCS_OK;
}

extern "C" size_t vcs_kv_append_batched_workspace_bytes(const vcs_kv_pool* pool, int n_cap, int B) {
  if (!pool || n_cap < 0 || B <= 0) return 0;
  const int tpb = append_tok_per_block(pool);
  return tpb == 0 ? 0 : append_ws_stream_bytes(pool, n_cap, tpb) * B;
}

extern "C" int vcs_kv_append_pages_batched(const vcs_kv_pool* pool, const void* k, const void* v, int64_t k_batch_stride,
                                           int64_t v_batch_stride, int64_t k_row_stride, int64_t v_row_stride,
                                           const int32_t* pos3, const int32_t* n_d, int n_cap,
                                           const int32_t* page_ids_d, int B, int32_t* status_d, void* workspace,
                                           size_t workspace_bytes, void* stream) {
  int rc = validate_pool(pool, true);
  if (rc != VCS_OK) return rc;
  if (B < 0 || B > 65535) VCS_FAIL(VCS_EINVAL, "kv_append_batched: B out of range");
  if (B == 0) return VCS_OK;
  if (!page_ids_d) VCS_FAIL(VCS_EINVAL, "kv_append_batched: NULL page ids");
  return append_launch(pool, k, v, k_batch_stride, v_batch_stride, k_row_stride, v_row_stride, pos3, n_d, n_cap, 0,
                       page_ids_d, B, 0, status_d, workspace, workspace_bytes, stream);
}

extern "C" int vcs_kv_append_pages(const vcs_kv_pool* pool, const void* k, const void* v, int64_t k_row_stride,
                                   int64_t v_row_stride, const int32_t* pos3, const int32_t* n_d, int n_cap,
                                   int32_t page_id, int32_t page_offset, int32_t* status_d, void* workspace,
                                   size_t workspace_bytes, void* stream) {
  int rc = validate_pool(pool, true);
  if (rc != VCS_OK) return rc;
  if (page_id < 0 || page_id >= pool->n_pages) VCS_FAIL(VCS_ECAP, "kv_append: page_id %d out of range [0,%d)", page_id, pool->n_pages);
  return append_launch(pool, k, v, 0, 0, k_row_stride, v_row_stride, pos3, n_d, n_cap, page_id, nullptr, 1, page_offset,
                       status_d, workspace, workspace_bytes, stream);
}
