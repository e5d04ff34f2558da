// Bounded-visual-attention prefill for sm_100a (mask Eq. 4 :140-145):
// flash-style online softmax, page-table-driven TMA loads of K/V tiles out of the chunk-granular
// paged KV pool, tcgen05 MMAs (kind::f16, bf16 x bf16 -> fp32) with accumulators in TMEM.
//
// One CTA = one 128-row query tile of one q head.  Every KV tile is handled by BOTH softmax
// warpgroups: warp w (lanes 32(w%4)..) of warpgroup 0 owns columns [0,64) of its 32 rows, warp w+4
// of warpgroup 1 owns columns [64,128) of the same rows; the two exchange their row maxima through
// shared memory (one 64-thread named barrier per warp pair and tile).  S is double-buffered in
// TMEM, so Q.K^T of tile j+1 runs on the tensor pipe while the softmax of tile j is computed, and
// there is ONE output accumulator: no partial-result merge, half the registers per thread.
// Warp roles (384 threads; setmaxnreg moves registers from the third warpgroup to the first two):
//   warps 0-7  softmax; together they also build the Q tile: load, rotate by M-RoPE on the fly,
//              store bf16 into the 128B-swizzled K-major layout the UMMA descriptor expects.
//   warp 8     TMA producer: walks the page table, issues cp.async.bulk.tensor for K and V tiles
//              (4-D map over [page][kv head][token][d], box 64 x 128, SWIZZLE_128B), 3-stage rings.
//   warp 9     MMA issuer (one elected lane) + TMEM allocator: S_b = Q K^T (SS), O += P_b V (TS: P is
//              read from TMEM, V straight from its TMA layout as an MN-major B operand).
// TMEM (512 columns): S_0 [0,128) | S_1 [128,256) | O [256,384).  P_b (bf16, 64 columns) overwrites
// the head of S_b once both halves of S_b sit in registers.  Issue order on the (in-order) tensor
// pipe: QK(0) QK(1) | PV(0) QK(2) | PV(1) QK(3) | ...: QK(j+2) may overwrite S_b only after PV(j)
// has read P_b.  The (lazy, threshold 2^8) rescale of O in tile j waits for S_FULL of tile j+1
// (issued after PV(j-1), so PV(j-1) has finished accumulating), the last tile for PV_DONE.
// K(u) and V(u-2) share one ring slot and one barrier pair: the MMA warp waits twice per tile.
#include "attn.cuh"

namespace vcs {

namespace tc {

constexpr int kBlockM = 128;      // query rows per CTA
constexpr int kBlockN = 128;      // KV tokens per tile
constexpr int kHeadDim = 128;
constexpr int kStages = 3;
#ifndef VCS_SOFTMAX_WGS
#define VCS_SOFTMAX_WGS 2
#endif
// softmax warpgroups: each thread owns kBlockN / kWGs columns of its row.  2 is the product setting;
// 4 (four warps per SM sub-partition, 32 columns each) was measured 7 % slower on config 2: the extra
// per-warp fixed work and the 4-way row-max exchange outweigh the better latency hiding.
constexpr int kWGs = VCS_SOFTMAX_WGS;
constexpr int kCols = kBlockN / kWGs;     // logits per thread and tile (also d columns of O per thread)
constexpr int kSoftmaxThreads = 128 * kWGs;
constexpr int kThreads = kSoftmaxThreads + 128;   // + one warpgroup holding the TMA and MMA warps; its registers move to the softmax ones
constexpr int kWarpTma = 4 * kWGs, kWarpMma = kWarpTma + 1;
constexpr int kRegsSoftmax = kWGs == 2 ? 224 : 104, kRegsOther = kWGs == 2 ? 48 : 40;   // inc must fit in what dec releases (per-CTA pool)
constexpr int kSlack = kWGs == 2 ? 1024 : 768;    // alignment slack of the dynamic shared memory (checked in the kernel)
constexpr int kHalfBytes = kBlockN * 128;            // one [128 rows x 64 bf16] swizzled region: 16 KB
constexpr int kTileBytes = 2 * kHalfBytes;           // 32 KB: a [128 x 128] bf16 tile as two d-halves
constexpr uint32_t kTmemCols = 512;
constexpr uint32_t kColS0 = 0, kColS1 = 128, kColO = 256;
constexpr float kRescaleThreshold = 8.0f;            // log2 units
constexpr int kPolyNum = 1, kPolyDen = 2;            // share of exp2 evaluations moved from MUFU to the FMA pipe

struct Smem {
  // offsets into the 1024-aligned dynamic shared memory
  static constexpr int q = 0;                        // Q tile; reused for the (m, l) exchange in the epilogue
  static constexpr int k = q + kTileBytes;
  static constexpr int v = k + kStages * kTileBytes;
  static constexpr int bar = v + kStages * kTileBytes;
  static constexpr int tmem_slot = bar + 192;
  static constexpr int xch = bar + 256;              // row-max exchange [2 halves][128 rows] floats
  static constexpr int total = xch + kWGs * kBlockM * 4;
};
enum Bar {
  Q_FULL = 0, KV_FULL = 1, KV_EMPTY = KV_FULL + kStages,
  S_FULL = KV_EMPTY + kStages, P_FULL = S_FULL + 2, PV_DONE = P_FULL + 2, ALL_DONE = PV_DONE + 1, NUM_BARS = ALL_DONE + 1
};
static_assert(NUM_BARS * 8 <= 192, "barrier region");

// ---- PTX wrappers ---------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t"
        "}"
        : "=r"(done)
        : "r"(bar), "r"(parity)
        : "memory");
  } while (!done);
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1, int c2, int c3) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];" ::"r"(dst),
      "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
      : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap* map) {
  asm volatile("prefetch.tensormap [%0];" ::"l"(map) : "memory");
}

__device__ __forceinline__ void tmem_alloc(uint32_t dst_smem, uint32_t cols) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(dst_smem), "r"(cols) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t cols) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(cols) : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// D[tmem] (+)= A[smem] * B[smem], bf16 inputs, fp32 accumulate
__device__ __forceinline__ void umma_bf16_ss(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t"
      "}" ::"r"(d_tmem),
      "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, float* v) {
  uint32_t* r = reinterpret_cast<uint32_t*>(v);
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
        "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]), "=r"(r[18]),
        "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]),
        "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr));
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const float* v) {
  const uint32_t* r = reinterpret_cast<const uint32_t*>(v);
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "
      "{%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};" ::"r"(taddr),
      "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]), "r"(r[10]),
      "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]), "r"(r[16]), "r"(r[17]), "r"(r[18]), "r"(r[19]), "r"(r[20]),
      "r"(r[21]), "r"(r[22]), "r"(r[23]), "r"(r[24]), "r"(r[25]), "r"(r[26]), "r"(r[27]), "r"(r[28]), "r"(r[29]), "r"(r[30]),
      "r"(r[31])
      : "memory");
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

__device__ __forceinline__ void sts_v4(uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
  asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}
__device__ __forceinline__ float ex2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// ---- packed fp32x2 arithmetic (sm_100: one FMA-pipe instruction for two lanes of a 64-bit register pair) ----
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float lo, float hi) {
  f32x2 r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void unpack2(f32x2 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
  f32x2 d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
  return d;
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) {
  f32x2 d;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  return d;
}
// 2^x for two lanes on the FMA pipe (no MUFU): x = n + r, n = rint(x) taken from the mantissa of
// x + 1.5*2^23, r in [-0.5, 0.5]; degree-2 minimax polynomial of 2^r (relative error 1.7e-3, below the
// 2^-9 = 2.0e-3 bf16 rounding of P that follows; the same p feeds the row sum, so weights stay normalised); n is added to the exponent field.  x is clamped at
// -126 (result ~1e-38 instead of exponent wrap-around); callers guarantee x <= 2^7.
__device__ __forceinline__ void exp2_poly2(f32x2 x2, float& p0, float& p1) {
  float x0, x1;
  unpack2(x2, x0, x1);
  x2 = pack2(fmaxf(x0, -126.f), fmaxf(x1, -126.f));
  const f32x2 t2 = add2(x2, pack2(12582912.f, 12582912.f));
  const f32x2 n2 = add2(t2, pack2(-12582912.f, -12582912.f));
  const f32x2 r2 = fma2(n2, pack2(-1.f, -1.f), x2);
  f32x2 q2 = fma2(pack2(0.23842722f, 0.23842722f), r2, pack2(0.70344825f, 0.70344825f));
  q2 = fma2(q2, r2, pack2(1.00044327f, 1.00044327f));
  float q0, q1, t0, t1;
  unpack2(q2, q0, q1);
  unpack2(t2, t0, t1);
  p0 = __int_as_float(__float_as_int(q0) + (__float_as_int(t0) << 23));
  p1 = __int_as_float(__float_as_int(q1) + (__float_as_int(t1) << 23));
}

// ---- UMMA descriptors (bit layout: cute/arch/mma_sm100_desc.hpp) --------------------------------
// shared-memory matrix descriptor, SWIZZLE_128B, version 1 (Blackwell)
__device__ __forceinline__ uint64_t smem_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr >> 4) & 0x3FFF);
  d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16;
  d |= (uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32;
  d |= (uint64_t)1 << 46;   // descriptor version
  d |= (uint64_t)2 << 61;   // layout type: SWIZZLE_128B
  return d;
}
// instruction descriptor: D fp32, A/B bf16, M x N, A K-major, B K-major or MN-major
__host__ __device__ constexpr uint32_t instr_desc(int M, int N, int b_mn_major) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)b_mn_major << 16) | ((uint32_t)(N >> 3) << 17) |
         ((uint32_t)(M >> 4) << 24);
}

// ---- visible-set walk (identical in every role) ---------------------------------------------
struct TileWalk {
  const AttnParams& p;
  int n_vis, q_hi;   // q_hi: last valid query row of this CTA's tile
  int pi, tok0, len, page;
  bool is_self;
  __device__ TileWalk(const AttnParams& p_, int n_vis_, int q_hi_) : p(p_), n_vis(n_vis_), q_hi(q_hi_), pi(-1), tok0(0), len(0), page(-1), is_self(false) {}
  __device__ __forceinline__ int page_length(int idx, int* page_out, bool* self_out) const {
    const bool self = idx == n_vis;
    const int pg = self ? p.self_page : p.page_table[idx];
    *page_out = pg;
    *self_out = self;
    if (pg < 0 || pg >= p.n_pages) return 0;
    int l = min(p.page_len[pg], p.page_cap);
    if (self) l = min(l, p.self_offset + q_hi + 1);   // tokens no row of this tile may see are skipped
    return max(l, 0);
  }
  __device__ int count() const {
    const int n_iter = n_vis + (p.self_page >= 0 ? 1 : 0);
    int n = 0, pg;
    bool sf;
    for (int i = 0; i < n_iter; ++i) n += (page_length(i, &pg, &sf) + kBlockN - 1) / kBlockN;
    return n;
  }
  __device__ void skip(int n) { for (int k = 0; k < n; ++k) next(); }
  // advance to the next tile; returns false when exhausted
  __device__ bool next() {
    const int n_iter = n_vis + (p.self_page >= 0 ? 1 : 0);
    if (pi >= 0 && tok0 + kBlockN < len) { tok0 += kBlockN; return true; }
    while (++pi < n_iter) {
      len = page_length(pi, &page, &is_self);
      if (len > 0) { tok0 = 0; return true; }
    }
    return false;
  }
};

// D[tmem] (+)= A[tmem] * B[smem]: A = P as packed bf16 pairs, lane = row, 8 columns per k-step of 16
__device__ __forceinline__ void umma_bf16_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t"
      "}" ::"r"(d_tmem),
      "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t* r) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
      "{%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" ::"r"(taddr),
      "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]), "r"(r[10]),
      "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
      : "memory");
}
// one lane of a fully converged warp (the compiler keeps tcgen05 operands in uniform registers
// without a per-instruction active-lane loop only when the guard comes from elect.sync)
__device__ __forceinline__ bool elect_one() {
  uint32_t pred;
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "elect.sync _|p, 0xffffffff;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t"
      "}"
      : "=r"(pred));
  return pred != 0;
}
template <int N> __device__ __forceinline__ void reg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N> __device__ __forceinline__ void reg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }
__device__ __forceinline__ void pair_bar_sync(int id) { asm volatile("bar.sync %0, %1;" ::"r"(id), "n"(32 * kWGs) : "memory"); }
__device__ __forceinline__ void softmax_bar_sync() { asm volatile("bar.sync 5, %0;" ::"n"(kSoftmaxThreads) : "memory"); }

#ifdef VCS_ATTN_TRACE
#define TRACE(slot, idx) do { if (trace_on) trace[(slot) * 64 + ((idx) < 64 ? (idx) : 63)] = clock64(); } while (0)
#else
#define TRACE(slot, idx) do { } while (0)
#endif

__global__ void __launch_bounds__(kThreads, 1)
attn_tc_kernel(const AttnParams p, const __grid_constant__ CUtensorMap tmap_k, const __grid_constant__ CUtensorMap tmap_v) {
  pdl_wait();
  pdl_launch_dependents();
  extern __shared__ uint8_t smem_raw[];

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  int h = blockIdx.y;
#ifdef VCS_ATTN_TRACE
  long long* trace = reinterpret_cast<long long*>(p.trace);
  const bool trace_on = trace && blockIdx.x == gridDim.x / 2 && blockIdx.y == 0 && lane == 0;
  long long* cta_log = trace ? trace + 18 * 64 + (blockIdx.y * gridDim.x + blockIdx.x) * 4 : nullptr;
  if (cta_log && threadIdx.x == 0) {
    unsigned long long t; unsigned smid;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
    cta_log[0] = (long long)t; cta_log[2] = smid;
  }
#endif
  int nq = p.nq_d ? *p.nq_d : p.nq_cap;
  if (nq > p.nq_cap) {
    nq = p.nq_cap;
    if (p.status && threadIdx.x == 0 && blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0) atomicOr(p.status, VCS_FLAG_COUNT_CLAMPED);
  }
  // ---- role of this CTA ----------------------------------------------------------------------
  // Normally CTA (x, y, z) = part z of n_split of item (q tile x, head y); CTAs with x beyond the
  // device count leave.  With tail_split (grids of a wave or more, n_split == 1) those spare CTAs
  // HELP instead: when the items leave an under-filled last wave (R = items mod SMs <= SMs / 2),
  // each of its R items is cut into s <= 4 KV parts, the owner keeps part 0 and spare CTAs (which
  // sit all over the launch order, so they run early) take the others; partials are merged by the
  // last CTA to finish, as in the host-chosen split.  The last wave then lasts 1/s of an item.
  int qx = blockIdx.x, part = blockIdx.z, n_eff = p.n_split, part_slot = -1;
  {
    const int q_act = (nq + kBlockM - 1) / kBlockM;
    int s_tail = 1, first_tail = 0x7fffffff, R = 0;
    if (p.tail_split && q_act * p.Hq > p.sm_count) {
      const int items = q_act * p.Hq, waves = items / p.sm_count;
      R = items - waves * p.sm_count;
      if (waves >= 1 && R > 0 && 2 * R <= p.sm_count) {
        const int spare = p.Hq * ((int)gridDim.x - q_act);
        s_tail = min(4, min(1 + spare / R, p.sm_count / R));
        first_tail = waves * p.sm_count;
      }
    }
    if (qx < q_act) {
      const int rank = h * q_act + qx;
      if (s_tail > 1 && rank >= first_tail) { part = 0; n_eff = s_tail; part_slot = (rank - first_tail) * 4; }
      else if (n_eff > 1) part_slot = (h * (int)gridDim.x + qx) * n_eff;
    } else {
      if (s_tail <= 1) return;   // uniform: whole CTA
      const int hidx = h * ((int)gridDim.x - q_act) + (qx - q_act);
      if (hidx >= R * (s_tail - 1)) return;
      const int tr = hidx / (s_tail - 1), rank = first_tail + tr;
      part = 1 + hidx % (s_tail - 1);
      n_eff = s_tail;
      part_slot = tr * 4;
      h = rank / q_act;
      qx = rank - h * q_act;
    }
  }
  const int kvh = h / (p.Hq / p.Hkv);
  const int q0 = qx * kBlockM;
  int n_vis = p.n_vis_d ? *p.n_vis_d : p.n_vis_cap;
  n_vis = max(0, min(n_vis, p.n_vis_cap));
  const int q_hi = min(q0 + kBlockM, nq) - 1;

  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  if (smem_base + Smem::total > smem_u32(smem_raw) + Smem::total + kSlack) __trap();   // raw base less aligned than assumed
  uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));
  const uint32_t sQ = smem_base + Smem::q, sK = smem_base + Smem::k, sV = smem_base + Smem::v;
  const uint32_t bars = smem_base + Smem::bar;
  auto bar = [&](int i) { return bars + 8u * i; };

  TileWalk walk0(p, n_vis, q_hi);
  const int n_total = walk0.count();
  // split-KV: this CTA handles tiles [t0, t0 + n_tiles) of the item's walk
  const int t0 = (int)((long long)part * n_total / n_eff);
  const int n_tiles = (int)((long long)(part + 1) * n_total / n_eff) - t0;

  if (threadIdx.x == 0) {
    mbar_init(bar(Q_FULL), kSoftmaxThreads);
    for (int s = 0; s < kStages; ++s) {
      mbar_init(bar(KV_FULL + s), 1);
      mbar_init(bar(KV_EMPTY + s), 1);
    }
    for (int w = 0; w < 2; ++w) {
      mbar_init(bar(S_FULL + w), 1);
      mbar_init(bar(P_FULL + w), kSoftmaxThreads);
    }
    mbar_init(bar(PV_DONE), 1);
    mbar_init(bar(ALL_DONE), 1);
    fence_barrier_init();
  }
  if (warp == kWarpMma) tmem_alloc(smem_base + Smem::tmem_slot, kTmemCols);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *reinterpret_cast<volatile uint32_t*>(smem_gen + Smem::tmem_slot);

  if (warp >= kWarpTma) {
  reg_dec<kRegsOther>();
  if (warp == kWarpTma) {
    // ===================== TMA producer =====================
    // Ring slot u % kStages (u = 0, 1, ...) holds { K(u) in its K part, V(u - 2) in its V part } under
    // ONE full / empty barrier pair: MMA iteration i = u - 2 consumes exactly V(i) and K(i + 2).
    // The whole warp walks the page table and waits; one elected lane issues the copies.
    if (n_tiles > 0) {
      if (elect_one()) {
        tma_prefetch_desc(&tmap_k);
        tma_prefetch_desc(&tmap_v);
      }
      TileWalk wk(p, n_vis, q_hi), wv(p, n_vis, q_hi);
      wk.skip(t0);
      wv.skip(t0);
      for (int u = 0; u < n_tiles + 2; ++u) {
        const int s = u % kStages;
        const bool has_k = u < n_tiles, has_v = u >= 2;
        if (has_k) wk.next();
        if (has_v) wv.next();
        mbar_wait(bar(KV_EMPTY + s), ((uint32_t)(u / kStages) & 1u) ^ 1u);
        if (elect_one()) {
          mbar_expect_tx(bar(KV_FULL + s), (has_k ? kTileBytes : 0) + (has_v ? kTileBytes : 0));
          if (has_k) {
            tma_load_4d(sK + s * kTileBytes, &tmap_k, bar(KV_FULL + s), 0, wk.tok0, kvh, wk.page);
            tma_load_4d(sK + s * kTileBytes + kHalfBytes, &tmap_k, bar(KV_FULL + s), 64, wk.tok0, kvh, wk.page);
          }
          if (has_v) {
            tma_load_4d(sV + s * kTileBytes, &tmap_v, bar(KV_FULL + s), 0, wv.tok0, kvh, wv.page);
            tma_load_4d(sV + s * kTileBytes + kHalfBytes, &tmap_v, bar(KV_FULL + s), 64, wv.tok0, kvh, wv.page);
          }
        }
        __syncwarp();
      }
    }
  } else if (warp == kWarpMma) {
    // ===================== MMA issuer =====================
    // The whole warp walks the loop (waits are warp-wide); one elected lane issues.  Descriptors are
    // built once and advanced by adding (byte offset >> 4) to their low word.  Per KV tile: two
    // waits (ring slot, P), one issue block (PV(i) then QK(i+2)), two commits.
    if (n_tiles > 0) {
      constexpr uint32_t idesc_qk = instr_desc(kBlockM, kBlockN, 0);
      constexpr uint32_t idesc_pv = instr_desc(kBlockM, kHeadDim, 1);
      const uint64_t descQ = smem_desc(sQ, 16, 1024), descK = smem_desc(sK, 16, 1024);
      const uint64_t descV = smem_desc(sV, kHalfBytes, 1024);
      // S_b[128 x 128] = Q[128 x d] . K_t[128 x d]^T : both K-major, 8 k-steps of 16 over d
      auto qk = [&](int t, int s, int k0, int k1) {
        const uint32_t col = (t & 1) ? kColS1 : kColS0;
        const uint64_t dk = descK + (uint64_t)((s * kTileBytes) >> 4);
#pragma unroll
        for (int kk = k0; kk < k1; ++kk) {
          const uint64_t off = (uint64_t)(((kk >> 2) * kHalfBytes + (kk & 3) * 32) >> 4);
          umma_bf16_ss(tmem + col, descQ + off, dk + off, idesc_qk, kk > 0);
        }
      };
      // One elected lane runs the whole loop (waits included).  The tensor pipe executes in order
      // and its queue is short, so everything that is not an MMA is kept off the tail of an
      // iteration: ring slot / phase are carried incrementally (no div/mod), the next slot's barrier
      // is polled before the last two Q.K^T k-steps are issued, and only the P wait + fence sit
      // between the last MMA of one iteration and the first of the next.
      if (elect_one()) {
        mbar_wait(bar(Q_FULL), 0);
        tc_fence_after();
        int s = 0;
        uint32_t ph = 0;
        mbar_wait(bar(KV_FULL + 0), 0);
        for (int u = 0; u < n_tiles + 2; ++u) {
          const int i = u - 2;
          if (i >= 0) mbar_wait(bar(P_FULL + (i & 1)), (uint32_t)(i >> 1) & 1u);
          tc_fence_after();
          TRACE(13, u);
          if (i >= 0) {
            // O[128 x d] (+)= P_b[128 x 128] . V_i[128 x d] : P from TMEM (8 columns per k-step), V MN-major
            // (d contiguous; 64-wide d groups 16 KB apart = LBO, 8-token groups 1 KB apart = SBO)
            const uint32_t colP = (i & 1) ? kColS1 : kColS0;
            const uint64_t dv = descV + (uint64_t)((s * kTileBytes) >> 4);
#pragma unroll
            for (int kk = 0; kk < kBlockN / 16; ++kk)
              umma_bf16_ts(tmem + kColO, tmem + colP + 8 * kk, dv + (uint64_t)((kk * 2048) >> 4), idesc_pv, (i > 0) | (kk > 0));
          }
          const int s_next = s + 1 == kStages ? 0 : s + 1;
          const uint32_t ph_next = s + 1 == kStages ? ph ^ 1u : ph;
          if (u < n_tiles) {
            qk(u, s, 0, 6);
            if (u + 1 < n_tiles + 2) mbar_wait(bar(KV_FULL + s_next), ph_next);
            qk(u, s, 6, 8);
            umma_commit(bar(KV_EMPTY + s));
            umma_commit(bar(S_FULL + (u & 1)));
          } else {
            umma_commit(bar(KV_EMPTY + s));
            umma_commit(bar(PV_DONE));   // no later QK whose S_FULL could tell the softmax that PV(i) is done
            if (u + 1 < n_tiles + 2) mbar_wait(bar(KV_FULL + s_next), ph_next);
          }
          s = s_next;
          ph = ph_next;
          TRACE(16, u);
        }
        umma_commit(bar(ALL_DONE));
      }
      __syncwarp();
    }
  }
  } else {
    reg_inc<kRegsSoftmax>();
    // ===================== softmax warpgroups (warps 0-3: even tiles, warps 4-7: odd tiles) ==========
    const int wg = warp >> 2;
    const int r = threadIdx.x & (kBlockM - 1);   // row in tile == TMEM lane
    const int i = q0 + r;                        // global query row
    const bool row_valid = i < nq;
    const uint32_t lane_addr = tmem + ((uint32_t)((warp & 3) * 32) << 16);
    const int c0 = kCols * wg;                      // first S column (token of the tile) / O column (d) of this thread
    float* xch = reinterpret_cast<float*>(smem_gen + Smem::xch);

    // ---- Q tile: load, M-RoPE, bf16, swizzled K-major store (each warpgroup: 32 of the 64 pairs) ----
    {
      const uint32_t row_off = (uint32_t)r * 128u;
      if (row_valid && n_tiles > 0) {
        const __nv_bfloat16* q = static_cast<const __nv_bfloat16*>(p.q) + (size_t)i * p.q_stride + (size_t)h * kHeadDim;
        const int pt = p.q_pos3[3 * i + 0], ph = p.q_pos3[3 * i + 1], pw = p.q_pos3[3 * i + 2];
#pragma unroll 2
        for (int cc = 0; cc < 8 / kWGs; ++cc) {
          const int c = (8 / kWGs) * wg + cc;
          const uint4 lo4 = ldg_nc_v4(q + 8 * c), hi4 = ldg_nc_v4(q + 64 + 8 * c);
          const uint32_t lo[4] = {lo4.x, lo4.y, lo4.z, lo4.w}, hi[4] = {hi4.x, hi4.y, hi4.z, hi4.w};
          uint32_t olo[4], ohi[4];
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            float rl[2], rh[2];
#pragma unroll
            for (int b = 0; b < 2; ++b) {
              const int m = 8 * c + 2 * e + b;
              const int ax = p.rope.axis_of[m];
              const int pos = ax == 0 ? pt : (ax == 1 ? ph : pw);
              float sn, cs;
              rope_sincos_fast(pos, p.rope.turn_frac[m], &sn, &cs);
              const float xl = b ? bf16_hi(lo[e]) : bf16_lo(lo[e]);
              const float xh = b ? bf16_hi(hi[e]) : bf16_lo(hi[e]);
              rl[b] = xl * cs - xh * sn;
              rh[b] = xh * cs + xl * sn;
            }
            olo[e] = pack_bf16(rl[0], rl[1]);
            ohi[e] = pack_bf16(rh[0], rh[1]);
          }
          const uint32_t sw = (uint32_t)((c ^ (r & 7)) << 4);
          sts_v4(sQ + row_off + sw, olo[0], olo[1], olo[2], olo[3]);
          sts_v4(sQ + kHalfBytes + row_off + sw, ohi[0], ohi[1], ohi[2], ohi[3]);
        }
      } else {
#pragma unroll
        for (int cc = 0; cc < 8 / kWGs; ++cc) {
          const int c = (8 / kWGs) * wg + cc;
          sts_v4(sQ + row_off + (c << 4), 0, 0, 0, 0);
          sts_v4(sQ + kHalfBytes + row_off + (c << 4), 0, 0, 0, 0);
        }
      }
      fence_proxy_async();
      mbar_arrive(bar(Q_FULL));
    }

    const float scale_log2 = p.scale * 1.4426950408889634f;
    float m_used = -INFINITY, l_run = 0.f;       // m_used is identical in both threads of a row; l_run is this half's sum
    TileWalk w(p, n_vis, q_hi);
    w.skip(t0);
    for (int j = 0; j < n_tiles && w.next(); ++j) {
      const int buf = j & 1;
      const uint32_t colS = buf ? kColS1 : kColS0;
      if ((warp & 3) == 0 && wg < 2) TRACE(wg * 6 + 0, j);
      mbar_wait(bar(S_FULL + buf), (uint32_t)(j >> 1) & 1u);
      tc_fence_after();
      if ((warp & 3) == 0 && wg < 2) TRACE(wg * 6 + 1, j);
#if defined(VCS_EXP) && (VCS_EXP & 2)
      if (j > 0) { tc_fence_before(); mbar_arrive(bar(P_FULL + buf)); continue; }
#endif
      float s[kCols];
#pragma unroll
      for (int c = 0; c < kCols / 32; ++c) tmem_ld32(lane_addr + colS + c0 + 32 * c, s + 32 * c);
      tmem_wait_ld();
      if ((warp & 3) == 0 && wg < 2) TRACE(wg * 6 + 2, j);

      // visible columns of this row in this tile: [0, limit) in tile coordinates, this thread owns [c0, c0 + 64)
      int limit = min(kBlockN, w.len - w.tok0);
      if (w.is_self) limit = min(limit, p.self_offset + i - w.tok0 + 1);
      limit -= c0;
      const bool masked = __any_sync(0xffffffffu, limit < kCols);   // warp-uniform: tail / diagonal tiles only
      if (masked) {
#pragma unroll
        for (int c = 0; c < kCols; ++c) s[c] = c < limit ? s[c] : -INFINITY;
      }
      float mx[8];
#pragma unroll
      for (int k = 0; k < 8; ++k) mx[k] = fmaxf(s[k], s[8 + k]);
#pragma unroll
      for (int c = 16; c < kCols; c += 16) {
#pragma unroll
        for (int k = 0; k < 8; ++k) mx[k] = fmaxf(fmaxf(mx[k], s[c + k]), s[c + 8 + k]);
      }
      const float m_half = fmaxf(fmaxf(fmaxf(mx[0], mx[1]), fmaxf(mx[2], mx[3])), fmaxf(fmaxf(mx[4], mx[5]), fmaxf(mx[6], mx[7])));
      // exchange with the thread that owns the other 64 columns of this row (warp +-4).  The first
      // pair barrier makes sure the partner has read the previous tile's value (it is long past that
      // point: the barrier is there for correctness, not waited on); after the second one BOTH
      // halves of S_buf are in registers, so P may overwrite S_buf.
      pair_bar_sync(1 + (warp & 3));
      xch[wg * kBlockM + r] = m_half;
      pair_bar_sync(1 + (warp & 3));
      float m_row = m_half;
#pragma unroll
      for (int g2 = 0; g2 < kWGs; ++g2) m_row = fmaxf(m_row, xch[g2 * kBlockM + r]);
      const float m_tile = m_row * scale_log2;
      const float m_new = fmaxf(m_used, m_tile);

      // lazy rescale, decided per warp (tcgen05.ld/st are warp-collective); both warps of a pair see
      // the same row maxima and take the same decision.  O must be idle: PV(j-1) has completed.
      const bool grow = (m_new - m_used) > kRescaleThreshold;   // true on the first visible tile (m_used = -inf)
      if (__any_sync(0xffffffffu, grow)) {
        const float alpha = (m_new == -INFINITY) ? 1.f : ex2(m_used - m_new);   // m_used = -inf -> 0
        l_run *= alpha;
        m_used = m_new;
        if (j > 0) {
          // PV(j-1) must have finished: QK(j+1) was issued after it, so S_FULL of tile j+1 implies it;
          // the last tile has no successor and waits for the first PV_DONE commit instead
          if (j + 1 < n_tiles) mbar_wait(bar(S_FULL + (buf ^ 1)), (uint32_t)((j + 1) >> 1) & 1u);
          else mbar_wait(bar(PV_DONE), 0);
          tc_fence_after();
#pragma unroll
          for (int c = 0; c < kCols / 32; ++c) {
            float o[32];
            tmem_ld32(lane_addr + kColO + c0 + 32 * c, o);
            tmem_wait_ld();
#pragma unroll
            for (int e = 0; e < 32; ++e) o[e] *= alpha;
            tmem_st32(lane_addr + kColO + c0 + 32 * c, o);
          }
        }
      }
      const float neg_m = (m_used == -INFINITY) ? 0.f : -m_used;
      if ((warp & 3) == 0 && wg < 2) TRACE(wg * 6 + 3, j);
      // P = 2^(s * scale_log2 - m_used) as bf16 pairs -> TMEM over the head of S_buf (this thread's 64
      // tokens = 32 packed columns at 32 * wg); row sums in four packed accumulators.  On unmasked
      // tiles kPolyNum of every kPolyDen column pairs take the FMA-pipe polynomial instead of MUFU.EX2
      // (the MUFU pipe, 16/clk/SM, would otherwise cost as many cycles per tile as the two MMAs).
      // Masked tiles hold -inf: MUFU only.
      const f32x2 scale2 = pack2(scale_log2, scale_log2), negm2 = pack2(neg_m, neg_m);
      f32x2 lsum[4] = {0ull, 0ull, 0ull, 0ull};
      if (!masked) {
#pragma unroll
        for (int c = 0; c < kCols / 32; ++c) {
          uint32_t pk[16];
#pragma unroll
          for (int e = 0; e < 32; e += 2) {
            const f32x2 x2 = fma2(pack2(s[32 * c + e], s[32 * c + e + 1]), scale2, negm2);
            float p0, p1;
            if (((e >> 1) % kPolyDen) < kPolyNum) {
              exp2_poly2(x2, p0, p1);
            } else {
              float x0, x1;
              unpack2(x2, x0, x1);
              p0 = ex2(x0);
              p1 = ex2(x1);
            }
            lsum[(e >> 1) & 3] = add2(lsum[(e >> 1) & 3], pack2(p0, p1));
            pk[e >> 1] = pack_bf16(p0, p1);
          }
          tmem_st16(lane_addr + colS + (kCols / 2) * wg + 16 * c, pk);
        }
      } else if (__all_sync(0xffffffffu, limit <= 0)) {
        // ragged page tail / diagonal: none of this warp's columns is visible to any of its rows -> P = 0
        uint32_t pk[16];
#pragma unroll
        for (int e = 0; e < 16; ++e) pk[e] = 0u;
#pragma unroll
        for (int c = 0; c < kCols / 32; ++c) tmem_st16(lane_addr + colS + (kCols / 2) * wg + 16 * c, pk);
      } else {
#pragma unroll
        for (int c = 0; c < kCols / 32; ++c) {
          uint32_t pk[16];
          if (c > 0 && __all_sync(0xffffffffu, limit <= 32 * c)) {   // this 32-column chunk is hidden from every row of the warp
#pragma unroll
            for (int e = 0; e < 16; ++e) pk[e] = 0u;
            tmem_st16(lane_addr + colS + (kCols / 2) * wg + 16 * c, pk);
            continue;
          }
#pragma unroll
          for (int e = 0; e < 32; e += 2) {
            const float p0 = ex2(fmaf(s[32 * c + e], scale_log2, neg_m));
            const float p1 = ex2(fmaf(s[32 * c + e + 1], scale_log2, neg_m));
            lsum[(e >> 1) & 3] = add2(lsum[(e >> 1) & 3], pack2(p0, p1));
            pk[e >> 1] = pack_bf16(p0, p1);
          }
          tmem_st16(lane_addr + colS + (kCols / 2) * wg + 16 * c, pk);
        }
      }
      {
        float a0, a1, b0, b1;
        unpack2(add2(lsum[0], lsum[1]), a0, a1);
        unpack2(add2(lsum[2], lsum[3]), b0, b1);
        l_run += (a0 + a1) + (b0 + b1);
      }
      if ((warp & 3) == 0 && wg < 2) TRACE(wg * 6 + 4, j);
      tmem_wait_st();
      tc_fence_before();
      mbar_arrive(bar(P_FULL + buf));
      if ((warp & 3) == 0 && wg < 2) TRACE(wg * 6 + 5, j);
    }

    // ---- epilogue: add the two halves' row sums, O / l -> bf16 -> global (each warpgroup: 64 d columns) ----
    if (n_tiles > 0) {
      mbar_wait(bar(ALL_DONE), 0);
      tc_fence_after();
    }
    float* ex = reinterpret_cast<float*>(smem_gen + Smem::q);   // Q tile no longer needed: every MMA has completed
    ex[wg * kBlockM + r] = l_run;
    softmax_bar_sync();
    float l_all = 0.f;
#pragma unroll
    for (int g2 = 0; g2 < kWGs; ++g2) l_all += ex[g2 * kBlockM + r];
    __nv_bfloat16* o_row = static_cast<__nv_bfloat16*>(p.out) + (size_t)i * p.out_stride + (size_t)h * kHeadDim;
    if (n_eff > 1) {
      // ---- split-KV: publish this CTA's unnormalised partial; the last CTA of the item merges ----
      constexpr int kPartFloats = kBlockM * kHeadDim + 2 * kBlockM;
      const int item = part_slot / (p.tail_split ? 4 : n_eff);          // ticket counter of this item
      float* pbuf = p.part + ((size_t)part_slot + part) * kPartFloats;
#pragma unroll
      for (int cc = 0; cc < kCols / 32; ++cc) {   // tcgen05.ld is warp-collective: load converged, store per valid row
        const int col = c0 + 32 * cc;
        float o[32];
        if (n_tiles > 0) {
          tmem_ld32(lane_addr + kColO + col, o);
          tmem_wait_ld();
        }
        if (row_valid) {
#pragma unroll
          for (int e = 0; e < 32; e += 4)
            *reinterpret_cast<float4*>(pbuf + (size_t)r * kHeadDim + col + e) =
                n_tiles > 0 ? make_float4(o[e], o[e + 1], o[e + 2], o[e + 3]) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
      }
      if (row_valid && wg == 0) {
        pbuf[kBlockM * kHeadDim + r] = m_used;
        pbuf[kBlockM * kHeadDim + kBlockM + r] = l_all;
      }
      __threadfence();
      softmax_bar_sync();
      int* flag = reinterpret_cast<int*>(smem_gen + Smem::q + 4096);
      if (threadIdx.x == 0) {
        const unsigned int t = atomicAdd(&p.part_counter[item], 1u);
        const int last = t == (unsigned)(n_eff - 1);
        if (last) p.part_counter[item] = 0u;   // self-reset for the next call
        *flag = last;
      }
      softmax_bar_sync();
      if (*flag && row_valid) {
        __threadfence();
        const float* base = p.part + (size_t)part_slot * kPartFloats;
        float m_all = -INFINITY;
        for (int z = 0; z < n_eff; ++z) m_all = fmaxf(m_all, __ldcg(base + (size_t)z * kPartFloats + kBlockM * kHeadDim + r));
        float acc[kCols];
#pragma unroll
        for (int e = 0; e < kCols; ++e) acc[e] = 0.f;
        float l_sum = 0.f;
        for (int z = 0; z < n_eff; ++z) {
          const float* pz = base + (size_t)z * kPartFloats;
          const float mz = __ldcg(pz + kBlockM * kHeadDim + r);
          const float wz = mz == -INFINITY ? 0.f : ex2(mz - m_all);
          l_sum = fmaf(__ldcg(pz + kBlockM * kHeadDim + kBlockM + r), wz, l_sum);
#pragma unroll
          for (int e = 0; e < kCols; e += 4) {
            const float4 v = __ldcg(reinterpret_cast<const float4*>(pz + (size_t)r * kHeadDim + c0 + e));
            acc[e] = fmaf(v.x, wz, acc[e]); acc[e + 1] = fmaf(v.y, wz, acc[e + 1]);
            acc[e + 2] = fmaf(v.z, wz, acc[e + 2]); acc[e + 3] = fmaf(v.w, wz, acc[e + 3]);
          }
        }
        const float inv = l_sum > 0.f ? 1.f / l_sum : 0.f;
#pragma unroll
        for (int e = 0; e < kCols; e += 8) {
          uint4 v;
          v.x = pack_bf16(acc[e] * inv, acc[e + 1] * inv);
          v.y = pack_bf16(acc[e + 2] * inv, acc[e + 3] * inv);
          v.z = pack_bf16(acc[e + 4] * inv, acc[e + 5] * inv);
          v.w = pack_bf16(acc[e + 6] * inv, acc[e + 7] * inv);
          stg_v4(o_row + c0 + e, v);
        }
        if (wg == 0 && p.lse)
          p.lse[(size_t)h * p.nq_cap + i] = l_sum > 0.f ? (m_all + log2f(l_sum)) * 0.6931471805599453f : -INFINITY;
      }
    } else {
    const float inv_l = l_all > 0.f ? 1.f / l_all : 0.f;
#pragma unroll
    for (int cc = 0; cc < kCols / 32; ++cc) {
      const int col = c0 + 32 * cc;
      float o[32];
      if (n_tiles > 0) {
        tmem_ld32(lane_addr + kColO + col, o);
        tmem_wait_ld();
      }
#pragma unroll
      for (int e = 0; e < 32; ++e) o[e] = n_tiles > 0 ? o[e] * inv_l : 0.f;
      if (row_valid) {
#pragma unroll
        for (int e = 0; e < 32; e += 8) {
          uint4 v;
          v.x = pack_bf16(o[e], o[e + 1]);
          v.y = pack_bf16(o[e + 2], o[e + 3]);
          v.z = pack_bf16(o[e + 4], o[e + 5]);
          v.w = pack_bf16(o[e + 6], o[e + 7]);
          stg_v4(o_row + col + e, v);
        }
      }
    }
    if (wg == 0 && row_valid && p.lse)
      p.lse[(size_t)h * p.nq_cap + i] = l_all > 0.f ? (m_used + log2f(l_all)) * 0.6931471805599453f : -INFINITY;
    }
    tc_fence_before();
  }

  __syncthreads();
#ifdef VCS_ATTN_TRACE
  if (cta_log && threadIdx.x == 0) {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    cta_log[1] = (long long)t; cta_log[3] = n_tiles;
  }
#endif
  if (warp == kWarpMma) {
    tc_fence_after();
    tmem_dealloc(tmem, kTmemCols);
  }
}

}  // namespace tc

bool attn_tc_supported(const vcs_kv_pool* pool) {
  if (!pool || !pool->opaque_h) return false;
  const PoolOpaque* o = reinterpret_cast<const PoolOpaque*>(pool->opaque_h);
  return o->magic == kPoolMagic && o->has_tma && pool->dtype == VCS_BF16 && pool->d == tc::kHeadDim;
}

// split-KV factor from HOST capacities only (device counts are unknown here): split when the
// (q tile, head) items cannot fill the SMs, never below ~4 KV tiles per split, at most 16.
static int attn_tc_sm_count() {
  static int sm_count = 0;
  if (sm_count == 0) {
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) {
      cudaGetLastError();
      n = 148;
    }
    sm_count = n;
  }
  return sm_count;
}

// grids that can reach a wave or more may end in an under-filled last wave: give them the buffers for
// the device-side tail split (at most SMs / 2 items x 4 parts)
static bool attn_tc_tail_capable(const vcs_kv_pool* pool, int nq_cap) {
  return (long long)((nq_cap + tc::kBlockM - 1) / tc::kBlockM) * pool->Hq > attn_tc_sm_count();
}

int attn_tc_splits(const vcs_kv_pool* pool, int nq_cap, int n_vis_cap) {
  const int sm_count = attn_tc_sm_count();
  const long long items = (long long)((nq_cap + tc::kBlockM - 1) / tc::kBlockM) * pool->Hq;
  if (items <= 0 || items * 4 >= (long long)sm_count * 3) return 1;
  const long long tiles_cap = (long long)(n_vis_cap + 1) * ((pool->page_cap + tc::kBlockN - 1) / tc::kBlockN);
  long long ns = sm_count / items;
  if (ns > tiles_cap / 4) ns = tiles_cap / 4;
  if (ns > 16) ns = 16;
  return ns < 1 ? 1 : (int)ns;
}

static size_t attn_tc_counter_bytes(const vcs_kv_pool* pool, int nq_cap) {
  return round_up((size_t)((nq_cap + tc::kBlockM - 1) / tc::kBlockM) * pool->Hq * sizeof(unsigned int), 256);
}
#ifdef VCS_ATTN_TRACE
constexpr size_t kTraceBytes = 18 * 64 * 8 + 4096 * 32;
#else
constexpr size_t kTraceBytes = 0;
#endif
// layout: [256 reserved][trace (debug builds)][item counters][partials: items x n_split x (128x128 + 256) floats]
size_t attn_tc_workspace_bytes(const vcs_kv_pool* pool, int nq_cap, int n_vis_cap) {
  const int ns = attn_tc_splits(pool, nq_cap, n_vis_cap);
  size_t b = 256 + kTraceBytes;
  const size_t part_bytes = (size_t)(tc::kBlockM * tc::kHeadDim + 2 * tc::kBlockM) * sizeof(float);
  if (ns > 1) {
    const size_t items = (size_t)((nq_cap + tc::kBlockM - 1) / tc::kBlockM) * pool->Hq;
    b += attn_tc_counter_bytes(pool, nq_cap) + items * ns * part_bytes;
  } else if (attn_tc_tail_capable(pool, nq_cap)) {
    b += attn_tc_counter_bytes(pool, nq_cap) + (size_t)(attn_tc_sm_count() / 2) * 4 * part_bytes;
  }
  return b;
}

int launch_attn_tc(const AttnParams& p_in, const vcs_kv_pool* pool, void* workspace, size_t, cudaStream_t st) {
  AttnParams p = p_in;
  char* ws = static_cast<char*>(workspace);
#ifdef VCS_ATTN_TRACE
  p.trace = ws + 256;
#endif
  p.n_split = attn_tc_splits(pool, p.nq_cap, p.n_vis_cap);
  p.sm_count = attn_tc_sm_count();
  p.tail_split = (p.n_split == 1 && attn_tc_tail_capable(pool, p.nq_cap)) ? 1 : 0;
  if (p.n_split > 1 || p.tail_split) {
    p.part_counter = reinterpret_cast<unsigned int*>(ws + 256 + kTraceBytes);
    p.part = reinterpret_cast<float*>(ws + 256 + kTraceBytes + attn_tc_counter_bytes(pool, p.nq_cap));
  }
  static bool attr_set = false;
  const int smem = tc::Smem::total + tc::kSlack;
  if (!attr_set) {
    VCS_CUDA_OK(cudaFuncSetAttribute(tc::attn_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    attr_set = true;
  }
  const PoolOpaque* o = reinterpret_cast<const PoolOpaque*>(pool->opaque_h);
  dim3 grid((p.nq_cap + tc::kBlockM - 1) / tc::kBlockM, p.Hq, p.n_split);
  cudaError_t err = launch_pdl(tc::attn_tc_kernel, grid, dim3(tc::kThreads), smem, st, p, o->tmap_k, o->tmap_v);
  if (err == cudaSuccess) err = cudaGetLastError();
  if (err != cudaSuccess) VCS_FAIL(VCS_ECUDA, "attention (tcgen05) launch: %s", cudaGetErrorString(err));
  return VCS_OK;
}

}  // namespace vcs
