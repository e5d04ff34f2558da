// Bounded-visual-attention prefill for sm_100a (mask Eq. 4 :140-145): flash-style
// online softmax, page-table-driven TMA loads of K/V tiles out of the chunk-granular paged KV pool,
// tcgen05 MMAs (kind::f16, bf16 x bf16 -> fp32) with accumulators in TMEM.
//
// Work decomposition (attn.cuh): per kv head the rows rho = i * g + hh (the g q heads of token i are
// adjacent rows) form 128-row q tiles; two adjacent q tiles (A, B) are one ITEM and share every K/V tile
// they read (GQA: K/V are loaded once for all q heads of the group, and once for two q tiles).  The
// flat range of (stream, kv head, item, KV tile) iterations is cut into one contiguous part per CTA
// (persistent grid = one CTA per SM, "stream-K"): no under-filled wave, no idle SM.  An item that is
// cut by a CTA boundary leaves unnormalised fp32 partials (O, m, l) in the workspace and a small
// descriptor; the combine kernel that follows (same stream, PDL) merges them.  No CTA ever waits for
// another CTA.
//
// One CTA = 512 threads, 16 warps:
//   warps 0-3   softmax of q tile A: one thread = one row, 64 logits per KV tile in registers;
//   warps 4-7   softmax of q tile B.  Both also build their Q tile at the start of a segment: load,
//               rotate by M-RoPE on the fly, store bf16 into the 128B-swizzled K-major UMMA layout.
//   warps 8-11  correction: rescale O in TMEM when a row maximum grew (lazily, threshold 2^8), and the
//               epilogue (O / l -> bf16 -> global, or the fp32 partial of a split item).
//   warp 12     TMA producer: walks the page table (lane-distributed window of 32 entries), issues
//               cp.async.bulk.tensor for K and V tiles (4-D map over [page][kv head][token][d], box
//               64 x 64, SWIZZLE_128B) into a ring of eight 16 KB slots in the order the MMAs consume
//               them (K0 K1 | V0 K2 | V1 K3 | ...), and publishes per-tile metadata (valid tokens,
//               causal origin) for the softmax warps.
//   warps 13,14 MMA issuers (one elected lane each): warp 13 for q tile A (+ TMEM allocator), warp 14 for q
//               tile B.  Per iteration j:
//                 P.V_t(j)   then   Q.K^T_t(j+2) into the S buffer that P_t(j) just left
//               S is DOUBLE-buffered per q tile, so Q.K^T of iteration j+1 is in TMEM before the softmax
//               of iteration j ends: no softmax latency sits between two MMAs of a tile, the loop is
//               bound by throughput (tensor pipe / instruction dispatch of the softmax), not by a chain.
// TMEM (512 columns): S_A0 [0,64) S_A1 [64,128) | S_B0 [128,192) S_B1 [192,256) | O_A [256,384) |
// O_B [384,512).  P (bf16, 32 columns) overwrites the head of its S buffer once the row sits in registers.
#include "attn.cuh"
#include <type_traits>

namespace vcs {

namespace tc {

constexpr int kBlockM = 128;      // rows per q tile
constexpr int kBlockN = kAttnKvTile;   // KV tokens per tile (64)
constexpr int kHeadDim = 128;
constexpr int kStages = 8;        // 16 KB ring slots (K and V tiles in consumption order)
constexpr int kThreads = 512;
constexpr int kWarpTma = 12, kWarpMma = 13;
constexpr int kRegsSoftmax = 160, kRegsCorr = 112, kRegsOther = 80;   // 256*160 + 128*112 + 128*80 = 64 K registers
constexpr int kQHalfBytes = kBlockM * 128;           // Q: one [128 rows x 64 bf16] swizzled region: 16 KB
constexpr int kQTileBytes = 2 * kQHalfBytes;         // 32 KB: a [128 x 128] bf16 q tile as two d-halves
constexpr int kHalfBytes = kBlockN * 128;            // K / V: one [64 tokens x 64 bf16] swizzled region: 8 KB
constexpr int kTileBytes = 2 * kHalfBytes;           // 16 KB: a [64 x 128] bf16 tile as two d-halves
constexpr uint32_t kTmemCols = 512;
constexpr uint32_t kColS = 0, kColO = 256;           // S: + 128 * tile + 64 * buffer;  O: + 128 * tile
constexpr float kRescaleThreshold = 8.0f;            // log2 units
constexpr int kPolyNum = 1, kPolyDen = 4;            // share of exp2 evaluations moved from MUFU to the FMA pipe
constexpr int kMetaRing = 8;
constexpr int kCombineSlices = 16;                   // row slices of an item in the combine kernel (16 rows each)

struct CtaRange {
  long long J_total, lo, hi;
  int b, kvh, p, t;      // item and iteration inside it where this CTA starts
  int G;                 // CTAs that share the range: min(grid, J_total), so that every one of them has work
};

struct Smem {
  // offsets into the 1024-aligned dynamic shared memory
  static constexpr int q = 0;                                  // [2 q tiles][32 KB]
  static constexpr int kv = q + 2 * kQTileBytes;               // [kStages][16 KB]
  static constexpr int bar = kv + kStages * kTileBytes;        // mbarriers
  static constexpr int tmem_slot = bar + 512;
  static constexpr int meta = tmem_slot + 16;                  // [kMetaRing] int4: valid tokens, causal origin
  static constexpr int scale = meta + kMetaRing * 16;          // [2 tiles][2 buffers][128] O rescale factors
  static constexpr int fin_m = scale + 4 * kBlockM * 4;        // [2][128] final row max (log2 units)
  static constexpr int fin_l = fin_m + 2 * kBlockM * 4;        // [2][128] final row sum
  static constexpr int range = fin_l + 2 * kBlockM * 4;        // CtaRange
  static constexpr int plan = range + 64;                      // StreamPlan[kAttnMaxStreams]
  static constexpr int rope_tf = plan + kAttnMaxStreams * (int)sizeof(StreamPlan);   // [64] Q0.64 turn fractions of the rotary pairs
  static constexpr int rope_ax = rope_tf + 64 * 8;             // [64] axis (t / h / w) of the rotary pairs
  static constexpr int stage = rope_ax + 64;                   // epilogue staging: [4 warps][32 rows][128 B], 16-byte pieces XOR-swizzled
  static constexpr int total = stage + 4 * 32 * 128;
};
constexpr int kSlack = 1024;
static_assert(sizeof(CtaRange) <= 64, "CtaRange");
static_assert(Smem::total + kSlack <= 227 * 1024, "shared memory budget");

enum Bar {
  Q_FULL = 0, Q_EMPTY = 1,
  KV_FULL = 2, KV_EMPTY = KV_FULL + kStages,
  S_FULL = KV_EMPTY + kStages,      // [2 tiles][2 buffers]: Q.K^T landed in TMEM
  P_FULL = S_FULL + 4,              // [2][2]: P stored (128 softmax threads) and O rescaled (128 correction threads)
  SCALE_FULL = P_FULL + 4,          // [2][2]: rescale factors of an iteration published by the softmax threads
  FIN_FULL = SCALE_FULL + 4,        // [2] tile: final (m, l) of a segment published
  PV_DONE = FIN_FULL + 2,           // [2] tile: a P.V finished (O may be rescaled)
  O_FULL = PV_DONE + 2,             // [2] tile: last P.V of the segment done
  O_FREE = O_FULL + 2,              // [2] tile: epilogue has read O
  META_FULL = O_FREE + 2,           // [kMetaRing]
  NUM_BARS = META_FULL + kMetaRing
};
static_assert(NUM_BARS * 8 <= 512, "barrier region");

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
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t* r) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
      "{%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" ::"r"(taddr),
      "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]), "r"(r[10]),
      "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
      : "memory");
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

__device__ __forceinline__ void sts_v4(uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
  asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}
__device__ __forceinline__ uint4 lds_v4(uint32_t addr) {
  uint4 v;
  asm volatile("ld.shared.v4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ void cp_async_16(uint32_t dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ float ex2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// 2^x on the FMA pipe (no MUFU): x = n + r, n = rint(x) taken from the mantissa of x + 1.5*2^23, r in
// [-0.5, 0.5]; degree-2 minimax polynomial of 2^r (relative error 1.7e-3, below the 2^-9 = 2.0e-3 bf16
// rounding of P that follows; the same p feeds the row sum, so weights stay normalised); n is added to the
// exponent field.  x is clamped at -126 (result ~1e-38 instead of exponent wrap-around); callers
// guarantee x <= 2^7.
__device__ __forceinline__ float exp2_poly(float x) {
  x = fmaxf(x, -126.f);
  const float t = x + 12582912.f;
  const float r = x - (t - 12582912.f);
  float q = fmaf(0.23842722f, r, 0.70344825f);
  q = fmaf(q, r, 1.00044327f);
  return __int_as_float(__float_as_int(q) + (__float_as_int(t) << 23));
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
// the same fields without the address (compile-time part), and a descriptor from its two words
__host__ __device__ constexpr uint64_t smem_desc_const(uint32_t lbo_bytes, uint32_t sbo_bytes) {
  return ((uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16) | ((uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32) | ((uint64_t)1 << 46) |
         ((uint64_t)2 << 61);
}
__device__ __forceinline__ uint64_t desc64(uint32_t lo, uint32_t hi) {
  uint64_t d;
  asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "r"(lo), "r"(hi));
  return d;
}
// instruction descriptor: D fp32, A/B bf16, M x N, A K-major, B K-major or MN-major
__host__ __device__ constexpr uint32_t instr_desc(int M, int N, int b_mn_major) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)b_mn_major << 16) | ((uint32_t)(N >> 3) << 17) |
         ((uint32_t)(M >> 4) << 24);
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

// ---- per-stream plan (computed by every CTA in its prologue; a warp per stream) -----------------
__device__ __forceinline__ int stream_self_page(const AttnParams& p, int b) {
  const int sp = p.self_pages_d ? p.self_pages_d[b] : p.self_page;
  return (sp < 0 || sp >= p.n_pages) ? -1 : sp;
}
__device__ __forceinline__ int page_valid_len(const AttnParams& p, int page) {
  if (page < 0 || page >= p.n_pages) return 0;
  return max(0, min(p.page_len[page], p.page_cap));
}

__device__ void plan_stream(const AttnParams& p, int b, int lane, StreamPlan* out) {
  const int g = p.Hq / p.Hkv;
  int nq = p.nq_d ? p.nq_d[b] : p.nq_cap;
  bool clamped = false;
  if (nq > p.nq_cap) { nq = p.nq_cap; clamped = true; }
  nq = max(nq, 0);
  int n_vis = p.n_vis_d ? p.n_vis_d[b] : p.n_vis_cap;
  n_vis = max(0, min(n_vis, p.n_vis_cap));
  const int sp = stream_self_page(p, b);
  const int self_len = sp >= 0 ? page_valid_len(p, sp) : 0;
  const int32_t* table = p.page_table + (size_t)b * p.n_vis_cap;
  int hist = 0;
  bool bad = false;
  for (int e = lane; e < n_vis; e += 32) {
    const int page = table[e];
    if (page != -1 && (page < 0 || page >= p.n_pages)) bad = true;    // -1 is padding, anything else out of range is flagged
    hist += plan_kv_tiles(page_valid_len(p, page));
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) hist += __shfl_xor_sync(0xffffffffu, hist, o);
  bad = __any_sync(0xffffffffu, bad);
  StreamPlan s;
  s.nq = nq; s.n_vis = n_vis; s.self_page = sp; s.self_len = self_len; s.hist_tiles = hist;
  s.R = g * nq;
  const int NT = plan_q_tiles(s.R);
  s.NP = (NT + 1) >> 1;
  long long J = 0;
  if (hist > 0 || self_len > 0) {
    for (int pp = lane; pp < s.NP; pp += 32) J += plan_item_len(s, g, p.self_offset, pp);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) J += __shfl_xor_sync(0xffffffffu, J, o);
  s.J = J;
  if (lane == 0) {
    *out = s;
    if (p.status && blockIdx.x == 0 && (clamped || bad))
      atomicOr(p.status, (clamped ? VCS_FLAG_COUNT_CLAMPED : 0) | (bad ? VCS_FLAG_BAD_PAGE : 0));
  }
}

// Walk of this CTA's segments; every role runs an identical copy.
struct SegIter {
  const StreamPlan* plans;
  int B, Hkv, g, self_off;
  int b, kvh, p, t0;
  long long remaining, pos;   // pos: absolute iteration index of (item, t0)
  int len, t1;                // current segment: iterations [t0, t1) of an item of `len` iterations
  __device__ SegIter(const StreamPlan* plans_, const CtaRange& r, const AttnParams& prm)
      : plans(plans_), B(prm.B), Hkv(prm.Hkv), g(prm.Hq / prm.Hkv), self_off(prm.self_offset), b(r.b), kvh(r.kvh), p(r.p),
        t0(r.t), remaining(r.hi - r.lo), pos(r.lo), len(0), t1(0) {}
  __device__ __forceinline__ bool valid() {
    if (remaining <= 0) return false;
    len = plan_item_len(plans[b], g, self_off, p);
    const long long e = (long long)t0 + remaining;
    t1 = e < (long long)len ? (int)e : len;
    return true;
  }
  __device__ __forceinline__ bool has_b() const { return 256 * p + 128 < plans[b].R; }
  __device__ __forceinline__ bool split() const { return t0 > 0 || t1 < len; }
  __device__ __forceinline__ void advance() {
    remaining -= t1 - t0;
    pos += t1 - t0;
    if (t1 < len) { t0 = t1; return; }     // only when remaining == 0
    t0 = 0;
    if (++p < plans[b].NP) return;
    p = 0;
    if (++kvh < Hkv) return;
    kvh = 0;
    do { ++b; } while (b < B && plans[b].J == 0);
  }
};

// KV-tile walk of one item, run by the whole TMA warp: lane l caches table entry win0 + l.
struct KvWalker {
  const AttnParams& prm;
  const int32_t* table;
  int n_vis, n_ent, self_page, self_lim, lane;
  int win0, my_page, my_len;
  int cur, tok0;
  __device__ KvWalker(const AttnParams& p_, int lane_) : prm(p_), lane(lane_) {}
  __device__ __forceinline__ void load_window(int w0) {
    win0 = w0;
    const int e = w0 + lane;
    my_page = -1;
    my_len = 0;
    if (e < n_ent) {
      if (e == n_vis) { my_page = self_page; my_len = self_lim; }
      else { my_page = table[e]; my_len = page_valid_len(prm, my_page); }
    }
  }
  // position the walk at iteration t of item (stream plan s, pair p)
  __device__ void seek(const StreamPlan& s, int b, int g, int p, int t) {
    table = prm.page_table + (size_t)b * prm.n_vis_cap;
    n_vis = s.n_vis;
    self_page = s.self_page;
    self_lim = s.self_len > 0 ? plan_self_limit(s.self_len, prm.self_offset, plan_item_last_token(s.R, g, p)) : 0;
    n_ent = n_vis + (self_lim > 0 ? 1 : 0);
    int acc = 0;
    for (int w0 = 0;; w0 += 32) {
      load_window(w0);
      const int tiles = plan_kv_tiles(my_len);
      int incl = tiles;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
      }
      const int tot = __shfl_sync(0xffffffffu, incl, 31);
      if (t < acc + tot || w0 + 32 >= n_ent) {
        const unsigned hit = __ballot_sync(0xffffffffu, acc + incl > t);
        const int L = hit ? __ffs(hit) - 1 : 0;
        const int excl = __shfl_sync(0xffffffffu, incl - tiles, L);
        cur = w0 + L;
        tok0 = (t - acc - excl) * kBlockN;
        return;
      }
      acc += tot;
    }
  }
  __device__ __forceinline__ void get(int& page, int& tok, int& valid, bool& is_self) const {
    const int L = cur - win0;
    page = __shfl_sync(0xffffffffu, my_page, L);
    const int len = __shfl_sync(0xffffffffu, my_len, L);
    tok = tok0;
    valid = min(kBlockN, len - tok0);
    is_self = self_lim > 0 && cur == n_vis;
  }
  __device__ __forceinline__ void advance() {
    int len = __shfl_sync(0xffffffffu, my_len, cur - win0);
    tok0 += kBlockN;
    if (tok0 < len) return;
    tok0 = 0;
    do {
      ++cur;
      if (cur >= n_ent) return;
      if (cur - win0 >= 32) load_window(cur);
      len = __shfl_sync(0xffffffffu, my_len, cur - win0);
    } while (len == 0);
  }
};

__global__ void __launch_bounds__(kThreads, 1)
attn_tc_kernel(const AttnParams p, const __grid_constant__ CUtensorMap tmap_k, const __grid_constant__ CUtensorMap tmap_v) {
  pdl_wait();
  pdl_launch_dependents();
  extern __shared__ uint8_t smem_raw[];

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));
  const uint32_t sQ = smem_base + Smem::q, sKV = smem_base + Smem::kv;
  const uint32_t bars = smem_base + Smem::bar;
  auto bar = [&](int i) { return bars + 8u * i; };
  StreamPlan* plans = reinterpret_cast<StreamPlan*>(smem_gen + Smem::plan);
  CtaRange* range = reinterpret_cast<CtaRange*>(smem_gen + Smem::range);
  const int g = p.Hq / p.Hkv;

  // ---- prologue: barriers, TMEM, per-stream plan, this CTA's range ---------------------------------
  if (threadIdx.x == 0) {
    mbar_init(bar(Q_FULL), 2 * kBlockM);
    mbar_init(bar(Q_EMPTY), 2);               // both MMA issuers
    for (int s = 0; s < kStages; ++s) {
      mbar_init(bar(KV_FULL + s), 1);
      mbar_init(bar(KV_EMPTY + s), 2);           // both MMA issuers
    }
    for (int t = 0; t < 4; ++t) {
      mbar_init(bar(S_FULL + t), 1);
      mbar_init(bar(P_FULL + t), 2 * kBlockM);
      mbar_init(bar(SCALE_FULL + t), kBlockM);
    }
    for (int t = 0; t < 2; ++t) {
      mbar_init(bar(FIN_FULL + t), kBlockM);
      mbar_init(bar(PV_DONE + t), 1);
      mbar_init(bar(O_FULL + t), 1);
      mbar_init(bar(O_FREE + t), kBlockM);
    }
    for (int s = 0; s < kMetaRing; ++s) mbar_init(bar(META_FULL + s), 1);
    fence_barrier_init();
  }
  if (warp == kWarpMma) tmem_alloc(smem_base + Smem::tmem_slot, kTmemCols);
  if (threadIdx.x < 64) {
    reinterpret_cast<unsigned long long*>(smem_gen + Smem::rope_tf)[threadIdx.x] = p.rope.turn_frac[threadIdx.x];
    reinterpret_cast<int8_t*>(smem_gen + Smem::rope_ax)[threadIdx.x] = p.rope.axis_of[threadIdx.x];
  }
  for (int b = warp; b < p.B; b += kThreads / 32) plan_stream(p, b, lane, plans + b);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *reinterpret_cast<volatile uint32_t*>(smem_gen + Smem::tmem_slot);

  if (warp == 0) {
    // total iterations, this CTA's share, and the (stream, kv head, item, iteration) where it starts
    long long J_total = 0;
    for (int b = 0; b < p.B; ++b) J_total += plans[b].J * p.Hkv;
    const int G = (int)(J_total < (long long)gridDim.x ? J_total : (long long)gridDim.x);
    const bool mine = (int)blockIdx.x < G;
    const long long lo = mine ? plan_cta_begin(J_total, G, blockIdx.x) : 0, hi = mine ? plan_cta_begin(J_total, G, blockIdx.x + 1) : 0;
    int sb = 0, skvh = 0, sp = 0, st = 0;
    if (hi > lo) {
      long long rem = lo;
      while (rem >= plans[sb].J * p.Hkv) { rem -= plans[sb].J * p.Hkv; ++sb; }   // J == 0 streams are skipped
      skvh = (int)(rem / plans[sb].J);
      rem -= (long long)skvh * plans[sb].J;
      // pair: first p whose inclusive prefix of item lengths exceeds rem (32 items per round)
      const StreamPlan s = plans[sb];
      long long acc = 0;
      for (int p0 = 0;; p0 += 32) {
        const int pp = p0 + lane;
        const int l = pp < s.NP ? plan_item_len(s, g, p.self_offset, pp) : 0;
        int incl = l;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
          const int v = __shfl_up_sync(0xffffffffu, incl, o);
          if (lane >= o) incl += v;
        }
        const int tot = __shfl_sync(0xffffffffu, incl, 31);
        if (rem < acc + tot || p0 + 32 >= s.NP) {
          const unsigned hit = __ballot_sync(0xffffffffu, acc + incl > rem);
          const int L = hit ? __ffs(hit) - 1 : 0;
          sp = p0 + L;
          st = (int)(rem - acc - __shfl_sync(0xffffffffu, incl - l, L));
          break;
        }
        acc += tot;
      }
    }
    if (lane == 0) {
      range->J_total = J_total; range->lo = lo; range->hi = hi;
      range->b = sb; range->kvh = skvh; range->p = sp; range->t = st; range->G = G;
    }
  }
  __syncthreads();

  // streams whose visible set is empty for every row (reading D29): zeros and lse = -inf, written by all CTAs
  for (int b = 0; b < p.B; ++b) {
    const StreamPlan s = plans[b];
    if (s.J != 0 || s.nq == 0) continue;
    __nv_bfloat16* ob = static_cast<__nv_bfloat16*>(p.out) + (size_t)b * p.out_bstride;
    const int vec_per_row = p.Hq * kHeadDim / 8;
    for (long long e = (long long)blockIdx.x * kThreads + threadIdx.x; e < (long long)s.nq * vec_per_row; e += (long long)gridDim.x * kThreads) {
      const int i = (int)(e / vec_per_row), v = (int)(e - (long long)i * vec_per_row);
      stg_v4(ob + (size_t)i * p.out_stride + 8 * v, make_uint4(0u, 0u, 0u, 0u));
    }
    if (p.lse)
      for (long long e = (long long)blockIdx.x * kThreads + threadIdx.x; e < (long long)s.nq * p.Hq; e += (long long)gridDim.x * kThreads) {
        const int h = (int)(e / s.nq), i = (int)(e - (long long)h * s.nq);
        p.lse[((size_t)b * p.Hq + h) * p.nq_cap + i] = -INFINITY;
      }
  }

  const CtaRange rg = *range;
  CombineDesc* desc = reinterpret_cast<CombineDesc*>(p.desc);

  if (warp >= 12) {
    reg_dec<kRegsOther>();
    if (warp == kWarpTma) {
      // ===================== TMA producer =====================
      // Ring slot = running tile number % kStages.  Per segment of n iterations the tiles are issued in the
      // order the MMA warp consumes them: K(0) K(1) | V(0) K(2) | V(1) K(3) | ... | V(n-1).
      if (elect_one()) {
        tma_prefetch_desc(&tmap_k);
        tma_prefetch_desc(&tmap_v);
      }
      SegIter sg(plans, rg, p);
      KvWalker wk(p, lane);
      int it = 0;              // iterations (K tiles) issued so far: index of the metadata ring
      uint32_t seq = 0;        // tiles issued so far
      bool wrote_desc = false;
      for (; sg.valid(); sg.advance()) {
        // combine descriptor of an item whose FIRST part ends this CTA's range (slot [c][1])
        if (sg.t0 == 0 && sg.t1 < sg.len && lane == 0) {
          const long long item_end = sg.pos + sg.len;     // pos = absolute index of the item's first iteration
          CombineDesc d;
          d.n_parts = plan_cta_of(rg.J_total, rg.G, item_end - 1) - (int)blockIdx.x + 1;
          d.b = sg.b; d.kvh = sg.kvh; d.p = sg.p;
          desc[blockIdx.x] = d;
          wrote_desc = true;
        }
        wk.seek(plans[sg.b], sg.b, g, sg.p, sg.t0);
        const int n = sg.t1 - sg.t0;
        int fpage[2] = {0, 0}, ftok[2] = {0, 0};     // coordinates of K(j), K(j+1): V(j) reads the same rows
        auto load_k = [&](int j) {
          int page, tok, valid;
          bool is_self;
          wk.get(page, tok, valid, is_self);
          wk.advance();
          fpage[j & 1] = page;
          ftok[j & 1] = tok;
          const int slot = (int)(seq % kStages);
          mbar_wait(bar(KV_EMPTY + slot), ((seq / kStages) & 1u) ^ 1u);
          if (elect_one()) {
            mbar_expect_tx(bar(KV_FULL + slot), kTileBytes);
            tma_load_4d(sKV + slot * kTileBytes, &tmap_k, bar(KV_FULL + slot), 0, tok, sg.kvh, page);
            tma_load_4d(sKV + slot * kTileBytes + kHalfBytes, &tmap_k, bar(KV_FULL + slot), 64, tok, sg.kvh, page);
            // metadata of this iteration for the softmax warps (ring of 8: the producer is never more than
            // six iterations ahead of them)
            int4* meta = reinterpret_cast<int4*>(smem_gen + Smem::meta) + (it & (kMetaRing - 1));
            *meta = make_int4(valid, is_self ? tok : -1, 0, 0);
            mbar_arrive(bar(META_FULL + (it & (kMetaRing - 1))));
          }
          __syncwarp();
          ++seq;
          ++it;
        };
        auto load_v = [&](int j) {
          const int slot = (int)(seq % kStages);
          mbar_wait(bar(KV_EMPTY + slot), ((seq / kStages) & 1u) ^ 1u);
          if (elect_one()) {
            mbar_expect_tx(bar(KV_FULL + slot), kTileBytes);
            tma_load_4d(sKV + slot * kTileBytes, &tmap_v, bar(KV_FULL + slot), 0, ftok[j & 1], sg.kvh, fpage[j & 1]);
            tma_load_4d(sKV + slot * kTileBytes + kHalfBytes, &tmap_v, bar(KV_FULL + slot), 64, ftok[j & 1], sg.kvh, fpage[j & 1]);
          }
          __syncwarp();
          ++seq;
        };
        load_k(0);
        if (n > 1) load_k(1);
        for (int j = 0; j < n; ++j) {
          load_v(j);
          if (j + 2 < n) load_k(j + 2);
        }
      }
      if (!wrote_desc && lane == 0) {
        CombineDesc d;
        d.n_parts = 0; d.b = 0; d.kvh = 0; d.p = 0;
        desc[blockIdx.x] = d;
      }
    } else if (warp == kWarpMma || warp == kWarpMma + 1) {
      // ===================== MMA issuers: warp 13 for q tile A, warp 14 for q tile B =====================
      // One issuer per q tile: a tile's P.V never queues behind the other tile's P_FULL wait, and the issue path
      // of one thread (barrier waits, descriptor words, eight Q.K^T and four P.V instructions, commits) is halved.
      // Both issuers walk the same ring; a slot is released by both (KV_EMPTY counts two).  The issuer of an
      // absent tile B (odd tile count) keeps pace through the KV_FULL waits and releases with a plain arrive.
      const int t = warp - kWarpMma;
      constexpr uint32_t idesc_qk = instr_desc(kBlockM, kBlockN, 0);
      constexpr uint32_t idesc_pv = instr_desc(kBlockM, kHeadDim, 1);
      if (elect_one()) {
        // descriptors as (low, high) words: only the 14-bit address field of the low word changes from one
        // instruction to the next (shared memory is < 256 KB, no carry), the high word is a constant
        constexpr uint32_t kDescHi = (uint32_t)(smem_desc_const(16, 1024) >> 32);
        const uint32_t q_lo = (uint32_t)smem_desc(sQ + t * kQTileBytes, 16, 1024);
        const uint32_t k_lo = (uint32_t)smem_desc(sKV, 16, 1024);
        const uint32_t v_lo = (uint32_t)smem_desc(sKV, kHalfBytes, 1024);
        static_assert((smem_desc_const(16, 1024) >> 32) == (smem_desc_const(kHalfBytes, 1024) >> 32), "descriptor high word");
        const uint32_t tS = tmem + kColS + 128 * t, tO = tmem + kColO + 128 * t;
        // S_t,b[128 x 64] = Q_t[128 x d] . K[64 x d]^T : both K-major, 8 k-steps of 16 over d
        auto qk = [&](int buf, uint32_t slot) {
          const uint32_t dk = k_lo + slot * (uint32_t)(kTileBytes >> 4);
#pragma unroll
          for (int kk = 0; kk < kHeadDim / 16; ++kk) {
            const uint32_t offq = (uint32_t)(((kk >> 2) * kQHalfBytes + (kk & 3) * 32) >> 4);
            const uint32_t offk = (uint32_t)(((kk >> 2) * kHalfBytes + (kk & 3) * 32) >> 4);
            umma_bf16_ss(tS + 64 * buf, desc64(q_lo + offq, kDescHi), desc64(dk + offk, kDescHi), idesc_qk, kk > 0);
          }
        };
        // O_t[128 x d] (+)= P_t,b[128 x 64] . V[64 x d] : P from TMEM (8 columns per k-step), V MN-major
        // (d contiguous; 64-wide d groups 8 KB apart = LBO, 8-token groups 1 KB apart = SBO)
        auto pv = [&](int buf, uint32_t slot, bool acc) {
          const uint32_t dv = v_lo + slot * (uint32_t)(kTileBytes >> 4);
#pragma unroll
          for (int kk = 0; kk < kBlockN / 16; ++kk)
            umma_bf16_ts(tO, tS + 64 * buf + 8 * kk, desc64(dv + (uint32_t)((kk * 2048) >> 4), kDescHi), idesc_pv, acc | (kk > 0));
        };
        auto wait_slot = [&](uint32_t sq) {
          mbar_wait(bar(KV_FULL + (int)(sq % kStages)), (sq / kStages) & 1u);
          tc_fence_after();
        };
        SegIter sg(plans, rg, p);
        uint32_t seg = 0;
        uint32_t seq = 0;                 // tiles consumed so far (ring position)
        uint32_t n_b0 = 0, n_b1 = 0;      // uses of this tile's S / P buffers
        uint32_t n_seg = 0;               // segments in which this tile was active (O_FULL / O_FREE phases)
        for (; sg.valid(); sg.advance(), ++seg) {
          const int n = sg.t1 - sg.t0;
          const bool act = t == 0 || sg.has_b();
          auto release = [&](int which) {
            if (act) umma_commit(bar(which)); else mbar_arrive(bar(which));
          };
          mbar_wait(bar(Q_FULL), seg & 1u);
          tc_fence_after();
          for (int jj = 0; jj < 2 && jj < n; ++jj) {     // Q.K^T of the first two iterations
            wait_slot(seq);
            if (act) {
              qk(jj, seq % kStages);
              umma_commit(bar(S_FULL + 2 * t + jj));
            }
            release(KV_EMPTY + (int)(seq % kStages));
            ++seq;
          }
          if (n <= 2) release(Q_EMPTY);
          // one iteration; the buffer index is a compile-time constant (two iterations per loop trip)
          auto step = [&](int j, auto buf_c) {
            constexpr int b = decltype(buf_c)::value;
            const bool more = j + 2 < n;
            const uint32_t vseq = seq, kseq = seq + 1;
            wait_slot(vseq);
            if (act) {
              if (j == 0 && n_seg > 0) mbar_wait(bar(O_FREE + t), (n_seg - 1) & 1u);
              uint32_t& n_b = b ? n_b1 : n_b0;
              mbar_wait(bar(P_FULL + 2 * t + b), n_b & 1u);
              ++n_b;
              tc_fence_after();
              pv(b, vseq % kStages, j > 0);
              umma_commit(bar(PV_DONE + t));
              if (more) {
                wait_slot(kseq);
                qk(b, kseq % kStages);
                umma_commit(bar(S_FULL + 2 * t + b));
              } else if (j == n - 1) {
                umma_commit(bar(O_FULL + t));
              }
            } else if (more) {
              wait_slot(kseq);
            }
            release(KV_EMPTY + (int)(vseq % kStages));
            ++seq;
            if (more) {
              release(KV_EMPTY + (int)(kseq % kStages));
              ++seq;
              if (j + 3 == n) release(Q_EMPTY);          // last Q.K^T of the segment issued
            }
          };
          for (int j = 0; j < n; j += 2) {
            step(j, std::integral_constant<int, 0>{});
            if (j + 1 < n) step(j + 1, std::integral_constant<int, 1>{});
          }
          if (act) ++n_seg;
        }
      }
      __syncwarp();
    }
  } else if (warp >= 8) {
    reg_dec<kRegsCorr>();
    // ===================== correction warpgroup: O rescale and epilogue =====================
    const int r = threadIdx.x & (kBlockM - 1);   // row in tile == TMEM lane
    const uint32_t lane_addr = tmem + ((uint32_t)((warp & 3) * 32) << 16);
    const float* sc_s = reinterpret_cast<const float*>(smem_gen + Smem::scale);
    const float* fm_s = reinterpret_cast<const float*>(smem_gen + Smem::fin_m);
    const float* fl_s = reinterpret_cast<const float*>(smem_gen + Smem::fin_l);
    SegIter sg(plans, rg, p);
    // The per-iteration handshakes are double-buffered by iteration parity like S itself: the softmax of
    // iteration j + 1 may publish before this warp has consumed iteration j, never iteration j + 2 (its
    // S needs P.V of iteration j, which needs our arrival on P_FULL).
    uint32_t n_sc[2][2] = {{0u, 0u}, {0u, 0u}}, n_seg[2] = {0u, 0u}, n_pv[2] = {0u, 0u};
    for (; sg.valid(); sg.advance()) {
      const int n = sg.t1 - sg.t0;
      const int n_t = sg.has_b() ? 2 : 1;
      for (int j = 0; j < n; ++j) {
        for (int t = 0; t < n_t; ++t) {
          mbar_wait(bar(SCALE_FULL + 2 * t + (j & 1)), n_sc[t][j & 1] & 1u);
          ++n_sc[t][j & 1];
          const float sc = sc_s[(2 * t + (j & 1)) * kBlockM + r];
          if (j > 0 && __any_sync(0xffffffffu, sc != 1.f)) {
            // O_t must be idle: P.V_t of iteration j - 1 (completion number n_pv[t] of PV_DONE) has finished, and
            // P.V_t of iteration j cannot start before P_FULL completes, which needs our arrival
            mbar_wait(bar(PV_DONE + t), (n_pv[t] - 1) & 1u);
            tc_fence_after();
#pragma unroll
            for (int c = 0; c < kHeadDim / 32; ++c) {
              float o[32];
              tmem_ld32(lane_addr + kColO + 128 * t + 32 * c, o);
              tmem_wait_ld();
#pragma unroll
              for (int e = 0; e < 32; ++e) o[e] *= sc;
              tmem_st32(lane_addr + kColO + 128 * t + 32 * c, o);
            }
            tmem_wait_st();
            tc_fence_before();
          }
          mbar_arrive(bar(P_FULL + 2 * t + (j & 1)));
          ++n_pv[t];
        }
      }
      // ---- epilogue of the segment ----
      const StreamPlan s = plans[sg.b];
      const bool split = sg.split();
      for (int t = 0; t < n_t; ++t) {
        mbar_wait(bar(FIN_FULL + t), n_seg[t] & 1u);      // final (m, l) of the rows
        const float m_fin = fm_s[t * kBlockM + r], l_fin = fl_s[t * kBlockM + r];
        mbar_wait(bar(O_FULL + t), n_seg[t] & 1u);
        ++n_seg[t];
        tc_fence_after();
        const int tile_row0 = (2 * sg.p + t) * kBlockM;
        const int rho = tile_row0 + r;
        const bool row_valid = rho < s.R;
        if (split) {
          // fp32 partial of a split item: O as [warp][4-column group][row in warp][4] so that every store
          // instruction writes 512 contiguous bytes, then m[128], l[128]
          float* slot = p.part + ((size_t)blockIdx.x * 2 + (sg.t0 == 0 ? 1 : 0)) * kPartSlotFloats + (size_t)t * kPartTileFloats;
          float* dst = slot + (size_t)(warp & 3) * (32 * 128) + lane * 4;
#pragma unroll
          for (int c = 0; c < kHeadDim / 32; ++c) {
            float o[32];
            tmem_ld32(lane_addr + kColO + 128 * t + 32 * c, o);
            tmem_wait_ld();
#pragma unroll
            for (int e = 0; e < 32; e += 4)
              *reinterpret_cast<float4*>(dst + (size_t)(8 * c + (e >> 2)) * 128) = make_float4(o[e], o[e + 1], o[e + 2], o[e + 3]);
          }
          slot[kBlockM * kHeadDim + r] = m_fin;
          slot[kBlockM * kHeadDim + kBlockM + r] = l_fin;
        } else {
          // bf16 output: rows are staged in shared memory (one 64-column half at a time) and written back with
          // lane = (group lane / 8 of 8 consecutive rows, 16-byte piece lane % 8): whole 128-byte lines per row
          const float inv_l = l_fin > 0.f ? 1.f / l_fin : 0.f;
          const uint32_t stg = smem_base + Smem::stage + (uint32_t)(warp & 3) * 4096u;
          __nv_bfloat16* ob = static_cast<__nv_bfloat16*>(p.out) + (size_t)sg.b * p.out_bstride + (size_t)(sg.kvh * g) * kHeadDim + 8 * (lane & 7);
#pragma unroll
          for (int half = 0; half < 2; ++half) {
#pragma unroll
            for (int cc = 0; cc < 2; ++cc) {
              float o[32];
              tmem_ld32(lane_addr + kColO + 128 * t + 64 * half + 32 * cc, o);
              tmem_wait_ld();
#pragma unroll
              for (int e = 0; e < 32; e += 8)
                sts_v4(stg + (uint32_t)lane * 128u + (uint32_t)(((4 * cc + (e >> 3)) ^ (lane & 7)) << 4),
                       pack_bf16(o[e] * inv_l, o[e + 1] * inv_l), pack_bf16(o[e + 2] * inv_l, o[e + 3] * inv_l),
                       pack_bf16(o[e + 4] * inv_l, o[e + 5] * inv_l), pack_bf16(o[e + 6] * inv_l, o[e + 7] * inv_l));
            }
            __syncwarp();
            {
              const int wrow0 = 8 * (lane >> 3);                       // this lane writes back 8 consecutive rows
              const int rk0 = tile_row0 + (warp & 3) * 32 + wrow0;
              int ik = rk0 / g, hk = rk0 - ik * g;
#pragma unroll
              for (int k = 0; k < 8; ++k) {
                const int row = wrow0 + k;
                const uint4 v = lds_v4(stg + (uint32_t)row * 128u + (uint32_t)(((lane & 7) ^ (row & 7)) << 4));
                if (rk0 + k < s.R) stg_v4(ob + (size_t)ik * p.out_stride + (size_t)hk * kHeadDim + 64 * half, v);
                if (++hk == g) { hk = 0; ++ik; }
              }
            }
            __syncwarp();
          }
          if (row_valid && p.lse) {
            const int i = rho / g, h = sg.kvh * g + (rho - i * g);
            p.lse[((size_t)sg.b * p.Hq + h) * p.nq_cap + i] = l_fin > 0.f ? (m_fin + log2f(l_fin)) * 0.6931471805599453f : -INFINITY;
          }
        }
        tc_fence_before();
        mbar_arrive(bar(O_FREE + t));
      }
    }
  } else {
    reg_inc<kRegsSoftmax>();
    // ===================== softmax warpgroups (warps 0-3: q tile A, warps 4-7: q tile B) ==========
    const int t = warp >> 2;
    const int r = threadIdx.x & (kBlockM - 1);   // row in tile == TMEM lane
    const uint32_t lane_addr = tmem + ((uint32_t)((warp & 3) * 32) << 16);
    const uint32_t colS = kColS + 128 * t;
    float* sc_s = reinterpret_cast<float*>(smem_gen + Smem::scale) + 2 * t * kBlockM + r;   // + 128 * buffer
    float* fm_s = reinterpret_cast<float*>(smem_gen + Smem::fin_m) + t * kBlockM + r;
    float* fl_s = reinterpret_cast<float*>(smem_gen + Smem::fin_l) + t * kBlockM + r;
    const float scale_log2 = p.scale * 1.4426950408889634f;
    SegIter sg(plans, rg, p);
    int it = 0, seg = 0;
    uint32_t n_buf[2] = {0u, 0u};   // uses of this tile's S / P buffers
    uint32_t n_act = 0;             // segments in which this tile was active
    for (; sg.valid(); sg.advance(), ++seg) {
      const int n = sg.t1 - sg.t0;
      const bool active = t == 0 || sg.has_b();
      const StreamPlan s = plans[sg.b];
      const int rho = (2 * sg.p + t) * kBlockM + r;
      const bool row_valid = active && rho < s.R;
      const int i = min(rho, s.R - 1) / g, hh = min(rho, s.R - 1) - i * g, h = sg.kvh * g + hh;

      // ---- Q tile: load, M-RoPE, bf16, swizzled K-major layout.  A warp builds its own 32 rows; lane = (group
      // lane / 8 of 8 CONSECUTIVE rows, 16-byte piece lane % 8 of the low and of the high d-half).  The raw
      // rows go straight to their final (swizzled) place with cp.async -- four whole 128-byte lines per
      // instruction, all 16 copies of a lane in flight, no registers -- and are then rotated IN PLACE by
      // the lane that copied them.  The g rows of a token share its rotation: with g >= 4 a lane's 8 rows
      // span at most three tokens, whose 3 x 8 sin / cos pairs are computed once, uniformly.  The loops
      // are rolled on purpose: this code runs once per segment, and as straight-line code it was 28 KB
      // whose instruction-cache misses cost more than its arithmetic (ncu: stall_no_instruction) ----
      if (seg > 0) mbar_wait(bar(Q_EMPTY), (uint32_t)(seg - 1) & 1u);
      if (active) {
        const int c = lane & 7, row0 = (warp & 3) * 32 + 8 * (lane >> 3);
        const int rho0 = (2 * sg.p + t) * kBlockM + row0;
        const int i0 = rho0 / g, hh0 = rho0 - i0 * g;
        const __nv_bfloat16* qb = static_cast<const __nv_bfloat16*>(p.q) + (size_t)sg.b * p.q_bstride + (size_t)(sg.kvh * g) * kHeadDim + 8 * c;
        const int32_t* qpb = p.q_pos3 + (size_t)sg.b * p.nq_cap * 3;
        const uint32_t qdst = sQ + t * kQTileBytes;
        {
          int ii = i0, hh = hh0;
#pragma unroll 1
          for (int k = 0; k < 8; ++k) {
            const int row = row0 + k;
            const uint32_t dst = qdst + (uint32_t)row * 128u + (uint32_t)((c ^ (row & 7)) << 4);
            if (rho0 + k < s.R) {
              const __nv_bfloat16* q = qb + (size_t)ii * p.q_stride + (size_t)hh * kHeadDim;
              cp_async_16(dst, q);
              cp_async_16(dst + kQHalfBytes, q + 64);
            } else {
              sts_v4(dst, 0u, 0u, 0u, 0u);
              sts_v4(dst + kQHalfBytes, 0u, 0u, 0u, 0u);
            }
            if (++hh == g) { hh = 0; ++ii; }
          }
          asm volatile("cp.async.commit_group;" ::: "memory");
        }
        unsigned long long tf[8];
        unsigned axbits = 0u;
#pragma unroll
        for (int e = 0; e < 8; ++e) {
          tf[e] = reinterpret_cast<const unsigned long long*>(smem_gen + Smem::rope_tf)[8 * c + e];
          axbits |= (unsigned)reinterpret_cast<const int8_t*>(smem_gen + Smem::rope_ax)[8 * c + e] << (2 * e);
        }
        // sin / cos of rotary pairs 8c .. 8c+7 for up to three tokens (g >= 4), or of the current token only
        float sn[3][8], cs[3][8];
        auto sincos8 = [&](int tok, float* sn_, float* cs_) {
          const int tk = min(tok, s.nq - 1);
          const int pt = __ldg(qpb + 3 * tk + 0), ph = __ldg(qpb + 3 * tk + 1), pw = __ldg(qpb + 3 * tk + 2);
#pragma unroll
          for (int e = 0; e < 8; ++e) {
            const unsigned ax = (axbits >> (2 * e)) & 3u;
            rope_sincos_fast(ax == 0u ? pt : (ax == 1u ? ph : pw), tf[e], &sn_[e], &cs_[e]);
          }
        };
        const bool shared_sets = g >= 4;
#pragma unroll 1
        for (int u = 0; u < (shared_sets ? 3 : 1); ++u) {
          float a_[8], b_[8];
          sincos8(i0 + u, a_, b_);
#pragma unroll
          for (int e = 0; e < 8; ++e) {
            if (u == 0) { sn[0][e] = a_[e]; cs[0][e] = b_[e]; }
            if (u == 1) { sn[1][e] = a_[e]; cs[1][e] = b_[e]; }
            if (u == 2) { sn[2][e] = a_[e]; cs[2][e] = b_[e]; }
          }
        }
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        {
          int set = 0, ii = i0, hh = hh0;
#pragma unroll 1
          for (int k = 0; k < 8; ++k) {
            const int row = row0 + k;
            const uint32_t dst = qdst + (uint32_t)row * 128u + (uint32_t)((c ^ (row & 7)) << 4);
            if (rho0 + k < s.R) {
              const uint4 lo4 = lds_v4(dst), hi4 = lds_v4(dst + kQHalfBytes);
              const uint32_t lo[4] = {lo4.x, lo4.y, lo4.z, lo4.w}, hi[4] = {hi4.x, hi4.y, hi4.z, hi4.w};
              uint32_t olo[4], ohi[4];
#pragma unroll
              for (int e = 0; e < 4; ++e) {
                float sv[2], cv[2];
#pragma unroll
                for (int u = 0; u < 2; ++u) {
                  sv[u] = set == 0 ? sn[0][2 * e + u] : (set == 1 ? sn[1][2 * e + u] : sn[2][2 * e + u]);
                  cv[u] = set == 0 ? cs[0][2 * e + u] : (set == 1 ? cs[1][2 * e + u] : cs[2][2 * e + u]);
                }
                const float xl0 = bf16_lo(lo[e]), xl1 = bf16_hi(lo[e]), xh0 = bf16_lo(hi[e]), xh1 = bf16_hi(hi[e]);
                olo[e] = pack_bf16(xl0 * cv[0] - xh0 * sv[0], xl1 * cv[1] - xh1 * sv[1]);
                ohi[e] = pack_bf16(xh0 * cv[0] + xl0 * sv[0], xh1 * cv[1] + xl1 * sv[1]);
              }
              sts_v4(dst, olo[0], olo[1], olo[2], olo[3]);
              sts_v4(dst + kQHalfBytes, ohi[0], ohi[1], ohi[2], ohi[3]);
            }
            if (++hh == g) {
              hh = 0;
              ++ii;
              if (shared_sets) ++set;
              else if (k < 7) sincos8(ii, sn[0], cs[0]);
            }
          }
        }
        fence_proxy_async();
      }
      mbar_arrive(bar(Q_FULL));
      if (!active) { it += n; continue; }
      // A short segment (n <= 2: all its Q.K^T are issued up front) needs nothing from the correction warps,
      // so this warpgroup could publish the rescale factors and the final (m, l) of TWO segments before they
      // have consumed the first (parity aliasing on the handshake barriers).  Wait until they have finished
      // the epilogue of this tile's previous segment; the Q build above already ran beside that epilogue.
      if (n_act > 0) mbar_wait(bar(O_FREE + t), (n_act - 1) & 1u);
      ++n_act;

      float m_used = -INFINITY, l_run = 0.f;
      auto read_meta = [&](int k) {      // metadata of iteration k of this CTA (ring written by the TMA warp)
        mbar_wait(bar(META_FULL + (k & (kMetaRing - 1))), (uint32_t)(k / kMetaRing) & 1u);
        return *reinterpret_cast<const int4*>(smem_gen + Smem::meta + 16 * (k & (kMetaRing - 1)));
      };
      int4 meta = read_meta(it);
      for (int j = 0; j < n; ++j, ++it) {
        const int b = j & 1;
        const uint32_t colSb = colS + 64 * b;
        // visible columns of this row in this tile: [0, limit)
        int limit = meta.x;
        if (meta.y >= 0) limit = min(limit, p.self_offset + i - meta.y + 1);
        mbar_wait(bar(S_FULL + 2 * t + b), n_buf[b] & 1u);
        ++n_buf[b];
        tc_fence_after();
        float s_[kBlockN];
#pragma unroll
        for (int c = 0; c < kBlockN / 32; ++c) tmem_ld32(lane_addr + colSb + 32 * c, s_ + 32 * c);
        if (j + 1 < n) meta = read_meta(it + 1);      // the next iteration's metadata, while the loads are in flight
        tmem_wait_ld();

        const bool masked = __any_sync(0xffffffffu, limit < kBlockN);   // warp-uniform: tail / diagonal tiles only
        if (masked) {
#pragma unroll
          for (int c = 0; c < kBlockN; ++c) s_[c] = c < limit ? s_[c] : -INFINITY;
        }
        float mx[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) mx[k] = fmaxf(s_[k], s_[8 + k]);
#pragma unroll
        for (int c = 16; c < kBlockN; c += 16) {
#pragma unroll
          for (int k = 0; k < 8; ++k) mx[k] = fmaxf(fmaxf(mx[k], s_[c + k]), s_[c + 8 + k]);
        }
        const float m_row = fmaxf(fmaxf(fmaxf(mx[0], mx[1]), fmaxf(mx[2], mx[3])), fmaxf(fmaxf(mx[4], mx[5]), fmaxf(mx[6], mx[7])));
        const float m_new = fmaxf(m_used, m_row * scale_log2);

        // lazy rescale, decided per row: the correction warp multiplies O by 2^(m_used - m_new) when the
        // maximum grew by more than 2^8, else by 1 (and skips the TMEM round trip when its 32 rows all say 1)
        float sc = 1.f;
        if ((m_new - m_used) > kRescaleThreshold) {     // true on the first visible tile (m_used = -inf)
          sc = (m_used == -INFINITY) ? 0.f : ex2(m_used - m_new);
          l_run *= sc;
          m_used = m_new;
          if (j == 0) sc = 1.f;
        }
        sc_s[b * kBlockM] = sc;
        tc_fence_before();
        mbar_arrive(bar(SCALE_FULL + 2 * t + b));

        const float neg_m = (m_used == -INFINITY) ? 0.f : -m_used;
        // P = 2^(s * scale_log2 - m_used) as bf16 pairs -> TMEM over the head of the S buffer (32 packed
        // columns); row sums in four accumulators.  Scalar FFMA / FADD on purpose: on sm_100 a packed f32x2
        // instruction (and IMAD, F2FP, FMNMX3) occupies the dispatch port for two cycles, a scalar FFMA for one
        // or less (measured), and the loop is bound by dispatch cycles.  On unmasked tiles
        // kPolyNum of every kPolyDen elements take the FMA-pipe polynomial instead of MUFU.EX2 (8 cycles of the
        // MUFU pipe per warp instruction).  Masked tiles hold -inf: MUFU only.
        float lsum[4] = {0.f, 0.f, 0.f, 0.f};
        if (!masked) {
#pragma unroll
          for (int c = 0; c < kBlockN / 32; ++c) {
            uint32_t pk[16];
#pragma unroll
            for (int e = 0; e < 32; e += 2) {
              float pe[2];
#pragma unroll
              for (int u = 0; u < 2; ++u) {
                const float x = fmaf(s_[32 * c + e + u], scale_log2, neg_m);
                pe[u] = (((e + u) % kPolyDen) < kPolyNum) ? exp2_poly(x) : ex2(x);
                lsum[((e >> 1) + u) & 3] += pe[u];
              }
              pk[e >> 1] = pack_bf16(pe[0], pe[1]);
            }
            tmem_st16(lane_addr + colSb + 16 * c, pk);
          }
        } else {
#pragma unroll
          for (int c = 0; c < kBlockN / 32; ++c) {
            uint32_t pk[16];
            if (__all_sync(0xffffffffu, limit <= 32 * c)) {   // this 32-column chunk is hidden from every row of the warp
#pragma unroll
              for (int e = 0; e < 16; ++e) pk[e] = 0u;
            } else {
#pragma unroll
              for (int e = 0; e < 32; e += 2) {
                const float p0 = ex2(fmaf(s_[32 * c + e], scale_log2, neg_m));
                const float p1 = ex2(fmaf(s_[32 * c + e + 1], scale_log2, neg_m));
                lsum[(e >> 1) & 3] += p0 + p1;
                pk[e >> 1] = pack_bf16(p0, p1);
              }
            }
            tmem_st16(lane_addr + colSb + 16 * c, pk);
          }
        }
        l_run += (lsum[0] + lsum[1]) + (lsum[2] + lsum[3]);
        tmem_wait_st();
        tc_fence_before();
        mbar_arrive(bar(P_FULL + 2 * t + b));
      }
      // final row statistics for the epilogue
      *fm_s = m_used;
      *fl_s = row_valid ? l_run : 0.f;
      mbar_arrive(bar(FIN_FULL + t));
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == kWarpMma) {
    tc_fence_after();
    tmem_dealloc(tmem, kTmemCols);
  }
}

// ---- combine: merge the partials of the items that a CTA boundary cut ------------------------------
// grid (attention CTAs, kCombineSlices): block (c, s) handles rows [16 s, 16 s + 16) of the 256 rows (two q
// tiles) of the item whose first part CTA c holds; a thread owns (row, 8-column group) pairs, 16
// consecutive rows per half warp so that every load reads 256 contiguous bytes of the partial layout.
// Part 0 lives in slot [c][1], part z > 0 in slot [c + z][0] (the first segment of the following CTAs).
__global__ void __launch_bounds__(256) attn_combine_kernel(const AttnParams p) {
  pdl_wait();
  pdl_launch_dependents();
  const CombineDesc d = reinterpret_cast<const CombineDesc*>(p.desc)[blockIdx.x];
  if (d.n_parts < 2) return;
  const int g = p.Hq / p.Hkv;
  int nq = p.nq_d ? p.nq_d[d.b] : p.nq_cap;
  nq = max(0, min(nq, p.nq_cap));
  const int R = g * nq;
  constexpr int kRowsPerBlock = 2 * kBlockM / kCombineSlices;
  const int rl = threadIdx.x & 15, cg = (threadIdx.x >> 4) & 15;
  auto slot_of = [&](int part, int t) {
    const size_t sidx = part == 0 ? (size_t)blockIdx.x * 2 + 1 : (size_t)(blockIdx.x + part) * 2;
    return p.part + sidx * kPartSlotFloats + (size_t)t * kPartTileFloats;
  };
  for (int r0 = 0; r0 < kRowsPerBlock; r0 += 16) {
    const int row = blockIdx.y * kRowsPerBlock + r0 + rl;            // 0..255 over both q tiles
    const int t = row >> 7, r = row & 127;
    const int rho = (2 * d.p + t) * kBlockM + r;
    if (rho >= R) continue;
    // O of a partial: [warp r / 32][4-column group][row r % 32][4]
    const size_t o_off = (size_t)(r >> 5) * (32 * 128) + (size_t)(2 * cg) * 128 + (r & 31) * 4;
    float m_all = -INFINITY, l_sum = 0.f;
    float acc[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) acc[e] = 0.f;
    for (int z0 = 0; z0 < d.n_parts; z0 += 4) {      // four parts per round: all their loads in flight at once
      float mz[4], lz[4];
      float4 v[4][2];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        mz[u] = -INFINITY; lz[u] = 0.f;
        v[u][0] = v[u][1] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (z0 + u < d.n_parts) {
          const float* sl = slot_of(z0 + u, t);
          mz[u] = __ldcg(sl + kBlockM * kHeadDim + r);
          lz[u] = __ldcg(sl + kBlockM * kHeadDim + kBlockM + r);
          v[u][0] = __ldcg(reinterpret_cast<const float4*>(sl + o_off));
          v[u][1] = __ldcg(reinterpret_cast<const float4*>(sl + o_off + 128));
        }
      }
      float m_new = m_all;
#pragma unroll
      for (int u = 0; u < 4; ++u) m_new = fmaxf(m_new, mz[u]);
      const float w_old = m_all == -INFINITY ? 0.f : exp2f(m_all - m_new);
      l_sum *= w_old;
#pragma unroll
      for (int e = 0; e < 8; ++e) acc[e] *= w_old;
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const float wz = mz[u] == -INFINITY ? 0.f : exp2f(mz[u] - m_new);
        l_sum = fmaf(lz[u], wz, l_sum);
        acc[0] = fmaf(v[u][0].x, wz, acc[0]); acc[1] = fmaf(v[u][0].y, wz, acc[1]);
        acc[2] = fmaf(v[u][0].z, wz, acc[2]); acc[3] = fmaf(v[u][0].w, wz, acc[3]);
        acc[4] = fmaf(v[u][1].x, wz, acc[4]); acc[5] = fmaf(v[u][1].y, wz, acc[5]);
        acc[6] = fmaf(v[u][1].z, wz, acc[6]); acc[7] = fmaf(v[u][1].w, wz, acc[7]);
      }
      m_all = m_new;
    }
    const int i = rho / g, hh = rho - i * g, h = d.kvh * g + hh;
    const float inv = l_sum > 0.f ? 1.f / l_sum : 0.f;
    __nv_bfloat16* o_row = static_cast<__nv_bfloat16*>(p.out) + (size_t)d.b * p.out_bstride + (size_t)i * p.out_stride +
                           (size_t)h * kHeadDim + 8 * cg;
    uint4 o;
    o.x = pack_bf16(acc[0] * inv, acc[1] * inv);
    o.y = pack_bf16(acc[2] * inv, acc[3] * inv);
    o.z = pack_bf16(acc[4] * inv, acc[5] * inv);
    o.w = pack_bf16(acc[6] * inv, acc[7] * inv);
    stg_v4(o_row, o);
    if (cg == 0 && p.lse)
      p.lse[((size_t)d.b * p.Hq + h) * p.nq_cap + i] = l_sum > 0.f ? (m_all + log2f(l_sum)) * 0.6931471805599453f : -INFINITY;
  }
}

}  // namespace tc

bool attn_tc_supported(const vcs_kv_pool* pool) {
  if (!pool || !pool->opaque_h) return false;
  const PoolOpaque* o = reinterpret_cast<const PoolOpaque*>(pool->opaque_h);
  return o->magic == kPoolMagic && o->has_tma && pool->dtype == VCS_BF16 && pool->d == tc::kHeadDim;
}

// layout: [combine descriptors: one per CTA][partial slots: 2 per CTA x 2 q tiles x (128x128 + 256) floats]
static size_t attn_tc_desc_bytes(int grid) { return round_up((size_t)grid * sizeof(CombineDesc), 256); }

size_t attn_tc_workspace_bytes(const vcs_kv_pool*) {
  const int grid = device_sm_count();
  return attn_tc_desc_bytes(grid) + (size_t)grid * 2 * kPartSlotFloats * sizeof(float);
}

int launch_attn_tc(const AttnParams& p_in, const vcs_kv_pool* pool, void* workspace, size_t, cudaStream_t st) {
  AttnParams p = p_in;
  char* ws = static_cast<char*>(workspace);
  p.grid = device_sm_count();
  if (p.grid <= 0) VCS_FAIL(VCS_ECUDA, "attention: cannot query the SM count of the current device");
  p.desc = ws;
  p.part = reinterpret_cast<float*>(ws + attn_tc_desc_bytes(p.grid));
  const int smem = tc::Smem::total + tc::kSlack;
  static PerDeviceOnce attr_once;
  int rc = attr_once.run([&]() { return cudaFuncSetAttribute(tc::attn_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem); });
  if (rc != VCS_OK) return rc;
  const PoolOpaque* o = reinterpret_cast<const PoolOpaque*>(pool->opaque_h);
  cudaError_t err = launch_pdl(tc::attn_tc_kernel, dim3(p.grid), dim3(tc::kThreads), smem, st, p, o->tmap_k, o->tmap_v);
  if (err == cudaSuccess) err = launch_pdl(tc::attn_combine_kernel, dim3(p.grid, tc::kCombineSlices), dim3(256), 0, st, p);
  if (err == cudaSuccess) err = cudaGetLastError();
  if (err != cudaSuccess) VCS_FAIL(VCS_ECUDA, "attention (tcgen05) launch: %s", cudaGetErrorString(err));
  return VCS_OK;
}

}  // namespace vcs

// ---- self-test hooks: the two approximations of the bf16 path evaluated on caller-supplied points, so that a test
// can pin their error by itself (the attention tolerance would otherwise be the only thing that bounds them) ------
namespace vcs {
__global__ void selftest_exp2_poly_kernel(const float* x, float* y, int n) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) y[i] = tc::exp2_poly(x[i]);
}
__global__ void selftest_rope_sincos_kernel(const int32_t* pos, int n, unsigned long long turn_frac, float* s, float* c) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) rope_sincos_fast(pos[i], turn_frac, s + i, c + i);
}
}  // namespace vcs

extern "C" int vcs_selftest_exp2_poly(const float* x_d, float* y_d, int n, void* stream) {
  if (n < 0 || (n > 0 && (!x_d || !y_d))) VCS_FAIL(VCS_EINVAL, "selftest_exp2_poly: bad arguments");
  if (n == 0) return VCS_OK;
  vcs::selftest_exp2_poly_kernel<<<(n + 255) / 256, 256, 0, (cudaStream_t)stream>>>(x_d, y_d, n);
  VCS_CUDA_OK(cudaGetLastError());
  return VCS_OK;
}

extern "C" int vcs_selftest_rope_sincos(const int32_t* pos_d, int n, double inv_freq, float* sin_d, float* cos_d, void* stream) {
  if (n < 0 || (n > 0 && (!pos_d || !sin_d || !cos_d)) || !(inv_freq >= 0.0))
    VCS_FAIL(VCS_EINVAL, "selftest_rope_sincos: bad arguments");
  if (n == 0) return VCS_OK;
  vcs::selftest_rope_sincos_kernel<<<(n + 255) / 256, 256, 0, (cudaStream_t)stream>>>(pos_d, n, vcs::turn_fraction_q64(inv_freq),
                                                                                      sin_d, cos_d);
  VCS_CUDA_OK(cudaGetLastError());
  return VCS_OK;
}
