// Shared parameter block of the bounded-attention kernels (SIMT and tcgen05) and the stream-K work
// partition of the tcgen05 kernel (plain integer arithmetic, usable from host and device).
#pragma once
#include "common.cuh"

namespace vcs {

constexpr int kAttnMaxStreams = 64;   // streams per batched launch (per-stream plan lives in shared memory)

struct AttnParams {
  const void* q;
  long long q_stride;      // elements between query rows
  long long q_bstride;     // elements between streams
  const int32_t* q_pos3;   // [B][nq_cap][3]
  const int32_t* nq_d;     // [B] or null (= nq_cap)
  int nq_cap;
  const int32_t* page_table;   // [B][n_vis_cap]
  const int32_t* n_vis_d;      // [B] or null (= n_vis_cap)
  int n_vis_cap;
  int self_page;                 // used when self_pages_d is null
  const int32_t* self_pages_d;   // [B] device self page ids (batched form) or null
  int self_offset;
  float scale;
  void* out;
  long long out_stride, out_bstride;
  float* lse;              // [B][Hq][nq_cap] or null
  int32_t* status;
  const void* k_pages;
  const void* v_pages;
  const int32_t* page_len;
  int n_pages, page_cap, Hkv, Hq, d;
  int B;
  RopeParams rope;
  // tcgen05 kernel only: persistent grid, partial slots of split items, descriptors for the combine kernel
  int grid;
  void* desc;
  float* part;
};

// ---- stream-K work partition (tcgen05 kernel) ------------------------------------------------------
// Rows of one kv head: rho = i * g + hh (token-major: the g q heads of a token are adjacent rows, they
// share the token's position and causal limit).  R = g * nq rows form NT = ceil(R / 128) q tiles, two
// adjacent q tiles form an ITEM (pair p = tiles 2p, 2p+1; the last item of a kv head may hold one tile).
// An item walks its visible KV tiles: the fully visible pages in table order, then the self page up to
// the causal limit of the item's last row.  One (item, KV tile) step is an ITERATION; all iterations of
// all (stream, kv head, item) in that order form one flat range that is cut into `grid` equal parts.
struct StreamPlan {
  int nq, n_vis, self_page, self_len, hist_tiles, R, NP;
  long long J;   // iterations of ONE kv head of this stream (all kv heads are alike)
};

#define VCS_HD __host__ __device__ __forceinline__

constexpr int kAttnKvTile = 64;      // KV tokens per iteration (S is double-buffered in TMEM: 2 q tiles x 2 x 64 columns)
VCS_HD int plan_kv_tiles(int len) { return (len + kAttnKvTile - 1) / kAttnKvTile; }
VCS_HD int plan_q_tiles(int rows) { return (rows + 127) >> 7; }

// last query token index of pair p (rows [256 p, 256 p + 256) clipped to R)
VCS_HD int plan_item_last_token(int R, int g, int p) {
  const int rho_end = R < 256 * (p + 1) ? R : 256 * (p + 1);
  return (rho_end - 1) / g;
}
// visible tokens of the self page for an item whose last token is i_hi
VCS_HD int plan_self_limit(int self_len, int self_off, int i_hi) {
  const int lim = self_off + i_hi + 1;
  return self_len < lim ? self_len : lim;
}
VCS_HD int plan_item_len(const StreamPlan& s, int g, int self_off, int p) {
  const int st = s.self_len > 0 ? plan_kv_tiles(plan_self_limit(s.self_len, self_off, plan_item_last_token(s.R, g, p))) : 0;
  return s.hist_tiles + st;
}
// first iteration of CTA c when J_total iterations are cut into G parts
VCS_HD long long plan_cta_begin(long long J_total, int G, int c) { return J_total * c / G; }
// the CTA that owns iteration x
VCS_HD int plan_cta_of(long long J_total, int G, long long x) { return (int)(((x + 1) * G + J_total - 1) / J_total) - 1; }

// descriptor of a split item, written by the CTA that holds the item's FIRST part (slot [c][1]); the
// other parts are the first segments (slot [c'][0]) of the following n_parts - 1 CTAs
struct CombineDesc {
  int n_parts;   // 0 / 1: nothing to merge
  int b, kvh, p;
};

constexpr int kPartTileFloats = 128 * 128 + 2 * 128;        // O[128][128], m[128], l[128]
constexpr int kPartSlotFloats = 2 * kPartTileFloats;        // two q tiles per item

int launch_attn_simt(const AttnParams& p, int dtype, cudaStream_t st);
// tcgen05 / TMA kernel (bf16, head_dim 128)
bool attn_tc_supported(const vcs_kv_pool* pool);
size_t attn_tc_workspace_bytes(const vcs_kv_pool* pool);
int launch_attn_tc(const AttnParams& p, const vcs_kv_pool* pool, void* workspace, size_t workspace_bytes,
                   cudaStream_t st);

}  // namespace vcs
