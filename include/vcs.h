/*
 * vcs.h -- C ABI of the B200-native ViCoStream per-chunk LLM-ingestion hot path.
 *
 * Paper: "ViCoStream: Streaming VideoLLMs Can Run Beyond 100 FPS with Stage-Wise Coordinated
 * Inference" (arxiv/paper_2606_19849); citations are PAPER.md:<line> of that text.
 * lists the readings (D1..D28) taken where the paper is silent.
 *
 * The four operations:
 *   vcs_temporal_drop         chunk-level temporal token dropping, Eq. 1-2
 *                             + stream compaction into a kept-index list
 *   vcs_kv_append_pages       write the retained tokens' K (M-RoPE rotated) and V into a
 *                             chunk-granular paged KV cache ("historical visual cache")
 *   vcs_bounded_prefill_attn  bounded visual attention / query-side attention
 *                             softmax(Q K^T / sqrt(d)) V over a visible page set (PAPER.md:129, :138,
 *                             mask Eq. 4)
 *   vcs_retrieval_score       query-chunk similarity + top-k, Eq. 3
 *
 * Conventions (every call):
 *   - Pointers are DEVICE pointers unless the name ends in `_h` (host).  Every buffer is
 *     allocated, owned and freed by the caller; the library holds no device memory (the one
 *     exception is the fixed scratch array of vcs_temporal_drop_static, see there), never
 *     allocates, frees or synchronises.  Scratch is passed as `workspace`, sized by the matching
 *     *_workspace_bytes() query.  The workspaces of vcs_temporal_drop, vcs_kv_append_pages*,
 *     vcs_retrieval_score and vcs_spatial_entropy_topk hold ticket counters: they must be ZEROED
 *     ONCE before first use and every call leaves them zeroed for the next one.  A workspace must
 *     not be shared by calls that may run concurrently.
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  A call only
 *     ENQUEUES work on it.  Counts that depend on dropping stay on the device (`*_d`, int32),
 *     with a host CAPACITY beside them that sizes grids and buffers.
 *   - Return value: VCS_OK or a negative error.  Argument errors visible from the host are
 *     reported synchronously BEFORE anything is enqueued; vcs_last_error() gives a thread-local
 *     message.  Device-side overflows (e.g. *n_d > n_cap) clamp and OR a VCS_FLAG_* bit into the
 *     optional `status_d` word.
 *   - 16-byte alignment is required of every data pointer and row stride (128-bit loads).
 *   - Kernels are launched with the programmatic-stream-serialization attribute and begin with
 *     griddepcontrol.wait (programmatic dependent launch): on one stream their order and visibility
 *     are those of plain launches, only the launch latency between consecutive vcs kernels is hidden.
 *     A foreign kernel that follows on the same stream WITHOUT that attribute waits for completion
 *     as usual; one launched WITH it must itself wait (cudaGridDependencySynchronize) before reading
 *     vcs outputs.
 *   - No CPU fallback exists: without a CUDA device the calls return VCS_ECUDA.
 */
#ifndef VCS_H_
#define VCS_H_

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define VCS_API __attribute__((visibility("default")))
#else
#define VCS_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

#define VCS_VERSION 101   /* 101: vcs_chunk_call / vcs_multi_call layout of round 2 (host_rows, prev_last_group_d) + size queries */

/* return codes */
#define VCS_OK            0
#define VCS_EINVAL       (-1)  /* null pointer, negative / inconsistent sizes            */
#define VCS_EALIGN       (-2)  /* pointer or stride not 16-byte aligned, D % 8 != 0 ...    */
#define VCS_ECAP         (-3)  /* capacity exceeded, page id out of range, workspace small */
#define VCS_EUNSUPPORTED (-4)  /* dtype / head_dim / implementation not available          */
#define VCS_ECUDA        (-5)  /* CUDA runtime / driver error                              */

/* element types */
#define VCS_F32  0             /* SIMT path (Tiny config)                                  */
#define VCS_BF16 1

/* device status bits (OR-ed into *status_d) */
#define VCS_FLAG_COUNT_CLAMPED 1   /* a device count exceeded its host capacity            */
#define VCS_FLAG_PAGE_OVERFLOW 2   /* page_offset + n > page_cap; the tail was not written */
#define VCS_FLAG_BAD_PAGE      4   /* a device-side page id was out of range; skipped      */

/* temporal-drop modes */
#define VCS_DROP_CHUNK_ALLPAIRS 0  /* Eq. 2: all pairs i<j, first group kept as anchor     */
#define VCS_DROP_CONSECUTIVE    1  /* PAPER.md:125 frame-level variant: vs previous group  */

/* attention implementation selector (flags argument of vcs_bounded_prefill_attn) */
#define VCS_ATTN_AUTO 0            /* tcgen05 kernel when dtype==BF16 && d==128, else SIMT */
#define VCS_ATTN_SIMT 1            /* force the fp32-accumulate SIMT kernel                */
#define VCS_ATTN_TC   2            /* force the tcgen05/TMA kernel (error if unsupported)  */

/*
 * Chunk-granular paged KV cache (GQA).  Host struct describing caller-owned device memory.
 *   k_pages, v_pages : [n_pages][Hkv][page_cap][d] elements of `dtype`; K is stored ALREADY
 *                      rotated by M-RoPE, V as given.
 *   page_len         : [n_pages] int32, valid tokens per page.
 *   k_sum            : [n_pages][Hkv][d] float, sum of the PRE-RoPE keys of the page (the
 *                      retrieval summary of Eq. 3 is k_sum / page_len; reading D19).
 *   rope_theta, rope_sections : M-RoPE base and rotary pairs per (t,h,w) axis, sum == d/2;
 *                      pair m rotates elements (m, m + d/2) by pos[axis(m)] * theta^(-2m/d).
 *   opaque_h         : HOST memory of vcs_pool_opaque_bytes() bytes filled by vcs_pool_init
 *                      (TMA tensor maps, inverse frequencies).  Caller-owned.
 */
typedef struct vcs_kv_pool {
  void    *k_pages;
  void    *v_pages;
  int32_t *page_len;
  float   *k_sum;
  int32_t  n_pages, page_cap, Hkv, Hq, d, dtype;
  float    rope_theta;
  int32_t  rope_sections[3];
  void    *opaque_h;
} vcs_kv_pool;

VCS_API int         vcs_version(void);
/* sizeof(vcs_chunk_call) / sizeof(vcs_multi_call) as the library was built: a caller (or a binding that mirrors
 * the structs) compares them with its own before the first call; a mismatch means another header version. */
VCS_API size_t      vcs_sizeof_chunk_call(void);
VCS_API size_t      vcs_sizeof_multi_call(void);
VCS_API const char *vcs_last_error(void);

/* Number of SMs / name of the current CUDA device (VCS_ECUDA if none).  name_h may be NULL. */
VCS_API int vcs_device_info(int *sm_count_h, int *cc_major_h, int *cc_minor_h, char *name_h, size_t name_bytes);

/*
 * vcs_visible_set -- step a6, vision side: the fully visible pages of chunk t of a stream (PAPER.md:129,
 * :140: V_vis(t) = { j : t - acn <= j <= t }; readings D11, D12, D14): the sink page (if >= 0)
 * followed by the pages of chunks max(0, t - W) .. t - 1 in stream order (W < 0: the whole history).  The
 * chunk's own page is the causal self page of the attention call and is not listed.  HOST arrays:
 * chunk_pages_h [n_chunks] (page of every chunk so far), table_out_h [table_cap] (the rest is padded with
 * -1).  Returns the number of entries (n_vis), or EINVAL / ECAP.  The query-side set (sink + recent +
 * retrieved, reading D21) is the same list with the top-k ids that vcs_retrieval_score writes on the device
 * appended to it.
 */
VCS_API int vcs_visible_set(int32_t t, int32_t W, int32_t sink_page, const int32_t *chunk_pages_h, int32_t n_chunks,
                            int32_t *table_out_h, int32_t table_cap);

/* Query side of step a6 (readings D14, D21): lays out the page table of a query prefill as
 * [sink_page (if >= 0)][recent_pages_h[0 .. n_recent)][k slots = -1][-1 padding up to table_cap] and returns the index
 * of the first of the k slots: pass table_d + that index as `topk_pages` of vcs_retrieval_score, which fills the
 * retrieved page ids in on the device; n_vis of the attention call is the return value + k (slots left at -1 are
 * skipped).  Host buffers.  Errors: EINVAL, ECAP (table_cap too small). */
VCS_API int vcs_visible_set_query(int32_t sink_page, const int32_t *recent_pages_h, int32_t n_recent, int32_t k,
                                  int32_t *table_out_h, int32_t table_cap);

/* Positions (reading D18).  vcs_next_position_base: *next_base_h = base + max(G*t_stride, Hg, Wg), the
 * pos_base of the chunk that follows one with `base` (the first chunk's base is the sink length).
 * vcs_text_positions: pos3_out_h[i] = (start+i, start+i, start+i) for i < n, the positions of sink and text
 * tokens (host buffer [n][3]; copy it to the device for vcs_kv_append_pages / vcs_bounded_prefill_attn).
 * Errors: EINVAL, ECAP (int32 overflow). */
VCS_API int vcs_next_position_base(int32_t G, int32_t Hg, int32_t Wg, int32_t t_stride, int32_t base, int32_t *next_base_h);
VCS_API int vcs_text_positions(int32_t start, int32_t n, int32_t *pos3_out_h);

VCS_API size_t vcs_pool_opaque_bytes(void);
/* Validates the pool description and fills opaque_h.  No device work, no allocation. */
VCS_API int    vcs_pool_init(vcs_kv_pool *pool_h);

/* ------------------------------------------------------------------------------------------
 * vcs_temporal_drop -- PAPER.md:111-121 (Eq. 1, Eq. 2), compaction PAPER.md:69.
 *
 * For each of B independent streams, one chunk of G temporal groups x P same-grid positions:
 *   S_ij(p) = <z_i(p), z_j(p)> / (|z_i(p)| |z_j(p)|)   (0 if a norm is 0), fp32 accumulation;
 *   mode 0: drop(p) <=> AND_{i<j} S_ij(p) > tau (strict); group 0 is the anchor and is always
 *           kept; a dropped position loses all tokens of groups >= 1.
 *   mode 1: token (g,p) is dropped iff S(z_{g-1}(p), z_g(p)) > tau, where z_{-1} is
 *           prev_last_group (the previous chunk's last group) or, if NULL, group 0 is kept.
 * Outputs per stream b (T = G*P):
 *   kept_idx  [B][T] int32 : ascending original indices g*P+p of kept tokens, then -1 padding
 *   kept_count[B]    int32
 *   keep_mask [B][T] uint8 : optional (NULL to skip), 1 = kept
 *   pos3      [B][T][3] int32 : optional; M-RoPE (t,h,w) of kept token j:
 *              (base + g*t_stride, base + r, base + c), p = r*Wg + c, base = pos_base_d[b];
 *              requires Hg*Wg == P.  Rows >= count are left untouched.
 * z: [B][G][P][D] contiguous, dtype VCS_F32 or VCS_BF16; prev_last_group: [B][P][D] or NULL.
 * Workspace: 16-byte aligned, zeroed once; it may then serve calls with any G, P, D as long as B stays the
 * same (the ticket counters of the B streams come first, the keep flags after them).
 * Errors: EINVAL (null/size), EALIGN (z or workspace not 16-B aligned, D*elem % 16 != 0), ECAP (workspace).
 */
VCS_API size_t vcs_temporal_drop_workspace_bytes(int B, int G, int P);
VCS_API int vcs_temporal_drop(const void *z, const void *prev_last_group,
                      int B, int G, int P, int D, int dtype, float tau, int mode,
                      int32_t *kept_idx, int32_t *kept_count, uint8_t *keep_mask,
                      int32_t *pos3, int Hg, int Wg, int t_stride, const int32_t *pos_base_d,
                      void *workspace, size_t workspace_bytes, void *stream);

/* ------------------------------------------------------------------------------------------
 * vcs_temporal_drop_static -- vcs_temporal_drop for callers that have no way to
 * provide the workspace: same inputs, same outputs, same kernel, no `workspace` argument.
 *
 * Who needs it: a serving process whose own pool already owns all of the HBM (a further cudaMalloc
 * fails), a per-frame loop that cannot afford the device-wide synchronisation cudaMalloc implies, a
 * plug-in that receives tensors but no allocator.  The ticket counters and keep flags then live in a
 * fixed array of VCS_DROP_STATIC_SCRATCH_BYTES (1 MiB) that is part of the library image: every GPU
 * that loads libvcs.so holds it until the process exits.  The call itself makes no cudaMalloc /
 * cudaFree and uses no allocating library routine; it enqueues one memset of the counters and the launch.
 *
 * Limit: vcs_temporal_drop_workspace_bytes(B, G, P) <= VCS_DROP_STATIC_SCRATCH_BYTES, i.e. about
 * B * (8192 + G*P) bytes (one 7B-shaped chunk of 4784 tokens: up to B = 80 streams).  Larger shapes
 * return VCS_ECAP with a message naming the sizes, before anything is enqueued; use vcs_temporal_drop.
 * First call on each device: looks up the array's device address (cudaGetSymbolAddress, with that
 * device current) and remembers it.  Make that first call outside any stream capture.
 * Sharing: there is ONE array per device.  Every call overwrites it, so two calls that can overlap on the
 * GPU (different streams without an ordering between them, or two host threads) race and give wrong lists;
 * calls on one stream, or ordered by events, are fine, in any mix of shapes.  An argument error found after
 * the size test may leave the clear of the library's own counters enqueued, nothing else.
 * Other errors: those of vcs_temporal_drop; VCS_ECUDA if the address lookup or the memset fails.
 */
#define VCS_DROP_STATIC_SCRATCH_BYTES (1u << 20)
VCS_API int vcs_temporal_drop_static(const void *z, const void *prev_last_group,
                      int B, int G, int P, int D, int dtype, float tau, int mode,
                      int32_t *kept_idx, int32_t *kept_count, uint8_t *keep_mask,
                      int32_t *pos3, int Hg, int Wg, int t_stride, const int32_t *pos_base_d,
                      void *stream);

/* ------------------------------------------------------------------------------------------
 * vcs_spatial_entropy_topk -- entropy-based spatial token selection (Table 8
 * middle).  For every token I(x) = -sum_m p_m log p_m, p = softmax(x) over the D
 * feature dimensions (reading D30; fp32, natural log); in every frame (temporal group)
 * of every stream the min(K, P) tokens with the highest entropy are retained, ties -> lower index.
 * z: [B][G][P][D] contiguous (VCS_F32 / VCS_BF16).  Outputs per stream b, Kp = min(K, P):
 *   kept_idx  [B][G*Kp] int32 : ascending original indices g*P+p (frame by frame)
 *   kept_count[B]       int32 : G*Kp
 *   entropy   [B][G][P] float : optional (NULL: the workspace holds it)
 *   pos3      [B][G*Kp][3]    : optional M-RoPE positions as in vcs_temporal_drop (needs Hg*Wg == P)
 * Errors: EINVAL, EALIGN, ECAP (workspace; P*4 bytes must fit one block's shared memory).
 */
VCS_API size_t vcs_spatial_entropy_topk_workspace_bytes(int B, int G, int P);
VCS_API int vcs_spatial_entropy_topk(const void *z, int B, int G, int P, int D, int dtype, int K,
                             int32_t *kept_idx, int32_t *kept_count, float *entropy,
                             int32_t *pos3, int Hg, int Wg, int t_stride, const int32_t *pos_base_d,
                             void *workspace, size_t workspace_bytes, void *stream);

/* ------------------------------------------------------------------------------------------
 * vcs_kv_append_pages -- KV cache write for the retained tokens (step a5).
 *
 * For i < n = min(*n_d, n_cap) and every kv head h:
 *   k_pages[page_id][h][page_offset+i][:] = round_dtype( MRoPE(k[i][h][:], pos3[i]) )
 *   v_pages[page_id][h][page_offset+i][:] = v[i][h][:]
 *   k_sum  [page_id][h][:] = (page_offset ? old : 0) + sum_i k[i][h][:]   (pre-RoPE, fp32,
 *                                                      fixed summation order: deterministic)
 *            The order is fixed for a given launch shape (n_cap, B, pool geometry): the same call repeated
 *            gives the same bits.  Launches whose key rows total at most 16 MiB (n_cap*B*Hkv*d*elem) add
 *            column-wise in token order, larger ones add per-block partial sums, so the SAME tokens appended
 *            with another n_cap or B may differ in the last bits of k_sum (and a retrieval tie may fall the
 *            other way).  Keep n_cap and B fixed for a stream if bit-identical summaries matter.
 *   page_len[page_id] = page_offset + n
 * k, v: [n_cap][Hkv][d] with `*_row_stride` ELEMENTS between consecutive tokens (heads are
 * contiguous, stride d).  pos3: [n_cap][3] int32.  n_d: device int32 (NULL = n_cap).
 * Tokens that would land beyond page_cap are not written (VCS_FLAG_PAGE_OVERFLOW).  The V rows from
 * page_offset + n up to the next multiple of 128 are zero-filled (the tcgen05 attention kernel reads whole
 * tiles of V).
 * Errors: EINVAL, EALIGN, ECAP (page_id out of range, page_offset > page_cap, workspace).
 */
VCS_API size_t vcs_kv_append_workspace_bytes(const vcs_kv_pool *pool_h, int n_cap);
VCS_API int vcs_kv_append_pages(const vcs_kv_pool *pool_h, const void *k, const void *v,
                        int64_t k_row_stride, int64_t v_row_stride,
                        const int32_t *pos3, const int32_t *n_d, int n_cap,
                        int32_t page_id, int32_t page_offset, int32_t *status_d,
                        void *workspace, size_t workspace_bytes, void *stream);

/*
 * Batched form (B independent streams, one launch; PAPER.md:73 -- several chunks in flight): stream
 * b appends rows [0, min(n_d[b], n_cap)) of k + b*k_batch_stride / v + b*v_batch_stride (ELEMENTS)
 * with pos3 + b*n_cap*3 into page page_ids_d[b] (DEVICE int32 [B]) at offset 0.  An out-of-range
 * page id writes nothing for that stream and sets VCS_FLAG_BAD_PAGE.  Same layouts, rounding and
 * deterministic k_sum as vcs_kv_append_pages; page ids must be distinct.
 */
VCS_API size_t vcs_kv_append_batched_workspace_bytes(const vcs_kv_pool *pool_h, int n_cap, int B);
VCS_API int vcs_kv_append_pages_batched(const vcs_kv_pool *pool_h, const void *k, const void *v,
                                int64_t k_batch_stride, int64_t v_batch_stride,
                                int64_t k_row_stride, int64_t v_row_stride,
                                const int32_t *pos3, const int32_t *n_d, int n_cap,
                                const int32_t *page_ids_d, int B, int32_t *status_d,
                                void *workspace, size_t workspace_bytes, void *stream);

/* ------------------------------------------------------------------------------------------
 * vcs_bounded_prefill_attn -- PAPER.md:129 (vision-side), :138 (query-side), Eq. 4 :140-145.
 *
 * For query row i < nq = min(*nq_d, nq_cap), q head h (kv head h / (Hq/Hkv)):
 *   out[i][h][:] = softmax_j( <MRoPE(q[i][h], q_pos3[i]), K_j> * scale ) V_j
 * over the visible set: every token t < page_len[p] of every page p = page_table_d[0..n_vis)
 * (n_vis = min(*n_vis_d, n_vis_cap); the table must hold no duplicates; an entry of -1 is padding
 * and is skipped, any other id outside [0, n_pages) is skipped and sets VCS_FLAG_BAD_PAGE), plus, if
 * self_page >= 0, tokens t <= self_offset + i (and t < page_len[self_page]) of the self page
 * (causal inside the current chunk).  The current chunk must have been appended first.
 * q: [nq_cap][Hq][d] PRE-RoPE, `q_row_stride` elements between rows; out likewise, pool dtype.
 * lse: optional [Hq][nq_cap] float, natural-log sum-exp of the scaled logits.
 * scale = 0 selects 1/sqrt(d).  Arithmetic: bf16 x bf16 -> fp32 (tcgen05 kind::f16), fp32
 * softmax, P rounded to bf16 before P*V, fp32 accumulation, output rounded to pool dtype.
 * A row with an empty visible set yields zeros and lse = -inf.
 * flags: VCS_ATTN_AUTO / VCS_ATTN_SIMT / VCS_ATTN_TC.
 * The tcgen05 kernel reads whole 128-token tiles: pool rows in [page_len, next multiple of 128) of a
 * visible page must hold FINITE values in v_pages (vcs_kv_append_pages zero-fills them; a pool that is
 * only ever written through vcs_kv_append_pages* satisfies this whatever its initial contents).
 * Workspace (tcgen05 kernel): partial results of work items cut by a CTA boundary and their
 * descriptors; its size depends on the device only, it needs no initialisation and carries no state
 * from one call to the next.
 * Errors: EINVAL, EALIGN, ECAP (self_page out of range, workspace), EUNSUPPORTED.
 */
VCS_API size_t vcs_bounded_prefill_attn_workspace_bytes(const vcs_kv_pool *pool_h, int nq_cap, int n_vis_cap);
VCS_API int vcs_bounded_prefill_attn(const vcs_kv_pool *pool_h, const void *q, int64_t q_row_stride,
                             const int32_t *q_pos3, const int32_t *nq_d, int nq_cap,
                             const int32_t *page_table_d, const int32_t *n_vis_d, int n_vis_cap,
                             int32_t self_page, int32_t self_offset, float softmax_scale,
                             void *out, int64_t out_row_stride, float *lse, int flags,
                             int32_t *status_d, void *workspace, size_t workspace_bytes,
                             void *stream);

/*
 * Batched form (B <= 64 independent streams in ONE launch; PAPER.md:73 -- several chunks in flight):
 * stream b reads q + b*q_batch_stride (ELEMENTS), q_pos3 + b*nq_cap*3, nq_d[b], the page table
 * page_tables_d + b*n_vis_cap with n_vis_d[b] entries and the causal self page self_pages_d[b]
 * (DEVICE int32 [B]; NULL or an id < 0: none), and writes out + b*out_batch_stride and
 * lse + b*Hq*nq_cap.  The streams' work items share one persistent grid, so a launch over many
 * small chunks fills the GPU like one large chunk.  Workspace as for the single-stream call.
 */
VCS_API int vcs_bounded_prefill_attn_batched(const vcs_kv_pool *pool_h, const void *q, int64_t q_batch_stride,
                             int64_t q_row_stride, const int32_t *q_pos3, const int32_t *nq_d, int nq_cap,
                             const int32_t *page_tables_d, const int32_t *n_vis_d, int n_vis_cap,
                             const int32_t *self_pages_d, int32_t self_offset, float softmax_scale,
                             void *out, int64_t out_batch_stride, int64_t out_row_stride, float *lse,
                             int B, int flags, int32_t *status_d, void *workspace, size_t workspace_bytes,
                             void *stream);

/* ------------------------------------------------------------------------------------------
 * vcs_retrieval_score -- Eq. 3, top-k.
 *
 * q_bar[kv][:] = mean over query rows i < nq and over the Hq/Hkv q heads of group kv of the
 * PRE-RoPE q; x_bar_c = k_sum[page_c] / page_len[page_c]; both flattened over (Hkv, d):
 *   scores[c] = <q_bar, x_bar_c>                       (normalize = 0, BASELINE config 5)
 *             = <q_bar, x_bar_c> / (|q_bar| |x_bar_c|)  (normalize = 1, Eq. 3; 0 if a norm is 0)
 * for c < n_cand, page_c = cand_pages_d[c].  An empty page scores 0.
 * topk_pages (optional, [k] int32, k <= 256): the k best pages not listed in exclude_pages_d, by
 * descending score, ties -> lower page id; -1 padding when fewer are eligible.  A page whose score
 * is NaN is never selected.
 * Errors: EINVAL, EALIGN, ECAP (workspace, k > 256).
 */
VCS_API size_t vcs_retrieval_score_workspace_bytes(const vcs_kv_pool *pool_h, int n_cand);
VCS_API int vcs_retrieval_score(const vcs_kv_pool *pool_h, const void *q, int64_t q_row_stride,
                        const int32_t *nq_d, int nq_cap,
                        const int32_t *cand_pages_d, int n_cand,
                        const int32_t *exclude_pages_d, int n_excl, int normalize,
                        float *scores, int k, int32_t *topk_pages,
                        void *workspace, size_t workspace_bytes, void *stream);

/*
 * vcs_retrieval_threshold -- threshold form of the query visibility, V_qry = { j : s_j >= tau_q }
 * (the rule the training mask of Eq. 4 uses), from scores written by
 * vcs_retrieval_score.  vis_pages[0 .. *vis_count_d) = pages cand_pages_d[c] with scores[c] >= tau_q
 * that are not in exclude_pages_d, in candidate order; the rest of vis_pages is -1; at most vis_cap
 * pages are written (the count is clamped).  The list can be used directly as the tail of an
 * attention page table with *vis_count_d added to its n_vis.  Errors: EINVAL.
 */
VCS_API int vcs_retrieval_threshold(const vcs_kv_pool *pool_h, const float *scores,
                            const int32_t *cand_pages_d, int n_cand,
                            const int32_t *exclude_pages_d, int n_excl, float tau_q,
                            int32_t *vis_pages, int vis_cap, int32_t *vis_count_d, void *stream);

/* ------------------------------------------------------------------------------------------
 * vcs_chunk_ingest / vcs_chunk_ingest_host -- one pass of the whole per-chunk hot path
 * (PAPER.md:57-71 restricted to token dropping -> KV append -> bounded prefill) for ONE stream:
 *   vcs_temporal_drop(z) -> kept_idx, kept_count, pos3
 *   vcs_kv_append_pages(k, v, pos3, kept_count) -> page `page_id` (offset 0)
 *   vcs_bounded_prefill_attn(q, pos3, kept_count; page_table; self_page = page_id) -> out
 * q/k/v hold T = G*P rows whose first kept_count rows belong to the kept tokens (the gather +
 * QKV projection between drop and append is the caller's, boundary step a4).
 * All members of vcs_chunk_call are caller-owned DEVICE buffers (see the three calls above for
 * shapes): z_d [G][P][D] of z_dtype; q_d [T][Hq][d], k_d / v_d [T][Hkv][d], out_d [T][Hq][d] of
 * the pool dtype, dense rows; kept_idx_d [T]; kept_count_d [1]; pos3_d [T][3]; pos_base_d [1].
 *
 * vcs_chunk_ingest       : inputs already resident in z_d / q_d / k_d / v_d; three launches.
 * vcs_chunk_ingest_host  : z_h, q_h, k_h, v_h are HOST buffers (pinned for true async) copied to
 *                          the staging members first; out_h [T][Hq][d], kept_idx_h [T] and
 *                          kept_count_h [1] are HOST buffers filled by device-to-host copies
 *                          enqueued after the kernels.  Nothing synchronises: the caller waits
 *                          on `stream` before reading the host outputs.
 * Errors: those of the three calls; EINVAL for NULL members.
 */
typedef struct vcs_chunk_call {
  int32_t G, P, D, Hg, Wg, t_stride, z_dtype, mode;
  float   tau;
  int32_t page_id, n_vis_cap, attn_flags;
  int32_t host_rows;   /* vcs_chunk_upload / _download: q, k, v and out rows copied (0 = all T rows); a caller that
                          knows the kept count on the host moves only the live rows */
  void *z_d, *q_d, *k_d, *v_d, *out_d;
  int32_t *kept_idx_d, *kept_count_d, *pos3_d;
  const int32_t *pos_base_d, *page_table_d, *n_vis_d;
  const void *prev_last_group_d;   /* mode VCS_DROP_CONSECUTIVE: the previous chunk's last group [P][D], or NULL */
  int32_t *status_d;
  void *ws_drop, *ws_append, *ws_attn;
  size_t ws_drop_bytes, ws_append_bytes, ws_attn_bytes;
} vcs_chunk_call;

/*
 * vcs_chunk_upload / vcs_chunk_download : the two copy halves of vcs_chunk_ingest_host as separate
 *                          calls, so that a caller can put them on their own streams and overlap the
 *                          H2D of chunk t+1 and the D2H of chunk t-1 with the kernels of chunk t
 *                          (double-buffered vcs_chunk_call staging members; the caller orders the
 *                          streams with events).  Only enqueue copies; same buffers as above.
 */
VCS_API int vcs_chunk_upload(const vcs_kv_pool *pool_h, const vcs_chunk_call *call_h,
                             const void *z_h, const void *q_h, const void *k_h, const void *v_h, void *stream);
VCS_API int vcs_chunk_download(const vcs_kv_pool *pool_h, const vcs_chunk_call *call_h,
                               void *out_h, int32_t *kept_idx_h, int32_t *kept_count_h, void *stream);
VCS_API int vcs_chunk_ingest(const vcs_kv_pool *pool_h, const vcs_chunk_call *call_h, void *stream);
VCS_API int vcs_chunk_ingest_host(const vcs_kv_pool *pool_h, const vcs_chunk_call *call_h,
                                  const void *z_h, const void *q_h, const void *k_h, const void *v_h,
                                  void *out_h, int32_t *kept_idx_h, int32_t *kept_count_h, void *stream);

/* ------------------------------------------------------------------------------------------
 * vcs_ingest_layers -- the hot path for L layers x B streams (several chunks in flight,
 * PAPER.md:73, :95): ONE token drop for the B streams (the drop sits before the LLM),
 * then for every layer l one batched KV append into pools_h[l] and one batched bounded prefill:
 * 1 + L x 3 launches (append, attention, combine) whatever B is, no host synchronisation.
 * pools_h: L host pool descriptors of identical geometry (one K/V pool per layer; page ids, page
 * lengths in use and page tables are shared by the layers: a chunk occupies the same page id in all).
 * Members of vcs_multi_call are caller-owned DEVICE buffers:
 *   z_d [B][G][P][D]; prev_last_group_d [B][P][D] or NULL (mode 1);
 *   q_d, out_d: layer l at + l*q_layer_stride / out_layer_stride ELEMENTS, then [B][T][Hq][d];
 *   k_d, v_d: layer l at + l*kv_layer_stride ELEMENTS, then [B][T][Hkv][d] (a stride of 0 feeds every
 *   layer the same rows); kept_idx_d [B][T], kept_count_d [B], pos3_d [B][T][3], pos_base_d [B];
 *   page_ids_d [B]: the page each stream's chunk is appended to (= its causal self page);
 *   page_tables_d [B][n_vis_cap], n_vis_d [B]: fully visible pages per stream (sink, window, retrieved).
 * Workspaces: ws_drop for B streams, ws_append = vcs_kv_append_batched_workspace_bytes(pool, T, B),
 * ws_attn as for vcs_bounded_prefill_attn; they are reused by the layers in turn.
 * Errors: those of the three calls; EINVAL for NULL members or pools of different geometry (heads, d, dtype,
 * n_pages, page_cap, rope).  Everything the host can see -- sizes, B <= 64, the page table, the size and
 * alignment of all three workspaces -- is checked BEFORE the first launch is enqueued, so an error return
 * leaves the pools, kept lists and positions untouched.
 */
typedef struct vcs_multi_call {
  int32_t B, L;
  int32_t G, P, D, Hg, Wg, t_stride, z_dtype, mode;
  float   tau;
  int32_t n_vis_cap, attn_flags;
  int64_t q_layer_stride, kv_layer_stride, out_layer_stride;
  void *z_d, *q_d, *k_d, *v_d, *out_d;
  const void *prev_last_group_d;
  int32_t *kept_idx_d, *kept_count_d, *pos3_d;
  const int32_t *pos_base_d, *page_ids_d, *page_tables_d, *n_vis_d;
  int32_t *status_d;
  void *ws_drop, *ws_append, *ws_attn;
  size_t ws_drop_bytes, ws_append_bytes, ws_attn_bytes;
} vcs_multi_call;

VCS_API int vcs_ingest_layers(const vcs_kv_pool *const *pools_h, const vcs_multi_call *call_h, void *stream);

/* ------------------------------------------------------------------------------------------
 * Self-test hooks.  The bf16 path uses two approximations whose error the attention tolerance alone
 * would bound only loosely; these calls evaluate them on caller-supplied points so that a test pins each:
 *   vcs_selftest_exp2_poly   y[i] = the degree-2 polynomial 2^x of the softmax (a quarter of the exponentials
 *                            run on the FMA pipe instead of MUFU); relative error <= 2e-3 for x in [-126, 8]
 *   vcs_selftest_rope_sincos sin / cos of pos[i] * inv_freq as the KV append and the Q build compute them
 *                            (Q0.64 turn fraction, 23-bit angle, MUFU sin / cos; reading D28);
 *                            absolute error <= 1e-6 for |pos| up to 2^20
 * x_d, y_d, sin_d, cos_d: device float[n]; pos_d: device int32[n].  Errors: EINVAL, ECUDA.
 */
VCS_API int vcs_selftest_exp2_poly(const float *x_d, float *y_d, int n, void *stream);
VCS_API int vcs_selftest_rope_sincos(const int32_t *pos_d, int n, double inv_freq, float *sin_d, float *cos_d, void *stream);

/* ------------------------------------------------------------------------------------------
 * CUDA-graph capture of a chain of calls (the launch-bound inner loop of a stream: 4 small launches per
 * chunk and layer).  Everything enqueued on `stream` between vcs_graph_begin and vcs_graph_end -- vcs
 * calls, and any other capturable stream work of the caller -- is recorded instead of executed;
 * vcs_graph_launch replays it with one launch (buffers and arguments are those of the recorded calls:
 * replay a graph only while they are alive).  The programmatic-dependent-launch edges between
 * consecutive vcs kernels are kept.  The handle owns host-side CUDA graph objects only; destroy it with
 * vcs_graph_destroy (called while the same thread is recording another graph, it is carried out when that
 * recording ends).  Capture is thread-local: other threads may keep using CUDA.  `stream` must be a
 * created stream (the legacy default stream cannot be captured).
 * Errors: ECUDA (capture / instantiate / launch), EINVAL.
 */
VCS_API int vcs_graph_begin(void *stream);
VCS_API int vcs_graph_end(void *stream, void **graph_out);
VCS_API int vcs_graph_launch(void *graph, void *stream);
VCS_API int vcs_graph_destroy(void *graph);

#ifdef __cplusplus
}
#endif
#endif /* VCS_H_ */
