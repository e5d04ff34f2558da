"""ORACLE -- TEST INFRASTRUCTURE ONLY.  Plain, slow, fp64 numpy restatement of ViCoStream's
per-chunk LLM-ingestion hot path, written from the paper (PAPER.md = /root/reference/PAPER.md,
arxiv/paper_2606_19849) and from the readings listed in DESIGN.md.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs may import this package.  It shares no code with the CUDA path
(`paper_2606_19849_b200/`), never imports it, and the product never imports this.

Everything is fp64 with explicit boolean masks; no blocking, fusion or reordering beyond what
the cited definition states.  Each function cites the passage it follows.

Pin status (tests/test_oracle_pins.py): every function below is pinned to closed forms,
textbook/library special cases, invariants or brute force.  PARITY UNPINNED: agreement with the
authors' released code on real video (their eps, token order, projector space, frames vs merged
temporal groups) -- nothing available offline can pin that; see DESIGN.md "Readings".
"""
from __future__ import annotations

from typing import Dict, Iterable, List, Optional, Sequence, Tuple

import numpy as np

F64 = np.float64


# ----------------------------------------------------------------------------------------------
# O1  temporal token dropping -- PAPER.md:111-121 (section 3 "Token Dropping", Eq. 1 and Eq. 2)
# ----------------------------------------------------------------------------------------------
def cosine_similarity(a: np.ndarray, b: np.ndarray) -> float:
    """Eq. 1: S = <a,b> / (||a|| ||b||).  Reading D6: S := 0 if either norm is 0.

    Reading D31: a cosine lies in [-1, 1] (Cauchy-Schwarz).  The fp64 quotient of a rounded dot
    product by two rounded square roots can land one ulp outside that interval -- it does so for
    about a quarter of random IDENTICAL token pairs, the static-pixel case the method exists for --
    and would then "exceed" tau = 1, against the paper's "s = 1.0 -> 0 % drop".  The
    quotient is therefore clamped to the interval the mathematics fixes."""
    a = np.asarray(a, dtype=F64)
    b = np.asarray(b, dtype=F64)
    na = np.sqrt(np.sum(a * a))
    nb = np.sqrt(np.sum(b * b))
    if na == 0.0 or nb == 0.0:
        return 0.0
    s = float(np.sum(a * b) / (na * nb))
    return min(1.0, max(-1.0, s))


def pairwise_similarity(Z: np.ndarray) -> np.ndarray:
    """Eq. 1 for every position and every pair: S[i, j, p] for i < j (other entries NaN).

    Z: [G][P][D] projected tokens z_t^{(i)}(p) of one chunk."""
    Z = np.asarray(Z, dtype=F64)
    G, P, _ = Z.shape
    S = np.full((G, G, P), np.nan, dtype=F64)
    for p in range(P):
        for i in range(G):
            for j in range(i + 1, G):
                S[i, j, p] = cosine_similarity(Z[i, p], Z[j, p])
    return S


def drop_predicate(Z: np.ndarray, tau: float) -> np.ndarray:
    """Eq. 2: drop(p) <=> AND_{i<j} [ S_{i->j}(p) > tau ]  (strict, reading D3).

    With G == 1 the conjunction is empty; reading D10: the only group is the anchor, so the
    predicate is irrelevant (returned False)."""
    Z = np.asarray(Z, dtype=F64)
    G, P, _ = Z.shape
    drop = np.zeros(P, dtype=bool)
    if G < 2:
        return drop
    S = pairwise_similarity(Z)
    for p in range(P):
        ok = True
        for i in range(G):
            for j in range(i + 1, G):
                ok = ok and bool(S[i, j, p] > tau)
        drop[p] = ok
    return drop


def temporal_keep_mask(Z: np.ndarray, tau: float, mode: int = 0,
                       prev_last_group: Optional[np.ndarray] = None) -> np.ndarray:
    """keep[g, p] for one chunk.

    mode 0 (chunk-level, the paper's rule): "we always preserve the first frame of each chunk as
    an anchor" -> keep[0, :] = True; a position that satisfies Eq. 2 loses
    all its non-anchor tokens (reading D2): keep[g>=1, p] = not drop(p).

    mode 1 (frame-level / consecutive variant): token (g, p) is pruned when its
    similarity to the previous group's token at p exceeds tau; the reference for g = 0 is the
    previous chunk's last group when supplied ("without a multi-frame chunk anchor"), otherwise
    group 0 is kept."""
    Z = np.asarray(Z, dtype=F64)
    G, P, _ = Z.shape
    keep = np.ones((G, P), dtype=bool)
    if mode == 0:
        drop = drop_predicate(Z, tau)
        for g in range(1, G):
            keep[g, :] = ~drop
    elif mode == 1:
        for g in range(G):
            for p in range(P):
                if g == 0:
                    if prev_last_group is None:
                        continue
                    ref = np.asarray(prev_last_group, dtype=F64)[p]
                else:
                    ref = Z[g - 1, p]
                keep[g, p] = not (cosine_similarity(ref, Z[g, p]) > tau)
    else:
        raise ValueError("mode must be 0 or 1")
    return keep


def compact(keep: np.ndarray) -> Tuple[np.ndarray, int]:
    """Stream compaction ("retained visual tokens Z_t"; reading D9): ascending
    original sequence index g*P + p of the kept tokens, and their count."""
    flat = np.asarray(keep, dtype=bool).reshape(-1)
    idx = np.array([i for i in range(flat.size) if flat[i]], dtype=np.int32)
    return idx, int(idx.size)


def temporal_drop(Z: np.ndarray, tau: float, mode: int = 0,
                  prev_last_group: Optional[np.ndarray] = None):
    """O1 end to end: (keep[G][P] bool, kept_idx int32 ascending, count)."""
    keep = temporal_keep_mask(Z, tau, mode, prev_last_group)
    idx, n = compact(keep)
    return keep, idx, n


# ----------------------------------------------------------------------------------------------
# O1b  entropy-based spatial token selection -- PAPER.md:109 (section 3 "Token Dropping", spatial
#      strategies; Table 8-middle).  Reading D30: "the normalized probability of the
#      m-th feature dimension" is the softmax of the token's features over its D dimensions; natural log.
# ----------------------------------------------------------------------------------------------
def feature_entropy(X: np.ndarray) -> np.ndarray:
    """I(x_j) = - sum_m p_jm log p_jm with p_j = softmax(x_j) over the feature dimension.  X: [n][D]."""
    X = np.asarray(X, dtype=F64)
    out = np.zeros(X.shape[0], dtype=F64)
    for j in range(X.shape[0]):
        x = X[j] - np.max(X[j])
        e = np.exp(x)
        pj = e / np.sum(e)
        nz = pj > 0.0
        out[j] = -np.sum(pj[nz] * np.log(pj[nz]))
    return out


def topk_by_score(scores: np.ndarray, K: int) -> np.ndarray:
    """Indices of the K highest scores (ties -> lower index wins), returned in ASCENDING index order
    (retained tokens keep their sequence order, reading D9)."""
    n = len(scores)
    order = sorted(range(n), key=lambda i: (-float(scores[i]), i))
    return np.array(sorted(order[:max(0, min(K, n))]), dtype=np.int32)


def spatial_entropy_select(Z: np.ndarray, K: int):
    """"Retains the top-K tokens with the highest entropy scores", "applied independently to each
    frame".  Z: [G][P][D] (G frames / temporal groups of one chunk).
    Returns (entropy[G][P], kept_idx ascending over g*P + p, count = G * min(K, P))."""
    Z = np.asarray(Z, dtype=F64)
    G, P, _ = Z.shape
    H = np.stack([feature_entropy(Z[g]) for g in range(G)], axis=0)
    idx = np.concatenate([g * P + topk_by_score(H[g], K) for g in range(G)]).astype(np.int32) if G else \
        np.zeros(0, dtype=np.int32)
    return H, idx, int(idx.size)


# ----------------------------------------------------------------------------------------------
# O2  positions (reading D18; the paper is silent, BASELINE.json: "M-RoPE (t,h,w) positions from
#     grid indices")
# ----------------------------------------------------------------------------------------------
def grid_positions(G: int, Hg: int, Wg: int, base: int, t_stride: int = 1) -> np.ndarray:
    """pos3[g*P + r*Wg + c] = (base + g*t_stride, base + r, base + c)."""
    pos = np.zeros((G * Hg * Wg, 3), dtype=np.int64)
    for g in range(G):
        for r in range(Hg):
            for c in range(Wg):
                pos[(g * Hg + r) * Wg + c] = (base + g * t_stride, base + r, base + c)
    return pos


def next_position_base(G: int, Hg: int, Wg: int, base: int, t_stride: int = 1) -> int:
    """b' = b + max(G*t_stride, Hg, Wg)."""
    return base + max(G * t_stride, Hg, Wg)


def text_positions(start: int, n: int) -> np.ndarray:
    """Text / sink token i: (start+i, start+i, start+i)."""
    i = np.arange(start, start + n, dtype=np.int64)
    return np.stack([i, i, i], axis=1)


# ----------------------------------------------------------------------------------------------
# O3  M-RoPE (reading D17: rotate-half pairs (m, m + d/2), pairs split into t/h/w sections)
# ----------------------------------------------------------------------------------------------
def mrope_rotate(x: np.ndarray, pos3: np.ndarray, theta: float, sections: Sequence[int]) -> np.ndarray:
    """x: [n][H][d]; pos3: [n][3] integer (t, h, w).  Pair m in [0, d/2): elements (m, m + d/2),
    frequency f_m = theta^(-2m/d), axis(m) = t for the first sections[0] pairs, h for the next
    sections[1], w for the last sections[2]; angle a = pos[axis(m)] * f_m;
    (x_m, x_{m+d/2}) <- (x_m cos a - x_{m+d/2} sin a,  x_{m+d/2} cos a + x_m sin a)."""
    x = np.asarray(x, dtype=F64)
    pos3 = np.asarray(pos3)
    n, H, d = x.shape
    half = d // 2
    assert sum(sections) == half
    axis_of = np.concatenate([np.full(sections[0], 0), np.full(sections[1], 1), np.full(sections[2], 2)])
    out = np.empty_like(x)
    for m in range(half):
        f_m = F64(theta) ** (-2.0 * m / d)
        a = pos3[:, axis_of[m]].astype(F64) * f_m                 # [n]
        c = np.cos(a)[:, None]
        s = np.sin(a)[:, None]
        lo = x[:, :, m]
        hi = x[:, :, m + half]
        out[:, :, m] = lo * c - hi * s
        out[:, :, m + half] = hi * c + lo * s
    return out


# ----------------------------------------------------------------------------------------------
# O4  chunk-granular paged KV state ("historical visual cache"; paging, GQA and the
#     per-page key summary come from BASELINE.json / readings D19, D27)
# ----------------------------------------------------------------------------------------------
class PagedKV:
    """page id -> K_rot[len][Hkv][d], V[len][Hkv][d], k_sum[Hkv][d] (sum of PRE-RoPE keys)."""

    def __init__(self, Hq: int, Hkv: int, d: int, theta: float, sections: Sequence[int]):
        self.Hq, self.Hkv, self.d = Hq, Hkv, d
        self.theta, self.sections = theta, tuple(sections)
        self.K: Dict[int, np.ndarray] = {}
        self.V: Dict[int, np.ndarray] = {}
        self.k_sum: Dict[int, np.ndarray] = {}

    def page_len(self, page: int) -> int:
        return 0 if page not in self.K else int(self.K[page].shape[0])

    def append(self, page: int, page_offset: int, K: np.ndarray, V: np.ndarray, pos3: np.ndarray):
        """Write K (rotated by M-RoPE at pos3) and V at [page_offset, page_offset + n) of `page`;
        page_offset == 0 starts the page afresh, otherwise it must equal the current length."""
        K = np.asarray(K, dtype=F64)
        V = np.asarray(V, dtype=F64)
        Kr = mrope_rotate(K, pos3, self.theta, self.sections)
        if page_offset == 0:
            self.K[page], self.V[page] = Kr, V.copy()
            self.k_sum[page] = K.sum(axis=0)
        else:
            assert page_offset == self.page_len(page)
            self.K[page] = np.concatenate([self.K[page], Kr], axis=0)
            self.V[page] = np.concatenate([self.V[page], V], axis=0)
            self.k_sum[page] = self.k_sum[page] + K.sum(axis=0)


# ----------------------------------------------------------------------------------------------
# O5  bounded visual attention -- PAPER.md:129 (Attn_v = softmax(Q K^T / sqrt(d)) V over the
#     chunks t-acn..t), PAPER.md:138 (query side), mask Eq. 4
# ----------------------------------------------------------------------------------------------
def bounded_attention(pool: PagedKV, Q: np.ndarray, q_pos3: np.ndarray,
                      page_table: Sequence[int], self_page: int = -1, self_offset: int = 0,
                      scale: Optional[float] = None, rows: Optional[Sequence[int]] = None,
                      return_probs: bool = False):
    """Q: [nq][Hq][d] PRE-RoPE queries (rotated here with q_pos3).

    Visible keys: every valid token of every page in `page_table` (fully visible: sink, the last
    W chunks, retrieved chunks), then the self page, where query row i sees tokens
    j_local <= self_offset + i (causal inside the current chunk, reading D13).  GQA (reading
    D16): q head h reads kv head h // (Hq/Hkv).  Scale 1/sqrt(d).
    `rows` restricts the computation to a subset of query rows (each row is independent).
    Returns O[nq'][Hq][d], lse[Hq][nq'] (natural log) and optionally P[Hq][nq'][N_tot]."""
    Q = np.asarray(Q, dtype=F64)
    nq, Hq, d = Q.shape
    g = Hq // pool.Hkv
    scale = (1.0 / np.sqrt(d)) if not scale else float(scale)
    Qr = mrope_rotate(Q, q_pos3, pool.theta, pool.sections)
    row_ids = np.arange(nq) if rows is None else np.asarray(list(rows), dtype=np.int64)

    Ks = [pool.K[p] for p in page_table]
    Vs = [pool.V[p] for p in page_table]
    n_full = int(sum(k.shape[0] for k in Ks))
    if self_page >= 0:
        Ks.append(pool.K[self_page])
        Vs.append(pool.V[self_page])
    K_cat = np.concatenate(Ks, axis=0) if Ks else np.zeros((0, pool.Hkv, d))
    V_cat = np.concatenate(Vs, axis=0) if Vs else np.zeros((0, pool.Hkv, d))
    N_tot = K_cat.shape[0]

    mask = np.zeros((row_ids.size, N_tot), dtype=bool)
    mask[:, :n_full] = True
    if self_page >= 0:
        j_local = np.arange(N_tot - n_full)
        mask[:, n_full:] = j_local[None, :] <= (self_offset + row_ids)[:, None]

    O = np.zeros((row_ids.size, Hq, d), dtype=F64)
    lse = np.zeros((Hq, row_ids.size), dtype=F64)
    probs = np.zeros((Hq, row_ids.size, N_tot), dtype=F64) if return_probs else None
    for h in range(Hq):
        kv = h // g
        L = (Qr[row_ids, h, :] @ K_cat[:, kv, :].T) * scale
        L = np.where(mask, L, -np.inf)
        # reading D29: a row with an EMPTY visible set (softmax undefined) yields zeros, lse = -inf
        vis_rows = mask.any(axis=1)
        lse[h, ~vis_rows] = -np.inf
        Lv = L[vis_rows]
        rowmax = np.max(Lv, axis=1, keepdims=True) if Lv.size else np.zeros((0, 1))
        Pm = np.exp(Lv - rowmax)
        rowsum = np.sum(Pm, axis=1, keepdims=True)
        Pm = Pm / rowsum
        O[vis_rows, h, :] = Pm @ V_cat[:, kv, :]
        lse[h, vis_rows] = (rowmax + np.log(rowsum))[:, 0]
        if return_probs:
            probs[h, vis_rows] = Pm
    if return_probs:
        return O, lse, probs
    return O, lse


def merge_partial_attention(O_a, lse_a, O_b, lse_b):
    """LSE merge of attention over two DISJOINT visible sets == attention over the union.
    O: [n][Hq][d], lse: [Hq][n]."""
    m = np.maximum(lse_a, lse_b)
    wa = np.exp(lse_a - m)
    wb = np.exp(lse_b - m)
    tot = wa + wb
    O = O_a * (wa / tot).T[:, :, None] + O_b * (wb / tot).T[:, :, None]
    return O, m + np.log(tot)


def eq4_visible(chunk_of_q: int, kind_q: str, chunk_of_k: int, kind_k: str, acn: int,
                retrieved: Iterable[int] = ()) -> bool:
    """Eq. 4 visibility of key chunk j for a query token of chunk i, at CHUNK
    granularity, extended with the sink of reading D14 and the recent window of reading D21:
      vision token:  t_j in V_vis(t_i) = { j : t_i - acn <= j <= t_i }
      query token:   t_j in V_qry (the retrieved set)
      sink keys are visible to everyone; a query additionally sees its own text chunk and, per
      BASELINE config 5, the recent window (passed in through `retrieved` by the caller)."""
    if kind_k == "sink":
        return True
    if kind_q == "vis":
        return kind_k == "vis" and (chunk_of_q - acn <= chunk_of_k <= chunk_of_q)
    if kind_q == "qry":
        if kind_k == "qry":
            return True
        return chunk_of_k in set(retrieved)
    raise ValueError(kind_q)


def eq4_mask(tok_chunk: Sequence[int], tok_kind: Sequence[str], acn: int,
             retrieved: Iterable[int] = ()) -> np.ndarray:
    """Token-level boolean mask over a whole stream laid out in sequence order: M[i, j] is True
    (additive 0) iff Eq. 4 exposes token j's chunk to token i AND j <= i (decoder causality,
    reading D13); False stands for the paper's -inf."""
    n = len(tok_chunk)
    M = np.zeros((n, n), dtype=bool)
    for i in range(n):
        for j in range(i + 1):
            M[i, j] = eq4_visible(tok_chunk[i], tok_kind[i], tok_chunk[j], tok_kind[j], acn, retrieved)
    return M


def masked_attention_dense(Qr: np.ndarray, Kr: np.ndarray, V: np.ndarray, M: np.ndarray,
                           scale: float) -> np.ndarray:
    """Textbook softmax(Q K^T * scale + mask) V for ONE head with an explicit boolean mask."""
    L = (np.asarray(Qr, F64) @ np.asarray(Kr, F64).T) * scale
    L = np.where(M, L, -np.inf)
    L = L - L.max(axis=1, keepdims=True)
    Pm = np.exp(L)
    Pm /= Pm.sum(axis=1, keepdims=True)
    return Pm @ np.asarray(V, F64)


# ----------------------------------------------------------------------------------------------
# O6  query-chunk retrieval -- PAPER.md:131-136 (Eq. 3), readings D19-D22
# ----------------------------------------------------------------------------------------------
def mean_query(Q: np.ndarray, Hkv: int) -> np.ndarray:
    """q_bar[kv][d] = mean over the query tokens and over the Hq/Hkv q heads of kv group `kv`
    of the PRE-RoPE queries (Eq. 3 "averaged into representative features", reading D19)."""
    Q = np.asarray(Q, dtype=F64)
    nq, Hq, d = Q.shape
    g = Hq // Hkv
    return Q.reshape(nq, Hkv, g, d).mean(axis=(0, 2))


def retrieval_scores(pool: PagedKV, Q: np.ndarray, cand_pages: Sequence[int],
                     normalize: bool = False) -> np.ndarray:
    """s_i for every candidate page: x_bar_i = k_sum[i] / page_len[i] (mean pre-RoPE key),
    flattened over (Hkv, d); s_i = <q_bar, x_bar_i> (BASELINE config 5, normalize=False) or the
    cosine of Eq. 3 (normalize=True; 0 if either norm is 0)."""
    qb = mean_query(Q, pool.Hkv).reshape(-1)
    out = np.zeros(len(cand_pages), dtype=F64)
    for c, page in enumerate(cand_pages):
        n = pool.page_len(page)
        xb = (pool.k_sum[page] / n).reshape(-1) if n > 0 else np.zeros_like(qb)
        s = float(np.sum(qb * xb))
        if normalize:
            nq_, nx_ = np.sqrt(np.sum(qb * qb)), np.sqrt(np.sum(xb * xb))
            s = 0.0 if (nq_ == 0.0 or nx_ == 0.0) else s / (nq_ * nx_)
        out[c] = s
    return out


def retrieve_topk(scores: np.ndarray, cand_pages: Sequence[int], k: int,
                  exclude_pages: Iterable[int] = ()) -> np.ndarray:
    """"Only the top-k chunks are exposed to query tokens".  Excluded pages
    (the recent window, reading D21) never win; order = descending score, ties -> lower page id
    (reading D22); fewer than k eligible candidates -> padded with -1."""
    excl = set(int(p) for p in exclude_pages)
    elig = [(-float(scores[c]), int(cand_pages[c])) for c in range(len(cand_pages))
            if int(cand_pages[c]) not in excl]
    elig.sort()
    out = np.full(k, -1, dtype=np.int32)
    for r, (_, page) in enumerate(elig[:k]):
        out[r] = page
    return out


def retrieve_threshold(scores: np.ndarray, cand_pages: Sequence[int], tau_q: float) -> List[int]:
    """Training-time visibility V_qry = { j : s_j >= tau_q }."""
    return [int(cand_pages[c]) for c in range(len(cand_pages)) if scores[c] >= tau_q]


# ----------------------------------------------------------------------------------------------
# throughput formula -- PAPER.md:77-83
# ----------------------------------------------------------------------------------------------
def fps_max(c: int, stage_ms: Sequence[float]) -> float:
    """FPS_max = 1000 * c / T_pipe,  T_pipe = max{T_vp, T_vit, T_drop, T_llm}."""
    return 1000.0 * c / max(stage_ms)
