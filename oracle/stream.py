"""ORACLE -- TEST INFRASTRUCTURE ONLY.  Per-chunk ingestion loop in the oracle: the control flow
of PAPER.md:57-71 / Fig. 2 restricted to the hot path (drop -> KV append -> bounded prefill) plus
the query-time path (retrieval -> query prefill), in fp64.  Shares nothing with the CUDA driver.
"""
from __future__ import annotations

from typing import Callable, List, Optional, Sequence

import numpy as np

from . import vicostream_oracle as vo


class OracleStream:
    """One video stream: sink page + one page per chunk; window W = paper's `acn`
    (visible set {t-W..t}; reading D11: current chunk PLUS W previous)."""

    def __init__(self, Hq: int, Hkv: int, d: int, theta: float, sections: Sequence[int],
                 G: int, Hg: int, Wg: int, tau: float, W: int, t_stride: int = 1, mode: int = 0):
        self.pool = vo.PagedKV(Hq, Hkv, d, theta, sections)
        self.G, self.Hg, self.Wg, self.t_stride = G, Hg, Wg, t_stride
        self.tau, self.W, self.mode = tau, W, mode
        self.sink_page: Optional[int] = None
        self.chunk_pages: List[int] = []
        self.pos_base = 0
        self.prev_last_group = None

    def add_sink(self, page: int, K: np.ndarray, V: np.ndarray):
        """Sink / system prefix (reading D14): S tokens at positions (i, i, i), own page."""
        n = K.shape[0]
        self.pool.append(page, 0, K, V, vo.text_positions(0, n))
        self.sink_page = page
        self.pos_base = n

    def visible_pages(self, t: Optional[int] = None) -> List[int]:
        """Fully visible pages for chunk index t (default: the next chunk): sink + chunks
        max(0, t-W)..t-1 (reading D12: clipped at stream start).  W < 0 = full history."""
        t = len(self.chunk_pages) if t is None else t
        lo = 0 if self.W < 0 else max(0, t - self.W)
        pages = [] if self.sink_page is None else [self.sink_page]
        return pages + self.chunk_pages[lo:t]

    def ingest_chunk(self, Z: np.ndarray, page: int,
                     qkv: Callable[[np.ndarray, int], tuple], attend: bool = True,
                     rows: Optional[Sequence[int]] = None):
        """One pass of the hot path over one chunk.  `qkv(kept_idx, n)` returns the PRE-RoPE
        Q[n][Hq][d], K[n][Hkv][d], V[n][Hkv][d] of the kept tokens (the boundary step a4)."""
        prev = self.prev_last_group if self.mode == 1 else None
        keep, kept_idx, n = vo.temporal_drop(Z, self.tau, self.mode, prev)
        pos_all = vo.grid_positions(self.G, self.Hg, self.Wg, self.pos_base, self.t_stride)
        pos3 = pos_all[kept_idx]
        Q, K, V = qkv(kept_idx, n)
        vis = self.visible_pages()
        self.pool.append(page, 0, K, V, pos3)
        out = dict(keep=keep, kept_idx=kept_idx, n=n, pos3=pos3, visible=vis, page=page)
        if attend:
            O, lse = vo.bounded_attention(self.pool, Q, pos3, vis, self_page=page, self_offset=0,
                                          rows=rows)
            out.update(O=O, lse=lse)
        self.chunk_pages.append(page)
        self.pos_base = vo.next_position_base(self.G, self.Hg, self.Wg, self.pos_base, self.t_stride)
        self.prev_last_group = np.asarray(Z)[-1]
        return out

    def query(self, Q: np.ndarray, K: np.ndarray, V: np.ndarray, text_page: int, k: int,
              recent: int, normalize: bool = False, cand_pages: Optional[Sequence[int]] = None):
        """Query-time path (reading D21): score every candidate chunk page,
        take the top-k outside the `recent` most recent chunks, then the text tokens attend to
        sink + recent + retrieved pages and causally to their own text page (reading D27)."""
        nq = Q.shape[0]
        recent_pages = self.chunk_pages[len(self.chunk_pages) - recent:] if recent > 0 else []
        cand = list(self.chunk_pages) if cand_pages is None else list(cand_pages)
        scores = vo.retrieval_scores(self.pool, Q, cand, normalize)
        top = vo.retrieve_topk(scores, cand, k, exclude_pages=recent_pages)
        pos3 = vo.text_positions(self.pos_base, nq)
        self.pool.append(text_page, 0, K, V, pos3)
        vis = ([] if self.sink_page is None else [self.sink_page]) + list(recent_pages) + \
            [int(p) for p in top if p >= 0]
        O, lse = vo.bounded_attention(self.pool, Q, pos3, vis, self_page=text_page, self_offset=0)
        return dict(scores=scores, topk=top, visible=vis, O=O, lse=lse, pos3=pos3)
