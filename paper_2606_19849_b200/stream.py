"""Per-chunk ingestion driver over the C ABI: drop -> KV append -> bounded prefill, and the
query-time path retrieval -> query prefill.  Marshalling and buffer
ownership only; all arithmetic runs in libvcs.so.  No host synchronisation between calls: kept
counts, page lengths and top-k page ids stay on the device.
"""
from __future__ import annotations

from typing import Callable, List, Optional, Sequence

import torch

from . import vcs


class VideoStream:
    """One video stream on one GPU.  Page ids are chosen by the caller (scattered is fine)."""

    def __init__(self, pool: vcs.KVPool, G: int, Hg: int, Wg: int, D: int, tau: float, W: int,
                 sink_page: int, chunk_pages: Sequence[int], sink_len: int, t_stride: int = 1,
                 mode: int = vcs.DROP_CHUNK_ALLPAIRS, attn_flags: int = vcs.ATTN_AUTO, device="cuda"):
        self.pool, self.G, self.Hg, self.Wg, self.D = pool, G, Hg, Wg, D
        self.P, self.T = Hg * Wg, G * Hg * Wg
        self.tau, self.W, self.mode, self.t_stride = float(tau), W, mode, t_stride
        self.attn_flags = attn_flags
        self.sink_page, self.chunk_pages, self.sink_len = sink_page, list(chunk_pages), sink_len
        self.dev = device
        n = len(self.chunk_pages)
        # visible-set tables (step a6): sink + chunks max(0,t-W)..t-1; W < 0 = full history
        cap = 1 + (n if W < 0 else min(W, n))
        tab = torch.full((max(n, 1), cap), -1, dtype=torch.int32)
        nvis = torch.zeros((max(n, 1),), dtype=torch.int32)
        for t in range(n):
            row, n_t = vcs.vcs_visible_set(t, W, sink_page, self.chunk_pages, cap)     # step a6 lives behind the C ABI
            tab[t] = torch.tensor(row, dtype=torch.int32)
            nvis[t] = n_t
        self.table_cap = cap
        self.tables = tab.to(device)
        self.n_vis = nvis.to(device)
        bases = [sink_len]                                     # reading D18: the rule lives behind the C ABI
        for _ in range(1, max(n, 1)):
            bases.append(vcs.vcs_next_position_base(G, Hg, Wg, bases[-1], t_stride))
        self.pos_base = torch.tensor(bases, dtype=torch.int32).to(device)
        self.kept_idx = torch.empty((1, self.T), dtype=torch.int32, device=device)
        self.kept_count = torch.zeros((1,), dtype=torch.int32, device=device)
        self.pos3 = torch.zeros((1, self.T, 3), dtype=torch.int32, device=device)
        self.status = torch.zeros((1,), dtype=torch.int32, device=device)
        self.ws_drop = vcs.workspace(vcs.vcs_temporal_drop_workspace_bytes(1, G, self.P), device)
        self.ws_append = vcs.workspace(vcs.vcs_kv_append_workspace_bytes(pool, max(self.T, sink_len)), device)
        self.ws_attn = vcs.workspace(vcs.vcs_bounded_prefill_attn_workspace_bytes(pool, self.T, cap + 16), device)
        self.t = 0
        self.prev_last_group: Optional[torch.Tensor] = None

    def add_sink(self, K: torch.Tensor, V: torch.Tensor):
        S = K.shape[0]
        pos = vcs.vcs_text_positions(0, S, self.dev)
        vcs.vcs_kv_append_pages(self.pool, K, V, pos, None, S, self.sink_page, 0, self.ws_append, self.status)

    def drop(self, z: torch.Tensor):
        """z: [G][P][D] device tensor of the chunk's projected tokens."""
        t = self.t
        prev = self.prev_last_group if self.mode == vcs.DROP_CONSECUTIVE else None
        vcs.vcs_temporal_drop(z.view(1, self.G, self.P, self.D), self.tau, self.kept_idx, self.kept_count,
                              self.ws_drop, mode=self.mode,
                              prev_last_group=None if prev is None else prev.view(1, self.P, self.D),
                              pos3=self.pos3, Hg=self.Hg, Wg=self.Wg, t_stride=self.t_stride,
                              pos_base=self.pos_base[t:t + 1])

    def append(self, K: torch.Tensor, V: torch.Tensor):
        vcs.vcs_kv_append_pages(self.pool, K, V, self.pos3[0], self.kept_count, self.T, self.chunk_pages[self.t], 0,
                                self.ws_append, self.status)

    def attend(self, Q: torch.Tensor, out: torch.Tensor, lse: Optional[torch.Tensor] = None):
        t = self.t
        vcs.vcs_bounded_prefill_attn(self.pool, Q, self.pos3[0], self.kept_count, self.T, self.tables[t],
                                     self.n_vis[t:t + 1], self.table_cap, self.chunk_pages[t], 0, out,
                                     self.ws_attn, lse=lse, flags=self.attn_flags, status=self.status)

    def ingest_chunk(self, z: torch.Tensor, qkv: Callable, out: torch.Tensor, lse: Optional[torch.Tensor] = None,
                     attend: bool = True):
        """One pass of the hot path.  `qkv(kept_idx[T] int32, kept_count[1] int32)` returns device
        Q[T][Hq][d], K[T][Hkv][d], V[T][Hkv][d] whose first count rows belong to the kept tokens
        (boundary step a4: gather + projection, or direct synthetic Q/K/V)."""
        self.drop(z)
        Q, K, V = qkv(self.kept_idx[0], self.kept_count)
        self.append(K, V)
        if attend:
            self.attend(Q, out, lse)
        self.prev_last_group = z[-1]
        self.t += 1


class QueryPath:
    """Query-time TTFT path (BASELINE config 5): score the bank, take top-k outside the recent
    window on the device, and prefill the text query over sink + recent + retrieved pages."""

    def __init__(self, pool: vcs.KVPool, sink_page: int, recent_pages: Sequence[int], cand_pages: Sequence[int],
                 k: int, nq_cap: int, text_page: int, text_pos_start: int, normalize: bool = False,
                 attn_flags: int = vcs.ATTN_AUTO, device="cuda"):
        self.pool, self.k, self.nq_cap, self.text_page, self.normalize = pool, k, nq_cap, text_page, normalize
        self.attn_flags = attn_flags
        tab, self.n_fixed = vcs.vcs_visible_set_query(sink_page, list(recent_pages), k)    # step a6, query side
        self.table = torch.tensor(tab, dtype=torch.int32, device=device)
        self.n_vis = torch.zeros((1,), dtype=torch.int32, device=device)
        self.cand = torch.tensor(list(cand_pages), dtype=torch.int32, device=device)
        self.excl = torch.tensor(list(recent_pages), dtype=torch.int32, device=device) if recent_pages else None
        self.scores = torch.zeros((len(cand_pages),), dtype=torch.float32, device=device)
        self.pos3 = vcs.vcs_text_positions(text_pos_start, nq_cap, device)
        self.status = torch.zeros((1,), dtype=torch.int32, device=device)
        self.ws_ret = vcs.workspace(vcs.vcs_retrieval_score_workspace_bytes(pool, len(cand_pages)), device)
        self.ws_append = vcs.workspace(vcs.vcs_kv_append_workspace_bytes(pool, nq_cap), device)
        self.ws_attn = vcs.workspace(vcs.vcs_bounded_prefill_attn_workspace_bytes(pool, nq_cap, len(tab)), device)

    def run(self, Q: torch.Tensor, K: torch.Tensor, V: torch.Tensor, out: torch.Tensor,
            lse: Optional[torch.Tensor] = None):
        # top-k page ids are written by the scorer straight into the tail of the page table
        vcs.vcs_retrieval_score(self.pool, Q, None, self.nq_cap, self.cand, self.scores, self.ws_ret, k=self.k,
                                topk_pages=self.table[self.n_fixed:], exclude_pages=self.excl,
                                normalize=self.normalize)
        vcs.vcs_kv_append_pages(self.pool, K, V, self.pos3, None, self.nq_cap, self.text_page, 0, self.ws_append,
                                self.status)
        # -1 padded entries (fewer than k eligible) are skipped by the kernels as bad pages
        vcs.vcs_bounded_prefill_attn(self.pool, Q, self.pos3, None, self.nq_cap, self.table, None,
                                     self.table.numel(), self.text_page, 0, out, self.ws_attn, lse=lse,
                                     flags=self.attn_flags, status=None)
