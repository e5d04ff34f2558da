"""GPU parity of vcs_ingest_layers (L layers x B streams, one drop + L x (batched append + batched bounded
prefill)) against L x B independent oracle streams, chunk after chunk, and of the CUDA-graph replay of the
same chain (vcs_graph_begin / _end / _launch)."""
import numpy as np
import pytest
import torch

import oracle as vo
import synth
from helpers import ATTN_MAX_ABS, ATTN_REL_L2, attn_errors, attn_max_abs_tol, dev, f64, i32

pytestmark = pytest.mark.gpu


def test_ingest_layers_streams_and_graph_replay():
    _layers_scene(synth.get_config("vl3b").with_(Hg=7, Wg=11, D=256, W=2), L=3, B=2, n_chunks=4, rows_of=None)


def test_ingest_layers_full_size_config2_grid():
    """The shape class bench.py times (config-2 grid 4 x 16 x 29, hidden 2048, 16 / 2 heads, sink 64, W = 4) at
    L = 4 layers x B = 4 streams over 6 chunks (the window fills at chunk 4 and slides twice); the oracle checks
    first / last 32 rows + every 23rd row of every layer and stream, under the flat north_star bar."""
    def rows_of(n):
        return sorted(set(list(range(min(32, n))) + list(range(max(0, n - 32), n)) + list(range(0, n, 23))))
    _layers_scene(synth.get_config("vl3b"), L=4, B=4, n_chunks=6, rows_of=rows_of)


def _layers_scene(cfg, L, B, n_chunks, rows_of):
    from paper_2606_19849_b200 import vcs
    T, bf = cfg.T, torch.bfloat16
    n_pages = 1 + B * n_chunks + 2
    ids = [int(p) for p in synth.gen_page_ids(n_pages, 1 + B * n_chunks, 11)]
    sink_page, chunk_pages = ids[0], [[ids[1 + b * n_chunks + t] for t in range(n_chunks)] for b in range(B)]
    pools = [vcs.KVPool(n_pages, cfg.page_cap, cfg.Hq, cfg.Hkv, cfg.d, bf, cfg.rope_theta, cfg.rope_sections) for _ in range(L)]
    ostreams = [[vo.OracleStream(cfg.Hq, cfg.Hkv, cfg.d, cfg.rope_theta, cfg.rope_sections, cfg.G, cfg.Hg, cfg.Wg, cfg.tau, cfg.W)
                 for _ in range(B)] for _ in range(L)]
    ws_app1 = vcs.workspace(vcs.vcs_kv_append_workspace_bytes(pools[0], T))
    rng = np.random.default_rng(3)
    i = torch.arange(cfg.sink, dtype=torch.int32, device="cuda")
    spos = torch.stack([i, i, i], 1).contiguous()
    for l in range(L):                                   # one sink page per layer, shared by the B streams
        sK = synth.bf16_round(rng.standard_normal((cfg.sink, cfg.Hkv, cfg.d)).astype(np.float32))
        sV = synth.bf16_round(rng.standard_normal((cfg.sink, cfg.Hkv, cfg.d)).astype(np.float32))
        vcs.vcs_kv_append_pages(pools[l], dev(sK, "bf16"), dev(sV, "bf16"), spos, None, cfg.sink, sink_page, 0, ws_app1)
        for b in range(B):
            ostreams[l][b].add_sink(sink_page, sK, sV)
    z = torch.empty((B, cfg.G, cfg.P, cfg.D), dtype=bf, device="cuda")
    q = torch.empty((L, B, T, cfg.Hq, cfg.d), dtype=bf, device="cuda")
    k = torch.empty((L, B, T, cfg.Hkv, cfg.d), dtype=bf, device="cuda")
    v = torch.empty_like(k)
    out = torch.zeros_like(q)
    kidx = torch.zeros((B, T), dtype=torch.int32, device="cuda")
    kcnt = torch.zeros((B,), dtype=torch.int32, device="cuda")
    pos3 = torch.zeros((B, T, 3), dtype=torch.int32, device="cuda")
    status = torch.zeros(1, dtype=torch.int32, device="cuda")
    ws_drop = vcs.workspace(vcs.vcs_temporal_drop_workspace_bytes(B, cfg.G, cfg.P))
    ws_app = vcs.workspace(vcs.vcs_kv_append_batched_workspace_bytes(pools[0], T, B))
    ws_attn = vcs.workspace(vcs.vcs_bounded_prefill_attn_workspace_bytes(pools[0], T, cfg.W + 1))
    step = max(cfg.G, cfg.Hg, cfg.Wg)
    pos_base = torch.zeros((B,), dtype=torch.int32, device="cuda")
    page_ids = torch.zeros((B,), dtype=torch.int32, device="cuda")
    tables = torch.full((B, cfg.W + 1), -1, dtype=torch.int32, device="cuda")
    n_vis = torch.zeros((B,), dtype=torch.int32, device="cuda")
    call = vcs.make_multi_call(pools, z, q, k, v, out, kidx, kcnt, pos3, pos_base, page_ids, tables, n_vis, cfg.Hg, cfg.Wg,
                               cfg.tau, ws_drop, ws_app, ws_attn, status)
    graph = None
    for t in range(n_chunks):
        Zs = [synth.gen_hidden_chunk(cfg, t, b)[0] for b in range(B)]
        qkv = [[synth.gen_qkv(cfg.with_(seed=100 + l), t, T, b) for b in range(B)] for l in range(L)]
        z.copy_(torch.stack([dev(Zb, "bf16") for Zb in Zs]))
        for l in range(L):
            for b in range(B):
                q[l, b].copy_(dev(qkv[l][b][0], "bf16")); k[l, b].copy_(dev(qkv[l][b][1], "bf16")); v[l, b].copy_(dev(qkv[l][b][2], "bf16"))
        vis = [[sink_page] + chunk_pages[b][max(0, t - cfg.W):t] for b in range(B)]
        tables.copy_(i32([vb + [-1] * (cfg.W + 1 - len(vb)) for vb in vis]))
        n_vis.copy_(i32([len(vb) for vb in vis]))
        page_ids.copy_(i32([chunk_pages[b][t] for b in range(B)]))
        pos_base.fill_(cfg.sink + step * t)
        if t < n_chunks - 1:
            vcs.vcs_ingest_layers(pools, call)
        else:
            # last chunk: record the chain once, then run it from the graph (1 + 3 L launches in one replay)
            side = torch.cuda.Stream()               # the legacy default stream cannot be captured
            torch.cuda.synchronize()
            with vcs.Graph.capture(side) as graph:
                vcs.vcs_ingest_layers(pools, call, stream=side)
            out.zero_(); kcnt.zero_()
            torch.cuda.synchronize()
            graph.launch(side)
        torch.cuda.synchronize()
        assert int(status) == 0
        for b in range(B):
            for l in range(L):
                Q, K, V = qkv[l][b]
                n_gpu = int(kcnt[b])
                rows = None if rows_of is None else rows_of(n_gpu)
                r = ostreams[l][b].ingest_chunk(Zs[b], chunk_pages[b][t], lambda idx, n: (Q[:n], K[:n], V[:n]), rows=rows)
                n = r["n"]
                assert r["visible"] == vis[b]
                assert n_gpu == n and np.array_equal(kidx[b, :n].cpu().numpy(), r["kept_idx"])
                ma, rl = attn_errors(f64(out[l, b])[:n] if rows is None else f64(out[l, b])[rows], r["O"])
                # reduced synthetic grids: reading D32; the full-size configuration: the flat north_star bar
                bar = attn_max_abs_tol(r["O"]) if rows_of is None else ATTN_MAX_ABS
                assert ma <= bar and rl <= ATTN_REL_L2, (t, l, b, ma, rl)
    # the same recorded chunk again: a replay is idempotent (appends start the page afresh at offset 0)
    ref = out.clone()
    out.zero_()
    torch.cuda.synchronize()
    graph.launch(side)
    torch.cuda.synchronize()
    assert torch.equal(out, ref)


def test_graph_destroyed_while_another_is_recorded():
    """A graph handle released while the same thread records the next graph (Python rebinding `g` inside the
    `with`) must not invalidate that recording: the destroy is carried out when the recording ends
    (include/vcs.h, graph section).  Both graphs replay the same drop and give the direct call's result."""
    from paper_2606_19849_b200 import vcs
    cfg = synth.get_config("tiny")
    Z, _ = synth.gen_hidden_chunk(cfg, 0)
    z = dev(Z, "bf16").unsqueeze(0).contiguous()
    T = cfg.T
    ws = vcs.workspace(vcs.vcs_temporal_drop_workspace_bytes(1, cfg.G, cfg.P))
    ref_idx = torch.full((1, T), -7, dtype=torch.int32, device="cuda")
    ref_cnt = torch.zeros((1,), dtype=torch.int32, device="cuda")
    vcs.vcs_temporal_drop(z, cfg.tau, ref_idx, ref_cnt, ws)
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    g = None
    for rep in range(3):
        idx = torch.full((1, T), -7, dtype=torch.int32, device="cuda")
        cnt = torch.zeros((1,), dtype=torch.int32, device="cuda")
        torch.cuda.synchronize()
        with vcs.Graph.capture(side) as g:                    # the previous graph dies here, inside the capture
            vcs.vcs_temporal_drop(z, cfg.tau, idx, cnt, ws, stream=side)
            vcs.vcs_temporal_drop(z, cfg.tau, idx, cnt, ws, stream=side)
        g.launch(side)
        side.synchronize()
        assert int(cnt) == int(ref_cnt) and torch.equal(idx, ref_idx), rep
