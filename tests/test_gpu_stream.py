"""GPU parity of the whole per-chunk path through the driver: drop -> append -> bounded prefill
for consecutive chunks (Tiny: every chunk, every row, fp32; 3B-shaped: reduced grid, bf16), and
the query-time path (retrieval -> query prefill) on a scattered bank."""
import numpy as np
import pytest
import torch

import oracle as vo
import synth
from helpers import ATTN_MAX_ABS, ATTN_REL_L2, F32_MAX_ABS, attn_errors, dev, f64, i32, tdtype

pytestmark = pytest.mark.gpu


def _streams(cfg, n_pool_pages, attn_flags=0, W=None):
    from paper_2606_19849_b200 import VideoStream, vcs
    W = cfg.W if W is None else W
    pages = [int(p) for p in synth.gen_page_ids(n_pool_pages, cfg.n_chunks + 2, cfg.seed)]
    pool = vcs.KVPool(n_pool_pages, cfg.page_cap, cfg.Hq, cfg.Hkv, cfg.d, tdtype(cfg.dtype), cfg.rope_theta,
                      cfg.rope_sections)
    gs = VideoStream(pool, cfg.G, cfg.Hg, cfg.Wg, cfg.D, cfg.tau, W, pages[0], pages[1:cfg.n_chunks + 1], cfg.sink,
                     t_stride=cfg.t_stride, attn_flags=attn_flags)
    os_ = vo.OracleStream(cfg.Hq, cfg.Hkv, cfg.d, cfg.rope_theta, cfg.rope_sections, cfg.G, cfg.Hg, cfg.Wg, cfg.tau,
                          W, cfg.t_stride)
    sK, sV = synth.gen_sink_kv(cfg)
    gs.add_sink(dev(sK, cfg.dtype), dev(sV, cfg.dtype))
    os_.add_sink(pages[0], sK, sV)
    return pool, gs, os_, pages


def test_tiny_stream_every_chunk_every_row():
    """BASELINE config 1: fp32, 6 chunks, projections as random N(0, 0.02) matrices (harness-side
    torch matmul = boundary step a4), plus the 'sharp' variant (Q/K std x7, logit std ~2.5) of SURVEY 8(c)."""
    cfg = synth.get_config("tiny")
    Z = synth.gen_hidden_tiny(cfg)
    for sharp in (1.0, 7.0):
        Wq, Wk, Wv = synth.gen_proj_weights_tiny(cfg)
        Wq, Wk = (Wq * sharp).astype(np.float32), (Wk * sharp).astype(np.float32)
        pool, gs, os_, pages = _streams(cfg, 16)
        Wq_d, Wk_d, Wv_d = dev(Wq, "f32"), dev(Wk, "f32"), dev(Wv, "f32")
        out = torch.zeros((cfg.T, cfg.Hq, cfg.d), dtype=torch.float32, device="cuda")
        lse = torch.zeros((cfg.Hq, cfg.T), dtype=torch.float32, device="cuda")
        for t in range(cfg.n_chunks):
            zt = dev(Z[t], "f32")

            def qkv_gpu(kept_idx, kept_count, zt=zt):
                X = zt.view(cfg.T, cfg.D).index_select(0, kept_idx.clamp(min=0).long())
                return ((X @ Wq_d).view(cfg.T, cfg.Hq, cfg.d), (X @ Wk_d).view(cfg.T, cfg.Hkv, cfg.d),
                        (X @ Wv_d).view(cfg.T, cfg.Hkv, cfg.d))

            def qkv_ref(idx, n, t=t):
                X = Z[t].reshape(cfg.T, cfg.D)[idx].astype(np.float64)
                return ((X @ Wq.astype(np.float64)).reshape(n, cfg.Hq, cfg.d),
                        (X @ Wk.astype(np.float64)).reshape(n, cfg.Hkv, cfg.d),
                        (X @ Wv.astype(np.float64)).reshape(n, cfg.Hkv, cfg.d))

            gs.ingest_chunk(zt, qkv_gpu, out, lse)
            r = os_.ingest_chunk(Z[t], pages[1 + t], qkv_ref)
            torch.cuda.synchronize()
            n = r["n"]
            assert int(gs.kept_count) == n
            assert np.array_equal(gs.kept_idx[0, :n].cpu().numpy(), r["kept_idx"])
            assert np.array_equal(gs.pos3[0, :n].cpu().numpy(), r["pos3"])
            ma, rl = attn_errors(f64(out)[:n], r["O"])
            # fp32 projections on the GPU vs fp64 in the oracle add ~1e-6 to Q/K/V themselves
            assert ma <= F32_MAX_ABS * (1.0 if sharp == 1.0 else 5.0), (t, sharp, ma)
            assert np.max(np.abs(f64(lse)[:, :n] - r["lse"])) <= 1e-3
        assert int(gs.status) == 0


@pytest.mark.parametrize("attn_flags", [pytest.param(1, id="simt"), pytest.param(0, id="auto")])
def test_vl3b_shaped_stream_reduced_grid(attn_flags):
    """3B-shaped layer (16/2 heads, d 128, bf16, W=4, sink 64) on a reduced grid so that the fp64
    oracle covers every row of 7 consecutive chunks (window slides past the stream start)."""
    cfg = synth.get_config("vl3b").with_(Hg=9, Wg=13, D=512, n_chunks=7)
    pool, gs, os_, pages = _streams(cfg, 24, attn_flags)
    out = torch.zeros((cfg.T, cfg.Hq, cfg.d), dtype=torch.bfloat16, device="cuda")
    worst = (0.0, 0.0)
    for t in range(cfg.n_chunks):
        Zt, _ = synth.gen_hidden_chunk(cfg, t)
        Q, K, V = synth.gen_qkv(cfg, t, cfg.T)
        Qd, Kd, Vd = dev(Q, "bf16"), dev(K, "bf16"), dev(V, "bf16")
        gs.ingest_chunk(dev(Zt, "bf16"), lambda idx, cnt: (Qd, Kd, Vd), out)
        r = os_.ingest_chunk(Zt, pages[1 + t], lambda idx, n: (Q[:n], K[:n], V[:n]))
        torch.cuda.synchronize()
        n = r["n"]
        assert int(gs.kept_count) == n and np.array_equal(gs.kept_idx[0, :n].cpu().numpy(), r["kept_idx"])
        assert r["visible"] == [pages[0]] + pages[1 + max(0, t - cfg.W):1 + t]
        ma, rl = attn_errors(f64(out)[:n], r["O"])
        assert ma <= ATTN_MAX_ABS and rl <= ATTN_REL_L2, (t, ma, rl)
        worst = (max(worst[0], ma), max(worst[1], rl))
    assert int(gs.status) == 0
    print("vl3b-shaped stream worst max-abs %.3e rel-L2 %.3e" % worst)


def test_full_history_vs_bounded_window():
    """Config 4 in miniature: W = inf sees every earlier chunk, W = 2 only the last two."""
    cfg = synth.get_config("sweep").with_(Hg=6, Wg=10, D=256, n_chunks=6)
    for W in (-1, 2):
        pool, gs, os_, pages = _streams(cfg, 16, W=W)
        out = torch.zeros((cfg.T, cfg.Hq, cfg.d), dtype=torch.bfloat16, device="cuda")
        for t in range(cfg.n_chunks):
            Zt, _ = synth.gen_hidden_chunk(cfg, t)
            Q, K, V = synth.gen_qkv(cfg, t, cfg.T)
            Qd, Kd, Vd = dev(Q, "bf16"), dev(K, "bf16"), dev(V, "bf16")
            gs.ingest_chunk(dev(Zt, "bf16"), lambda idx, cnt: (Qd, Kd, Vd), out)
            r = os_.ingest_chunk(Zt, pages[1 + t], lambda idx, n: (Q[:n], K[:n], V[:n]))
            torch.cuda.synchronize()
            assert len(r["visible"]) == 1 + (t if W < 0 else min(t, 2))
            ma, rl = attn_errors(f64(out)[:r["n"]], r["O"])
            assert ma <= ATTN_MAX_ABS and rl <= ATTN_REL_L2, (W, t, ma, rl)


def test_query_path_scattered_bank():
    """Config 5 in miniature: 48 text tokens, sink + recent 4 + top-8 of a 40-page scattered bank."""
    from paper_2606_19849_b200 import QueryPath, vcs
    cfg = synth.get_config("ttft")
    n_bank, k, recent, nq = 40, 8, 4, synth.configs.TTFT_NQ
    page_cap = 384
    pages = [int(p) for p in synth.gen_page_ids(64, n_bank + 2, 5)]
    pool = vcs.KVPool(64, page_cap, cfg.Hq, cfg.Hkv, cfg.d, torch.bfloat16, cfg.rope_theta, cfg.rope_sections)
    os_ = vo.OracleStream(cfg.Hq, cfg.Hkv, cfg.d, cfg.rope_theta, cfg.rope_sections, cfg.G, cfg.Hg, cfg.Wg, cfg.tau, cfg.W)
    ws = vcs.workspace(vcs.vcs_kv_append_workspace_bytes(pool, page_cap))
    sK, sV = synth.gen_sink_kv(cfg)
    sp = vo.text_positions(0, cfg.sink)
    vcs.vcs_kv_append_pages(pool, dev(sK, "bf16"), dev(sV, "bf16"), i32(sp), None, cfg.sink, pages[0], 0, ws)
    os_.add_sink(pages[0], sK, sV)
    lens, page_kv = synth.gen_bank(cfg, n_bank, 150, page_cap)
    rng = np.random.default_rng(0)
    base = cfg.sink
    for i in range(n_bank):
        K, V = page_kv(i)
        pos = (base + rng.integers(0, 46, size=(int(lens[i]), 3))).astype(np.int32)
        vcs.vcs_kv_append_pages(pool, dev(K, "bf16"), dev(V, "bf16"), i32(pos), None, int(lens[i]), pages[1 + i], 0, ws)
        os_.pool.append(pages[1 + i], 0, K, V, pos)
        os_.chunk_pages.append(pages[1 + i])
        base += 46
    os_.pos_base = base
    Q, K, V = synth.gen_query(cfg, nq)
    text_page = pages[n_bank + 1]
    qp = QueryPath(pool, pages[0], os_.chunk_pages[-recent:], os_.chunk_pages, k, nq, text_page, base)
    out = torch.zeros((nq, cfg.Hq, cfg.d), dtype=torch.bfloat16, device="cuda")
    qp.run(dev(Q, "bf16"), dev(K, "bf16"), dev(V, "bf16"), out)
    torch.cuda.synchronize()
    r = os_.query(Q, K, V, text_page, k, recent)
    srt = np.sort(r["scores"][:-recent])[::-1]
    assert srt[k - 1] - srt[k] >= 1e-4                             # seeded gap between 8th and 9th score
    assert qp.table.cpu().tolist() == r["visible"]
    assert np.max(np.abs(f64(qp.scores) - r["scores"])) <= 1e-5 * np.max(np.abs(r["scores"])) + 1e-6
    ma, rl = attn_errors(f64(out), r["O"])
    assert ma <= ATTN_MAX_ABS and rl <= ATTN_REL_L2, (ma, rl)


def test_frame_level_mode1_stream_with_previous_chunk_reference():
    """Frame-level / consecutive dropping (mode 1) through the driver AND through the one-call
    vcs_chunk_ingest: the first group of chunk t is compared with the last group of chunk t-1 (no anchor),
    so tokens that stay static across a chunk boundary are dropped there too."""
    from paper_2606_19849_b200 import VideoStream, vcs
    cfg = synth.get_config("vl3b").with_(Hg=6, Wg=10, D=256, n_chunks=4, W=2)
    rng = np.random.default_rng(17)
    frames = np.empty((cfg.n_chunks * cfg.G, cfg.P, cfg.D), dtype=np.float32)
    frames[0] = rng.standard_normal((cfg.P, cfg.D))
    for f in range(1, frames.shape[0]):
        static = rng.random(cfg.P) < 0.6
        frames[f] = np.where(static[:, None], frames[f - 1] + 0.05 * rng.standard_normal((cfg.P, cfg.D)),
                             rng.standard_normal((cfg.P, cfg.D)))
    frames = synth.bf16_round(frames)
    Zs = frames.reshape(cfg.n_chunks, cfg.G, cfg.P, cfg.D)
    pages = [int(p) for p in synth.gen_page_ids(16, 2 * cfg.n_chunks + 2, 5)]
    pool = vcs.KVPool(16, cfg.page_cap, cfg.Hq, cfg.Hkv, cfg.d, torch.bfloat16, cfg.rope_theta, cfg.rope_sections)
    sK, sV = synth.gen_sink_kv(cfg)
    gs = VideoStream(pool, cfg.G, cfg.Hg, cfg.Wg, cfg.D, cfg.tau, cfg.W, pages[0], pages[1:cfg.n_chunks + 1], cfg.sink,
                     mode=vcs.DROP_CONSECUTIVE)
    os_ = vo.OracleStream(cfg.Hq, cfg.Hkv, cfg.d, cfg.rope_theta, cfg.rope_sections, cfg.G, cfg.Hg, cfg.Wg, cfg.tau, cfg.W,
                          mode=1)
    gs.add_sink(dev(sK, "bf16"), dev(sV, "bf16"))
    os_.add_sink(pages[0], sK, sV)
    out = torch.zeros((cfg.T, cfg.Hq, cfg.d), dtype=torch.bfloat16, device="cuda")
    out2 = torch.zeros_like(out)
    kidx2 = torch.zeros((cfg.T,), dtype=torch.int32, device="cuda")
    kcnt2 = torch.zeros((1,), dtype=torch.int32, device="cuda")
    pos2 = torch.zeros((cfg.T, 3), dtype=torch.int32, device="cuda")
    dropped_at_boundary = 0
    for t in range(cfg.n_chunks):
        Q, K, V = synth.gen_qkv(cfg, t, cfg.T)
        Qd, Kd, Vd, Zd = dev(Q, "bf16"), dev(K, "bf16"), dev(V, "bf16"), dev(Zs[t], "bf16")
        prev = gs.prev_last_group
        gs.ingest_chunk(Zd, lambda idx, cnt: (Qd, Kd, Vd), out)
        r = os_.ingest_chunk(Zs[t], pages[1 + t], lambda idx, n: (Q[:n], K[:n], V[:n]))
        torch.cuda.synchronize()
        n = r["n"]
        assert int(gs.kept_count) == n and np.array_equal(gs.kept_idx[0, :n].cpu().numpy(), r["kept_idx"])
        ma, rl = attn_errors(f64(out)[:n], r["O"])
        assert ma <= ATTN_MAX_ABS and rl <= ATTN_REL_L2, (t, ma, rl)
        if t > 0:
            dropped_at_boundary += int((~r["keep"][0]).sum())
        # the same chunk again through ONE C call (vcs_chunk_call.prev_last_group_d) into a second page
        vis = r["visible"]
        tab = i32(vis + [-1] * (cfg.W + 1 - len(vis)))
        call = vcs.make_chunk_call(pool, Zd, Qd, Kd, Vd, out2, kidx2, kcnt2, pos2, gs.pos_base[t:t + 1], tab, i32([len(vis)]),
                                   pages[cfg.n_chunks + 1 + t], cfg.Hg, cfg.Wg, cfg.tau, gs.ws_drop, gs.ws_append, gs.ws_attn,
                                   gs.status, mode=vcs.DROP_CONSECUTIVE, prev_last_group=prev)
        vcs.vcs_chunk_ingest(pool, call)
        torch.cuda.synchronize()
        assert int(kcnt2) == n and np.array_equal(kidx2[:n].cpu().numpy(), r["kept_idx"])
        ma, rl = attn_errors(f64(out2)[:n], r["O"])
        assert ma <= ATTN_MAX_ABS and rl <= ATTN_REL_L2, (t, ma, rl)
    assert dropped_at_boundary > 50 and int(gs.status) == 0
