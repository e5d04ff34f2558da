"""GPU parity of the one-call forms of the hot path: vcs_chunk_ingest_host (host buffers in and out,
one stream) and vcs_chunk_upload / vcs_chunk_ingest / vcs_chunk_download (copy halves on their own
streams) against the oracle stream, chunk by chunk."""
import ctypes as C

import numpy as np
import pytest
import torch

import oracle as vo
import synth
from helpers import ATTN_MAX_ABS, ATTN_REL_L2, attn_errors, dev, f64

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("split_streams", [False, True])
def test_chunk_ingest_host_forms(split_streams):
    from paper_2606_19849_b200 import vcs
    L = vcs.lib()
    cfg = synth.get_config("vl3b").with_(Hg=9, Wg=13, D=512, n_chunks=4, W=2)
    T, bf = cfg.T, torch.bfloat16
    pages = [int(p) for p in synth.gen_page_ids(12, cfg.n_chunks + 1, 3)]
    pool = vcs.KVPool(12, cfg.page_cap, cfg.Hq, cfg.Hkv, cfg.d, bf, cfg.rope_theta, cfg.rope_sections)
    os_ = vo.OracleStream(cfg.Hq, cfg.Hkv, cfg.d, cfg.rope_theta, cfg.rope_sections, cfg.G, cfg.Hg, cfg.Wg, cfg.tau, cfg.W)
    ws_app = vcs.workspace(vcs.vcs_kv_append_workspace_bytes(pool, T))
    status = torch.zeros(1, dtype=torch.int32, device="cuda")
    sK, sV = synth.gen_sink_kv(cfg)
    i = torch.arange(cfg.sink, dtype=torch.int32, device="cuda")
    vcs.vcs_kv_append_pages(pool, dev(sK, "bf16"), dev(sV, "bf16"), torch.stack([i, i, i], 1).contiguous(), None, cfg.sink,
                            pages[0], 0, ws_app, status)
    os_.add_sink(pages[0], sK, sV)
    ws_drop = vcs.workspace(vcs.vcs_temporal_drop_workspace_bytes(1, cfg.G, cfg.P))
    ws_attn = vcs.workspace(vcs.vcs_bounded_prefill_attn_workspace_bytes(pool, T, cfg.W + 1))
    z_d = torch.empty((cfg.G, cfg.P, cfg.D), dtype=bf, device="cuda")
    q_d = torch.empty((T, cfg.Hq, cfg.d), dtype=bf, device="cuda")
    k_d = torch.empty((T, cfg.Hkv, cfg.d), dtype=bf, device="cuda")
    v_d = torch.empty_like(k_d)
    out_d = torch.zeros_like(q_d)
    kidx = torch.zeros((T,), dtype=torch.int32, device="cuda")
    kcnt = torch.zeros((1,), dtype=torch.int32, device="cuda")
    pos3 = torch.zeros((T, 3), dtype=torch.int32, device="cuda")
    out_h = torch.zeros((T, cfg.Hq, cfg.d), dtype=bf).pin_memory()
    idx_h = torch.zeros((T,), dtype=torch.int32).pin_memory()
    cnt_h = torch.zeros((1,), dtype=torch.int32).pin_memory()
    step = max(cfg.G, cfg.Hg, cfg.Wg)
    s_main = torch.cuda.current_stream()
    s_up, s_dn = torch.cuda.Stream(), torch.cuda.Stream()
    for t in range(cfg.n_chunks):
        Z, _ = synth.gen_hidden_chunk(cfg, t)
        Q, K, V = synth.gen_qkv(cfg, t, T)
        hz, hq, hk, hv = (synth.to_torch(a, "bf16").pin_memory() for a in (Z, Q, K, V))
        vis = [pages[0]] + pages[1 + max(0, t - cfg.W):1 + t]
        tab = torch.tensor(vis + [-1] * (cfg.W + 1 - len(vis)), dtype=torch.int32, device="cuda")
        nvis = torch.tensor([len(vis)], dtype=torch.int32, device="cuda")
        base = torch.tensor([cfg.sink + step * t], dtype=torch.int32, device="cuda")
        call = vcs.make_chunk_call(pool, z_d, q_d, k_d, v_d, out_d, kidx, kcnt, pos3, base, tab, nvis, pages[1 + t],
                                   cfg.Hg, cfg.Wg, cfg.tau, ws_drop, ws_app, ws_attn, status)
        if not split_streams:
            vcs.vcs_chunk_ingest_host(pool, call, hz, hq, hk, hv, out_h, idx_h, cnt_h)
        else:
            s_up.wait_stream(s_main)
            rc = L.vcs_chunk_upload(pool.ref, C.byref(call), hz.data_ptr(), hq.data_ptr(), hk.data_ptr(), hv.data_ptr(),
                                    C.c_void_p(s_up.cuda_stream))
            s_main.wait_stream(s_up)
            vcs.vcs_chunk_ingest(pool, call)
            s_dn.wait_stream(s_main)
            rc |= L.vcs_chunk_download(pool.ref, C.byref(call), out_h.data_ptr(), idx_h.data_ptr(), cnt_h.data_ptr(),
                                       C.c_void_p(s_dn.cuda_stream))
            assert rc == 0
            s_main.wait_stream(s_dn)
        torch.cuda.synchronize()
        r = os_.ingest_chunk(Z, pages[1 + t], lambda idx, n: (Q[:n], K[:n], V[:n]))
        n = r["n"]
        assert int(cnt_h) == n and np.array_equal(idx_h[:n].numpy(), r["kept_idx"])
        assert r["visible"] == vis
        ma, rl = attn_errors(f64(out_h)[:n], r["O"])
        assert ma <= ATTN_MAX_ABS and rl <= ATTN_REL_L2, (t, ma, rl)
    assert int(status) == 0


def test_stage_overlap_schedule_matches_oracle():
    """bench.py's headline schedule: drop + append of chunk t+1 on a second stream under the attention
    of chunk t (double-buffered kept_idx / kept_count / pos3 / drop workspace, events for the two
    dependencies).  No host sync inside the loop; every chunk's results are checked afterwards."""
    from paper_2606_19849_b200 import vcs
    cfg = synth.get_config("vl3b").with_(Hg=9, Wg=13, D=512, n_chunks=7, W=2)
    T, bf, n_ch = cfg.T, torch.bfloat16, cfg.n_chunks
    ring = [int(p) for p in synth.gen_page_ids(12, cfg.W + 5, 4)]       # sink + W + 4 ring pages
    sink_page, ring = ring[0], ring[1:]
    R = len(ring)
    pool = vcs.KVPool(12, cfg.page_cap, cfg.Hq, cfg.Hkv, cfg.d, bf, cfg.rope_theta, cfg.rope_sections)
    os_ = vo.OracleStream(cfg.Hq, cfg.Hkv, cfg.d, cfg.rope_theta, cfg.rope_sections, cfg.G, cfg.Hg, cfg.Wg, cfg.tau, cfg.W)
    ws_app = vcs.workspace(vcs.vcs_kv_append_workspace_bytes(pool, T))
    ws_attn = vcs.workspace(vcs.vcs_bounded_prefill_attn_workspace_bytes(pool, T, cfg.W + 1))
    status = torch.zeros(1, dtype=torch.int32, device="cuda")
    sK, sV = synth.gen_sink_kv(cfg)
    i = torch.arange(cfg.sink, dtype=torch.int32, device="cuda")
    vcs.vcs_kv_append_pages(pool, dev(sK, "bf16"), dev(sV, "bf16"), torch.stack([i, i, i], 1).contiguous(), None, cfg.sink,
                            sink_page, 0, ws_app, status)
    os_.add_sink(sink_page, sK, sV)
    sets = [dict(kidx=torch.zeros((1, T), dtype=torch.int32, device="cuda"), kcnt=torch.zeros(1, dtype=torch.int32, device="cuda"),
                 pos3=torch.zeros((1, T, 3), dtype=torch.int32, device="cuda"),
                 ws=vcs.workspace(vcs.vcs_temporal_drop_workspace_bytes(1, cfg.G, cfg.P))) for _ in range(2)]
    ins = []
    for t in range(n_ch):
        Z, _ = synth.gen_hidden_chunk(cfg, t)
        Q, K, V = synth.gen_qkv(cfg, t, T)
        ins.append((Z, Q, K, V, dev(Z, "bf16")[None], dev(Q, "bf16"), dev(K, "bf16"), dev(V, "bf16")))
    outs = [torch.zeros((T, cfg.Hq, cfg.d), dtype=bf, device="cuda") for _ in range(n_ch)]
    kept = [torch.zeros((T,), dtype=torch.int32, device="cuda") for _ in range(n_ch)]
    cnts = torch.zeros((n_ch,), dtype=torch.int32, device="cuda")
    step = max(cfg.G, cfg.Hg, cfg.Wg)
    bases = (cfg.sink + step * torch.arange(n_ch, dtype=torch.int32)).cuda()
    tabs, nvis = [], []
    for t in range(n_ch):
        vis = [sink_page] + [ring[j % R] for j in range(max(0, t - cfg.W), t)]
        tabs.append(torch.tensor(vis + [-1] * (cfg.W + 1 - len(vis)), dtype=torch.int32, device="cuda"))
        nvis.append(torch.tensor([len(vis)], dtype=torch.int32, device="cuda"))
    main, side = torch.cuda.current_stream(), torch.cuda.Stream()
    side.wait_stream(main)
    ev_side, ev_attn = {}, {}
    for t in range(n_ch):
        s = sets[t % 2]
        if t - 2 in ev_attn:
            side.wait_event(ev_attn[t - 2])
        with torch.cuda.stream(side):
            vcs.vcs_temporal_drop(ins[t][4], cfg.tau, s["kidx"], s["kcnt"], s["ws"], pos3=s["pos3"], Hg=cfg.Hg, Wg=cfg.Wg,
                                  pos_base=bases[t:t + 1])
            vcs.vcs_kv_append_pages(pool, ins[t][6], ins[t][7], s["pos3"][0], s["kcnt"], T, ring[t % R], 0, ws_app, status)
            ev_side[t] = torch.cuda.Event(); ev_side[t].record(side)
        main.wait_event(ev_side[t])
        vcs.vcs_bounded_prefill_attn(pool, ins[t][5], s["pos3"][0], s["kcnt"], T, tabs[t], nvis[t], cfg.W + 1, ring[t % R], 0,
                                     outs[t], ws_attn, status=status)
        kept[t].copy_(s["kidx"][0], non_blocking=True)
        cnts[t:t + 1].copy_(s["kcnt"], non_blocking=True)
        ev_attn[t] = torch.cuda.Event(); ev_attn[t].record(main)
    torch.cuda.synchronize()
    assert int(status) == 0
    for t in range(n_ch):
        Z, Q, K, V = ins[t][:4]
        r = os_.ingest_chunk(Z, ring[t % R] + 100 * (t // R), lambda idx, n: (Q[:n], K[:n], V[:n]))
        n = r["n"]
        assert int(cnts[t]) == n and np.array_equal(kept[t][:n].cpu().numpy(), r["kept_idx"]), t
        ma, rl = attn_errors(f64(outs[t])[:n], r["O"])
        assert ma <= ATTN_MAX_ABS and rl <= ATTN_REL_L2, (t, ma, rl)
