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
