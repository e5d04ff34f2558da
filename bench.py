#!/usr/bin/env python
"""bench.py -- per-chunk LLM-ingestion hot path of ViCoStream on B200.

A step = one pass of the whole hot path over one chunk of a running stream:
    vcs_temporal_drop -> vcs_kv_append_pages -> vcs_bounded_prefill_attn
on BASELINE.json config 2 (Qwen2.5-VL-3B-shaped layer: 16 q / 2 kv heads, d 128, hidden 2048,
chunk = 4 groups x 464 merged tokens, sink 64, window W = 4 chunks, page = 1 chunk, bf16).
Metric: visual tokens/s (pre-drop tokens of the chunk / step time).  The dominant kernel is the
bounded-prefill attention (tensor-bound); its TFLOP/s is measured live with CUDA events.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl vcs|reference]
"""
from __future__ import annotations

import argparse
import ctypes as C
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import synth  # noqa: E402

WORKLOAD = "vl3b"           # BASELINE.json configs[1]
NBUF = 16                   # rotating chunk input sets: 16 x 17.1 MB = 274 MB > 2 x L2 (126 MB)
RING = 8                    # physical pages cycled by the stream (>= W + 2)
POOL_PAGES = 24
NCU_ATTN_DRAM_BYTES = 9875712   # one ncu --set full capture of this command, see profiles/r01f_ncu_full.md


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return dict(hbm=d["hbm_gbs"], tensor=d["bf16_tflops"], tensor_sustained=d["bf16_tflops_sustained"],
                    source="measured (MEASURED_PEAKS.json)")
    return dict(hbm=6650.0, tensor=1590.0, tensor_sustained=1400.0, source="fallback (B200_PROFILING.md)")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float):
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        time.sleep(0.05)
        self.proc.terminate()
        sm, smax, reasons = [], None, set()
        rows = [r for (t, r) in self.rows if t0 <= t <= t1 + 0.05] or [r for (_, r) in self.rows[-3:]]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0])); smax = float(f[1])
            except (ValueError, IndexError):
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=smax, reasons=sorted(reasons),
                    samples=len(sm))


# --------------------------------------------------------------------------------------------
def gen_inputs(cfg, n_sets):
    """n_sets seeded chunks: hidden tokens + Q/K/V rows (T-row capacity), storage-exact float32."""
    sets = []
    for b in range(n_sets):
        Z, static = synth.gen_hidden_chunk(cfg, b)
        Q, K, V = synth.gen_qkv(cfg, b, cfg.T)
        n = cfg.P + (cfg.G - 1) * int((~static).sum())      # kept count implied by the recipe
        sets.append(dict(Z=Z, Q=Q, K=K, V=V, n=n))
    return sets


def flops_attn(cfg, n, n_hist):
    """Algorithmic attention flops of one launch: 4 d Hq sum_i vis(i), causal half counted exactly."""
    return 4.0 * cfg.d * cfg.Hq * (n * n_hist + n * (n + 1) / 2.0)


def bytes_drop(cfg, n):
    return cfg.T * cfg.D * 2 + 4 * n + 4 + 12 * n


def bytes_append(cfg, n):
    return 2 * (n * cfg.Hkv * cfg.d * 2 * 2) + 12 * n + cfg.Hkv * cfg.d * 4


def run_vcs(args, rank, world):
    import torch
    from paper_2606_19849_b200 import vcs
    L = vcs.lib()
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", 0)))
    dev = torch.device("cuda")
    cfg = synth.get_config(WORKLOAD)
    T, W = cfg.T, cfg.W
    steps, warmup = args.steps, max(args.warmup, 3)
    prefill = W + 1
    total = prefill + warmup + 2 * steps + 8  # headline pass + event-split pass (+ e2e warm-up steps)

    sets = gen_inputs(cfg, NBUF)
    bf = torch.bfloat16
    z_d = [synth.to_torch(s["Z"], "bf16").to(dev) for s in sets]
    q_d = [synth.to_torch(s["Q"], "bf16").to(dev) for s in sets]
    k_d = [synth.to_torch(s["K"], "bf16").to(dev) for s in sets]
    v_d = [synth.to_torch(s["V"], "bf16").to(dev) for s in sets]
    out_d = [torch.zeros((T, cfg.Hq, cfg.d), dtype=bf, device=dev) for _ in range(2)]

    pages = [int(p) for p in synth.gen_page_ids(POOL_PAGES, RING + 1, cfg.seed)]   # scattered ids
    sink_page, ring = pages[0], pages[1:]
    pool = vcs.KVPool(POOL_PAGES, cfg.page_cap, cfg.Hq, cfg.Hkv, cfg.d, bf, cfg.rope_theta, cfg.rope_sections)
    ws_drop = vcs.workspace(vcs.vcs_temporal_drop_workspace_bytes(1, cfg.G, cfg.P))
    ws_app = vcs.workspace(vcs.vcs_kv_append_workspace_bytes(pool, T))
    ws_attn = vcs.workspace(vcs.vcs_bounded_prefill_attn_workspace_bytes(pool, T, W + 1))
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    sK, sV = synth.gen_sink_kv(cfg)
    i = torch.arange(cfg.sink, dtype=torch.int32, device=dev)
    vcs.vcs_kv_append_pages(pool, synth.to_torch(sK, "bf16").to(dev), synth.to_torch(sV, "bf16").to(dev),
                            torch.stack([i, i, i], 1).contiguous(), None, cfg.sink, sink_page, 0, ws_app, status)

    # per-step device state: visible-set tables (step a6), position bases
    tab = torch.full((RING, W + 1), -1, dtype=torch.int32)
    for r in range(RING):
        tab[r] = torch.tensor([sink_page] + [ring[(r - W + j) % RING] for j in range(W)], dtype=torch.int32)
    tab = tab.to(dev)
    n_vis_full = torch.tensor([W + 1], dtype=torch.int32, device=dev)
    n_vis_pre = torch.arange(1, W + 2, dtype=torch.int32, device=dev)           # stream start: clipped window
    step_pos = max(cfg.G * cfg.t_stride, cfg.Hg, cfg.Wg)
    pos_base = (cfg.sink + step_pos * torch.arange(total, dtype=torch.int32)).to(dev)
    kept_idx = torch.zeros((T,), dtype=torch.int32, device=dev)
    kept_cnt = torch.zeros((1,), dtype=torch.int32, device=dev)
    pos3 = torch.zeros((T, 3), dtype=torch.int32, device=dev)

    def call_for(s, zt, qt, kt, vt, ot, kidx=None, kcnt=None, p3=None, wsd=None):
        wsd = ws_drop if wsd is None else wsd
        kidx = kept_idx if kidx is None else kidx
        kcnt = kept_cnt if kcnt is None else kcnt
        p3 = pos3 if p3 is None else p3
        r = s % RING
        if s < W:   # first chunks: window holds only s earlier chunks; table = sink + last s ring pages
            t = torch.tensor([sink_page] + [ring[j] for j in range(s)] + [-1] * (W - s), dtype=torch.int32, device=dev)
            nv = n_vis_pre[s:s + 1]
            keep_alive.append(t)
        else:
            t, nv = tab[r], n_vis_full
        return vcs.make_chunk_call(pool, zt, qt, kt, vt, ot, kidx, kcnt, p3, pos_base[s:s + 1], t, nv, ring[r],
                                   cfg.Hg, cfg.Wg, cfg.tau, wsd, ws_app, ws_attn, status)

    keep_alive = []
    calls = [call_for(s, z_d[s % NBUF], q_d[s % NBUF], k_d[s % NBUF], v_d[s % NBUF], out_d[s % 2]) for s in range(total)]
    stream = torch.cuda.current_stream()
    sh = C.c_void_p(stream.cuda_stream)
    pref = pool.ref
    kv_stride, q_stride = cfg.Hkv * cfg.d, cfg.Hq * cfg.d

    def launch_split(c, ev):
        """The three launches of vcs_chunk_ingest, issued one by one so events can sit between."""
        ev[0].record(stream)
        rc = L.vcs_temporal_drop(c.z_d, None, 1, c.G, c.P, c.D, c.z_dtype, c.tau, c.mode, c.kept_idx_d, c.kept_count_d,
                                 None, c.pos3_d, c.Hg, c.Wg, c.t_stride, c.pos_base_d, c.ws_drop, c.ws_drop_bytes, sh)
        ev[1].record(stream)
        rc |= L.vcs_kv_append_pages(pref, c.k_d, c.v_d, kv_stride, kv_stride, c.pos3_d, c.kept_count_d, T, c.page_id, 0,
                                    c.status_d, c.ws_append, c.ws_append_bytes, sh)
        ev[2].record(stream)
        rc |= L.vcs_bounded_prefill_attn(pref, c.q_d, q_stride, c.pos3_d, c.kept_count_d, T, c.page_table_d, c.n_vis_d,
                                         c.n_vis_cap, c.page_id, 0, 0.0, c.out_d, q_stride, None, c.attn_flags,
                                         c.status_d, c.ws_attn, c.ws_attn_bytes, sh)
        ev[3].record(stream)
        if rc != 0:
            raise RuntimeError("vcs call failed: " + L.vcs_last_error().decode())

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timed region: K steps through vcs_chunk_ingest (3 launches per step, no
    # host sync, no events between kernels), then the same K steps again with events between the
    # three kernels for the per-kernel breakdown / roofline (event records add launch gaps) -------
    for s in range(prefill + warmup):
        rc = L.vcs_chunk_ingest(pref, C.byref(calls[s]), sh)
        assert rc == 0, L.vcs_last_error()
    sampler = ClockSampler(torch.cuda.current_device())
    sampler.start()
    time.sleep(0.15)
    barrier()
    t0 = time.time()
    w0, w1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    w0.record(stream)
    for k in range(steps):
        rc = L.vcs_chunk_ingest(pref, C.byref(calls[prefill + warmup + k]), sh)
        if rc != 0:
            raise RuntimeError("vcs call failed: " + L.vcs_last_error().decode())
    w1.record(stream)
    barrier()
    total_ms = w0.elapsed_time(w1)
    # ---- stage overlap across chunks (the paper's stage-wise pipelining, on streams):
    # the token drop and the KV append of chunk t+1 run on a second stream under the attention of chunk t
    # (the page of chunk t+1 is not in chunk t's visible set: the ring holds W + 4 pages).  Two sets of
    # (kept_idx, kept_count, pos3, drop workspace); events order drop(t), append(t) -> attn(t) and
    # attn(t) -> drop(t+2) (buffer reuse).  Same kernels, same work per chunk.
    s_drop = torch.cuda.Stream()
    h_drop = C.c_void_p(s_drop.cuda_stream)
    psets = [(torch.zeros_like(kept_idx), torch.zeros_like(kept_cnt), torch.zeros_like(pos3),
              vcs.workspace(vcs.vcs_temporal_drop_workspace_bytes(1, cfg.G, cfg.P))) for _ in range(2)]

    # argument blocks and events are built before the timed region: the host only enqueues inside it
    def overlapped_call(k):
        s = prefill + warmup + steps + k
        ki_, kc_, p3_, wsd_ = psets[k % 2]
        return call_for(s, z_d[s % NBUF], q_d[s % NBUF], k_d[s % NBUF], v_d[s % NBUF], out_d[s % 2], kidx=ki_, kcnt=kc_,
                        p3=p3_, wsd=wsd_)
    ov_calls = [overlapped_call(k) for k in range(steps)]
    ov_events = [(torch.cuda.Event(), torch.cuda.Event()) for _ in range(steps)]

    def run_overlapped(first, count):
        ev_drop, ev_attn = {}, {}
        for k in range(first, first + count):
            c = ov_calls[k]
            if k - 2 in ev_attn:
                s_drop.wait_event(ev_attn[k - 2])
            rc = L.vcs_temporal_drop(c.z_d, None, 1, c.G, c.P, c.D, c.z_dtype, c.tau, c.mode, c.kept_idx_d, c.kept_count_d,
                                     None, c.pos3_d, c.Hg, c.Wg, c.t_stride, c.pos_base_d, c.ws_drop, c.ws_drop_bytes, h_drop)
            rc |= L.vcs_kv_append_pages(pref, c.k_d, c.v_d, kv_stride, kv_stride, c.pos3_d, c.kept_count_d, T, c.page_id, 0,
                                        c.status_d, c.ws_append, c.ws_append_bytes, h_drop)
            ev_drop[k] = ov_events[k][0]; ev_drop[k].record(s_drop)
            stream.wait_event(ev_drop[k])
            rc |= L.vcs_bounded_prefill_attn(pref, c.q_d, q_stride, c.pos3_d, c.kept_count_d, T, c.page_table_d, c.n_vis_d,
                                             c.n_vis_cap, c.page_id, 0, 0.0, c.out_d, q_stride, None, c.attn_flags,
                                             c.status_d, c.ws_attn, c.ws_attn_bytes, sh)
            ev_attn[k] = ov_events[k][1]; ev_attn[k].record(stream)
            if rc != 0:
                raise RuntimeError("vcs call failed: " + L.vcs_last_error().decode())

    barrier()
    o0, o1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    s_drop.wait_stream(stream)
    o0.record(stream)
    s_drop.wait_event(o0)
    th0 = time.perf_counter()
    run_overlapped(0, steps)
    host_issue_us = (time.perf_counter() - th0) * 1e6 / steps   # host time to ENQUEUE one step (no sync inside)
    o1.record(stream)
    s_drop.synchronize()
    barrier()
    t1 = time.time()
    clocks = sampler.stop(t0, t1)            # sampled over both timed passes (one-stream and overlapped)
    overlap_ms = o0.elapsed_time(o1)
    assert int(status) == 0

    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(steps)]
    for k in range(steps):
        launch_split(calls[prefill + warmup + steps + k], evs[k])
    barrier()
    t_drop = np.array([e[0].elapsed_time(e[1]) for e in evs])
    t_app = np.array([e[1].elapsed_time(e[2]) for e in evs])
    t_att = np.array([e[2].elapsed_time(e[3]) for e in evs])
    assert int(status) == 0, "device status flags set"

    # algorithmic work per step from the kept counts the stream actually produced
    ns = [sets[s % NBUF]["n"] for s in range(total)]
    fl, bd, ba = [], [], []
    for k in range(steps):
        s = prefill + warmup + steps + k
        hist = cfg.sink + sum(ns[s - W:s])
        fl.append(flops_attn(cfg, ns[s], hist)); bd.append(bytes_drop(cfg, ns[s])); ba.append(bytes_append(cfg, ns[s]))
    peaks = _peaks()
    att_tflops = float(np.mean(fl) / (np.mean(t_att) * 1e-3) / 1e12)

    # ---- end-to-end: the same steps from pinned HOST buffers through the public calls
    # vcs_chunk_upload -> vcs_chunk_ingest -> vcs_chunk_download on three streams with double-buffered
    # staging: every step's inputs cross PCIe host->device and its results device->host inside the
    # timed region; the H2D of chunk t+1 and the D2H of chunk t-1 overlap the kernels of chunk t -------
    e_steps = min(steps, 200)
    hz = [synth.to_torch(s["Z"], "bf16").pin_memory() for s in sets]
    hq = [synth.to_torch(s["Q"], "bf16").pin_memory() for s in sets]
    hk = [synth.to_torch(s["K"], "bf16").pin_memory() for s in sets]
    hv = [synth.to_torch(s["V"], "bf16").pin_memory() for s in sets]
    ho = [torch.zeros((T, cfg.Hq, cfg.d), dtype=bf).pin_memory() for _ in range(2)]
    hidx = [torch.zeros((T,), dtype=torch.int32).pin_memory() for _ in range(2)]
    hcnt = [torch.zeros((1,), dtype=torch.int32).pin_memory() for _ in range(2)]
    stage = [[torch.empty_like(z_d[0]), torch.empty_like(q_d[0]), torch.empty_like(k_d[0]), torch.empty_like(v_d[0]),
              torch.empty_like(out_d[0]), torch.zeros_like(kept_idx), torch.zeros_like(kept_cnt), torch.zeros_like(pos3)]
             for _ in range(2)]
    base_s = prefill + warmup
    ecalls = [call_for(base_s + k, *stage[k % 2][:5], kidx=stage[k % 2][5], kcnt=stage[k % 2][6], p3=stage[k % 2][7])
              for k in range(e_steps + 3)]
    s_up, s_dn = torch.cuda.Stream(), torch.cuda.Stream()
    h_up, h_dn = C.c_void_p(s_up.cuda_stream), C.c_void_p(s_dn.cuda_stream)

    def e2e_run(first, count):
        ev_up, ev_cp, ev_dn = {}, {}, {}
        for k in range(first, first + count):
            b, c = (base_s + k) % NBUF, ecalls[k]
            if k - 2 in ev_cp:
                s_up.wait_event(ev_cp[k - 2])                 # staging set k % 2 was read by chunk k-2's kernels
            rc = L.vcs_chunk_upload(pref, C.byref(c), hz[b].data_ptr(), hq[b].data_ptr(), hk[b].data_ptr(), hv[b].data_ptr(), h_up)
            ev_up[k] = torch.cuda.Event(); ev_up[k].record(s_up)
            stream.wait_event(ev_up[k])
            if k - 2 in ev_dn:
                stream.wait_event(ev_dn[k - 2])               # output set k % 2 has been copied out
            rc |= L.vcs_chunk_ingest(pref, C.byref(c), sh)
            ev_cp[k] = torch.cuda.Event(); ev_cp[k].record(stream)
            s_dn.wait_event(ev_cp[k])
            rc |= L.vcs_chunk_download(pref, C.byref(c), ho[k % 2].data_ptr(), hidx[k % 2].data_ptr(), hcnt[k % 2].data_ptr(), h_dn)
            ev_dn[k] = torch.cuda.Event(); ev_dn[k].record(s_dn)
            assert rc == 0, L.vcs_last_error()

    barrier()
    e2e_run(0, 3)                                              # warm-up
    for st_ in (s_up, s_dn):
        st_.synchronize()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    s_up.wait_stream(stream)
    e0.record(s_up)
    e2e_run(3, e_steps)
    e1.record(s_dn)
    for st_ in (s_up, s_dn):
        st_.synchronize()
    barrier()
    e2e_ms = e0.elapsed_time(e1)
    last = 3 + e_steps - 1
    assert int(hcnt[last % 2]) == ns[base_s + last], (int(hcnt[last % 2]), ns[base_s + last])
    h2d = T * cfg.D * 2 + T * cfg.Hq * cfg.d * 2 + 2 * T * cfg.Hkv * cfg.d * 2
    d2h = T * cfg.Hq * cfg.d * 2 + T * 4 + 4

    # max over ranks of the timed regions; whole-job throughput = all ranks' tokens / that time
    from paper_2606_19849_b200.replicas import aggregate_throughput
    (dev_ms, e_ms, ser_ms), (value, e2e_value, serial_value) = aggregate_throughput(
        [overlap_ms, e2e_ms, total_ms], [T * steps, T * e_steps, T * steps], world, dev)

    line = {
        "metric": "visual tokens/s per chunk prefill (drop + KV append + bounded attention, one layer)",
        "value": value, "unit": "visual tokens/s", "n_gpus": world, "steps": steps, "warmup": warmup,
        "ms_per_step": dev_ms / steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16", "data": "synthetic",
        "config": {"workload": "config2 Qwen2.5-VL-3B-shaped layer: 16q/2kv heads d128 hidden 2048, chunk 4x464 tokens, "
                               "rho 0.6 tau 0.95, sink 64, W=4, page=1 chunk, M-RoPE, steady-state stream",
                   "tokens_per_chunk": T, "kept_per_chunk_mean": float(np.mean(ns)),
                   "visible_kv_mean": float(cfg.sink + W * np.mean(ns)),
                   "l2": f"inputs rotate through {NBUF} chunk sets (274 MB > 2x L2); KV window (5 MB) is L2-resident by design",
                   "pipelining": "stage overlap across chunks as in PAPER.md:73-83: the token drop and KV append of chunk t+1 run on a "
                                 "second stream under the attention of chunk t; every chunk still passes drop -> append -> "
                                 "attention (3 launches); the one-stream figure is under 'serial'",
                   "parallelism": "replicas only" if world > 1 else "single GPU"},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": "visual tokens/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "steps": e_steps, "ms_per_step": e_ms / e_steps, "api": "vcs_chunk_upload / vcs_chunk_ingest / vcs_chunk_download on three streams, pinned host buffers, double-buffered staging"},
        "gpu_launches": 3 * steps,
        "roofline": {"bound": "tensor", "kernel": "attn_tc_kernel (vcs_bounded_prefill_attn)", "achieved": att_tflops,
                     "peak": peaks["tensor_sustained"], "unit": "TFLOP/s", "frac": att_tflops / peaks["tensor_sustained"],
                     "frac_of_burst_peak": att_tflops / peaks["tensor"],
                     "peak_source": peaks["source"] + ": sustained bf16 figure (the kernel is timed inside a long step)",
                     "traffic": NCU_ATTN_DRAM_BYTES, "traffic_source": "profiles/r01f_ncu_full.md (dram__bytes_read.sum + dram__bytes_write.sum of one attn_tc_kernel launch; K/V window and output stay in L2)",
                     "flops_per_launch": float(np.mean(fl)), "us_per_launch": float(np.mean(t_att) * 1e3),
                     "share_of_step": float(np.sum(t_att) / (np.sum(t_att) + np.sum(t_drop) + np.sum(t_app)))},
        "kernels": {
            "drop": {"us": float(np.mean(t_drop) * 1e3), "GBps": float(np.mean(bd) / (np.mean(t_drop) * 1e-3) / 1e9),
                     "frac_hbm": float(np.mean(bd) / (np.mean(t_drop) * 1e-3) / 1e9 / peaks["hbm"])},
            "append": {"us": float(np.mean(t_app) * 1e3), "GBps": float(np.mean(ba) / (np.mean(t_app) * 1e-3) / 1e9),
                       "frac_hbm": float(np.mean(ba) / (np.mean(t_app) * 1e-3) / 1e9 / peaks["hbm"])},
            "attn": {"us": float(np.mean(t_att) * 1e3), "TFLOPs": att_tflops,
                     "us_min": float(np.min(t_att) * 1e3), "us_max": float(np.max(t_att) * 1e3)}},
        "serial": {"value": serial_value, "unit": "visual tokens/s", "ms_per_step": ser_ms / steps,
                   "what": "same K steps on ONE stream through vcs_chunk_ingest (no overlap between chunks)"},
        "host_issue_us_per_step": host_issue_us,       # host time to enqueue one overlapped step (the GPU must be the slower one)
        "fps_equiv": 1000.0 * 8 / (dev_ms / steps),      # PAPER.md:81 with c = 8 frames per chunk, one layer
    }
    if rank == 0:
        if world == 1 and not args.no_extras:
            line["extras"] = extras(peaks)
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = cpu_baseline(cfg, sets, budget_s=args.cpu_budget)
        print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------------------------
def extras(peaks):
    """Side measurements reported beside the headline (not part of `value`): the HBM-bound kernels
    cold and batched (SURVEY 8d protocol: inputs rotate through > 2x L2), and the attention kernel
    on the config-3 (7B-shaped) steady-state window."""
    import torch
    from paper_2606_19849_b200 import vcs
    dev, bf = torch.device("cuda"), torch.bfloat16
    out = {}

    def timed(fn, n):
        for i in range(3):
            fn(i)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for i in range(n):
            fn(3 + i)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) * 1e-3 / n

    # (1) drop + compaction, B = 32 config-2 chunks per launch (243 MB), two input sets
    c2 = synth.get_config("vl3b")
    B = 32
    zs = [torch.randn((B, c2.G, c2.P, c2.D), device=dev, dtype=torch.float32).to(bf) for _ in range(2)]
    ki = torch.zeros((B, c2.T), dtype=torch.int32, device=dev)
    kc = torch.zeros((B,), dtype=torch.int32, device=dev)
    p3 = torch.zeros((B, c2.T, 3), dtype=torch.int32, device=dev)
    pb = torch.zeros((B,), dtype=torch.int32, device=dev)
    wsd = vcs.workspace(vcs.vcs_temporal_drop_workspace_bytes(B, c2.G, c2.P))
    t = timed(lambda i: vcs.vcs_temporal_drop(zs[i & 1], c2.tau, ki, kc, wsd, pos3=p3, Hg=c2.Hg, Wg=c2.Wg, pos_base=pb), 20)
    nbytes = B * c2.T * c2.D * 2 + int(kc.sum()) * 16 + 4 * B
    out["drop_batched_cold"] = {"B": B, "bytes": nbytes, "us": t * 1e6, "GBps": nbytes / t / 1e9,
                                "frac_hbm": nbytes / t / 1e9 / peaks["hbm"]}
    del zs

    # (2) KV append, config-3 chunk (2093 kept x 4 kv heads), 32 rotating K/V input sets and pages
    c3 = synth.get_config("vl7b")
    n3 = int(round(c3.T * (1 - c3.rho * (c3.G - 1) / c3.G)))
    NP = 34
    pool = vcs.KVPool(NP, c3.page_cap, c3.Hq, c3.Hkv, c3.d, bf, c3.rope_theta, c3.rope_sections)
    ks = [torch.randn((n3, c3.Hkv, c3.d), device=dev).to(bf) for _ in range(32)]
    vs = [torch.randn((n3, c3.Hkv, c3.d), device=dev).to(bf) for _ in range(32)]
    i3 = torch.arange(n3, dtype=torch.int32, device=dev)
    pos = torch.stack([i3 // 1196, (i3 % 1196) // 46, i3 % 46], 1).contiguous()
    wsa = vcs.workspace(vcs.vcs_kv_append_workspace_bytes(pool, n3))
    st = torch.zeros(1, dtype=torch.int32, device=dev)
    t = timed(lambda i: vcs.vcs_kv_append_pages(pool, ks[i % 32], vs[i % 32], pos, None, n3, 1 + i % 32, 0, wsa, st), 64)
    nbytes = 2 * (n3 * c3.Hkv * c3.d * 2 * 2) + 12 * n3 + c3.Hkv * c3.d * 4
    out["append_cfg3_cold"] = {"n": n3, "bytes": nbytes, "us": t * 1e6, "GBps": nbytes / t / 1e9,
                               "frac_hbm": nbytes / t / 1e9 / peaks["hbm"]}

    # (2b) batched append: B = 32 config-3 chunks per launch (275 MB of traffic), two input sets / page sets
    Bb = 32
    pool_b = vcs.KVPool(2 * Bb, c3.page_cap, c3.Hq, c3.Hkv, c3.d, bf, c3.rope_theta, c3.rope_sections)
    kb = [torch.randn((Bb, n3, c3.Hkv, c3.d), device=dev).to(bf) for _ in range(2)]
    vb = [torch.randn((Bb, n3, c3.Hkv, c3.d), device=dev).to(bf) for _ in range(2)]
    posb = pos.unsqueeze(0).expand(Bb, -1, -1).contiguous()
    pids = [torch.arange(j * Bb, (j + 1) * Bb, dtype=torch.int32, device=dev) for j in range(2)]
    wsb = vcs.workspace(vcs.vcs_kv_append_batched_workspace_bytes(pool_b, n3, Bb))
    t = timed(lambda i: vcs.vcs_kv_append_pages_batched(pool_b, kb[i & 1], vb[i & 1], posb, None, n3, pids[i & 1], wsb, st), 20)
    out["append_batched_cold"] = {"B": Bb, "bytes": nbytes * Bb, "us": t * 1e6, "GBps": nbytes * Bb / t / 1e9,
                                  "frac_hbm": nbytes * Bb / t / 1e9 / peaks["hbm"]}
    del pool_b, kb, vb

    # (3) attention on the config-3 steady-state window: sink 128 + 8 pages + causal self page
    sk = torch.randn((c3.sink, c3.Hkv, c3.d), device=dev).to(bf)
    vcs.vcs_kv_append_pages(pool, sk, sk, pos[:c3.sink].contiguous(), None, c3.sink, 0, 0, wsa, st)
    tab = torch.arange(0, c3.W + 1, dtype=torch.int32, device=dev)
    nv = torch.tensor([c3.W + 1], dtype=torch.int32, device=dev)
    nq = torch.tensor([n3], dtype=torch.int32, device=dev)
    q = torch.randn((c3.T, c3.Hq, c3.d), device=dev).to(bf)
    qp = torch.zeros((c3.T, 3), dtype=torch.int32, device=dev)
    qp[:n3] = pos
    o = torch.zeros((c3.T, c3.Hq, c3.d), dtype=bf, device=dev)
    wst = vcs.workspace(vcs.vcs_bounded_prefill_attn_workspace_bytes(pool, c3.T, c3.W + 1))
    t = timed(lambda i: vcs.vcs_bounded_prefill_attn(pool, q, qp, nq, c3.T, tab, nv, c3.W + 1, c3.W + 1, 0, o, wst, status=st), 10)
    fl = flops_attn(c3, n3, c3.sink + c3.W * n3)
    out["attn_cfg3"] = {"flops": fl, "us": t * 1e6, "TFLOPs": fl / t / 1e12, "frac_tensor": fl / t / 1e12 / peaks["tensor"]}
    assert int(st) == 0
    return out


# --------------------------------------------------------------------------------------------
def _oracle_stream(cfg, sets, n_hist_chunks):
    """Oracle stream in steady state: sink + the last W chunks appended (no attention yet)."""
    import oracle as vo
    st = vo.OracleStream(cfg.Hq, cfg.Hkv, cfg.d, cfg.rope_theta, cfg.rope_sections, cfg.G, cfg.Hg, cfg.Wg, cfg.tau,
                         cfg.W, cfg.t_stride)
    sK, sV = synth.gen_sink_kv(cfg)
    st.add_sink(0, sK, sV)
    for t in range(n_hist_chunks):
        s = sets[t % len(sets)]
        st.ingest_chunk(s["Z"], 1 + t, lambda idx, n, s=s: (s["Q"][:n], s["K"][:n], s["V"][:n]), attend=False)
    return st


def _oracle_step(cfg, st, s, page, row_frac):
    """One oracle pass over one chunk; attention on the first ceil(row_frac * n) query rows."""
    t0 = time.perf_counter()
    rows = None if row_frac >= 1.0 else list(range(max(1, int(np.ceil(row_frac * s["n"])))))
    r = st.ingest_chunk(s["Z"], page, lambda idx, n: (s["Q"][:n], s["K"][:n], s["V"][:n]), rows=rows)
    dt = time.perf_counter() - t0
    frac = 1.0 if rows is None else len(rows) / r["n"]
    return dt, frac


def _blas_threads():
    try:
        from threadpoolctl import threadpool_info
        return max([p.get("num_threads", 1) for p in threadpool_info()] or [1])
    except Exception:
        return os.cpu_count()


def cpu_baseline(cfg, sets, budget_s=15.0):
    """The oracle as it stands, timed on this host's cores on a bounded sample of the workload:
    whole chunks (every query row, every head) of the steady-state stream until ~budget_s of CPU work."""
    st = _oracle_stream(cfg, sets[:cfg.W + 1], cfg.W)
    tot, toks, n, page = 0.0, 0.0, 0, 100
    while tot < budget_s and n < 64:
        s = sets[(cfg.W + n) % len(sets)]
        dt, frac = _oracle_step(cfg, st, s, page, 1.0)
        tot += dt; toks += cfg.T * frac; n += 1; page += 1
    return {"value": toks / tot, "unit": "visual tokens/s", "cores": _blas_threads(), "kind": "oracle",
            "host_cpus": os.cpu_count(), "seconds": tot,
            "sample": f"{n} consecutive config-2 chunks in steady state (sink + W=4 history): full drop + append + "
                      f"attention on every kept query row and all 16 heads, fp64 numpy"}


def run_reference(args, rank, world):
    """--impl reference: the oracle on the host cores, same metric/config; rank 0 only.  Each step is
    a bounded SAMPLE of one steady-state config-2 chunk: the same fraction f of every stage's units
    (positions for the drop, kept tokens for the append arithmetic, evenly spaced query rows for the
    attention over the full window), f sized so that K + W steps end within ~2 minutes; the tokens
    of a step are f * T."""
    if rank != 0:
        return
    import oracle as vo
    cfg = synth.get_config(WORKLOAD)
    steps, warmup = args.steps, args.warmup
    sets = gen_inputs(cfg, min(NBUF, cfg.W + 3))
    st = _oracle_stream(cfg, sets, cfg.W)                      # sink + W history chunks
    cur = sets[cfg.W % len(sets)]
    r = st.ingest_chunk(cur["Z"], 100, lambda idx, n: (cur["Q"][:n], cur["K"][:n], cur["V"][:n]), attend=False)
    n, pos3, vis = r["n"], r["pos3"], r["visible"]
    Q, K, V = cur["Q"][:n], cur["K"][:n], cur["V"][:n]

    def sample_step(f):
        ps = max(1, int(round(f * cfg.P)))
        ns = max(1, int(round(f * n)))
        rows = sorted(set(int(x) for x in np.linspace(0, n - 1, ns)))
        t0 = time.perf_counter()
        vo.temporal_drop(cur["Z"][:, :ps, :], cfg.tau)                                     # drop + compaction
        scratch = vo.PagedKV(cfg.Hq, cfg.Hkv, cfg.d, cfg.rope_theta, cfg.rope_sections)
        scratch.append(0, 0, K[:ns], V[:ns], pos3[:ns])                                    # M-RoPE + page write + key sum
        vo.bounded_attention(st.pool, Q, pos3, vis, self_page=100, self_offset=0, rows=rows)   # full window, sampled rows
        return time.perf_counter() - t0, ps / cfg.P

    dt_cal, f_cal = sample_step(0.05)
    per_step = 120.0 / max(1, steps + warmup)
    f = min(1.0, max(1.0 / cfg.P, f_cal * per_step / max(dt_cal, 1e-4) * 0.9))
    for _ in range(warmup):
        sample_step(f)
    tot, toks = 0.0, 0.0
    for _ in range(steps):
        dt, fe = sample_step(f)
        tot += dt; toks += cfg.T * fe
    value = toks / tot
    sample = (f"each step = the fraction {f:.4f} of one steady-state config-2 chunk in every stage (drop positions, appended "
              f"tokens, evenly spaced attention rows over the full sink + W=4 window, all 16 heads); tokens scaled by it")
    print(json.dumps({
        "impl": "reference", "metric": "visual tokens/s per chunk prefill (drop + KV append + bounded attention, one layer)",
        "value": value, "unit": "visual tokens/s", "n_gpus": world, "steps": steps, "warmup": warmup,
        "ms_per_step": 1e3 * tot / max(steps, 1), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "config2 Qwen2.5-VL-3B-shaped layer (fp64 numpy oracle on host cores)"},
        "cpu_baseline": {"value": value, "unit": "visual tokens/s", "cores": _blas_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "visual tokens/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=50)
    ap.add_argument("--impl", default="vcs", choices=["vcs", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true")
    ap.add_argument("--cpu-budget", type=float, default=12.0)
    args = ap.parse_args()
    rank, world = int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))
    if args.impl == "reference":
        return run_reference(args, rank, world)
    if world > 1:
        import torch
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", 0)))
        dist.init_process_group("nccl")
    run_vcs(args, rank, world)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
