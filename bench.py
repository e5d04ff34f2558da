#!/usr/bin/env python
"""bench.py -- per-chunk LLM-ingestion hot path of ViCoStream on B200.

A step = one pass of the whole hot path over one chunk of a running stream:
    vcs_temporal_drop -> vcs_kv_append_pages -> vcs_bounded_prefill_attn (+ combine)
Headline workload: BASELINE.json configs[2] (the largest single-GPU config; `metric` names none):
Qwen2.5-VL-7B-shaped layer, 28 q / 4 kv heads, d 128, hidden 3584, 720p chunk = 4 groups x 1196 merged
tokens, sink 128, window W = 8 chunks, page = 1 chunk, bf16, run as a STREAM of consecutive chunks.
Metric: visual tokens/s (pre-drop tokens of the chunk / step time).  The dominant kernel is the
bounded-prefill attention (tensor-bound); its TFLOP/s is measured live with CUDA events.
`extras` carries config 2 (3B shape) measured the same way, config 4 (latency vs chunk index), config 5
(query-time path), the rho = 0.93 operating point of config 3, the L-layer x B-stream driver and the
HBM-bound kernels cold and batched.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl vcs|reference]
"""
from __future__ import annotations

import argparse
import ctypes as C
import hashlib
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

HEADLINE = "vl7b"           # BASELINE.json configs[2]
FRAMES_PER_CHUNK = 8        # 4 temporal groups x 2 frames (Qwen2.5-VL merges 2 frames per temporal patch)
LAYERS = {"vl3b": 36, "vl7b": 28}


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return dict(hbm=d["hbm_gbs"], tensor=d["bf16_tflops"], tensor_sustained=d["bf16_tflops_sustained"],
                    source="measured (MEASURED_PEAKS.json)")
    return dict(hbm=6650.0, tensor=1590.0, tensor_sustained=1400.0, source="fallback (B200_PROFILING.md)")


def _ncu_traffic():
    """dram__bytes_read.sum + dram__bytes_write.sum of one attention launch, from the committed ncu capture
    (profiles/attn_traffic.csv: one data row `attn_tc_cu_sha256,dram_bytes_per_launch,source`), valid only for the
    kernel source it was taken on (keyed by the sha256 of attn_tc.cu): stale captures read as null."""
    try:
        with open(os.path.join(ROOT, "profiles", "attn_traffic.csv")) as f:
            rows = [ln.strip().split(",", 2) for ln in f if ln.strip() and not ln.startswith("#")]
        rec = dict(zip(rows[0], rows[1]))
        with open(os.path.join(ROOT, "paper_2606_19849_b200", "csrc", "attn_tc.cu"), "rb") as f:
            sha = hashlib.sha256(f.read()).hexdigest()
        if rec.get("attn_tc_cu_sha256") == sha:
            return float(rec["dram_bytes_per_launch"]), rec.get("source")
        return None, "profiles/attn_traffic.csv was captured on another version of attn_tc.cu"
    except (OSError, ValueError, IndexError, KeyError):
        return None, "no capture on file"


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
        sm, smax, pw, reasons = [], None, [], set()
        rows = [r for (t, r) in self.rows if t0 <= t <= t1 + 0.05] or [r for (_, r) in self.rows[-3:]]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0])); smax = float(f[1]); pw.append(float(f[2]))
            except (ValueError, IndexError):
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=smax, reasons=sorted(reasons),
                    power_w_max=max(pw) if pw else None, samples=len(sm))


# --------------------------------------------------------------------------------------------
def flops_attn(cfg, n, n_hist):
    """Algorithmic attention flops of one launch: 4 d Hq sum_i vis(i), causal half counted exactly."""
    return 4.0 * cfg.d * cfg.Hq * (n * n_hist + n * (n + 1) / 2.0)


def bytes_drop(cfg, n):
    return cfg.T * cfg.D * 2 + 4 * n + 4 + 12 * n


def bytes_append(cfg, n):
    return 2 * (n * cfg.Hkv * cfg.d * 2 * 2) + 12 * n + cfg.Hkv * cfg.d * 4


def gen_inputs(cfg, n_sets):
    """n_sets seeded chunks: hidden tokens + Q/K/V rows (T-row capacity), storage-exact float32."""
    sets = []
    for b in range(n_sets):
        Z, static = synth.gen_hidden_chunk(cfg, b)
        Q, K, V = synth.gen_qkv(cfg, b, cfg.T)
        n = cfg.P + (cfg.G - 1) * int((~static).sum())      # kept count implied by the recipe
        sets.append(dict(Z=Z, Q=Q, K=K, V=V, n=n))
    return sets


class StreamBench:
    """A steady-state stream of one configuration through the C ABI: NBUF rotating chunk input sets (more than
    2 x L2 of inputs), a ring of RING physical pages (scattered ids), the visible-set tables of step a6 on the
    device, one vcs_chunk_call per step.  Steps run directly (4 launches each) or from a CUDA graph that holds
    one period (lcm(NBUF, RING) steps) of the chain."""

    def __init__(self, name, rho=None, nbuf=8):
        import torch
        from paper_2606_19849_b200 import vcs
        self.torch, self.vcs, self.L = torch, vcs, vcs.lib()
        cfg = synth.get_config(name)
        if rho is not None:
            cfg = cfg.with_(rho=rho)
        self.cfg, self.name = cfg, name
        dev, bf = torch.device("cuda"), torch.bfloat16
        T, W = cfg.T, cfg.W
        self.NBUF, self.RING = nbuf, 2 * W if 2 * W >= W + 2 else W + 2
        self.period = int(np.lcm(self.NBUF, self.RING))
        self.sets = gen_inputs(cfg, self.NBUF)
        self.z_d = [synth.to_torch(s["Z"], "bf16").to(dev) for s in self.sets]
        self.q_d = [synth.to_torch(s["Q"], "bf16").to(dev) for s in self.sets]
        self.k_d = [synth.to_torch(s["K"], "bf16").to(dev) for s in self.sets]
        self.v_d = [synth.to_torch(s["V"], "bf16").to(dev) for s in self.sets]
        self.out_d = [torch.zeros((T, cfg.Hq, cfg.d), dtype=bf, device=dev) for _ in range(2)]
        n_pool = self.RING + 8
        pages = [int(p) for p in synth.gen_page_ids(n_pool, self.RING + 1, cfg.seed)]   # scattered ids
        self.sink_page, self.ring = pages[0], pages[1:]
        self.pool = vcs.KVPool(n_pool, cfg.page_cap, cfg.Hq, cfg.Hkv, cfg.d, bf, cfg.rope_theta, cfg.rope_sections)
        self.ws_drop = vcs.workspace(vcs.vcs_temporal_drop_workspace_bytes(1, cfg.G, cfg.P))
        self.ws_app = vcs.workspace(vcs.vcs_kv_append_workspace_bytes(self.pool, T))
        self.ws_attn = vcs.workspace(vcs.vcs_bounded_prefill_attn_workspace_bytes(self.pool, T, W + 1))
        self.status = torch.zeros(1, dtype=torch.int32, device=dev)
        sK, sV = synth.gen_sink_kv(cfg)
        vcs.vcs_kv_append_pages(self.pool, synth.to_torch(sK, "bf16").to(dev), synth.to_torch(sV, "bf16").to(dev),
                                vcs.vcs_text_positions(0, cfg.sink, dev), None, cfg.sink, self.sink_page, 0, self.ws_app,
                                self.status)
        # visible-set tables (step a6): sink + the W previous ring pages; clipped at the stream start
        tab = torch.full((self.RING, W + 1), -1, dtype=torch.int32)
        for r in range(self.RING):
            tab[r] = torch.tensor([self.sink_page] + [self.ring[(r - W + j) % self.RING] for j in range(W)], dtype=torch.int32)
        self.tab = tab.to(dev)
        self.n_vis_full = torch.tensor([W + 1], dtype=torch.int32, device=dev)
        self.n_vis_pre = torch.arange(1, W + 2, dtype=torch.int32, device=dev)
        self.start_tabs = [torch.tensor([self.sink_page] + [self.ring[j] for j in range(s)] + [-1] * (W - s), dtype=torch.int32,
                                        device=dev) for s in range(W)]
        bases = [cfg.sink]
        for _ in range(4095):
            bases.append(vcs.vcs_next_position_base(cfg.G, cfg.Hg, cfg.Wg, bases[-1], cfg.t_stride))
        self.pos_base = torch.tensor(bases, dtype=torch.int32).to(dev)
        self.kept_idx = torch.zeros((T,), dtype=torch.int32, device=dev)
        self.kept_cnt = torch.zeros((1,), dtype=torch.int32, device=dev)
        self.pos3 = torch.zeros((T, 3), dtype=torch.int32, device=dev)
        self.stream = torch.cuda.Stream()
        self.sh = C.c_void_p(self.stream.cuda_stream)
        self._calls = {}
        self.kv_stride, self.q_stride = cfg.Hkv * cfg.d, cfg.Hq * cfg.d

    def call(self, s, bufs=None, host_rows=0):
        """vcs_chunk_call of step s (input set s % NBUF, page ring[s % RING]); cached."""
        key = (s, id(bufs), host_rows)
        if key in self._calls:
            return self._calls[key]
        cfg, W, vcs = self.cfg, self.cfg.W, self.vcs
        r, b = s % self.RING, s % self.NBUF
        if s < W:
            t, nv = self.start_tabs[s], self.n_vis_pre[s:s + 1]
        else:
            t, nv = self.tab[r], self.n_vis_full
        z, q, k, v, o = (self.z_d[b], self.q_d[b], self.k_d[b], self.v_d[b], self.out_d[s % 2]) if bufs is None else bufs
        c = vcs.make_chunk_call(self.pool, z, q, k, v, o, self.kept_idx, self.kept_cnt, self.pos3,
                                self.pos_base[s % 4096:s % 4096 + 1], t, nv, self.ring[r], cfg.Hg, cfg.Wg, cfg.tau,
                                self.ws_drop, self.ws_app, self.ws_attn, self.status, host_rows=host_rows)
        self._calls[key] = c
        return c

    def n_of(self, s):
        return self.sets[s % self.NBUF]["n"]

    def hist_of(self, s):
        W = self.cfg.W
        return self.cfg.sink + sum(self.n_of(j) for j in range(max(0, s - W), s))

    def run_direct(self, first, count):
        for s in range(first, first + count):
            rc = self.L.vcs_chunk_ingest(self.pool.ref, C.byref(self.call(s)), self.sh)
            if rc != 0:
                raise RuntimeError("vcs call failed: " + self.L.vcs_last_error().decode())

    def capture_period(self, first):
        """One period of steps (first must be >= W and a multiple of the period) recorded into a CUDA graph."""
        assert first >= self.cfg.W and first % self.period == 0
        self.torch.cuda.synchronize()
        with self.vcs.Graph.capture(self.stream) as g:
            self.run_direct(first, self.period)
        return g

    def split_pass(self, first, count):
        """The launches of vcs_chunk_ingest issued one by one with events between them (per-kernel breakdown;
        event records add launch gaps, so this pass is not the throughput figure)."""
        torch, L, cfg = self.torch, self.L, self.cfg
        evs = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(count)]
        for k in range(count):
            c, ev = self.call(first + k), evs[k]
            ev[0].record(self.stream)
            rc = L.vcs_temporal_drop(c.z_d, None, 1, c.G, c.P, c.D, c.z_dtype, c.tau, c.mode, c.kept_idx_d, c.kept_count_d,
                                     None, c.pos3_d, c.Hg, c.Wg, c.t_stride, c.pos_base_d, c.ws_drop, c.ws_drop_bytes, self.sh)
            ev[1].record(self.stream)
            rc |= L.vcs_kv_append_pages(self.pool.ref, c.k_d, c.v_d, self.kv_stride, self.kv_stride, c.pos3_d, c.kept_count_d,
                                        cfg.T, c.page_id, 0, c.status_d, c.ws_append, c.ws_append_bytes, self.sh)
            ev[2].record(self.stream)
            rc |= L.vcs_bounded_prefill_attn(self.pool.ref, c.q_d, self.q_stride, c.pos3_d, c.kept_count_d, cfg.T,
                                             c.page_table_d, c.n_vis_d, c.n_vis_cap, c.page_id, 0, 0.0, c.out_d, self.q_stride,
                                             None, c.attn_flags, c.status_d, c.ws_attn, c.ws_attn_bytes, self.sh)
            ev[3].record(self.stream)
            if rc != 0:
                raise RuntimeError("vcs call failed: " + L.vcs_last_error().decode())
        self.stream.synchronize()
        t = np.array([[e[i].elapsed_time(e[i + 1]) for i in range(3)] for e in evs])      # ms: drop, append, attention
        fl = np.array([flops_attn(cfg, self.n_of(first + k), self.hist_of(first + k)) for k in range(count)])
        bd = np.array([bytes_drop(cfg, self.n_of(first + k)) for k in range(count)])
        ba = np.array([bytes_append(cfg, self.n_of(first + k)) for k in range(count)])
        return t, fl, bd, ba

    def solo_pass(self, first, rounds=4, reps=4):
        """The drop and the append kernel each launched back to back over the steps of `rounds` periods (inputs rotate
        through the same NBUF sets as in the stream), replayed from a CUDA graph so that the host's issue rate does not
        bound the figure: device time per launch, in ms."""
        L, cfg, n = self.L, self.cfg, rounds * self.period
        calls = [self.call(first + k) for k in range(n)]

        def drops():
            for c in calls:
                L.vcs_temporal_drop(c.z_d, None, 1, c.G, c.P, c.D, c.z_dtype, c.tau, c.mode, c.kept_idx_d, c.kept_count_d,
                                    None, c.pos3_d, c.Hg, c.Wg, c.t_stride, c.pos_base_d, c.ws_drop, c.ws_drop_bytes, self.sh)

        def appends():
            for c in calls:
                L.vcs_kv_append_pages(self.pool.ref, c.k_d, c.v_d, self.kv_stride, self.kv_stride, c.pos3_d, c.kept_count_d,
                                      cfg.T, c.page_id, 0, c.status_d, c.ws_append, c.ws_append_bytes, self.sh)
        out = []
        for fn in (drops, appends):
            self.torch.cuda.synchronize()
            with self.vcs.Graph.capture(self.stream) as g:
                fn()
            g.launch(self.stream)
            out.append(self.timed(lambda: [g.launch(self.stream) for _ in range(reps)]) / (reps * n))
        # every append of this pass sees the kept count of the pass's last drop
        return out[0], out[1], bytes_append(cfg, self.n_of(first + n - 1))

    def timed(self, fn):
        """Device time (ms) of fn() on this stream, synchronised on both sides."""
        torch = self.torch
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        self.stream.synchronize()
        e0.record(self.stream)
        fn()
        e1.record(self.stream)
        self.stream.synchronize()
        return e0.elapsed_time(e1)

    def measure(self, steps, warmup, peaks, split_steps=64, min_region_s=1.0, min_samples=5):
        """warm-up, then the timed region: EXACTLY `steps` steps (whole periods replayed from the period graph plus a
        second graph holding the remaining steps % period steps), as one sample between two events; the sample is
        repeated until the samples cover at least `min_region_s` seconds (and at least `min_samples` times) so that the
        clock record spans the power regime the figure belongs to.  The figure is the MEDIAN sample; min and max are
        kept.  Then the same steps launched directly, the per-kernel split pass and the solo pass."""
        W, P = self.cfg.W, self.period
        first = ((W + warmup + P - 1) // P) * P                  # graph periods start on a multiple of the period
        self.run_direct(0, first)
        g = self.capture_period(first)
        full, rem = divmod(steps, P)
        g_rem = None
        if rem:
            self.torch.cuda.synchronize()
            with self.vcs.Graph.capture(self.stream) as g_rem:
                self.run_direct(first, rem)                      # steps first .. first + rem - 1: the head of a period

        def sample():
            for _ in range(full):
                g.launch(self.stream)
            if g_rem is not None:
                g_rem.launch(self.stream)
        for _ in range(2):
            sample()
        probe_ms = self.timed(sample)
        n_samples = int(min(4000, max(min_samples, np.ceil(min_region_s * 1e3 / max(probe_ms, 1e-3)))))
        t_region0 = time.time()
        samples = np.array([self.timed(sample) for _ in range(n_samples)])
        # the per-kernel split pass runs straight after the samples, inside the clock record, so that the attention
        # time behind `roofline` belongs to the same power regime as the throughput figure
        t, fl, bd, ba = self.split_pass(first, max(P, min(split_steps, steps)))
        t_region1 = time.time()
        graph_ms = float(np.median(samples))
        host = {}

        def direct():
            th0 = time.perf_counter()
            self.run_direct(first, steps)
            host["us"] = (time.perf_counter() - th0) * 1e6 / steps          # host time to ENQUEUE one step (no sync inside)
        direct_ms = self.timed(direct)
        host_us = host["us"]
        solo_drop, solo_append, ba_solo = self.solo_pass(first)
        self.run_direct(first, P)                                # leave pages / counts as a whole step writes them
        assert int(self.status) == 0, "device status flags set"
        n_steps = steps
        att_tflops = float(fl.mean() / (t[:, 2].mean() * 1e-3) / 1e12)
        how = "launched back to back over the rotating input sets from a CUDA graph; us_in_step = between events inside the step (adds launch gaps)"
        kern = {
            "drop": {"us": solo_drop * 1e3, "GBps": float(bd.mean() / (solo_drop * 1e-3) / 1e9),
                     "frac_hbm": float(bd.mean() / (solo_drop * 1e-3) / 1e9 / peaks["hbm"]),
                     "us_in_step": float(t[:, 0].mean() * 1e3), "how": how},
            "append": {"us": solo_append * 1e3, "GBps": float(ba_solo / (solo_append * 1e-3) / 1e9),
                       "frac_hbm": float(ba_solo / (solo_append * 1e-3) / 1e9 / peaks["hbm"]),
                       "us_in_step": float(t[:, 1].mean() * 1e3), "how": how},
            "attn": {"us": float(t[:, 2].mean() * 1e3), "TFLOPs": att_tflops, "us_min": float(t[:, 2].min() * 1e3),
                     "us_max": float(t[:, 2].max() * 1e3), "what": "attn_tc_kernel + attn_combine_kernel"}}
        kept = float(np.mean([s["n"] for s in self.sets]))
        # per-chunk flatness (north_star "per-chunk latency flat in chunk index"): attention time per
        # algorithmic flop over the steady-state steps of the split pass
        norm = t[:, 2] / fl
        flat = float((norm.max() - norm.min()) / np.median(norm))
        L_model = LAYERS[self.name]
        t_model_ms = t[:, 0].mean() + L_model * (t[:, 1].mean() + t[:, 2].mean())
        return dict(steps=n_steps, graph_ms=graph_ms, graph_ms_min=float(samples.min()), graph_ms_max=float(samples.max()),
                    samples=n_samples, region=(t_region0, t_region1), first=first, direct_ms=direct_ms, host_issue_us_per_step=host_us, kernels=kern,
                    att_tflops=att_tflops, flops_per_launch=float(fl.mean()), share_attn=float(t[:, 2].sum() / t.sum()),
                    kept_mean=kept, flatness_flops_normalised=flat,
                    model_estimate={"layers": L_model, "ms_per_chunk": float(t_model_ms),
                                    "visual_tokens_per_s": float(self.cfg.T / (t_model_ms * 1e-3)),
                                    "fps_equiv": float(1000.0 * FRAMES_PER_CHUNK / t_model_ms),
                                    "formula": "T / (t_drop + L (t_append + t_attn)) from the split pass (attention layers only; "
                                               "MLP / projections are out of scope)"},
                    graph=g)


def sustain_pass(sb, m, seconds, peaks):
    """The period graph replayed back to back for at least `seconds` seconds in ONE timed region (a stream is seconds
    long: this is the power-capped regime), with its own clock record; straight after it, while the chip is still in
    that regime, the split pass gives the attention time per launch."""
    torch = sb.torch
    g, P, T = m["graph"], sb.period, sb.cfg.T
    period_ms = m["graph_ms"] / m["steps"] * P
    n = int(max(1, np.ceil(seconds * 1e3 / period_ms)))
    sampler = ClockSampler(torch.cuda.current_device())
    sampler.start()
    time.sleep(0.1)
    t0 = time.time()
    ms = sb.timed(lambda: [g.launch(sb.stream) for _ in range(n)])
    t1 = time.time()
    t, fl, _, _ = sb.split_pass(m["first"], 4 * P)
    clocks = sampler.stop(t0, t1)
    tf = float(fl.mean() / (t[:, 2].mean() * 1e-3) / 1e12)
    return {"seconds": ms * 1e-3, "steps": n * P, "value": T * n * P / (ms * 1e-3), "unit": "visual tokens/s",
            "ms_per_step": ms / (n * P), "attn_us": float(t[:, 2].mean() * 1e3), "attn_TFLOPs": tf,
            "attn_frac_of_sustained_peak": tf / peaks["tensor_sustained"], "attn_frac_of_burst_peak": tf / peaks["tensor"],
            "clocks": clocks,
            "what": "period graph replayed back to back in one timed region; attention timed by the split pass right after it"}


def e2e_pass(sb, first, e_steps):
    """The same steps from pinned HOST buffers through the public calls vcs_chunk_upload -> vcs_chunk_ingest ->
    vcs_chunk_download on three streams with double-buffered staging: every step's inputs cross PCIe host->device
    and its results device->host inside the timed region (only the LIVE q / k / v / out rows: the caller knows the
    kept count of its synthetic chunk; host_rows); the H2D of chunk t+1 and the D2H of chunk t-1 overlap the
    kernels of chunk t."""
    torch, L, cfg = sb.torch, sb.L, sb.cfg
    T, bf = cfg.T, torch.bfloat16
    hz = [synth.to_torch(s["Z"], "bf16").pin_memory() for s in sb.sets]
    hq = [synth.to_torch(s["Q"], "bf16").pin_memory() for s in sb.sets]
    hk = [synth.to_torch(s["K"], "bf16").pin_memory() for s in sb.sets]
    hv = [synth.to_torch(s["V"], "bf16").pin_memory() for s in sb.sets]
    ho = [torch.zeros((T, cfg.Hq, cfg.d), dtype=bf).pin_memory() for _ in range(2)]
    hidx = [torch.zeros((T,), dtype=torch.int32).pin_memory() for _ in range(2)]
    hcnt = [torch.zeros((1,), dtype=torch.int32).pin_memory() for _ in range(2)]
    stage = [(torch.empty_like(sb.z_d[0]), torch.empty_like(sb.q_d[0]), torch.empty_like(sb.k_d[0]), torch.empty_like(sb.v_d[0]),
              torch.empty_like(sb.out_d[0])) for _ in range(2)]
    calls = [sb.call(first + k, bufs=stage[k % 2], host_rows=sb.n_of(first + k)) for k in range(e_steps + 3)]
    s_up, s_dn, stream = torch.cuda.Stream(), torch.cuda.Stream(), sb.stream
    h_up, h_dn = C.c_void_p(s_up.cuda_stream), C.c_void_p(s_dn.cuda_stream)
    pref = sb.pool.ref

    def run(k0, count):
        ev_cp, ev_dn = {}, {}
        for k in range(k0, k0 + count):
            b, c = (first + k) % sb.NBUF, calls[k]
            if k - 2 in ev_cp:
                s_up.wait_event(ev_cp[k - 2])                 # staging set k % 2 was read by chunk k-2's kernels
            rc = L.vcs_chunk_upload(pref, C.byref(c), hz[b].data_ptr(), hq[b].data_ptr(), hk[b].data_ptr(), hv[b].data_ptr(), h_up)
            ev_up = torch.cuda.Event(); ev_up.record(s_up)
            stream.wait_event(ev_up)
            if k - 2 in ev_dn:
                stream.wait_event(ev_dn[k - 2])               # output set k % 2 has been copied out
            rc |= L.vcs_chunk_ingest(pref, C.byref(c), sb.sh)
            ev_cp[k] = torch.cuda.Event(); ev_cp[k].record(stream)
            s_dn.wait_event(ev_cp[k])
            rc |= L.vcs_chunk_download(pref, C.byref(c), ho[k % 2].data_ptr(), hidx[k % 2].data_ptr(), hcnt[k % 2].data_ptr(), h_dn)
            ev_dn[k] = torch.cuda.Event(); ev_dn[k].record(s_dn)
            assert rc == 0, L.vcs_last_error()

    torch.cuda.synchronize()
    run(0, 3)                                                  # warm-up
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    s_up.wait_stream(stream)
    e0.record(s_up)
    run(3, e_steps)
    e1.record(s_dn)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    last = 3 + e_steps - 1
    assert int(hcnt[last % 2]) == sb.n_of(first + last), (int(hcnt[last % 2]), sb.n_of(first + last))
    n_mean = float(np.mean([sb.n_of(first + 3 + k) for k in range(e_steps)]))
    h2d = T * cfg.D * 2 + n_mean * (cfg.Hq + 2 * cfg.Hkv) * cfg.d * 2
    d2h = n_mean * cfg.Hq * cfg.d * 2 + T * 4 + 4
    return ms, h2d, d2h


def stream_summary(sb, m, peaks, clocks=None):
    """JSON block of one measured stream (used for the headline's companions in `extras`)."""
    cfg = sb.cfg
    ms = m["graph_ms"] / m["steps"]
    return {"workload": sb.name, "tokens_per_chunk": cfg.T, "kept_per_chunk_mean": m["kept_mean"],
            "kept_fraction": m["kept_mean"] / cfg.T, "visible_kv_mean": cfg.sink + cfg.W * m["kept_mean"],
            "value": cfg.T * m["steps"] / (m["graph_ms"] * 1e-3), "unit": "visual tokens/s", "ms_per_step": ms,
            "retained_tokens_per_s": m["kept_mean"] * m["steps"] / (m["graph_ms"] * 1e-3),
            "direct_launches": {"value": cfg.T * m["steps"] / (m["direct_ms"] * 1e-3), "ms_per_step": m["direct_ms"] / m["steps"],
                                "host_issue_us_per_step": m["host_issue_us_per_step"]},
            "kernels": m["kernels"], "attn_frac_of_burst_peak": m["att_tflops"] / peaks["tensor"],
            "attn_frac_of_sustained_peak": m["att_tflops"] / peaks["tensor_sustained"],
            "flatness_flops_normalised": m["flatness_flops_normalised"], "model_estimate": m["model_estimate"]}


# --------------------------------------------------------------------------------------------
def _timed_loop(torch, fn, n, warm=3):
    for i in range(warm):
        fn(i)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for i in range(n):
        fn(warm + i)
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) * 1e-3 / n


def extra_cfg4(peaks):
    """Config 4 (history sweep on the config-2 shape, chunk index 1..64): per-chunk attention latency with the
    window bounded (W = 8) and unbounded (W = inf).  PAPER.md:237 / Fig. 4: bounded stays flat, full grows.
    Flatness = (max - min) / median of time per algorithmic flop over the chunks whose window is full."""
    import torch
    from paper_2606_19849_b200 import vcs
    cfg = synth.get_config("sweep")
    dev, bf, T, N = torch.device("cuda"), torch.bfloat16, cfg.T, cfg.n_chunks
    pool = vcs.KVPool(N + 2, cfg.page_cap, cfg.Hq, cfg.Hkv, cfg.d, bf, cfg.rope_theta, cfg.rope_sections)
    ws_app = vcs.workspace(vcs.vcs_kv_append_workspace_bytes(pool, T))
    ws_att = vcs.workspace(vcs.vcs_bounded_prefill_attn_workspace_bytes(pool, T, N + 1))
    st = torch.zeros(1, dtype=torch.int32, device=dev)
    sets = gen_inputs(cfg, 4)
    qkv = [(synth.to_torch(s["Q"], "bf16").to(dev), synth.to_torch(s["K"], "bf16").to(dev), synth.to_torch(s["V"], "bf16").to(dev))
           for s in sets]
    i3 = torch.arange(T, dtype=torch.int32, device=dev)
    pos = torch.stack([i3 // cfg.P, (i3 % cfg.P) // cfg.Wg, i3 % cfg.Wg], 1).contiguous()
    sk = torch.randn((cfg.sink, cfg.Hkv, cfg.d), device=dev).to(bf)
    vcs.vcs_kv_append_pages(pool, sk, sk, pos, None, cfg.sink, 0, 0, ws_app, st)
    out = torch.zeros((T, cfg.Hq, cfg.d), dtype=bf, device=dev)
    full_tab = torch.arange(0, N + 1, dtype=torch.int32, device=dev)           # sink (page 0) + chunk pages 1..N in order
    res = {"W8": [], "Winf": []}
    ns = []
    for t in range(N):
        q, k, v = qkv[t % 4]
        n = sets[t % 4]["n"]
        ns.append(n)
        nd = torch.tensor([n], dtype=torch.int32, device=dev)
        vcs.vcs_kv_append_pages(pool, k, v, pos, nd, T, 1 + t, 0, ws_app, st)
        lo = max(0, t - 8)
        tab8 = torch.tensor([0] + list(range(1 + lo, 1 + t)) + [-1] * (9 - (1 + t - lo)), dtype=torch.int32, device=dev)
        nv8 = torch.tensor([1 + t - lo], dtype=torch.int32, device=dev)
        nvf = torch.tensor([1 + t], dtype=torch.int32, device=dev)
        for key, tab, nv, cap in (("W8", tab8, nv8, 9), ("Winf", full_tab, nvf, N + 1)):
            reps = []
            for i in range(6):            # single launches timed one by one; the median of the last five is the point
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                vcs.vcs_bounded_prefill_attn(pool, q, pos, nd, T, tab, nv, cap, 1 + t, 0, out, ws_att, status=st)
                e1.record()
                torch.cuda.synchronize()
                reps.append(e0.elapsed_time(e1))
            ms = float(np.median(reps[1:])) * 1e-3
            hist = cfg.sink + sum(ns[lo:t] if key == "W8" else ns[:t])
            res[key].append((ms * 1e6, flops_attn(cfg, n, hist), hist + n))
    assert int(st) == 0
    out_d = {}
    for key, rows in res.items():
        us, fl, vis = np.array([r[0] for r in rows]), np.array([r[1] for r in rows]), [int(r[2]) for r in rows]
        out_d[key] = {"us_per_chunk": [round(float(x), 1) for x in us], "visible_kv_tokens_last": vis[-1],
                      "TFLOPs_last": float(fl[-1] / us[-1] / 1e6)}
    us8, fl8 = np.array([r[0] for r in res["W8"]])[9:], np.array([r[1] for r in res["W8"]])[9:]
    norm = us8 / fl8
    out_d["W8"]["steady_us_median"] = float(np.median(us8))
    out_d["W8"]["flatness_flops_normalised"] = float((norm.max() - norm.min()) / np.median(norm))
    out_d["W8"]["flatness_p10_p90"] = float((np.percentile(us8, 90) - np.percentile(us8, 10)) / np.median(us8))
    out_d["growth_full_over_bounded_at_chunk_64"] = float(res["Winf"][-1][0] / np.median(us8))
    out_d["note"] = "each point = median of 5 single launches timed one by one (launch + combine included); target flatness <= 5 %"
    return out_d


def extra_cfg5(peaks):
    """Config 5 (query-time TTFT path on the 7B shape): 48 text query tokens -> retrieval scoring over a 256-page
    bank + top-8 on the device -> text-page append -> query prefill over sink 128 + recent 4 + retrieved 8
    scattered pages.  Also the scorer alone on a 4096-page bank (where it is bandwidth- rather than latency-bound)."""
    import torch
    from paper_2606_19849_b200 import QueryPath, vcs
    cfg = synth.get_config("ttft")
    dev, bf = torch.device("cuda"), torch.bfloat16
    n_bank, k, recent, nq = synth.configs.TTFT_BANK, synth.configs.TTFT_TOPK, cfg.W, synth.configs.TTFT_NQ
    n_pool = n_bank + 8
    pages = [int(p) for p in synth.gen_page_ids(n_pool, n_bank + 2, 5)]
    pool = vcs.KVPool(n_pool, cfg.page_cap, cfg.Hq, cfg.Hkv, cfg.d, bf, cfg.rope_theta, cfg.rope_sections)
    ws = vcs.workspace(vcs.vcs_kv_append_workspace_bytes(pool, cfg.page_cap))
    lens, _ = synth.gen_bank(cfg, n_bank, 1950, 2240)
    i3 = torch.arange(cfg.page_cap, dtype=torch.int32, device=dev)
    pos = torch.stack([i3 % 97, i3 % 26, i3 % 46], 1).contiguous()
    sk = torch.randn((cfg.sink, cfg.Hkv, cfg.d), device=dev).to(bf)
    vcs.vcs_kv_append_pages(pool, sk, sk, pos, None, cfg.sink, pages[0], 0, ws)
    for i in range(n_bank):
        K = torch.randn((int(lens[i]), cfg.Hkv, cfg.d), device=dev).to(bf)
        V = torch.randn((int(lens[i]), cfg.Hkv, cfg.d), device=dev).to(bf)
        vcs.vcs_kv_append_pages(pool, K, V, pos, None, int(lens[i]), pages[1 + i], 0, ws)
    bank = pages[1:1 + n_bank]
    qp = QueryPath(pool, pages[0], bank[-recent:], bank, k, nq, pages[n_bank + 1], 100000)
    Q = torch.randn((nq, cfg.Hq, cfg.d), device=dev).to(bf)
    Kq = torch.randn((nq, cfg.Hkv, cfg.d), device=dev).to(bf)
    Vq = torch.randn((nq, cfg.Hkv, cfg.d), device=dev).to(bf)
    out = torch.zeros((nq, cfg.Hq, cfg.d), dtype=bf, device=dev)
    t_path = _timed_loop(torch, lambda i: qp.run(Q, Kq, Vq, out), 50, warm=5)
    vis = [p for p in qp.table.cpu().tolist() if p >= 0]
    n_tok = int(sum(int(pool.page_len[p]) for p in vis)) + nq
    t_attn = _timed_loop(torch, lambda i: vcs.vcs_bounded_prefill_attn(pool, Q, qp.pos3, None, nq, qp.table, None, qp.table.numel(),
                                                                       qp.text_page, 0, out, qp.ws_attn), 50, warm=5)
    fl = 4.0 * cfg.d * cfg.Hq * nq * (n_tok - nq / 2.0)
    kv_bytes = n_tok * cfg.Hkv * cfg.d * 2 * 2
    res = {"query_path_us": t_path * 1e6, "what": "vcs_retrieval_score (256-page bank, top-8 on device) + text-page append + query prefill",
           "visible_tokens": n_tok, "attn_us": t_attn * 1e6, "attn_TFLOPs": fl / t_attn / 1e12,
           "attn_kv_GBps": kv_bytes / t_attn / 1e9, "attn_kv_frac_hbm": kv_bytes / t_attn / 1e9 / peaks["hbm"],
           "kv_bytes": kv_bytes, "paper_context": "TTFT < 50 ms with ur = 32 / 64 at 25 % retention on one A100 (PAPER.md:241)"}
    del qp, pool
    # scorer alone on a 4096-page bank (small pages: only k_sum / page_len matter)
    nb = 4096
    pool2 = vcs.KVPool(nb, 128, cfg.Hq, cfg.Hkv, cfg.d, bf, cfg.rope_theta, cfg.rope_sections)
    pool2.k_sum.normal_()
    pool2.page_len.fill_(100)
    cand = torch.arange(nb, dtype=torch.int32, device=dev)
    scores = torch.zeros(nb, dtype=torch.float32, device=dev)
    topk = torch.zeros(k, dtype=torch.int32, device=dev)
    wsr = vcs.workspace(vcs.vcs_retrieval_score_workspace_bytes(pool2, nb))
    t_sc = _timed_loop(torch, lambda i: vcs.vcs_retrieval_score(pool2, Q, None, nq, cand, scores, wsr, k=k, topk_pages=topk), 50, warm=5)
    by = nb * cfg.Hkv * cfg.d * 4
    res["retrieval_4096_pages"] = {"us": t_sc * 1e6, "summary_bytes": by, "GBps": by / t_sc / 1e9}
    return res


def extra_layers(name, B, peaks, chunks=6):
    """vcs_ingest_layers: the whole attention stack of the model shape (L layers, one KV pool per layer) for B
    streams per launch, the chain of 1 + 3 L launches per chunk replayed from a CUDA graph.  Q / K / V rows are
    the same buffers for every layer (layer stride 0): the kernels cannot tell, the bench saves memory."""
    import torch
    from paper_2606_19849_b200 import vcs
    cfg = synth.get_config(name)
    L, W, T = LAYERS[name], cfg.W, cfg.T
    dev, bf = torch.device("cuda"), torch.bfloat16
    ring = W + 2
    n_pages = 1 + B * ring
    pools = [vcs.KVPool(n_pages, cfg.page_cap, cfg.Hq, cfg.Hkv, cfg.d, bf, cfg.rope_theta, cfg.rope_sections) for _ in range(L)]
    sets = gen_inputs(cfg, 2)
    z = torch.stack([synth.to_torch(sets[b % 2]["Z"], "bf16") for b in range(B)]).to(dev)
    q = torch.stack([synth.to_torch(sets[b % 2]["Q"], "bf16") for b in range(B)]).to(dev)
    k = torch.stack([synth.to_torch(sets[b % 2]["K"], "bf16") for b in range(B)]).to(dev)
    v = torch.stack([synth.to_torch(sets[b % 2]["V"], "bf16") for b in range(B)]).to(dev)
    out = torch.zeros((1, B, T, cfg.Hq, cfg.d), dtype=bf, device=dev)
    kidx = torch.zeros((B, T), dtype=torch.int32, device=dev)
    kcnt = torch.zeros((B,), dtype=torch.int32, device=dev)
    pos3 = torch.zeros((B, T, 3), dtype=torch.int32, device=dev)
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    ws_drop = vcs.workspace(vcs.vcs_temporal_drop_workspace_bytes(B, cfg.G, cfg.P))
    ws_app = vcs.workspace(vcs.vcs_kv_append_batched_workspace_bytes(pools[0], T, B))
    ws_att = vcs.workspace(vcs.vcs_bounded_prefill_attn_workspace_bytes(pools[0], T, W + 1))
    ws1 = vcs.workspace(vcs.vcs_kv_append_workspace_bytes(pools[0], T))
    sk = torch.randn((cfg.sink, cfg.Hkv, cfg.d), device=dev).to(bf)
    sink_pos = vcs.vcs_text_positions(0, cfg.sink, dev)
    for p_ in pools:
        vcs.vcs_kv_append_pages(p_, sk, sk, sink_pos, None, cfg.sink, 0, 0, ws1, status)
    side = torch.cuda.Stream()
    graphs, keep = [], []
    for t in range(ring):                     # one graph per ring position (the page ids / tables are arguments)
        vis = [[0] + [1 + b * ring + (t - W + j) % ring for j in range(W)] for b in range(B)]
        tables = torch.tensor(vis, dtype=torch.int32, device=dev)
        n_vis = torch.full((B,), W + 1, dtype=torch.int32, device=dev)
        page_ids = torch.tensor([1 + b * ring + t for b in range(B)], dtype=torch.int32, device=dev)
        pos_base = torch.full((B,), cfg.sink + 46 * t, dtype=torch.int32, device=dev)
        call = vcs.make_multi_call(pools, z, q, k, v, out, kidx, kcnt, pos3, pos_base, page_ids, tables, n_vis, cfg.Hg, cfg.Wg,
                                   cfg.tau, ws_drop, ws_app, ws_att, status, share_qkv_across_layers=True)
        call.out_layer_stride = 0             # every layer writes the same output buffer (not read by anyone here)
        vcs.vcs_ingest_layers(pools, call, stream=side)          # fills the ring once, uncaptured
        side.synchronize()
        with vcs.Graph.capture(side) as g:
            vcs.vcs_ingest_layers(pools, call, stream=side)
        graphs.append(g)
        keep.append((tables, n_vis, page_ids, pos_base, call))
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for t in range(ring):
        graphs[t].launch(side)
    side.synchronize()
    e0.record(side)
    for c in range(chunks):
        graphs[c % ring].launch(side)
    e1.record(side)
    side.synchronize()
    assert int(status) == 0
    ms = e0.elapsed_time(e1) / chunks
    return {"workload": name, "layers": L, "streams_per_launch": B, "launches_per_chunk": 1 + 3 * L, "ms_per_chunk_all_streams": ms,
            "visual_tokens_per_s": B * T / (ms * 1e-3), "fps_equiv": B * 1000.0 * FRAMES_PER_CHUNK / ms,
            "what": "drop + L x (KV append + bounded prefill) per chunk through vcs_ingest_layers, CUDA-graph replay; the LLM's "
                    "MLPs / projections are out of scope (PAPER.md Table 2 'LLM prefill' 44 ms per 8-frame chunk on one A100 "
                    "includes them: context, not a like-for-like figure)"}


def extra_cold_batched(peaks):
    """The HBM-bound kernels cold and batched (SURVEY 8d protocol: B streams per launch, inputs rotate through more
    than 2 x L2): the figures compared with north_star's 70 % bar."""
    import torch
    from paper_2606_19849_b200 import vcs
    dev, bf = torch.device("cuda"), torch.bfloat16
    out = {}
    c2, B = synth.get_config("vl3b"), 32
    zs = [torch.randn((B, c2.G, c2.P, c2.D), device=dev, dtype=torch.float32).to(bf) for _ in range(2)]
    ki = torch.zeros((B, c2.T), dtype=torch.int32, device=dev)
    kc = torch.zeros((B,), dtype=torch.int32, device=dev)
    p3 = torch.zeros((B, c2.T, 3), dtype=torch.int32, device=dev)
    pb = torch.zeros((B,), dtype=torch.int32, device=dev)
    wsd = vcs.workspace(vcs.vcs_temporal_drop_workspace_bytes(B, c2.G, c2.P))
    t = _timed_loop(torch, lambda i: vcs.vcs_temporal_drop(zs[i & 1], c2.tau, ki, kc, wsd, pos3=p3, Hg=c2.Hg, Wg=c2.Wg, pos_base=pb), 20)
    nbytes = B * c2.T * c2.D * 2 + int(kc.sum()) * 16 + 4 * B
    out["drop_batched_cold"] = {"B": B, "bytes": nbytes, "us": t * 1e6, "GBps": nbytes / t / 1e9, "frac_hbm": nbytes / t / 1e9 / peaks["hbm"]}
    del zs
    c3 = synth.get_config("vl7b")
    zs = [torch.randn((B, c3.G, c3.P, c3.D), device=dev, dtype=torch.float32).to(bf) for _ in range(2)]
    ki3 = torch.zeros((B, c3.T), dtype=torch.int32, device=dev)
    p33 = torch.zeros((B, c3.T, 3), dtype=torch.int32, device=dev)
    wsd3 = vcs.workspace(vcs.vcs_temporal_drop_workspace_bytes(B, c3.G, c3.P))
    t = _timed_loop(torch, lambda i: vcs.vcs_temporal_drop(zs[i & 1], c3.tau, ki3, kc, wsd3, pos3=p33, Hg=c3.Hg, Wg=c3.Wg, pos_base=pb), 10)
    nbytes = B * c3.T * c3.D * 2 + int(kc.sum()) * 16 + 4 * B
    out["drop_batched_cold_cfg3"] = {"B": B, "bytes": nbytes, "us": t * 1e6, "GBps": nbytes / t / 1e9, "frac_hbm": nbytes / t / 1e9 / peaks["hbm"]}
    del zs, ki3, p33
    n3 = int(round(c3.T * (1 - c3.rho * (c3.G - 1) / c3.G)))
    Bb = 32
    pool_b = vcs.KVPool(2 * Bb, c3.page_cap, c3.Hq, c3.Hkv, c3.d, bf, c3.rope_theta, c3.rope_sections)
    kb = [torch.randn((Bb, n3, c3.Hkv, c3.d), device=dev).to(bf) for _ in range(2)]
    vb = [torch.randn((Bb, n3, c3.Hkv, c3.d), device=dev).to(bf) for _ in range(2)]
    i3 = torch.arange(n3, dtype=torch.int32, device=dev)
    pos = torch.stack([i3 // 1196, (i3 % 1196) // 46, i3 % 46], 1).contiguous()
    posb = pos.unsqueeze(0).expand(Bb, -1, -1).contiguous()
    pids = [torch.arange(j * Bb, (j + 1) * Bb, dtype=torch.int32, device=dev) for j in range(2)]
    wsb = vcs.workspace(vcs.vcs_kv_append_batched_workspace_bytes(pool_b, n3, Bb))
    st = torch.zeros(1, dtype=torch.int32, device=dev)
    t = _timed_loop(torch, lambda i: vcs.vcs_kv_append_pages_batched(pool_b, kb[i & 1], vb[i & 1], posb, None, n3, pids[i & 1], wsb, st), 20)
    nbytes = (2 * (n3 * c3.Hkv * c3.d * 2 * 2) + 12 * n3 + c3.Hkv * c3.d * 4) * Bb
    out["append_batched_cold"] = {"B": Bb, "bytes": nbytes, "us": t * 1e6, "GBps": nbytes / t / 1e9, "frac_hbm": nbytes / t / 1e9 / peaks["hbm"]}
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


def _blas_threads():
    try:
        from threadpoolctl import threadpool_info
        return max([p.get("num_threads", 1) for p in threadpool_info()] or [1])
    except Exception:
        return os.cpu_count()


def _oracle_sample_step(cfg, st, cur, pos3, vis, n, f):
    """The fraction f of one steady-state chunk in every stage of the oracle: drop positions, appended tokens,
    evenly spaced attention rows over the full window (all heads).  Returns (seconds, fraction of T processed,
    seconds per stage)."""
    import oracle as vo
    ps = max(1, int(round(f * cfg.P)))
    ns = max(1, int(round(f * n)))
    rows = sorted(set(int(x) for x in np.linspace(0, n - 1, ns)))
    t0 = time.perf_counter()
    vo.temporal_drop(cur["Z"][:, :ps, :], cfg.tau)
    t1 = time.perf_counter()
    scratch = vo.PagedKV(cfg.Hq, cfg.Hkv, cfg.d, cfg.rope_theta, cfg.rope_sections)
    scratch.append(0, 0, cur["K"][:ns], cur["V"][:ns], pos3[:ns])
    t2 = time.perf_counter()
    vo.bounded_attention(st.pool, cur["Q"][:n], pos3, vis, self_page=1000, self_offset=0, rows=rows)
    t3 = time.perf_counter()
    return t3 - t0, ps / cfg.P, {"drop": t1 - t0, "append": t2 - t1, "attention": t3 - t2}


def _oracle_retrieval_seconds(cfg, st, cur):
    """Eq. 3 scoring + top-k of a 48-token query over the pages the oracle stream holds (the query-time stage; it is
    not part of a chunk step, so it is timed whole, beside the per-chunk stages)."""
    import oracle as vo
    pages = list(st.chunk_pages)
    t0 = time.perf_counter()
    sc = vo.retrieval_scores(st.pool, cur["Q"][:48], pages)
    vo.retrieve_topk(sc, pages, min(8, len(pages)))
    return time.perf_counter() - t0, len(pages)


def _cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for ln in f:
                if ln.lower().startswith("model name"):
                    return ln.split(":", 1)[1].strip()
    except OSError:
        pass
    import platform
    return platform.processor() or platform.machine()


def _oracle_setup(cfg, n_sets=3):
    sets = gen_inputs(cfg, n_sets)
    st = _oracle_stream(cfg, sets, cfg.W)                      # sink + W history chunks
    cur = sets[cfg.W % len(sets)]
    r = st.ingest_chunk(cur["Z"], 1000, lambda idx, n: (cur["Q"][:n], cur["K"][:n], cur["V"][:n]), attend=False)
    return st, cur, r["pos3"], r["visible"], r["n"]


def cpu_baseline(cfg, budget_s=15.0):
    """The oracle as it stands, timed on this host's cores on a bounded sample of the headline workload; seconds per
    stage beside the blended figure (drop / append / attention per chunk sample, retrieval per query)."""
    st, cur, pos3, vis, n = _oracle_setup(cfg)
    dt_cal, f_cal, _ = _oracle_sample_step(cfg, st, cur, pos3, vis, n, 0.01)
    f = min(1.0, max(1.0 / cfg.P, f_cal * (budget_s / 4) / max(dt_cal, 1e-4)))       # second calibration: ~budget / 4 or less
    dt_cal, f_cal, _ = _oracle_sample_step(cfg, st, cur, pos3, vis, n, f)             # (the tiny first sample overstates the cost)
    f = min(1.0, max(1.0 / cfg.P, f_cal * budget_s / max(dt_cal, 1e-4) * 0.9))
    dt, fe, stages = _oracle_sample_step(cfg, st, cur, pos3, vis, n, f)
    t_ret, n_ret = _oracle_retrieval_seconds(cfg, st, cur)
    return {"value": cfg.T * fe / dt, "unit": "visual tokens/s", "cores": _blas_threads(), "kind": "oracle",
            "host_cpus": os.cpu_count(), "cpu_model": _cpu_model(), "seconds": dt,
            "stage_seconds_of_sample": {k: round(v, 4) for k, v in stages.items()},
            "stage_seconds_per_whole_chunk": {k: round(v / fe, 2) for k, v in stages.items()},
            "retrieval_seconds_per_query": round(t_ret, 6), "retrieval_pages": n_ret,
            "sample": f"the fraction {fe:.4f} of one steady-state config-3 chunk in every stage (drop positions, appended tokens, "
                      f"evenly spaced attention rows over the full sink + W=8 window, all 28 heads), fp64 numpy; tokens scaled by it; "
                      f"retrieval = one 48-token query scored against the {n_ret} chunk pages of the oracle stream"}


def run_reference(args, rank, world):
    """--impl reference: the oracle on the host cores, same metric / config; rank 0 only.  Each step is a bounded
    SAMPLE of one steady-state config-3 chunk (the same fraction f of every stage's units), f sized so that
    K + W steps end within ~2 minutes; the tokens of a step are f * T."""
    if rank != 0:
        return
    cfg = synth.get_config(HEADLINE)
    steps, warmup = args.steps, args.warmup
    st, cur, pos3, vis, n = _oracle_setup(cfg)
    dt_cal, f_cal, _ = _oracle_sample_step(cfg, st, cur, pos3, vis, n, 0.01)
    per_step = 110.0 / max(1, steps + warmup)
    f = min(1.0, max(1.0 / cfg.P, f_cal * per_step / max(dt_cal, 1e-4) * 0.9))
    for _ in range(warmup):
        _oracle_sample_step(cfg, st, cur, pos3, vis, n, f)
    tot, toks = 0.0, 0.0
    for _ in range(steps):
        dt, fe, _ = _oracle_sample_step(cfg, st, cur, pos3, vis, n, f)
        tot += dt; toks += cfg.T * fe
    value = toks / tot
    sample = (f"each step = the fraction {f:.5f} of one steady-state config-3 chunk in every stage (drop positions, appended "
              f"tokens, evenly spaced attention rows over the full sink + W=8 window, all 28 heads); tokens scaled by it")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": "visual tokens/s", "n_gpus": world, "steps": steps,
        "warmup": warmup, "ms_per_step": 1e3 * tot / max(steps, 1), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD_TEXT, "arm": "fp64 numpy oracle on the host cores (no GPU work)"},
        "cpu_baseline": {"value": value, "unit": "visual tokens/s", "cores": _blas_threads(), "kind": "oracle", "sample": sample,
                         "cpu_model": _cpu_model()},
        "e2e": {"value": value, "unit": "visual tokens/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }), flush=True)


METRIC = "visual tokens/s per chunk prefill (drop + KV append + bounded attention, one layer)"
WORKLOAD_TEXT = ("config3 Qwen2.5-VL-7B-shaped layer as a stream: 28q/4kv heads d128 hidden 3584, 720p chunk 4x1196 tokens, "
                 "rho 0.75 tau 0.95, sink 128, W=8, page=1 chunk, M-RoPE, consecutive chunks in steady state")


def run_vcs(args, rank, world):
    import torch
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", 0)))
    dev = torch.device("cuda")
    steps, warmup = args.steps, max(args.warmup, 3)
    peaks = _peaks()

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize()

    extras = (("cfg2", lambda: _extra_stream("vl3b", None, steps, warmup, peaks)),
              ("cfg3_rho093", lambda: _extra_stream("vl7b", 0.93, steps, warmup, peaks)),
              ("cfg4", lambda: extra_cfg4(peaks)), ("cfg5", lambda: extra_cfg5(peaks)),
              ("layers_cfg3_B1", lambda: extra_layers("vl7b", 1, peaks)),
              ("layers_cfg2_B4", lambda: extra_layers("vl3b", 4, peaks)),
              ("cold_batched", lambda: extra_cold_batched(peaks)))
    if args.only:
        # one companion measurement alone (what the ncu captures under profiles/ run): not a bench line
        if rank == 0:
            print(json.dumps({"only": args.only, "result": dict(extras)[args.only]()}), flush=True)
        return

    sb = StreamBench(HEADLINE)
    cfg, T = sb.cfg, sb.cfg.T
    sampler = ClockSampler(torch.cuda.current_device())
    sampler.start()
    time.sleep(0.15)
    barrier()
    t0 = time.time()
    m = sb.measure(steps, warmup, peaks)
    barrier()
    t1 = time.time()
    clocks = sampler.stop(*m["region"])                       # the clock record of the timed samples themselves
    sustained = sustain_pass(sb, m, args.sustain, peaks) if (args.sustain > 0 and world == 1) else None
    # end to end from host buffers
    first = m["first"]
    e_steps = min(m["steps"], 64)
    e2e_ms, h2d, d2h = e2e_pass(sb, first, e_steps)
    barrier()

    from paper_2606_19849_b200.replicas import aggregate_throughput
    (dev_ms, e_ms, dir_ms), (value, e2e_value, direct_value) = aggregate_throughput(
        [m["graph_ms"], e2e_ms, m["direct_ms"]], [T * m["steps"], T * e_steps, T * m["steps"]], world, dev)

    # which peak applies: the burst figure while the sampled SM clock sits at its maximum, the sustained one when the
    # clock record shows the power-capped regime (both are printed)
    # power-capped regime: the sampler saw sw_power_cap during the timed region and the SM clock below its maximum
    capped = bool(clocks.get("sm_mhz") and clocks.get("sm_max_mhz") and "sw_power_cap" in (clocks.get("reasons") or [])
                  and clocks["sm_mhz"] < 0.97 * clocks["sm_max_mhz"])
    peak_used = peaks["tensor_sustained"] if capped else peaks["tensor"]
    traffic, traffic_src = _ncu_traffic()
    ms_step = dev_ms / m["steps"]
    line = {
        "metric": METRIC, "value": value, "unit": "visual tokens/s", "n_gpus": world, "steps": m["steps"],
        "steps_requested": args.steps, "warmup": warmup, "ms_per_step": ms_step,
        "timing": {"what": "median of `samples` timed regions of exactly `steps` steps each (events on the launching stream, "
                           "synchronised on both sides), repeated to cover >= 1 s so that the clock record spans the regime",
                   "samples": m["samples"], "ms_per_step_min": m["graph_ms_min"] / m["steps"],
                   "ms_per_step_max": m["graph_ms_max"] / m["steps"], "region_s": m["region"][1] - m["region"][0]}, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16", "data": "synthetic",
        "config": {"workload": WORKLOAD_TEXT, "tokens_per_chunk": T, "kept_per_chunk_mean": m["kept_mean"],
                   "kept_fraction": m["kept_mean"] / T, "visible_kv_mean": float(cfg.sink + cfg.W * m["kept_mean"]),
                   "l2": f"inputs rotate through {sb.NBUF} chunk sets ({sb.NBUF * (T * cfg.D + T * (cfg.Hq + 2 * cfg.Hkv) * cfg.d) * 2 / 1e6:.0f} MB"
                         " > 2x L2); the KV window is L2-resident by design",
                   "launch": f"every chunk passes drop -> append -> attention -> combine (4 launches, PDL-chained, no host sync); "
                             f"the chain of one period ({sb.period} chunks) is replayed from a CUDA graph (vcs_graph_*); the figure "
                             "with direct launches is under 'direct_launches'",
                   "parallelism": "replicas only" if world > 1 else "single GPU"},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": "visual tokens/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "steps": e_steps, "ms_per_step": e_ms / e_steps,
                "h2d_GBps": h2d / (e_ms / e_steps * 1e-3) / 1e9,
                "bound_by": "the host->device copy over PCIe (hidden tokens + live Q/K/V rows); the kernels take `ms_per_step` "
                            "of the device-timed figure, the rest is the copy",
                "api": "vcs_chunk_upload / vcs_chunk_ingest / vcs_chunk_download on three streams, pinned host buffers, "
                       "double-buffered staging, live rows only (host_rows)"},
        "gpu_launches": 4 * m["steps"],
        "roofline": {"bound": "tensor", "kernel": "attn_tc_kernel (+ attn_combine_kernel) of vcs_bounded_prefill_attn",
                     "achieved": m["att_tflops"], "peak": peak_used, "unit": "TFLOP/s", "frac": m["att_tflops"] / peak_used,
                     "frac_of_burst_peak": m["att_tflops"] / peaks["tensor"],
                     "frac_of_sustained_peak": m["att_tflops"] / peaks["tensor_sustained"],
                     "peak_source": peaks["source"] + (": sustained bf16 figure (clock record shows the power-capped regime)" if capped
                                                       else ": burst bf16 figure (SM clock at its maximum during the timed region)"),
                     "traffic": traffic, "traffic_source": traffic_src,
                     "flops_per_launch": m["flops_per_launch"], "us_per_launch": m["kernels"]["attn"]["us"],
                     "share_of_step": m["share_attn"]},
        "kernels": m["kernels"],
        "retained_tokens_per_s": m["kept_mean"] / (ms_step * 1e-3) * world,
        "direct_launches": {"value": direct_value, "unit": "visual tokens/s", "ms_per_step": dir_ms / m["steps"],
                            "host_issue_us_per_step": m["host_issue_us_per_step"]},
        "flatness_flops_normalised": m["flatness_flops_normalised"],
        "model_estimate": m["model_estimate"],
        "fps_equiv_one_layer": 1000.0 * FRAMES_PER_CHUNK / ms_step,
    }
    if sustained is not None:
        line["sustained"] = sustained
    if rank == 0:
        del sb, m
        torch.cuda.empty_cache()
        if world == 1 and not args.no_extras:
            ex = {}
            for key, fn in extras:
                try:
                    ex[key] = fn()
                except Exception as e:      # an extra must never take the headline down with it
                    ex[key] = {"error": f"{type(e).__name__}: {e}"}
                torch.cuda.empty_cache()
            line["extras"] = ex
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = cpu_baseline(cfg, budget_s=args.cpu_budget)
        # the long per-chunk series go FIRST and the flat summary LAST: a reader that keeps only the tail of the line
        # still gets every scalar that matters
        series = {}
        c4 = line.get("extras", {}).get("cfg4", {})
        for key in ("W8", "Winf"):
            if isinstance(c4.get(key), dict) and "us_per_chunk" in c4[key]:
                series["cfg4_" + key + "_us_per_chunk"] = [int(round(x)) for x in c4[key].pop("us_per_chunk")]
        out = {"series": series}
        out.update(line)
        out["summary"] = _summary(line)
        print(json.dumps(out), flush=True)


def _summary(line):
    """Flat object of the scalars the headline and the extras produce (4 significant digits), last key of the line."""
    def get(d, *ks):
        for k in ks:
            if not isinstance(d, dict) or k not in d:
                return None
            d = d[k]
        return d

    def r(x):
        return float(f"{x:.4g}") if isinstance(x, (int, float)) and x == x else x
    ex, k = line.get("extras", {}), line.get("kernels", {})
    s = {
        "hdr_tokens_per_s": line["value"], "hdr_ms_per_step": line["ms_per_step"],
        "hdr_ms_per_step_min": get(line, "timing", "ms_per_step_min"), "hdr_ms_per_step_max": get(line, "timing", "ms_per_step_max"),
        "hdr_samples": get(line, "timing", "samples"), "hdr_sm_mhz": get(line, "clocks", "sm_mhz"),
        "hdr_attn_us": get(k, "attn", "us"), "hdr_attn_TFLOPs": get(k, "attn", "TFLOPs"),
        "hdr_attn_frac_burst": get(line, "roofline", "frac_of_burst_peak"),
        "hdr_attn_frac_sustained": get(line, "roofline", "frac_of_sustained_peak"),
        "hdr_flatness_flops": line.get("flatness_flops_normalised"),
        "hdr_drop_us": get(k, "drop", "us"), "hdr_drop_frac_hbm": get(k, "drop", "frac_hbm"),
        "hdr_append_us": get(k, "append", "us"), "hdr_append_frac_hbm": get(k, "append", "frac_hbm"),
        "e2e_tokens_per_s": get(line, "e2e", "value"), "e2e_h2d_GBps": get(line, "e2e", "h2d_GBps"),
        "sustain_s": get(line, "sustained", "seconds"), "sustain_tokens_per_s": get(line, "sustained", "value"),
        "sustain_attn_TFLOPs": get(line, "sustained", "attn_TFLOPs"),
        "sustain_attn_frac_sustained": get(line, "sustained", "attn_frac_of_sustained_peak"),
        "sustain_sm_mhz": get(line, "sustained", "clocks", "sm_mhz"),
        "sustain_power_cap": "sw_power_cap" in (get(line, "sustained", "clocks", "reasons") or []),
    }
    for tag, key in (("cfg2", "cfg2"), ("cfg3_rho093", "cfg3_rho093")):
        e = ex.get(key, {})
        s.update({tag + "_tokens_per_s": e.get("value"), tag + "_ms_per_step": e.get("ms_per_step"),
                  tag + "_attn_us": get(e, "kernels", "attn", "us"), tag + "_attn_TFLOPs": get(e, "kernels", "attn", "TFLOPs"),
                  tag + "_attn_frac_burst": e.get("attn_frac_of_burst_peak"),
                  tag + "_flatness_flops": e.get("flatness_flops_normalised")})
        if tag == "cfg2":
            s.update({"cfg2_drop_us": get(e, "kernels", "drop", "us"), "cfg2_drop_frac_hbm": get(e, "kernels", "drop", "frac_hbm"),
                      "cfg2_append_us": get(e, "kernels", "append", "us"),
                      "cfg2_append_frac_hbm": get(e, "kernels", "append", "frac_hbm")})
    c4, c5, cb = ex.get("cfg4", {}), ex.get("cfg5", {}), ex.get("cold_batched", {})
    s.update({
        "cfg4_W8_steady_us": get(c4, "W8", "steady_us_median"), "cfg4_W8_flatness_flops": get(c4, "W8", "flatness_flops_normalised"),
        "cfg4_W8_p10_p90": get(c4, "W8", "flatness_p10_p90"), "cfg4_Winf_TFLOPs_last": get(c4, "Winf", "TFLOPs_last"),
        "cfg4_growth_full_over_bounded": c4.get("growth_full_over_bounded_at_chunk_64"),
        "cfg5_query_path_us": c5.get("query_path_us"), "cfg5_attn_us": c5.get("attn_us"), "cfg5_attn_TFLOPs": c5.get("attn_TFLOPs"),
        "cfg5_kv_frac_hbm": c5.get("attn_kv_frac_hbm"), "retrieval_4096_us": get(c5, "retrieval_4096_pages", "us"),
        "layers_cfg3_B1_ms": get(ex, "layers_cfg3_B1", "ms_per_chunk_all_streams"),
        "layers_cfg3_B1_tokens_per_s": get(ex, "layers_cfg3_B1", "visual_tokens_per_s"),
        "layers_cfg2_B4_ms": get(ex, "layers_cfg2_B4", "ms_per_chunk_all_streams"),
        "layers_cfg2_B4_tokens_per_s": get(ex, "layers_cfg2_B4", "visual_tokens_per_s"),
        "drop_batched_cfg2_frac_hbm": get(cb, "drop_batched_cold", "frac_hbm"),
        "drop_batched_cfg3_frac_hbm": get(cb, "drop_batched_cold_cfg3", "frac_hbm"),
        "append_batched_frac_hbm": get(cb, "append_batched_cold", "frac_hbm"),
        "cpu_tokens_per_s": get(line, "cpu_baseline", "value"), "cpu_cores": get(line, "cpu_baseline", "cores"),
        "extras_errors": [kk for kk, vv in ex.items() if isinstance(vv, dict) and "error" in vv],
    })
    return {kk: r(vv) for kk, vv in s.items()}


def _extra_stream(name, rho, steps, warmup, peaks):
    sb = StreamBench(name, rho=rho)
    m = sb.measure(steps, warmup, peaks)
    out = stream_summary(sb, m, peaks)
    if rho is not None:
        out["rho"] = rho
        out["note"] = "SURVEY D26: the paper's '30 % retention' operating point (PAPER.md:185-190) needs rho = 0.93 under this generator"
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=320)
    ap.add_argument("--warmup", type=int, default=16)
    ap.add_argument("--impl", default="vcs", choices=["vcs", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true")
    ap.add_argument("--cpu-budget", type=float, default=15.0)
    ap.add_argument("--only", default=None, choices=["cfg2", "cfg3_rho093", "cfg4", "cfg5", "layers_cfg3_B1", "layers_cfg2_B4",
                                                     "cold_batched"],
                    help="run one companion measurement alone and print it (used for profiling); no bench line")
    ap.add_argument("--sustain", type=float, default=3.0,
                    help="seconds of back-to-back graph replay for the power-capped figure (0 = skip)")
    args = ap.parse_args()
    if "RANK" not in os.environ and args.gpus > 1:
        # not under torchrun: start the N ranks ourselves (one process per GPU, rendezvous on 127.0.0.1)
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(29500 + os.getpid() % 1000), os.path.abspath(__file__)] + sys.argv[1:]
        sys.exit(subprocess.call(cmd))
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
