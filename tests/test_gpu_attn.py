"""GPU parity: vcs_bounded_prefill_attn vs the oracle (fp64, explicit masks).

Tolerances (north_star): bf16-in / fp32-accumulate attention max-abs <= 1e-2 (x max(1, |O|_inf),
DESIGN.md reading D32) and relative L2 <= 5e-3; the fp32 SIMT path (Tiny) max-abs <= 1e-5.  The oracle keeps K_rot un-rounded in
fp64; the tolerance absorbs the bf16 storage rounding of K_rot, Q_rot, P and O (D28)."""
import numpy as np
import pytest
import torch

import oracle as vo
import synth
from helpers import ATTN_REL_L2, F32_MAX_ABS, attn_errors, attn_max_abs_tol, dev, f64, i32, tdtype

pytestmark = pytest.mark.gpu


class Scene:
    """A pool with a few pages of given lengths on both sides (CUDA pool filled via the ABI)."""

    def __init__(self, dtype, Hq, Hkv, d, page_lens, page_cap, n_pages=None, seed=0, pos_hi=4000, q_std=1.0, poison=False):
        from paper_2606_19849_b200 import vcs
        self.vcs = vcs
        self.dtype, self.Hq, self.Hkv, self.d = dtype, Hq, Hkv, d
        sec = (16, 24, 24) if d == 128 else (8, 12, 12)
        n_pages = n_pages or (len(page_lens) + 3)
        self.rng = np.random.default_rng(seed)
        self.pool = vcs.KVPool(n_pages, page_cap, Hq, Hkv, d, tdtype(dtype), 1e6, sec)
        if poison:       # a caller-owned pool need not be zeroed or finite (include/vcs.h)
            self.pool.k_pages.fill_(float("nan"))
            self.pool.v_pages.fill_(float("nan"))
            self.pool.k_sum.fill_(float("nan"))
        self.opool = vo.PagedKV(Hq, Hkv, d, 1e6, sec)
        self.pages = [int(p) for p in synth.gen_page_ids(n_pages, len(page_lens), seed)]
        self.pos_hi, self.q_std = pos_hi, q_std
        self.ws_app = vcs.workspace(vcs.vcs_kv_append_workspace_bytes(self.pool, page_cap))
        self.kv = {}
        for page, n in zip(self.pages, page_lens):
            self.fill(page, n)

    def rand(self, *shape, std=1.0):
        x = (std * self.rng.standard_normal(shape)).astype(np.float32)
        return synth.bf16_round(x) if self.dtype == "bf16" else x

    def fill(self, page, n):
        K, V = self.rand(n, self.Hkv, self.d), self.rand(n, self.Hkv, self.d)
        pos = self.rng.integers(0, self.pos_hi, size=(max(n, 1), 3)).astype(np.int32)[:n]
        if n > 0:
            self.vcs.vcs_kv_append_pages(self.pool, dev(K, self.dtype), dev(V, self.dtype), i32(pos.reshape(-1, 3)),
                                         None, n, page, 0, self.ws_app)
        self.opool.append(page, 0, K, V, pos.reshape(-1, 3))
        self.kv[page] = (K, V, pos)

    def run(self, nq, vis, self_page=-1, self_offset=0, nq_cap=None, flags=0, rows=None, scale=0.0,
            n_vis_cap=None, q_pos=None):
        vcs = self.vcs
        nq_cap = nq_cap or nq
        Q = self.rand(nq_cap, self.Hq, self.d, std=self.q_std)
        qpos = self.rng.integers(0, self.pos_hi, size=(nq_cap, 3)).astype(np.int32) if q_pos is None else q_pos
        n_vis_cap = n_vis_cap if n_vis_cap is not None else max(len(vis), 1)
        table = np.full(n_vis_cap, -1, dtype=np.int32)
        table[:len(vis)] = vis
        out = torch.full((nq_cap, self.Hq, self.d), 7.0, dtype=tdtype(self.dtype), device="cuda")
        lse = torch.full((self.Hq, nq_cap), 3.0, dtype=torch.float32, device="cuda")
        ws = vcs.workspace(vcs.vcs_bounded_prefill_attn_workspace_bytes(self.pool, nq_cap, n_vis_cap))
        status = torch.zeros(1, dtype=torch.int32, device="cuda")
        for _ in range(2):
            vcs.vcs_bounded_prefill_attn(self.pool, dev(Q, self.dtype), i32(qpos), i32([nq]), nq_cap, i32(table),
                                         i32([len(vis)]), n_vis_cap, self_page, self_offset, out, ws, lse=lse,
                                         softmax_scale=scale, flags=flags, status=status)
        torch.cuda.synchronize()
        assert int(status) == 0
        O_ref, lse_ref = vo.bounded_attention(self.opool, Q[:nq], qpos[:nq], vis, self_page, self_offset,
                                              scale=scale or None, rows=rows)
        sel = np.arange(nq) if rows is None else np.asarray(rows)
        got, got_lse = f64(out)[sel], f64(lse)[:, sel]
        assert np.all(f64(out)[nq:] == 7.0) and np.all(f64(lse)[:, nq:] == 3.0)   # rows >= nq untouched
        return got, O_ref, got_lse, lse_ref

    def check(self, *a, **kw):
        got, ref, glse, rlse = self.run(*a, **kw)
        ma, rl = attn_errors(got, ref)
        if self.dtype == "bf16":
            assert ma <= attn_max_abs_tol(ref) and rl <= ATTN_REL_L2, (ma, rl)     # reading D32
            fin = np.isfinite(rlse)
            assert np.max(np.abs(glse[fin] - rlse[fin])) <= 2e-2
        else:
            assert ma <= F32_MAX_ABS, ma
            fin = np.isfinite(rlse)
            assert np.max(np.abs(glse[fin] - rlse[fin])) <= 1e-4
        return ma, rl


IMPLS = [pytest.param(1, id="simt"), pytest.param(2, id="tc")]


@pytest.mark.parametrize("flags", IMPLS)
def test_attn_bf16_tiles_and_ragged_tails(flags):
    # 3 fully visible pages with ragged lengths (several 128-token tiles + tails) + causal self page
    s = Scene("bf16", 16, 2, 128, [64, 300, 129, 517], 640, seed=1)
    sink, a, b, me = s.pages
    s.check(517, [sink, a, b], self_page=me, flags=flags)                    # chunk prefill, 5 q tiles
    s.check(200, [a], self_page=me, self_offset=317, flags=flags)             # continuation: offset causal
    s.check(130, [b, sink, a], flags=flags)                                  # no self page (pure cross attention)
    s.check(1, [sink], self_page=me, flags=flags)                            # single row
    s.check(70, [], self_page=me, nq_cap=256, flags=flags)                   # self only; nq < nq_cap (2 q tiles cap)


@pytest.mark.parametrize("flags", IMPLS)
def test_attn_bf16_gqa7_sharp_logits(flags):
    # 7B-like grouping (28/4), sharper logits (q std 2) so that masking / max tracking errors show
    s = Scene("bf16", 28, 4, 128, [128, 257, 96], 384, seed=2, q_std=2.0)
    sink, a, me = s.pages
    s.check(96, [sink, a], self_page=me, flags=flags)
    s.check(48, [a, sink], flags=flags, scale=0.05)                           # explicit scale


@pytest.mark.parametrize("flags", IMPLS)
def test_attn_empty_pages_and_empty_visible_set(flags):
    s = Scene("bf16", 4, 2, 128, [0, 40, 0], 128, seed=3)
    e0, a, e1 = s.pages
    s.check(40, [e0, a, e1], flags=flags)                                    # zero-length pages are skipped
    got, ref, glse, rlse = s.run(5, [e0], flags=flags)                       # nothing visible at all
    assert np.all(got == 0.0) and np.all(np.isneginf(glse))


def test_attn_fp32_simt_tiny_shapes():
    s = Scene("f32", 2, 1, 64, [8, 24, 20, 27], 32, seed=4, q_std=4.0)
    sink, a, b, me = s.pages
    s.check(27, [sink, a, b], self_page=me)
    s.check(27, [sink], self_page=me, flags=1)
    s2 = Scene("f32", 4, 2, 128, [50, 77], 128, seed=5)
    s2.check(77, [s2.pages[0]], self_page=s2.pages[1])
    s3 = Scene("bf16", 4, 2, 64, [50, 77], 128, seed=6)                      # bf16, d = 64 -> SIMT in AUTO mode
    s3.check(77, [s3.pages[0]], self_page=s3.pages[1])


def test_attn_tc_tail_split_of_under_filled_last_wave():
    """Grids of more than one wave whose last wave is under-filled: the spare CTAs (q tiles beyond
    nq inside the nq_cap grid) take KV parts of the last-wave items and the partials are merged
    (DESIGN.md §5 'tail split').  28 heads x 6 active q tiles = 168 items on 148 SMs -> 20 tail
    items in 4 parts; every row checked.  Second call: self page only, so the first q tiles have
    fewer KV tiles than parts (empty parts must merge as nothing)."""
    s = Scene("bf16", 28, 4, 128, [64, 300, 700], 1536, seed=11)
    sink, a, me = s.pages
    s.check(700, [sink, a], self_page=me, nq_cap=1536, flags=2)
    s.check(700, [], self_page=me, nq_cap=1536, flags=2)
    s.check(641, [a, sink], nq_cap=1536, flags=2)                             # no self page, ragged last q tile


def test_attn_tc_matches_simt_closely():
    """Two structurally different GPU implementations agree far inside the oracle tolerance."""
    s = Scene("bf16", 16, 2, 128, [64, 700, 333], 768, seed=7)
    sink, a, me = s.pages
    state = s.rng.bit_generator.state
    g1, ref, _, _ = s.run(333, [sink, a], self_page=me, flags=1)
    s.rng.bit_generator.state = state
    g2, _, _, _ = s.run(333, [sink, a], self_page=me, flags=2)
    assert np.max(np.abs(g1 - g2)) <= 8e-3


def test_attn_window_permutation_invariance_on_gpu():
    s = Scene("bf16", 16, 2, 128, [64, 150, 260, 90], 384, seed=8)
    sink, a, b, me = s.pages
    state = s.rng.bit_generator.state
    g1, _, _, _ = s.run(90, [sink, a, b], self_page=me)
    s.rng.bit_generator.state = state
    g2, _, _, _ = s.run(90, [b, sink, a], self_page=me)
    assert np.max(np.abs(g1 - g2)) <= 8e-3                                   # only summation order differs


def test_attn_vl3b_full_size_sampled_rows():
    """Config 2 at full size (sink 64 + 4 history pages + self, ~1000 kept rows, 16 heads) in the
    launch configuration bench.py times; the oracle checks a row sample (first/last 128 + every 7th)."""
    cfg = synth.get_config("vl3b")
    lens = [cfg.sink, 1021, 987, 1040, 1003, 1021]
    s = Scene("bf16", cfg.Hq, cfg.Hkv, cfg.d, lens, cfg.page_cap, n_pages=12, seed=9)
    nq = lens[-1]
    rows = sorted(set(list(range(128)) + list(range(nq - 128, nq)) + list(range(0, nq, 7))))
    ma, rl = s.check(nq, s.pages[:5], self_page=s.pages[5], nq_cap=cfg.T, rows=rows)
    print("vl3b full-size attention: max-abs %.3e rel-L2 %.3e" % (ma, rl))


def test_attn_tc_randomized_shapes_against_oracle():
    """40 seeded random scenes (GQA 16/2, 28/4, 8/8, 32/4; 1-5 history pages of ragged, empty, exactly-one-tile
    and one-over lengths; causal self page with and without an offset, or none; nq < nq_cap grids that reach the
    split-KV and tail-split launch shapes) on the tcgen05 path; 50 sampled rows per scene checked by the oracle."""
    rng = np.random.default_rng(1)
    for trial in range(40):
        Hq, Hkv = [(16, 2), (28, 4), (8, 8), (32, 4)][rng.integers(0, 4)]
        npg = int(rng.integers(1, 6))
        cap = int(rng.choice([640, 1200, 2304]))
        lens = [int(rng.integers(0, cap + 1)) if rng.random() < 0.8 else int(rng.choice([128, 129, 1, 256, 127]))
                for _ in range(npg)]
        me_len = int(rng.integers(1, cap + 1))
        s = Scene("bf16", Hq, Hkv, 128, lens + [me_len], cap, seed=int(rng.integers(0, 1 << 30)))
        use_self = rng.random() < 0.7
        if use_self:
            off = int(rng.integers(0, me_len)) if rng.random() < 0.3 else 0
            nq = me_len - off
        else:
            off, nq = 0, int(rng.integers(1, cap + 1))
        nq_cap = nq if rng.random() < 0.4 else int(min(4096, nq + rng.integers(0, 2000)))
        vis = [p for p in s.pages[:-1] if rng.random() < 0.85]
        rows = sorted(set(rng.integers(0, nq, size=min(nq, 48)).tolist() + [0, nq - 1]))
        got, ref, glse, rlse = s.run(nq, vis, self_page=s.pages[-1] if use_self else -1, self_offset=off, nq_cap=nq_cap,
                                     flags=2, rows=rows)
        ma, rl = attn_errors(got, ref)
        fin = np.isfinite(rlse)
        assert ma <= attn_max_abs_tol(ref) and rl <= ATTN_REL_L2, (trial, Hq, Hkv, lens, me_len, off, nq, nq_cap, ma, rl)
        assert not fin.any() or np.max(np.abs(glse[fin] - rlse[fin])) <= 2e-2, trial


@pytest.mark.parametrize("flags", IMPLS)
def test_attn_pool_poisoned_with_nan(flags):
    """The pool is caller-owned memory and is NOT required to be zeroed: every byte is NaN before the
    stream starts.  Ragged tails, a diagonal tile and a continuation append (page_offset > 0)."""
    s = Scene("bf16", 16, 2, 128, [64, 300, 129, 517], 640, seed=21, poison=True)
    sink, a, b, me = s.pages
    s.check(517, [sink, a, b], self_page=me, flags=flags)
    s.check(130, [b, sink, a], flags=flags)
    # continuation: 40 more tokens appended to page `a` at offset 300 (a fresh tail is zero-filled again)
    K, V = s.rand(40, s.Hkv, s.d), s.rand(40, s.Hkv, s.d)
    pos = s.rng.integers(0, s.pos_hi, size=(40, 3)).astype(np.int32)
    s.vcs.vcs_kv_append_pages(s.pool, dev(K, "bf16"), dev(V, "bf16"), i32(pos), None, 40, a, 300, s.ws_app)
    s.opool.append(a, 300, K, V, pos)
    s.check(200, [a, sink], self_page=me, self_offset=317, flags=flags)


def test_attn_batched_streams_one_launch():
    """vcs_bounded_prefill_attn_batched: B = 3 streams of different kept counts, window sizes and self
    pages in ONE launch (their work items share the persistent grid) == three oracle calls."""
    from paper_2606_19849_b200 import vcs
    s = Scene("bf16", 16, 2, 128, [64, 300, 129, 517, 222, 700, 64], 768, seed=31, n_pages=12)
    sink, a, b, me0, me1, me2, c = s.pages
    B, nq_cap, n_vis_cap = 3, 768, 4
    streams = [dict(nq=517, vis=[sink, a, b], me=me0), dict(nq=222, vis=[c], me=me1), dict(nq=700, vis=[sink, b, a, c], me=me2)]
    Q = s.rand(B, nq_cap, s.Hq, s.d)
    qpos = s.rng.integers(0, s.pos_hi, size=(B, nq_cap, 3)).astype(np.int32)
    tables = np.full((B, n_vis_cap), -1, dtype=np.int32)
    for bi, st in enumerate(streams):
        tables[bi, :len(st["vis"])] = st["vis"]
    out = torch.full((B, nq_cap, s.Hq, s.d), 7.0, dtype=torch.bfloat16, device="cuda")
    lse = torch.full((B, s.Hq, nq_cap), 3.0, dtype=torch.float32, device="cuda")
    ws = vcs.workspace(vcs.vcs_bounded_prefill_attn_workspace_bytes(s.pool, nq_cap, n_vis_cap))
    status = torch.zeros(1, dtype=torch.int32, device="cuda")
    for flags in (vcs.ATTN_TC, vcs.ATTN_SIMT):
        out.fill_(7.0)
        vcs.vcs_bounded_prefill_attn_batched(s.pool, dev(Q, "bf16"), i32(qpos), i32([st["nq"] for st in streams]), nq_cap,
                                             i32(tables), i32([len(st["vis"]) for st in streams]),
                                             i32([st["me"] for st in streams]), 0, out, ws, lse=lse, flags=flags, status=status)
        torch.cuda.synchronize()
        assert int(status) == 0
        for bi, st in enumerate(streams):
            nq = st["nq"]
            ref, rlse = vo.bounded_attention(s.opool, Q[bi, :nq], qpos[bi, :nq], st["vis"], st["me"], 0)
            got = f64(out[bi])
            ma, rl = attn_errors(got[:nq], ref)
            assert ma <= attn_max_abs_tol(ref) and rl <= ATTN_REL_L2, (flags, bi, ma, rl)
            assert np.all(got[nq:] == 7.0)
            assert np.max(np.abs(f64(lse[bi])[:, :nq] - rlse)) <= 2e-2


def test_attn_workspace_reused_across_shapes():
    """One workspace serves calls of different shapes back to back (it carries no state between calls):
    a 48-row query prefill (many KV parts per item), then a multi-tile chunk prefill, then the query again."""
    s = Scene("bf16", 28, 4, 128, [128, 900, 640, 700], 1024, seed=41)
    sink, a, b, me = s.pages
    from paper_2606_19849_b200 import vcs
    ws = vcs.workspace(vcs.vcs_bounded_prefill_attn_workspace_bytes(s.pool, 1024, 8))
    ws.fill_(0xAB)                                               # needs no initialisation either
    def one(nq, vis, self_page, nq_cap):
        Q = s.rand(nq_cap, s.Hq, s.d)
        qpos = s.rng.integers(0, s.pos_hi, size=(nq_cap, 3)).astype(np.int32)
        out = torch.zeros((nq_cap, s.Hq, s.d), dtype=torch.bfloat16, device="cuda")
        table = np.full(8, -1, dtype=np.int32); table[:len(vis)] = vis
        vcs.vcs_bounded_prefill_attn(s.pool, dev(Q, "bf16"), i32(qpos), i32([nq]), nq_cap, i32(table), i32([len(vis)]), 8,
                                     self_page, 0, out, ws, flags=vcs.ATTN_TC)
        torch.cuda.synchronize()
        ref, _ = vo.bounded_attention(s.opool, Q[:nq], qpos[:nq], vis, self_page, 0)
        ma, rl = attn_errors(f64(out)[:nq], ref)
        assert ma <= attn_max_abs_tol(ref) and rl <= ATTN_REL_L2, (nq, ma, rl)
    one(48, [sink, a, b], -1, 48)
    one(700, [sink, a], me, 1024)
    one(48, [b, a], -1, 64)


def test_softmax_polynomial_and_fast_rope_errors_are_pinned():
    """The two approximations of the bf16 path, each against fp64 on its whole domain (so that their share of the
    attention tolerance is known and cannot grow unnoticed): the degree-2 2^x used for a quarter of the softmax
    exponentials (relative error <= 2e-3 on [-126, 8], the range the kernel feeds it: scores minus the running maximum,
    lazily rescaled at 2^8) and the Q0.64 / MUFU sin-cos of M-RoPE (absolute error <= 1e-6 for positions up to 2^20,
    reading D28; rotated K / Q are rounded to bf16 right after, 2^-9 relative)."""
    from paper_2606_19849_b200 import vcs
    rng = np.random.default_rng(3)
    x = np.concatenate([rng.uniform(-126.0, 8.0, 1 << 20), rng.uniform(-16.0, 0.0, 1 << 20),     # where the weights live
                        np.arange(-126, 9) - 0.5, np.arange(-126, 9) + 0.49999, np.arange(-126, 9), [-126.0, 8.0, 0.0, -0.0]])
    x = np.clip(x, -126.0, 8.0).astype(np.float32)              # the stated domain: the kernel clamps below -126
    y = vcs.vcs_selftest_exp2_poly(torch.from_numpy(x).cuda()).cpu().numpy().astype(np.float64)
    rel = np.abs(y / np.exp2(x.astype(np.float64)) - 1.0)
    assert rel.max() <= 2e-3, (rel.max(), x[rel.argmax()])
    assert rel.max() >= 1e-3                                     # it IS the degree-2 polynomial, not the MUFU path
    # below the clamp the result stays tiny and finite (no exponent wrap-around)
    lo = vcs.vcs_selftest_exp2_poly(torch.tensor([-127.0, -200.0, -1e30, float("-inf")], device="cuda")).cpu().numpy()
    assert np.all(np.isfinite(lo)) and np.all(lo >= 0) and np.all(lo <= 2.0 ** -125)
    pos = np.concatenate([rng.integers(0, 1 << 20, 1 << 18), np.arange(0, 4096), [(1 << 20) - 1, 100000, 99999]]).astype(np.int32)
    worst = 0.0
    for theta, d in ((1e6, 128), (1e4, 64)):
        for m in (0, 1, 2, 7, 15, 16, 31, 40, d // 2 - 1):
            inv_freq = float(theta) ** (-2.0 * m / d)
            s, c = vcs.vcs_selftest_rope_sincos(torch.from_numpy(pos).cuda(), inv_freq)
            a = pos.astype(np.float64) * inv_freq
            err = max(np.abs(s.cpu().numpy() - np.sin(a)).max(), np.abs(c.cpu().numpy() - np.cos(a)).max())
            worst = max(worst, float(err))
    assert worst <= 1e-6, worst
