"""GPU parity: vcs_temporal_drop vs the oracle, bit-exact kept indices / counts / masks / pos3."""
import numpy as np
import pytest
import torch

import oracle as vo
import synth
from helpers import dev, i32

pytestmark = pytest.mark.gpu


def _run_drop(Z, dtype, tau, mode=0, prev=None, want_mask=True, grid=None, base=None, t_stride=1):
    """Z: numpy [B][G][P][D] storage-exact float32.  Returns numpy outputs of the CUDA path."""
    from paper_2606_19849_b200 import vcs
    B, G, P, D = Z.shape
    z = dev(Z, dtype)
    T = G * P
    kept_idx = torch.full((B, T), -7, dtype=torch.int32, device="cuda")
    cnt = torch.full((B,), -7, dtype=torch.int32, device="cuda")
    mask = torch.full((B, T), 9, dtype=torch.uint8, device="cuda") if want_mask else None
    pos3 = torch.full((B, T, 3), -5, dtype=torch.int32, device="cuda") if grid else None
    ws = vcs.workspace(vcs.vcs_temporal_drop_workspace_bytes(B, G, P))
    for _ in range(2):   # twice: the workspace must come back zeroed (self-resetting counters)
        vcs.vcs_temporal_drop(z, tau, kept_idx, cnt, ws, mode=mode,
                              prev_last_group=None if prev is None else dev(prev, dtype), keep_mask=mask,
                              pos3=pos3, Hg=grid[0] if grid else 0, Wg=grid[1] if grid else 0, t_stride=t_stride,
                              pos_base=None if base is None else i32(base))
    torch.cuda.synchronize()
    assert int(ws[:4 * B].view(torch.int32).abs().sum()) == 0
    return (kept_idx.cpu().numpy(), cnt.cpu().numpy(), None if mask is None else mask.cpu().numpy(),
            None if pos3 is None else pos3.cpu().numpy())


def _check(Z, dtype, tau, mode=0, prev=None, grid=None, base=None, t_stride=1, want_mask=True):
    B, G, P, D = Z.shape
    idx, cnt, mask, pos3 = _run_drop(Z, dtype, tau, mode, prev, want_mask, grid, base, t_stride)
    for b in range(B):
        keep, ref_idx, n = vo.temporal_drop(Z[b], tau, mode, None if prev is None else prev[b])
        assert cnt[b] == n, (b, cnt[b], n)
        assert np.array_equal(idx[b, :n], ref_idx)
        assert np.all(idx[b, n:] == -1)
        if want_mask:
            assert np.array_equal(mask[b].astype(bool), keep.ravel())
        if grid:
            ref_pos = vo.grid_positions(G, grid[0], grid[1], 0 if base is None else int(base[b]), t_stride)[ref_idx]
            assert np.array_equal(pos3[b, :n], ref_pos)
            assert np.all(pos3[b, n:] == -5)                     # rows >= count untouched


def _mixed(B, G, P, D, seed, rho=0.5, bf16=True):
    rng = np.random.default_rng(seed)
    static = rng.random((B, 1, P, 1)) < rho
    base = rng.standard_normal((B, 1, P, D))
    Z = np.where(static, base + 0.05 * rng.standard_normal((B, G, P, D)), rng.standard_normal((B, G, P, D)))
    Z = Z.astype(np.float32)
    return synth.bf16_round(Z) if bf16 else Z


def test_drop_tiny_all_chunks_fp32():
    cfg = synth.get_config("tiny")
    Z = synth.gen_hidden_tiny(cfg)
    for t in range(cfg.n_chunks):
        _check(Z[t][None], "f32", cfg.tau, grid=(cfg.Hg, cfg.Wg), base=[cfg.sink + 4 * t])
    _check(Z, "f32", cfg.tau)                                    # all six chunks as a batch B=6
    _check(Z[1:], "f32", cfg.tau, mode=1, prev=Z[:-1, -1])      # frame-level variant with prev


def test_drop_vl3b_full_chunk_bf16():
    cfg = synth.get_config("vl3b")
    for t in range(2):
        Z, static = synth.gen_hidden_chunk(cfg, t)
        _check(Z[None], "bf16", cfg.tau, grid=(cfg.Hg, cfg.Wg), base=[cfg.sink + 29 * t])
        idx, cnt, _, _ = _run_drop(Z[None], "bf16", cfg.tau)
        assert cnt[0] == cfg.P + (cfg.G - 1) * int((~static).sum())


def test_drop_vl7b_batch_bf16():
    cfg = synth.get_config("vl7b")
    Zs = np.stack([synth.gen_hidden_chunk(cfg, t)[0] for t in range(2)])
    _check(Zs, "bf16", cfg.tau, grid=(cfg.Hg, cfg.Wg), base=[128, 174], want_mask=False)


@pytest.mark.parametrize("G", [1, 2, 3, 5, 8, 9, 10, 12])
def test_drop_group_counts(G):
    Z = _mixed(2, G, 37, 264, seed=G)
    _check(Z, "bf16", 0.9)
    _check(Z, "bf16", 0.9, mode=1)
    prev = _mixed(2, 1, 37, 264, seed=100 + G)[:, 0]
    prev[:, ::2] = Z[:, 0, ::2]                                   # half the positions repeat the previous frame
    _check(Z, "bf16", 0.9, mode=1, prev=prev)


@pytest.mark.parametrize("shape", [(1, 4, 1, 8), (3, 4, 5, 8), (1, 2, 300, 2048), (2, 4, 129, 3584), (1, 4, 33, 520),
                                   (5, 3, 64, 72)])
def test_drop_ragged_shapes(shape):
    B, G, P, D = shape
    Z = _mixed(B, G, P, D, seed=P + D)
    _check(Z, "bf16", 0.95)
    _check(_mixed(B, G, P, max(4, D // 2), seed=P, bf16=False), "f32", 0.95)


def test_drop_threshold_extremes_and_degenerate():
    Z = _mixed(1, 4, 40, 128, seed=1)
    idx, cnt, mask, _ = _run_drop(Z, "bf16", 1.0)               # tau >= 1 keeps everything (paper s = 1.0)
    assert cnt[0] == 160 and np.array_equal(idx[0], np.arange(160))
    idx, cnt, mask, _ = _run_drop(Z, "bf16", -1.5)              # only the anchor group survives
    assert cnt[0] == 40 and np.array_equal(idx[0, :40], np.arange(40)) and mask[0, :40].all() and not mask[0, 40:].any()
    Zz = Z.copy()
    Zz[0, 2, 5] = 0.0                                            # zero-norm token: S := 0
    _check(Zz, "bf16", 0.5)
    _check(Zz, "bf16", -0.5)
    Zi = np.repeat(Z[:, :1], 4, axis=1).copy()                   # identical groups: S = 1 (reading D31: |S| <= 1)
    _check(Zi, "bf16", 0.999)
    _check(Zi, "bf16", 1.0)                                      # paper: s = 1.0 -> 0 % drop
    _check(Zi, "bf16", 1.0, mode=1, prev=Zi[:, 0])
    _check(Zi * np.array([1.0, 2.0, 0.5, 4.0], dtype=np.float32)[None, :, None, None], "bf16", 1.0)   # parallel tokens


def test_drop_empty_inputs():
    from paper_2606_19849_b200 import vcs
    cnt = torch.full((2,), 5, dtype=torch.int32, device="cuda")
    z = torch.zeros((2, 4, 0, 64), dtype=torch.bfloat16, device="cuda")
    vcs.vcs_temporal_drop(z, 0.9, torch.zeros((2, 0), dtype=torch.int32, device="cuda"), cnt, vcs.workspace(256))
    torch.cuda.synchronize()
    assert cnt.tolist() == [0, 0]


@pytest.mark.parametrize("G,P", [(8, 1196), (16, 1196), (9, 1000)])
def test_drop_more_than_8192_tokens_stays_ascending(G, P):
    """T = G * P > 8192 (720p grid at c = 16 / 32 frames, Table 2): the compacted list must stay in
    ascending sequence order (reading D9) on the templated (G <= 8) and the generic path; pos3 with it."""
    Z = _mixed(1, G, P, 64, seed=G * P, rho=0.6)
    grid = (26, 46) if P == 1196 else (25, 40)
    _check(Z, "bf16", 0.9, grid=grid, base=[77])
    _check(Z, "bf16", 0.9, mode=1)
    idx, cnt, _, _ = _run_drop(Z, "bf16", 2.0)                   # nothing dropped: the identity list
    assert cnt[0] == G * P and np.array_equal(idx[0], np.arange(G * P))


def test_drop_workspace_reused_with_other_shapes():
    """One (zeroed once) workspace serves calls of different G, P, D at the same B (include/vcs.h): stale
    flags of a larger earlier call must not leak into the padding of a later, smaller one."""
    from paper_2606_19849_b200 import vcs
    ws = vcs.workspace(vcs.vcs_temporal_drop_workspace_bytes(2, 8, 300))
    for (B, G, P, D, tau) in [(2, 8, 300, 64, 2.0), (2, 3, 37, 64, 0.9), (2, 4, 129, 128, 0.9), (2, 3, 37, 64, 0.9)]:
        Z = _mixed(B, G, P, D, seed=B * G * P)
        T = G * P
        idx = torch.full((B, T), -7, dtype=torch.int32, device="cuda")
        cnt = torch.full((B,), -7, dtype=torch.int32, device="cuda")
        vcs.vcs_temporal_drop(dev(Z, "bf16"), tau, idx, cnt, ws)
        torch.cuda.synchronize()
        for b in range(B):
            _, ref_idx, n = vo.temporal_drop(Z[b], tau)
            assert int(cnt[b]) == n and np.array_equal(idx[b, :n].cpu().numpy(), ref_idx), (B, G, P)
