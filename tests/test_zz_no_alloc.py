"""vcs_temporal_drop_static: temporal dropping for callers that cannot allocate device memory.

A serving process that handed all of the HBM to its own pool, a per-frame loop that may not call
cudaMalloc, or a plug-in without an allocator cannot give vcs_temporal_drop its workspace.  They call
vcs_temporal_drop_static, which keeps the ticket counters and keep flags in a 1 MiB array inside
libvcs.so.  It launches the same kernel, so its lists, counts, masks and positions must equal those of
vcs_temporal_drop bit for bit (the bar every drop test uses: integer work is exact).

The array is shared by every call and keeps the last call's contents, so the check runs two calls in a
row with DIFFERENT shapes: the second one starts on the first one's leftovers.  This file is named to be
collected last: with `pytest -x` a failure here cannot hide a test of the existing paths.
"""
import numpy as np
import pytest
import torch

import synth
from helpers import dev, i32


def _scene(B, G, P, D, seed, rho=0.5):
    """Half-static synthetic chunk [B][G][P][D], bf16-exact values (recipe of tests/test_gpu_drop.py)."""
    rng = np.random.default_rng(seed)
    static = rng.random((B, 1, P, 1)) < rho
    base = rng.standard_normal((B, 1, P, D))
    Z = np.where(static, base + 0.05 * rng.standard_normal((B, G, P, D)), rng.standard_normal((B, G, P, D)))
    return synth.bf16_round(Z.astype(np.float32))


def _outputs(B, T, grid):
    return dict(kept_idx=torch.full((B, T), -7, dtype=torch.int32, device="cuda"),
                kept_count=torch.full((B,), -7, dtype=torch.int32, device="cuda"),
                keep_mask=torch.full((B, T), 9, dtype=torch.uint8, device="cuda"),
                pos3=torch.full((B, T, 3), -5, dtype=torch.int32, device="cuda") if grid else None)


def _both_paths(vcs, Z, tau, mode=0, prev=None, grid=None, base=None):
    """Run the caller-workspace path and the static-scratch path on the same inputs; return both output sets."""
    B, G, P, D = Z.shape
    z = dev(Z, "bf16")
    kw = dict(mode=mode, prev_last_group=None if prev is None else dev(prev, "bf16"),
              Hg=grid[0] if grid else 0, Wg=grid[1] if grid else 0, t_stride=2,
              pos_base=None if base is None else i32(base))
    ref, got = _outputs(B, G * P, grid), _outputs(B, G * P, grid)
    ws = vcs.workspace(vcs.vcs_temporal_drop_workspace_bytes(B, G, P))
    vcs.vcs_temporal_drop(z, tau, ref["kept_idx"], ref["kept_count"], ws, keep_mask=ref["keep_mask"], pos3=ref["pos3"], **kw)
    vcs.vcs_temporal_drop_static(z, tau, got["kept_idx"], got["kept_count"], keep_mask=got["keep_mask"], pos3=got["pos3"], **kw)
    torch.cuda.synchronize()
    return ref, got


def _assert_same(ref, got):
    assert int(ref["kept_count"].min()) >= 0
    for name in ref:
        if ref[name] is not None:
            assert torch.equal(ref[name], got[name]), name


@pytest.mark.gpu
def test_static_scratch_matches_workspace_path_on_two_calls_in_a_row():
    from paper_2606_19849_b200 import vcs
    # call 1: two streams, four groups, 37 x 13 = 481 positions (several blocks per stream, ragged last block)
    ref, got = _both_paths(vcs, _scene(2, 4, 481, 256, seed=11), 0.9, grid=(37, 13), base=np.array([5, 1000]))
    _assert_same(ref, got)
    assert 0 < int(ref["kept_count"][0]) < 4 * 481            # the scene really drops some and keeps some
    # call 2, straight after, on the array call 1 dirtied: other B / G / P (its flag rows start elsewhere), the
    # frame-level rule with a previous chunk's last group, and more than one 4096-token compaction pass
    Z2 = _scene(3, 3, 1501, 128, seed=12)
    prev = Z2[:, 0] + synth.bf16_round(0.02 * np.random.default_rng(13).standard_normal(Z2[:, 0].shape).astype(np.float32))
    ref, got = _both_paths(vcs, Z2, 0.8, mode=vcs.DROP_CONSECUTIVE, prev=synth.bf16_round(prev))
    _assert_same(ref, got)
    # and the first shape again: nothing of call 2 leaks into it
    ref, got = _both_paths(vcs, _scene(2, 4, 481, 256, seed=14), 0.9, grid=(37, 13))
    _assert_same(ref, got)


@pytest.mark.gpu
def test_static_scratch_empty_chunk_and_limit_on_device():
    from paper_2606_19849_b200 import vcs
    cnt = torch.full((2,), -7, dtype=torch.int32, device="cuda")
    vcs.vcs_temporal_drop_static(torch.zeros((2, 4, 0, 64), dtype=torch.bfloat16, device="cuda"), 0.9,
                                 torch.zeros((2, 0), dtype=torch.int32, device="cuda"), cnt)
    torch.cuda.synchronize()
    assert cnt.tolist() == [0, 0]
    # the largest B that still fits a 7B-shaped chunk (4784 tokens) is accepted, one more is refused
    G, P = 2, 2392
    B = 1
    while vcs.vcs_temporal_drop_workspace_bytes(B + 1, G, P) <= vcs.DROP_STATIC_SCRATCH_BYTES:
        B += 1
    Z = _scene(B, G, P, 16, seed=15)
    ref, got = _both_paths(vcs, Z, 0.9)
    _assert_same(ref, got)
    z = torch.zeros((B + 1, G, P, 16), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(vcs.VcsError) as e:
        vcs.vcs_temporal_drop_static(z, 0.9, torch.zeros((B + 1, G * P), dtype=torch.int32, device="cuda"),
                                     torch.zeros((B + 1,), dtype=torch.int32, device="cuda"))
    assert e.value.code == vcs.ECAP


def test_static_scratch_size_limit_is_refused_without_a_device():
    """The size test runs before any CUDA call: too large a shape answers VCS_ECAP with the sizes in the message."""
    from paper_2606_19849_b200 import build, vcs
    build.build_library()
    lib = vcs.lib()
    assert lib.vcs_temporal_drop_workspace_bytes(1, 8, 200000) > vcs.DROP_STATIC_SCRATCH_BYTES
    rc = lib.vcs_temporal_drop_static(16, None, 1, 8, 200000, 64, vcs.BF16, 0.9, 0, 16, 16, None, None, 0, 0, 1, None, None)
    assert rc == vcs.ECAP
    msg = lib.vcs_last_error().decode()
    assert "P=200000" in msg and str(vcs.DROP_STATIC_SCRATCH_BYTES) in msg
