"""GPU parity: vcs_kv_append_pages vs the oracle (K rotated by M-RoPE, V copy, key sums, lengths)."""
import numpy as np
import pytest
import torch

import oracle as vo
import synth
from helpers import dev, f64, i32, tdtype

pytestmark = pytest.mark.gpu


def k_rot_tol(Kref):
    """Stored K (reading D28): one bf16 rounding (2^-8 relative, the ulp) of a rotation whose sin / cos
    come from the fp32 fast path -- angle good to 2 pi 2^-24 = 3.7e-7 rad plus ~5e-7 absolute from MUFU sin / cos,
    i.e. <= 2e-6 times the length r of the rotated pair (m, m + d/2), which the rotation preserves."""
    half = Kref.shape[-1] // 2
    r = np.hypot(Kref[..., :half], Kref[..., half:])
    return 2.0 ** -8 * np.abs(Kref) + 2e-6 * np.concatenate([r, r], axis=-1)


def _pool(n_pages, page_cap, Hq, Hkv, d, dtype):
    from paper_2606_19849_b200 import vcs
    sec = (16, 24, 24) if d == 128 else (8, 12, 12)
    return vcs.KVPool(n_pages, page_cap, Hq, Hkv, d, tdtype(dtype), 1e6, sec), sec


def _check_page(pool, opool, page, dtype):
    n = opool.page_len(page)
    assert int(pool.page_len[page]) == n
    K = f64(pool.k_pages[page, :, :n]).transpose(1, 0, 2)
    V = f64(pool.v_pages[page, :, :n]).transpose(1, 0, 2)
    Kref, Vref = opool.K[page], opool.V[page]
    assert np.array_equal(V, Vref)                               # V is a bit-exact copy
    if n == 0:
        assert float(pool.k_sum[page].abs().sum()) == 0.0
        return
    if dtype == "bf16":
        assert np.all(np.abs(K - Kref) <= k_rot_tol(Kref))
    else:
        assert np.max(np.abs(K - Kref)) <= 2e-6 * max(1.0, np.max(np.abs(Kref)))
    ks = f64(pool.k_sum[page])
    assert np.max(np.abs(ks - opool.k_sum[page])) <= 1e-5 * max(1.0, np.sqrt(n)) * max(1.0, np.max(np.abs(Kref)))


@pytest.mark.parametrize("dtype,Hq,Hkv,d", [("bf16", 16, 2, 128), ("bf16", 28, 4, 128), ("f32", 2, 1, 64), ("bf16", 4, 2, 64),
                                             ("f32", 4, 2, 128)])
def test_append_parity(dtype, Hq, Hkv, d):
    from paper_2606_19849_b200 import vcs
    rng = np.random.default_rng(d + Hkv)
    pool, sec = _pool(6, 256, Hq, Hkv, d, dtype)
    opool = vo.PagedKV(Hq, Hkv, d, 1e6, sec)
    ws = vcs.workspace(vcs.vcs_kv_append_workspace_bytes(pool, 256))
    status = torch.zeros(1, dtype=torch.int32, device="cuda")
    for page, n, n_cap in [(4, 201, 256), (1, 1, 8), (3, 37, 37), (0, 0, 16)]:
        K = rng.standard_normal((n_cap, Hkv, d)).astype(np.float32)
        V = rng.standard_normal((n_cap, Hkv, d)).astype(np.float32)
        if dtype == "bf16":
            K, V = synth.bf16_round(K), synth.bf16_round(V)
        pos = rng.integers(0, 100000, size=(n_cap, 3)).astype(np.int32)   # large positions: fp64 angle reduction
        vcs.vcs_kv_append_pages(pool, dev(K, dtype), dev(V, dtype), i32(pos), i32([n]), n_cap, page, 0, ws, status)
        opool.append(page, 0, K[:n], V[:n], pos[:n])
        torch.cuda.synchronize()
        _check_page(pool, opool, page, dtype)
    assert int(status) == 0
    # untouched tails stay zero; other pages untouched
    assert float(pool.k_pages[4, :, 201:].abs().sum()) == 0.0 and int(pool.page_len[2]) == 0 and int(pool.page_len[5]) == 0


def test_append_offset_strided_and_overflow():
    from paper_2606_19849_b200 import vcs
    rng = np.random.default_rng(3)
    Hq, Hkv, d = 16, 2, 128
    pool, sec = _pool(3, 128, Hq, Hkv, d, "bf16")
    opool = vo.PagedKV(Hq, Hkv, d, 1e6, sec)
    ws = vcs.workspace(vcs.vcs_kv_append_workspace_bytes(pool, 128))
    status = torch.zeros(1, dtype=torch.int32, device="cuda")
    # K and V as slices of one fused [n][ (Hq + 2 Hkv) * d ] projection output (row stride != Hkv*d)
    fused = synth.bf16_round(rng.standard_normal((100, (Hq + 2 * Hkv) * d)).astype(np.float32))
    fd = dev(fused, "bf16")
    kd = fd[:, Hq * d:(Hq + Hkv) * d].view(100, Hkv, d)
    vd = fd[:, (Hq + Hkv) * d:].view(100, Hkv, d)
    assert kd.stride(0) == (Hq + 2 * Hkv) * d
    K = fused[:, Hq * d:(Hq + Hkv) * d].reshape(100, Hkv, d)
    V = fused[:, (Hq + Hkv) * d:].reshape(100, Hkv, d)
    pos = rng.integers(0, 5000, size=(100, 3)).astype(np.int32)
    pd = i32(pos)
    vcs.vcs_kv_append_pages(pool, kd, vd, pd, None, 60, 2, 0, ws, status)               # n_d = NULL -> n_cap
    vcs.vcs_kv_append_pages(pool, kd[60:], vd[60:], pd[60:], i32([40]), 40, 2, 60, ws, status)
    opool.append(2, 0, K[:60], V[:60], pos[:60])
    opool.append(2, 60, K[60:], V[60:], pos[60:])
    torch.cuda.synchronize()
    _check_page(pool, opool, 2, "bf16")
    assert int(status) == 0
    # count above capacity clamps; page overflow truncates and flags
    vcs.vcs_kv_append_pages(pool, kd, vd, pd, i32([500]), 100, 1, 0, ws, status)
    torch.cuda.synchronize()
    assert int(status) == vcs.FLAG_COUNT_CLAMPED and int(pool.page_len[1]) == 100
    status.zero_()
    vcs.vcs_kv_append_pages(pool, kd, vd, pd, None, 100, 0, 50, ws, status)
    torch.cuda.synchronize()
    assert int(status) == vcs.FLAG_PAGE_OVERFLOW and int(pool.page_len[0]) == 128
    assert np.array_equal(f64(pool.v_pages[0, :, 50:128]).transpose(1, 0, 2), V[:78])
    with pytest.raises(vcs.VcsError) as e:
        vcs.vcs_kv_append_pages(pool, kd, vd, pd, None, 10, 3, 0, ws, status)
    assert e.value.code == vcs.ECAP


def test_append_batched_matches_oracle_and_flags_bad_page():
    """B streams in one launch: ragged device counts, scattered page ids, one out-of-range id."""
    from paper_2606_19849_b200 import vcs
    Hq, Hkv, d, cap, B, n_cap = 16, 2, 128, 640, 5, 600
    sec = (16, 24, 24)
    pool = vcs.KVPool(12, cap, Hq, Hkv, d, torch.bfloat16, 1e6, sec)
    rng = np.random.default_rng(11)
    K = synth.bf16_round(rng.standard_normal((B, n_cap, Hkv, d)).astype(np.float32))
    V = synth.bf16_round(rng.standard_normal((B, n_cap, Hkv, d)).astype(np.float32))
    pos = rng.integers(0, 5000, size=(B, n_cap, 3)).astype(np.int32)
    ns = np.array([600, 1, 333, 0, 129], dtype=np.int32)
    page_ids = np.array([7, 2, 99, 5, 0], dtype=np.int32)            # stream 2: bad page id
    status = torch.zeros(1, dtype=torch.int32, device="cuda")
    ws = vcs.workspace(vcs.vcs_kv_append_batched_workspace_bytes(pool, n_cap, B))
    for _ in range(2):                                               # twice: the workspace resets itself
        vcs.vcs_kv_append_pages_batched(pool, dev(K, "bf16"), dev(V, "bf16"), i32(pos), i32(ns), n_cap, i32(page_ids), ws, status)
    torch.cuda.synchronize()
    assert int(status) == vcs.FLAG_BAD_PAGE
    for b in range(B):
        if b == 2:
            continue
        n, page = int(ns[b]), int(page_ids[b])
        op = vo.PagedKV(Hq, Hkv, d, 1e6, sec)
        op.append(page, 0, K[b, :n], V[b, :n], pos[b, :n])
        assert int(pool.page_len[page]) == n
        got_k = f64(pool.k_pages[page, :, :n]).transpose(1, 0, 2)
        assert np.max(np.abs(got_k - op.K[page])) <= 2.0 ** -7 * max(1.0, np.max(np.abs(op.K[page]))) if n else True
        assert np.array_equal(f64(pool.v_pages[page, :, :n]).transpose(1, 0, 2), op.V[page])
        assert np.max(np.abs(f64(pool.k_sum[page]) - op.k_sum[page])) <= 1e-4 * max(1.0, n ** 0.5)
    assert int(pool.page_len.sum()) == int(ns.sum() - ns[2])        # nothing written for the bad stream


@pytest.mark.parametrize("strided", [False, True])
def test_append_batched_many_token_groups_per_block(strided):
    """B x n_cap large enough that every block walks several token groups (here 6, more than the V ring has
    slots, so the ring wraps and slots are refilled) with ragged per-stream counts; contiguous rows (one bulk
    copy per group) and strided rows (one per token).  V bit-exact, K within a bf16 ulp, k_sum, untouched tails."""
    from paper_2606_19849_b200 import vcs
    Hq, Hkv, d, cap, B, n_cap = 28, 4, 128, 1100, 16, 1024
    sec = (16, 24, 24)
    pool = vcs.KVPool(B + 2, cap, Hq, Hkv, d, torch.bfloat16, 1e6, sec)
    rng = np.random.default_rng(21 + int(strided))
    width = Hkv * d * (3 if strided else 1)                          # strided: K / V rows are slices of a wider row
    Kw = synth.bf16_round(rng.standard_normal((B, n_cap, width)).astype(np.float32))
    Vw = synth.bf16_round(rng.standard_normal((B, n_cap, width)).astype(np.float32))
    kd = dev(Kw, "bf16")[:, :, Hkv * d * int(strided):Hkv * d * (int(strided) + 1)].unflatten(2, (Hkv, d))
    vd = dev(Vw, "bf16")[:, :, Hkv * d * int(strided):Hkv * d * (int(strided) + 1)].unflatten(2, (Hkv, d))
    K = Kw[:, :, Hkv * d * int(strided):Hkv * d * (int(strided) + 1)].reshape(B, n_cap, Hkv, d)
    V = Vw[:, :, Hkv * d * int(strided):Hkv * d * (int(strided) + 1)].reshape(B, n_cap, Hkv, d)
    assert kd.stride(1) == width and kd.stride(0) == n_cap * width
    pos = rng.integers(0, 20000, size=(B, n_cap, 3)).astype(np.int32)
    ns = rng.integers(0, n_cap + 1, size=B).astype(np.int32)
    ns[0], ns[1], ns[2] = n_cap, 0, 1017                              # full, empty, ragged last group
    page_ids = rng.permutation(B + 2)[:B].astype(np.int32)
    status = torch.zeros(1, dtype=torch.int32, device="cuda")
    ws = vcs.workspace(vcs.vcs_kv_append_batched_workspace_bytes(pool, n_cap, B))
    vcs.vcs_kv_append_pages_batched(pool, kd, vd, i32(pos), i32(ns), n_cap, i32(page_ids), ws, status)
    torch.cuda.synchronize()
    assert int(status) == 0
    for b in range(B):
        n, page = int(ns[b]), int(page_ids[b])
        assert int(pool.page_len[page]) == n
        assert float(pool.v_pages[page, :, n:].abs().sum()) == 0.0 and float(pool.k_pages[page, :, n:].abs().sum()) == 0.0
        if n == 0:
            continue
        op = vo.PagedKV(Hq, Hkv, d, 1e6, sec)
        op.append(page, 0, K[b, :n], V[b, :n], pos[b, :n])
        assert np.array_equal(f64(pool.v_pages[page, :, :n]).transpose(1, 0, 2), op.V[page]), b
        got_k = f64(pool.k_pages[page, :, :n]).transpose(1, 0, 2)
        assert np.all(np.abs(got_k - op.K[page]) <= k_rot_tol(op.K[page])), b
        assert np.max(np.abs(f64(pool.k_sum[page]) - op.k_sum[page])) <= 1e-4 * max(1.0, n ** 0.5), b
