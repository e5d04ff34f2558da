"""GPU parity: vcs_retrieval_score vs the oracle (scores, exact top-k sets and order)."""
import numpy as np
import pytest
import torch

import oracle as vo
import synth
from helpers import dev, f64, i32, tdtype

pytestmark = pytest.mark.gpu


def _bank(dtype, Hq, Hkv, d, n_pages, page_cap, seed):
    from paper_2606_19849_b200 import vcs
    rng = np.random.default_rng(seed)
    sec = (16, 24, 24) if d == 128 else (8, 12, 12)
    pool = vcs.KVPool(n_pages, page_cap, Hq, Hkv, d, tdtype(dtype), 1e6, sec)
    opool = vo.PagedKV(Hq, Hkv, d, 1e6, sec)
    ws = vcs.workspace(vcs.vcs_kv_append_workspace_bytes(pool, page_cap))
    for page in range(n_pages):
        n = int(rng.integers(1, page_cap + 1)) if page % 7 != 3 else 0
        K = rng.standard_normal((n, Hkv, d)).astype(np.float32) + 0.3 * rng.standard_normal((1, Hkv, d)).astype(np.float32)
        V = rng.standard_normal((n, Hkv, d)).astype(np.float32)
        if dtype == "bf16":
            K, V = synth.bf16_round(K), synth.bf16_round(V)
        pos = rng.integers(0, 999, size=(n, 3)).astype(np.int32)
        if n:
            vcs.vcs_kv_append_pages(pool, dev(K, dtype), dev(V, dtype), i32(pos), None, n, page, 0, ws)
        opool.append(page, 0, K, V, pos)
    return vcs, pool, opool, rng


@pytest.mark.parametrize("dtype,Hq,Hkv,d,normalize", [("bf16", 28, 4, 128, False), ("bf16", 28, 4, 128, True),
                                                       ("f32", 2, 1, 64, True), ("bf16", 16, 2, 128, False)])
def test_retrieval_scores_and_topk(dtype, Hq, Hkv, d, normalize):
    vcs, pool, opool, rng = _bank(dtype, Hq, Hkv, d, 40, 64, seed=Hq + d)
    nq = 48
    Q = rng.standard_normal((nq, Hq, d)).astype(np.float32)
    Q = synth.bf16_round(Q) if dtype == "bf16" else Q
    cand = rng.permutation(40)[:33].astype(np.int32)
    excl = cand[[2, 9, 30]]
    k = 8
    scores = torch.zeros(33, dtype=torch.float32, device="cuda")
    topk = torch.full((k,), -9, dtype=torch.int32, device="cuda")
    ws = vcs.workspace(vcs.vcs_retrieval_score_workspace_bytes(pool, 33))
    for _ in range(2):
        vcs.vcs_retrieval_score(pool, dev(Q, dtype), i32([nq]), nq, i32(cand), scores, ws, k=k, topk_pages=topk,
                                exclude_pages=i32(excl), normalize=normalize)
    torch.cuda.synchronize()
    ref = vo.retrieval_scores(opool, Q, cand, normalize)
    # fp32 means and dots over Hkv*d terms: absolute error relative to |q_bar||x_bar|
    qb = vo.mean_query(Q, Hkv).ravel()
    bound = np.array([np.linalg.norm(qb) * (np.linalg.norm(opool.k_sum[int(p)]) / max(opool.page_len(int(p)), 1))
                      for p in cand])
    tol = 1e-5 * (bound if not normalize else 1.0) + 1e-7
    assert np.all(np.abs(f64(scores) - ref) <= tol)
    ref_top = vo.retrieve_topk(ref, cand, k, exclude_pages=excl)
    srt = np.sort(ref[~np.isin(cand, excl)])[::-1]
    assert np.min(np.abs(np.diff(srt[:k + 1]))) > 1e-6           # seeded gap: the order is well defined
    assert topk.cpu().numpy().tolist() == ref_top.tolist()


def test_retrieval_ties_padding_and_no_topk():
    vcs, pool, opool, rng = _bank("bf16", 4, 2, 128, 12, 32, seed=1)
    Q = np.zeros((4, 4, 128), dtype=np.float32)                  # all scores 0 -> ties -> ascending page id
    cand = np.array([7, 2, 9, 4, 11], dtype=np.int32)
    scores = torch.ones(5, dtype=torch.float32, device="cuda")
    topk = torch.full((7,), -9, dtype=torch.int32, device="cuda")
    ws = vcs.workspace(vcs.vcs_retrieval_score_workspace_bytes(pool, 5))
    vcs.vcs_retrieval_score(pool, dev(Q, "bf16"), None, 4, i32(cand), scores, ws, k=7, topk_pages=topk,
                            exclude_pages=i32([9]))
    torch.cuda.synchronize()
    assert scores.cpu().tolist() == [0.0] * 5
    assert topk.cpu().tolist() == [2, 4, 7, 11, -1, -1, -1]
    vcs.vcs_retrieval_score(pool, dev(Q, "bf16"), None, 4, i32(cand), scores, ws)   # scores only
    torch.cuda.synchronize()


def test_retrieval_threshold_visibility():
    """V_qry = {j : s_j >= tau_q}: GPU list == oracle list (candidate order, exclusions,
    clamped capacity, -1 padding); tau_q is placed in the widest score gap so fp32 vs fp64 cannot flip it."""
    vcs, pool, opool, rng = _bank("bf16", 28, 4, 128, 300, 64, seed=9)
    nq = 48
    Q = synth.bf16_round(rng.standard_normal((nq, 28, 128)).astype(np.float32))
    cand = [int(p) for p in rng.permutation(300)[:280]]
    excl = cand[5:9]
    ref = vo.retrieval_scores(opool, Q, cand)
    scores = torch.zeros(len(cand), dtype=torch.float32, device="cuda")
    ws = vcs.workspace(vcs.vcs_retrieval_score_workspace_bytes(pool, len(cand)))
    vcs.vcs_retrieval_score(pool, dev(Q, "bf16"), None, nq, i32(cand), scores, ws)
    srt = np.sort(ref)
    for frac in (0.05, 0.4, 0.75):
        lo = int(frac * len(cand))
        g = int(np.argmax(srt[lo + 1:lo + 61] - srt[lo:lo + 60])) + lo     # widest gap after the quantile (empty pages tie at 0)
        tau_q = 0.5 * (srt[g] + srt[g + 1])
        assert srt[g + 1] - srt[g] > 1e-5 * max(1.0, np.max(np.abs(ref)))
        want = [p for p in vo.retrieve_threshold(ref, cand, tau_q) if p not in excl]
        for cap in (len(cand), 7):
            vis = torch.full((cap,), 123, dtype=torch.int32, device="cuda")
            cnt = torch.zeros(1, dtype=torch.int32, device="cuda")
            vcs.vcs_retrieval_threshold(pool, scores, i32(cand), tau_q, vis, cnt, exclude_pages=i32(excl))
            torch.cuda.synchronize()
            n = min(len(want), cap)
            assert int(cnt) == n
            assert vis.cpu().tolist() == want[:n] + [-1] * (cap - n)
    # tau above every score: nothing visible; below: everything not excluded
    vis = torch.zeros(len(cand), dtype=torch.int32, device="cuda")
    cnt = torch.ones(1, dtype=torch.int32, device="cuda")
    vcs.vcs_retrieval_threshold(pool, scores, i32(cand), 1e30, vis, cnt)
    assert int(cnt) == 0 and bool((vis == -1).all())
    vcs.vcs_retrieval_threshold(pool, scores, i32(cand), -1e30, vis, cnt, exclude_pages=i32(excl))
    assert int(cnt) == len(cand) - len(excl)


_BIG = {}


def _big_bank():
    """4112 small pages (1..8 tokens, every 11th empty, every page with id % 5 == 1 a copy of its predecessor so that
    equal scores exist), built once per process on both sides."""
    if not _BIG:
        from paper_2606_19849_b200 import vcs
        rng = np.random.default_rng(77)
        Hq, Hkv, d, n_pages, cap = 28, 4, 128, 4112, 8
        pool = vcs.KVPool(n_pages, cap, Hq, Hkv, d, torch.bfloat16, 1e6, (16, 24, 24))
        opool = vo.PagedKV(Hq, Hkv, d, 1e6, (16, 24, 24))
        ws = vcs.workspace(vcs.vcs_kv_append_workspace_bytes(pool, cap))
        prev = None
        for page in range(n_pages):
            if page % 5 == 1 and prev is not None and prev[0].shape[0] > 0:
                K, V, pos = prev
            else:
                n = 0 if page % 11 == 7 else int(rng.integers(1, cap + 1))
                K = synth.bf16_round((rng.standard_normal((n, Hkv, d)) + 0.5 * rng.standard_normal((1, Hkv, d))).astype(np.float32))
                V = synth.bf16_round(rng.standard_normal((n, Hkv, d)).astype(np.float32))
                pos = rng.integers(0, 999, size=(n, 3)).astype(np.int32)
            n = K.shape[0]
            if n:
                vcs.vcs_kv_append_pages(pool, dev(K, "bf16"), dev(V, "bf16"), i32(pos), None, n, page, 0, ws)
            opool.append(page, 0, K, V, pos)
            prev = (K, V, pos)
        Q = synth.bf16_round(rng.standard_normal((48, Hq, d)).astype(np.float32))
        _BIG.update(vcs=vcs, pool=pool, opool=opool, Q=Q)
    return _BIG["vcs"], _BIG["pool"], _BIG["opool"], _BIG["Q"]


@pytest.mark.parametrize("n_cand,k", [(257, 1), (257, 256), (1000, 8), (1000, 256), (4096, 1), (4096, 8), (4096, 256)])
def test_topk_over_more_than_256_candidates(n_cand, k):
    """"Only the top-k chunks are exposed to query tokens" on banks larger than one block of threads:
    the k-rounds-of-arg-max branch of score_topk_kernel, with excluded pages, equal scores (copied pages, ties go to
    the lower page id, reading D22), empty pages, NaN summaries on the pages that would otherwise win, and fewer
    eligible candidates than k (-1 padding).  Scores are compared with the oracle's within the fp32 bound; the LIST is
    the oracle's retrieve_topk taken on the device's own fp32 scores (both sides decide in the same precision), and
    every listed page must also be a defensible winner under the oracle's fp64 scores."""
    vcs, pool, opool, Q = _big_bank()
    rng = np.random.default_rng(n_cand * 1000 + k)
    cand = rng.permutation(4112)[:n_cand].astype(np.int32)
    ref = vo.retrieval_scores(opool, Q, cand)
    order = np.argsort(-ref)
    nan_pages = cand[order[[0, 3]]]                               # the best and the fourth best page get NaN summaries
    excl = np.concatenate([cand[order[[1, 6]]], cand[rng.permutation(n_cand)[:6]]]).astype(np.int32)
    saved = pool.k_sum[torch.as_tensor(nan_pages.astype(np.int64), device="cuda")].clone()
    scores = torch.zeros(n_cand, dtype=torch.float32, device="cuda")
    topk = torch.full((k,), -9, dtype=torch.int32, device="cuda")
    ws = vcs.workspace(vcs.vcs_retrieval_score_workspace_bytes(pool, n_cand))
    try:
        pool.k_sum[torch.as_tensor(nan_pages.astype(np.int64), device="cuda")] = float("nan")
        for _ in range(2):                                        # twice: the eligibility flags cleared by a round are rebuilt
            vcs.vcs_retrieval_score(pool, dev(Q, "bf16"), None, 48, i32(cand), scores, ws, k=k, topk_pages=topk,
                                    exclude_pages=i32(excl))
        torch.cuda.synchronize()
    finally:
        pool.k_sum[torch.as_tensor(nan_pages.astype(np.int64), device="cuda")] = saved
    got_s, got = f64(scores), topk.cpu().numpy()
    is_nan = np.isin(cand, nan_pages)
    assert np.isnan(got_s[is_nan]).all() and not np.isnan(got_s[~is_nan]).any()
    qb = vo.mean_query(Q, 4).ravel()
    bound = np.array([np.linalg.norm(qb) * (np.linalg.norm(opool.k_sum[int(p)]) / max(opool.page_len(int(p)), 1)) for p in cand])
    tol = 1e-5 * bound + 1e-7
    assert np.all(np.abs(got_s - ref)[~is_nan] <= tol[~is_nan])
    out = np.concatenate([excl, nan_pages])
    want = vo.retrieve_topk(np.where(is_nan, 0.0, got_s), cand, k, exclude_pages=out)
    assert got.tolist() == want.tolist()
    n_elig = int((~np.isin(cand, out)).sum())
    assert (got >= 0).sum() == min(k, n_elig)
    if k == 256 and n_cand == 257:
        assert n_elig < k and got[-1] == -1                       # the padding case really occurs
    # under the oracle's own scores: nobody outside the list beats the weakest listed page by more than the bound
    listed = got[got >= 0]
    s_of = {int(p): ref[c] for c, p in enumerate(cand)}
    if len(listed) < n_elig:
        weakest = min(s_of[int(p)] for p in listed)
        rest = [s_of[int(p)] for p in cand if p not in set(listed.tolist()) and p not in set(out.tolist())]
        assert max(rest) <= weakest + 2 * tol.max()
    # equal scores exist among the winners of the large lists and resolve to ascending page id
    if k == 256 and n_cand >= 1000:
        gs = {int(p): got_s[c] for c, p in enumerate(cand)}
        ties = [(a, b) for a, b in zip(listed[:-1], listed[1:]) if gs[int(a)] == gs[int(b)]]
        assert ties and all(a < b for a, b in ties)
