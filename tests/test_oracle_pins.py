"""Pins for the oracle (CPU, -m "not gpu"): the oracle is checked against what the paper and the
mathematics fix -- printed values (tests/golden), closed forms, invariants, special cases that
reduce to a textbook / library routine, brute force on tiny inputs.  Nothing here touches the
CUDA path.  SURVEY.md section 8(c) "What pins each part" is the checklist.
"""
import itertools
import os

import numpy as np
import pytest
import torch

import oracle as vo
import synth

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
SEC128 = (16, 24, 24)
SEC64 = (8, 12, 12)


def _rows(path):
    with open(os.path.join(GOLDEN, path)) as f:
        return [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]


# ------------------------------------------------------------------ similarity (Eq. 1) --------
def test_cosine_hand_cases():
    assert vo.cosine_similarity([1, 0], [1, 0]) == 1.0
    assert vo.cosine_similarity([1, 0], [0, 1]) == 0.0
    assert abs(vo.cosine_similarity([1, 0], [1, 1]) - 0.70710678118654752) < 1e-15
    assert vo.cosine_similarity([1, 0], [-2, 0]) == -1.0
    assert vo.cosine_similarity([0, 0], [1, 1]) == 0.0          # reading D6


def test_cosine_matches_library_and_scale_invariance():
    rng = np.random.default_rng(1)
    for _ in range(20):
        a, b = rng.standard_normal(37), rng.standard_normal(37)
        lib = np.dot(a, b) / (np.linalg.norm(a) * np.linalg.norm(b))
        assert abs(vo.cosine_similarity(a, b) - lib) < 1e-14
        assert abs(vo.cosine_similarity(3.5 * a, 0.01 * b) - lib) < 1e-14
        assert abs(vo.cosine_similarity(b, a) - lib) < 1e-14


def test_pairwise_similarity_indexing():
    # tokens in the plane at chosen angles: S[i,j,p] must be cos(angle_i - angle_j) at THAT p
    ang = np.array([[0.0, 0.3], [0.5, 1.0], [2.0, -1.0]])       # [G=3][P=2]
    Z = np.stack([np.cos(ang), np.sin(ang)], axis=-1) * np.array([1.0, 2.0, 0.5])[:, None, None]
    S = vo.pairwise_similarity(Z)
    for p in range(2):
        for i, j in [(0, 1), (0, 2), (1, 2)]:
            assert abs(S[i, j, p] - np.cos(ang[i, p] - ang[j, p])) < 1e-14
    assert np.isnan(S[1, 0, 0]) and np.isnan(S[0, 0, 0])


# ------------------------------------------------------------------ drop rule (Eq. 2) ---------
def _random_chunk(G=4, P=12, D=16, seed=0, rho=0.5):
    rng = np.random.default_rng(seed)
    static = rng.random(P) < rho
    base = rng.standard_normal((P, D))
    Z = rng.standard_normal((G, P, D))
    Z = np.where(static[None, :, None], base[None] + 0.05 * rng.standard_normal((G, P, D)), Z)
    return Z, static


def test_tau_one_keeps_everything_paper_s1():
    # Table 8-left: "Baseline (s=1.0, 0%)": cosine <= 1 can never exceed tau = 1.
    # IDENTICAL tokens (static pixels) are the case that matters: the raw fp64 quotient lands at
    # 1 + 1 ulp for a good share of them (reading D31: the oracle clamps to [-1, 1]).
    Z, _ = _random_chunk()
    Z[:, 0, :] = Z[0, 0, :]                                     # identical tokens: S = 1 exactly
    keep, idx, n = vo.temporal_drop(Z, 1.0)
    assert keep.all() and n == Z.shape[0] * Z.shape[1]
    assert np.array_equal(idx, np.arange(n))
    Z[:, 1, :] = 0.0
    Z[:, 1, 3] = [1.0, 2.0, 4.0, 0.5]                           # parallel tokens: S = 1 exactly
    assert vo.temporal_drop(Z, 1.0)[0].all()


def test_cosine_bound_on_identical_and_opposite_tokens_d31():
    # |S| <= 1 (Cauchy-Schwarz) must hold for EVERY input, rounding included: 2000 random identical /
    # opposite / scaled pairs in several dimensions; every group of a chunk identical -> nothing can be
    # dropped at tau = 1 and everything non-anchor is dropped just below 1 (strictness, reading D3).
    rng = np.random.default_rng(2)
    over = 0
    for k in range(2000):
        D = int(rng.choice([3, 16, 128, 2048]))
        a = rng.standard_normal(D)
        raw = np.sum(a * a) / (np.sqrt(np.sum(a * a)) * np.sqrt(np.sum(a * a)))
        over += raw > 1.0
        assert vo.cosine_similarity(a, a) <= 1.0
        assert vo.cosine_similarity(a, -a) >= -1.0
        assert vo.cosine_similarity(a, 3.0 * a) <= 1.0
        assert vo.cosine_similarity(a, a) > 1.0 - 1e-15
    assert over > 100                                            # the unclamped quotient does exceed 1: the pin bites
    Z = np.repeat(rng.standard_normal((1, 12, 64)), 4, axis=0)    # four identical groups
    keep, idx, n = vo.temporal_drop(Z, 1.0)
    assert keep.all() and n == 48
    keep, idx, n = vo.temporal_drop(Z, 1.0 - 1e-9)
    assert n == 12 and keep[0].all() and not keep[1:].any()
    assert vo.temporal_keep_mask(Z, 1.0, mode=1, prev_last_group=Z[0]).all()


def test_tau_below_minus_one_drops_all_non_anchor():
    # every similarity > tau  =>  only the anchor group survives: count = P, rate = (G-1)/G,
    # the bound behind the paper's 74 % < 75 % at c=4
    Z, _ = _random_chunk(G=4, P=12)
    keep, idx, n = vo.temporal_drop(Z, -1.5)
    assert n == 12 and np.array_equal(idx, np.arange(12))
    assert keep[0].all() and not keep[1:].any()
    assert 1.0 - n / keep.size == 0.75


def test_golden_table8_rule_properties():
    rows = [(float(s), float(r)) for s, r in _rows("table8_drop_rates.txt")]
    assert rows[0] == (1.0, 0.0)
    rates = [r for _, r in rows]
    assert all(a < b for a, b in zip(rates, rates[1:]))          # rate grows as s falls
    assert max(rates) < 75.0                                     # anchor bound (G-1)/G at c=4
    # the oracle obeys the same three properties on a mixed chunk
    rng = np.random.default_rng(5)
    G, P, D = 4, 64, 24
    base = rng.standard_normal((P, D))
    noise = rng.random(P)[None, :, None] * 2.0                   # graded redundancy per position
    Z = base[None] + noise * rng.standard_normal((G, P, D))
    prev = -1.0
    for s, _ in rows:
        keep, _, n = vo.temporal_drop(Z, s)
        rate = 1.0 - n / keep.size
        assert keep[0].all()
        assert rate >= prev and rate <= 0.75
        prev = rate
    assert vo.temporal_drop(Z, 1.0)[2] == G * P


def test_strict_inequality_and_zero_norm():
    e0, e1 = np.array([1.0, 0.0]), np.array([0.0, 1.0])
    Z = np.stack([np.stack([e0, e0]), np.stack([e0, e1])])      # [G=2][P=2]: S = (1, 0)
    assert vo.drop_predicate(Z, 1.0).tolist() == [False, False]   # S == tau is NOT dropped
    assert vo.drop_predicate(Z, 0.0).tolist() == [True, False]
    assert vo.drop_predicate(Z, -1e-9).tolist() == [True, True]
    Zz = np.stack([np.stack([e0, np.zeros(2)]), np.stack([e0, e1])])
    assert vo.drop_predicate(Zz, 0.5).tolist() == [True, False]   # zero norm: S := 0 (D6)
    assert vo.drop_predicate(Zz, -0.5).tolist() == [True, True]


def test_drop_predicate_group_permutation_invariant():
    Z, _ = _random_chunk(G=4, P=20, seed=3)
    ref = vo.drop_predicate(Z, 0.95)
    assert ref.any() and not ref.all()
    for perm in itertools.permutations(range(4)):
        assert np.array_equal(vo.drop_predicate(Z[list(perm)], 0.95), ref)


def test_all_pairs_not_just_consecutive():
    # angles 0, 20, 40 deg: consecutive cos = 0.94 > 0.9 but cos(0,40 deg) = 0.766 < 0.9
    a = np.deg2rad([0.0, 20.0, 40.0])
    Z = np.stack([np.cos(a), np.sin(a)], axis=-1)[:, None, :]   # [G=3][P=1][2]
    assert vo.drop_predicate(Z, 0.9).tolist() == [False]        # Eq. 2 is over ALL pairs i<j
    assert vo.drop_predicate(Z, 0.75).tolist() == [True]
    keep1 = vo.temporal_keep_mask(Z, 0.9, mode=1)               # consecutive variant differs
    assert keep1[:, 0].tolist() == [True, False, False]


def test_brute_force_all_patterns():
    # every subset of P = 4 positions made "redundant" by construction; G = 3
    G, P = 3, 4
    for pattern in itertools.product([False, True], repeat=P):
        Z = np.zeros((G, P, 2))
        for p, red in enumerate(pattern):
            spread = 0.02 if red else 1.2                        # radians between groups
            for g in range(G):
                Z[g, p] = (1 + g) * np.array([np.cos(p + g * spread), np.sin(p + g * spread)])
        keep, idx, n = vo.temporal_drop(Z, 0.95)
        assert keep[0].all()
        for p, red in enumerate(pattern):
            assert keep[1:, p].tolist() == [not red] * (G - 1)
        expect = [g * P + p for g in range(G) for p in range(P) if g == 0 or not pattern[p]]
        assert idx.tolist() == expect and n == len(expect)


def test_compaction_matches_flatnonzero():
    rng = np.random.default_rng(7)
    for _ in range(10):
        keep = rng.random((3, 17)) < 0.4
        idx, n = vo.compact(keep)
        assert np.array_equal(idx, np.flatnonzero(keep.ravel()))
        assert n == int(keep.sum()) and np.all(np.diff(idx) > 0)
    idx, n = vo.compact(np.zeros((2, 5), dtype=bool))
    assert n == 0 and idx.size == 0


def test_modes_agree_for_two_groups_and_mode1_prev():
    Z, _ = _random_chunk(G=2, P=30, seed=9)
    k0 = vo.temporal_keep_mask(Z, 0.9, mode=0)
    k1 = vo.temporal_keep_mask(Z, 0.9, mode=1)
    assert np.array_equal(k0, k1) and not k0.all()
    prev = Z[0] * 2.0                                            # cos(prev, Z[0]) = 1 > tau
    k1p = vo.temporal_keep_mask(Z, 0.9, mode=1, prev_last_group=prev)
    assert not k1p[0].any() and np.array_equal(k1p[1], k1[1])   # no anchor in frame-level mode
    Z1 = Z[:1]
    assert vo.temporal_keep_mask(Z1, 0.9, mode=0).all()          # G = 1: anchor only (D10)


def test_generator_expected_kept_fraction_and_margin():
    # E[kept] = 1 - rho (G-1)/G under the DESIGN.md recipe; similarities stay 1e-4 away from tau
    cfg = synth.get_config("vl3b").with_(Hg=8, Wg=12, D=256)
    tot = kept = 0
    for t in range(6):
        Z, static = synth.gen_hidden_chunk(cfg, t)
        S = vo.pairwise_similarity(Z)
        vals = S[~np.isnan(S)]
        assert np.min(np.abs(vals - cfg.tau)) >= 1e-4
        keep, idx, n = vo.temporal_drop(Z, cfg.tau)
        assert np.array_equal(~keep[1], static)                  # static positions are the dropped ones
        assert np.array_equal(keep, vo.temporal_keep_mask(Z, cfg.tau, mode=1))
        tot += keep.size
        kept += n
    assert abs(kept / tot - (1 - cfg.rho * (cfg.G - 1) / cfg.G)) < 0.05


def test_tiny_generator_margin():
    cfg = synth.get_config("tiny")
    Z = synth.gen_hidden_tiny(cfg)
    fr = []
    for t in range(cfg.n_chunks):
        S = vo.pairwise_similarity(Z[t])
        assert np.min(np.abs(S[~np.isnan(S)] - cfg.tau)) >= 1e-4
        fr.append(vo.temporal_drop(Z[t], cfg.tau)[2] / cfg.T)
    assert 0.55 < np.mean(fr) < 0.95                             # ~ 1 - 0.5*(1/2) = 0.75


# ------------------------------------------------------------------ positions (O2) ------------
def test_grid_positions_and_base():
    pos = vo.grid_positions(G=2, Hg=2, Wg=3, base=10, t_stride=1)
    assert pos.shape == (12, 3)
    assert pos[0].tolist() == [10, 10, 10]
    assert pos[2].tolist() == [10, 10, 12]
    assert pos[3].tolist() == [10, 11, 10]
    assert pos[6 + 5].tolist() == [11, 11, 12]
    assert vo.next_position_base(2, 2, 3, 10) == 13
    assert vo.next_position_base(4, 16, 29, 64) == 64 + 29
    assert vo.next_position_base(40, 16, 29, 0, t_stride=1) == 40
    assert vo.text_positions(5, 3).tolist() == [[5, 5, 5], [6, 6, 6], [7, 7, 7]]


# ------------------------------------------------------------------ M-RoPE (O3) ---------------
def _textbook_rope_1d(x, n, theta):
    """1-D rotary embedding written with complex numbers: (x_m + i x_{m+d/2}) * exp(i n f_m)."""
    d = x.shape[-1]
    half = d // 2
    f = theta ** (-2.0 * np.arange(half) / d)
    z = (x[..., :half] + 1j * x[..., half:]) * np.exp(1j * n[:, None, None] * f)
    return np.concatenate([z.real, z.imag], axis=-1)


def test_mrope_reduces_to_1d_rope():
    rng = np.random.default_rng(11)
    x = rng.standard_normal((9, 3, 128))
    n = rng.integers(0, 5000, size=9)
    pos3 = np.stack([n, n, n], axis=1)
    got = vo.mrope_rotate(x, pos3, 1e6, SEC128)
    assert np.max(np.abs(got - _textbook_rope_1d(x, n.astype(float), 1e6))) < 1e-9


def test_mrope_identity_norm_shift_sections():
    rng = np.random.default_rng(12)
    x = rng.standard_normal((6, 2, 64))
    pos = rng.integers(0, 300, size=(6, 3))
    assert np.array_equal(vo.mrope_rotate(x, np.zeros((6, 3), int), 1e6, SEC64), x)
    r = vo.mrope_rotate(x, pos, 1e6, SEC64)
    assert np.allclose(np.linalg.norm(r, axis=-1), np.linalg.norm(x, axis=-1), atol=1e-12)
    # relative property: <rot(q,p+D), rot(k,p'+D)> == <rot(q,p), rot(k,p')> for a common shift D
    q, k = rng.standard_normal((6, 2, 64)), rng.standard_normal((6, 2, 64))
    pq, pk = rng.integers(0, 300, (6, 3)), rng.integers(0, 300, (6, 3))
    shift = np.array([17, 5, 123])
    a = np.sum(vo.mrope_rotate(q, pq, 1e6, SEC64) * vo.mrope_rotate(k, pk, 1e6, SEC64), -1)
    b = np.sum(vo.mrope_rotate(q, pq + shift, 1e6, SEC64) * vo.mrope_rotate(k, pk + shift, 1e6, SEC64), -1)
    assert np.max(np.abs(a - b)) < 1e-9
    # section assignment: changing only h moves only the h-section pairs (pairs 8..19 for d=64)
    p2 = pos.copy()
    p2[:, 1] += 7
    diff = np.abs(vo.mrope_rotate(x, p2, 1e6, SEC64) - r).max(axis=(0, 1))
    moved = np.flatnonzero(diff > 1e-12)
    expect = np.concatenate([np.arange(8, 20), 32 + np.arange(8, 20)])
    assert np.array_equal(moved, expect)


def test_mrope_direction_and_frequency():
    # pair 0 has f = 1: rotating (1, 0) by position n gives (cos n, sin n) -- sign convention
    x = np.zeros((1, 1, 64))
    x[0, 0, 0] = 1.0
    r = vo.mrope_rotate(x, np.array([[2, 0, 0]]), 1e6, SEC64)
    assert abs(r[0, 0, 0] - np.cos(2.0)) < 1e-15 and abs(r[0, 0, 32] - np.sin(2.0)) < 1e-15
    # pair m = 8 is the first h pair with f = theta^(-16/64)
    x = np.zeros((1, 1, 64))
    x[0, 0, 8] = 1.0
    r = vo.mrope_rotate(x, np.array([[9, 3, 0]]), 1e6, SEC64)
    a = 3 * 1e6 ** (-0.25)
    assert abs(r[0, 0, 8] - np.cos(a)) < 1e-15 and abs(r[0, 0, 40] - np.sin(a)) < 1e-15


# ------------------------------------------------------------------ attention (O5) ------------
def _mini_stream(n_chunks=4, W=2, sink=5, Hq=4, Hkv=2, d=64, seed=0, lens=(7, 9, 4, 11, 6, 8), sharp=3.0):
    """Sink + chunks appended to an oracle pool with scattered page ids; returns everything."""
    rng = np.random.default_rng(seed)
    pool = vo.PagedKV(Hq, Hkv, d, 1e6, SEC64 if d == 64 else SEC128)
    pages = synth.gen_page_ids(32, n_chunks + 1, seed)
    Ks, Vs, Qs, Ps = [], [], [], []
    K, V = rng.standard_normal((sink, Hkv, d)), rng.standard_normal((sink, Hkv, d))
    pos = vo.text_positions(0, sink)
    pool.append(int(pages[0]), 0, K, V, pos)
    Ks.append(K); Vs.append(V); Ps.append(pos); Qs.append(np.zeros((sink, Hq, d)))
    base = sink
    for t in range(n_chunks):
        n = lens[t]
        pos = np.stack([base + rng.integers(0, 3, n), base + rng.integers(0, 9, n), base + rng.integers(0, 9, n)], 1)
        Q = sharp * rng.standard_normal((n, Hq, d))
        K, V = rng.standard_normal((n, Hkv, d)), rng.standard_normal((n, Hkv, d))
        pool.append(int(pages[t + 1]), 0, K, V, pos)
        Ks.append(K); Vs.append(V); Ps.append(pos); Qs.append(Q)
        base += 9
    return pool, pages, Qs, Ks, Vs, Ps


def test_softmax_rows_sum_to_one_and_lse():
    pool, pages, Qs, Ks, Vs, Ps = _mini_stream()
    O, lse, P = vo.bounded_attention(pool, Qs[3], Ps[3], [int(pages[0]), int(pages[1]), int(pages[2])],
                                     self_page=int(pages[3]), return_probs=True)
    assert np.max(np.abs(P.sum(axis=2) - 1.0)) < 1e-13
    n_full = 5 + 7 + 9
    for i in range(Qs[3].shape[0]):                               # causal part of the self page
        assert np.all(P[:, i, n_full + i + 1:] == 0.0) and np.all(P[:, i, :n_full + i + 1] > 0.0)
    # lse definition: log sum exp of the scaled visible logits, recomputed directly for one row
    Qr = vo.mrope_rotate(Qs[3], Ps[3], 1e6, SEC64)
    Kc = np.concatenate([pool.K[int(p)] for p in pages[:4]], 0)
    i, h = 2, 3
    logits = (Kc[:n_full + i + 1, h // 2] @ Qr[i, h]) / np.sqrt(64)
    assert abs(lse[h, i] - np.log(np.sum(np.exp(logits)))) < 1e-12


def test_unbounded_window_equals_full_causal_sdpa():
    """W = inf, no retrieval == textbook full causal attention over sink + all chunks; checked
    against torch's scaled_dot_product_attention (library routine) in fp64 on CPU."""
    pool, pages, Qs, Ks, Vs, Ps = _mini_stream(n_chunks=4)
    Hq, Hkv, d = 4, 2, 64
    Qall = vo.mrope_rotate(np.concatenate(Qs), np.concatenate(Ps), 1e6, SEC64)
    Kall = vo.mrope_rotate(np.concatenate(Ks), np.concatenate(Ps), 1e6, SEC64)
    Vall = np.concatenate(Vs)
    q = torch.from_numpy(Qall).permute(1, 0, 2)[None]
    k = torch.from_numpy(np.repeat(Kall, Hq // Hkv, axis=1)).permute(1, 0, 2)[None]
    v = torch.from_numpy(np.repeat(Vall, Hq // Hkv, axis=1)).permute(1, 0, 2)[None]
    ref = torch.nn.functional.scaled_dot_product_attention(q, k, v, is_causal=True)[0].permute(1, 0, 2).numpy()
    start = 5
    for t in range(4):
        n = Qs[t + 1].shape[0]
        vis = [int(p) for p in pages[:t + 1]]
        O, _ = vo.bounded_attention(pool, Qs[t + 1], Ps[t + 1], vis, self_page=int(pages[t + 1]))
        assert np.max(np.abs(O - ref[start:start + n])) < 1e-12
        start += n


def test_page_table_mask_equals_eq4_mask():
    """The paged visible-set construction reproduces the paper's Eq. 4 staircase mask
    (V_vis(t) = {t-acn..t}) + sink + causality, for acn = 1 and 2."""
    for acn in (1, 2):
        pool, pages, Qs, Ks, Vs, Ps = _mini_stream(n_chunks=5, W=acn, seed=3)
        chunk_of, kind = [], []
        for c, K in enumerate(Ks):
            chunk_of += [c - 1] * K.shape[0]
            kind += ["sink" if c == 0 else "vis"] * K.shape[0]
        M = vo.eq4_mask(chunk_of, kind, acn)
        Qall = vo.mrope_rotate(np.concatenate(Qs), np.concatenate(Ps), 1e6, SEC64)
        Kall = vo.mrope_rotate(np.concatenate(Ks), np.concatenate(Ps), 1e6, SEC64)
        Vall = np.concatenate(Vs)
        start = 5
        for t in range(5):
            n = Qs[t + 1].shape[0]
            lo = max(0, t - acn)
            vis = [int(pages[0])] + [int(p) for p in pages[1 + lo:1 + t]]
            O, _ = vo.bounded_attention(pool, Qs[t + 1], Ps[t + 1], vis, self_page=int(pages[t + 1]))
            for h in range(4):
                ref = vo.masked_attention_dense(Qall[start:start + n, h], Kall[:, h // 2], Vall[:, h // 2],
                                                M[start:start + n], 1 / 8.0)
                assert np.max(np.abs(O[:, h] - ref)) < 1e-12
            start += n
        # staircase: a row of chunk 4 must NOT see chunk 4-acn-1
        row = 5 + sum(Q.shape[0] for Q in Qs[1:5])
        far = 5 + sum(Q.shape[0] for Q in Qs[1:1 + (4 - acn - 1)])
        assert not M[row, far] and M[row, 0]


def test_attention_page_permutation_and_physical_ids():
    pool, pages, Qs, Ks, Vs, Ps = _mini_stream(n_chunks=4)
    vis = [int(p) for p in pages[:4]]
    O, lse = vo.bounded_attention(pool, Qs[4], Ps[4], vis, self_page=int(pages[4]))
    O2, lse2 = vo.bounded_attention(pool, Qs[4], Ps[4], vis[::-1], self_page=int(pages[4]))
    assert np.max(np.abs(O - O2)) < 1e-12 and np.max(np.abs(lse - lse2)) < 1e-12
    pool2 = vo.PagedKV(4, 2, 64, 1e6, SEC64)                      # same content, other page ids
    for c in range(5):
        pool2.append(100 + c, 0, Ks[c], Vs[c], Ps[c])
    O3, _ = vo.bounded_attention(pool2, Qs[4], Ps[4], [103, 100, 102, 101], self_page=104)
    assert np.max(np.abs(O - O3)) < 1e-12


def test_zero_query_gives_mean_of_visible_values():
    pool, pages, Qs, Ks, Vs, Ps = _mini_stream(n_chunks=3)
    n = Qs[3].shape[0]
    vis = [int(pages[0]), int(pages[2])]                          # sink + chunk 1 (skip chunk 0)
    O, lse = vo.bounded_attention(pool, np.zeros_like(Qs[3]), Ps[3], vis, self_page=int(pages[3]), self_offset=0)
    Vfull = np.concatenate([Vs[0], Vs[2]])
    for i in range(n):
        allv = np.concatenate([Vfull, Vs[3][:i + 1]])
        for h in range(4):
            assert np.max(np.abs(O[i, h] - allv[:, h // 2].mean(axis=0))) < 1e-13
        assert np.allclose(lse[:, i], np.log(allv.shape[0]))
    # self_offset shifts the causal limit: row i sees self tokens [0, off + i]
    O2, _ = vo.bounded_attention(pool, np.zeros((2, 4, 64)), Ps[3][:2], [], self_page=int(pages[3]), self_offset=2)
    assert np.max(np.abs(O2[0, 0] - Vs[3][:3, 0].mean(axis=0))) < 1e-13
    assert np.max(np.abs(O2[1, 3] - Vs[3][:4, 1].mean(axis=0))) < 1e-13


def test_single_key_and_negligible_page_and_gqa():
    rng = np.random.default_rng(21)
    pool = vo.PagedKV(4, 2, 64, 1e6, SEC64)
    K1, V1 = rng.standard_normal((1, 2, 64)), rng.standard_normal((1, 2, 64))
    pool.append(3, 0, K1, V1, np.zeros((1, 3), int))
    Q = rng.standard_normal((5, 4, 64))
    zero = np.zeros((5, 3), int)
    O, _ = vo.bounded_attention(pool, Q, zero, [3])
    for h in range(4):
        assert np.max(np.abs(O[:, h] - V1[0, h // 2])) < 1e-14     # single visible key, GQA map (D16)
    # a page whose logits are <= -1e4 below the rest changes nothing
    Kb = rng.standard_normal((6, 2, 64))
    pool.append(5, 0, Kb, rng.standard_normal((6, 2, 64)), np.zeros((6, 3), int))
    qdir = Q.reshape(5, 2, 2, 64).sum(axis=(0, 2))
    Kneg = np.repeat((-1e4 * qdir / np.sum(qdir * qdir, -1, keepdims=True))[None], 3, 0)
    Qpos = np.abs(rng.standard_normal((5, 4, 1))) * np.repeat(qdir, 2, axis=0)[None] + 0.0
    pool.append(9, 0, Kneg, 1e3 * rng.standard_normal((3, 2, 64)), np.zeros((3, 3), int))
    Oa, _ = vo.bounded_attention(pool, Qpos, zero, [3, 5])
    Ob, _ = vo.bounded_attention(pool, Qpos, zero, [3, 9, 5])
    assert np.max(np.abs(Oa - Ob)) < 1e-12
    # GQA: q head h must read kv head h // g -- recompute one head by hand from the other kv head
    Oc, _ = vo.bounded_attention(pool, Q, zero, [5])
    h = 2
    L = (Q[:, h] @ Kb[:, 1].T) / 8.0
    P = np.exp(L - L.max(1, keepdims=True)); P /= P.sum(1, keepdims=True)
    assert np.max(np.abs(Oc[:, h] - P @ pool.V[5][:, 1])) < 1e-13


def test_empty_visible_set_reading_d29():
    pool, pages, Qs, Ks, Vs, Ps = _mini_stream(n_chunks=2)
    pool.append(30, 0, np.zeros((0, 2, 64)), np.zeros((0, 2, 64)), np.zeros((0, 3), int))
    O, lse = vo.bounded_attention(pool, Qs[1], Ps[1], [30])
    assert np.all(O == 0.0) and np.all(np.isneginf(lse))
    O2, lse2 = vo.bounded_attention(pool, Qs[1], Ps[1], [30, int(pages[0])])
    O3, lse3 = vo.bounded_attention(pool, Qs[1], Ps[1], [int(pages[0])])
    assert np.array_equal(O2, O3) and np.array_equal(lse2, lse3)


def test_lse_merge_equals_union():
    pool, pages, Qs, Ks, Vs, Ps = _mini_stream(n_chunks=4)
    a = [int(pages[0]), int(pages[1])]
    b = [int(pages[2]), int(pages[3])]
    Oa, la = vo.bounded_attention(pool, Qs[4], Ps[4], a)
    Ob, lb = vo.bounded_attention(pool, Qs[4], Ps[4], b, self_page=int(pages[4]))
    Ou, lu = vo.bounded_attention(pool, Qs[4], Ps[4], a + b, self_page=int(pages[4]))
    Om, lm = vo.merge_partial_attention(Oa, la, Ob, lb)
    assert np.max(np.abs(Om - Ou)) < 1e-12 and np.max(np.abs(lm - lu)) < 1e-12


def test_append_offset_equals_single_append():
    rng = np.random.default_rng(4)
    K, V = rng.standard_normal((10, 2, 64)), rng.standard_normal((10, 2, 64))
    pos = rng.integers(0, 50, (10, 3))
    a, b = vo.PagedKV(4, 2, 64, 1e6, SEC64), vo.PagedKV(4, 2, 64, 1e6, SEC64)
    a.append(0, 0, K, V, pos)
    b.append(0, 0, K[:4], V[:4], pos[:4])
    b.append(0, 4, K[4:], V[4:], pos[4:])
    assert np.array_equal(a.K[0], b.K[0]) and np.array_equal(a.V[0], b.V[0])
    assert np.allclose(a.k_sum[0], b.k_sum[0], atol=1e-13) and a.page_len(0) == 10
    assert np.allclose(a.k_sum[0], K.sum(0))                     # summary is of PRE-RoPE keys
    assert np.array_equal(a.V[0], V)                             # V untouched by RoPE


# ------------------------------------------------------------------ retrieval (O6) ------------
def _bank(n_pages=12, seed=0):
    rng = np.random.default_rng(seed)
    pool = vo.PagedKV(4, 2, 64, 1e6, SEC64)
    for p in range(n_pages):
        n = int(rng.integers(3, 9))
        pool.append(p, 0, rng.standard_normal((n, 2, 64)), rng.standard_normal((n, 2, 64)), rng.integers(0, 9, (n, 3)))
    return pool, rng


def test_retrieval_scores_cosine_and_planted_page():
    pool, rng = _bank()
    Q = rng.standard_normal((6, 4, 64))
    qb = vo.mean_query(Q, 2)
    assert np.allclose(qb[1], Q[:, 2:4].mean(axis=(0, 1)))        # head folding h -> h // g
    # a page whose mean key is alpha * q_bar scores cosine 1 and ranks first under both scores
    pool.append(20, 0, np.repeat(3.0 * qb[None], 5, 0), np.zeros((5, 2, 64)), np.zeros((5, 3), int))
    cand = list(range(12)) + [20]
    s_cos = vo.retrieval_scores(pool, Q, cand, normalize=True)
    s_dot = vo.retrieval_scores(pool, Q, cand, normalize=False)
    assert abs(s_cos[-1] - 1.0) < 1e-12 and np.all(s_cos[:-1] < 1.0) and np.all(s_cos >= -1.0)
    assert abs(s_dot[-1] - 3.0 * np.sum(qb * qb)) < 1e-10
    assert vo.retrieve_topk(s_cos, cand, 1)[0] == 20 and vo.retrieve_topk(s_dot, cand, 1)[0] == 20
    # library cross-check of one score
    xb = (pool.k_sum[4] / pool.page_len(4)).ravel()
    assert abs(s_cos[4] - np.dot(qb.ravel(), xb) / np.linalg.norm(qb) / np.linalg.norm(xb)) < 1e-14


def test_topk_matches_argsort_order_invariance_exclusion_ties():
    pool, rng = _bank()
    Q = rng.standard_normal((6, 4, 64))
    cand = list(range(12))
    s = vo.retrieval_scores(pool, Q, cand)
    top = vo.retrieve_topk(s, cand, 5)
    assert top.tolist() == np.argsort(-s, kind="stable")[:5].tolist()
    perm = rng.permutation(12)
    s2 = vo.retrieval_scores(pool, Q, [cand[i] for i in perm])
    assert np.allclose(s2, s[perm], atol=0)
    assert vo.retrieve_topk(s2, [cand[i] for i in perm], 5).tolist() == top.tolist()
    excl = [int(top[0]), int(top[2])]
    top_e = vo.retrieve_topk(s, cand, 3, exclude_pages=excl)
    assert top_e.tolist() == [p for p in np.argsort(-s, kind="stable").tolist() if p not in excl][:3]
    assert vo.retrieve_topk(np.array([1.0, 2.0, 2.0, 0.5]), [7, 9, 4, 1], 3).tolist() == [4, 9, 7]
    assert vo.retrieve_topk(np.array([1.0, 2.0]), [3, 5], 4).tolist() == [5, 3, -1, -1]
    assert vo.retrieve_threshold(np.array([0.1, 0.7, 0.5]), [4, 2, 9], 0.5) == [2, 9]


# ------------------------------------------------------------------ stream driver -------------
def test_oracle_stream_window_and_query_sets():
    cfg = synth.get_config("tiny")
    Z = synth.gen_hidden_tiny(cfg)
    Wq, Wk, Wv = synth.gen_proj_weights_tiny(cfg)
    st = vo.OracleStream(cfg.Hq, cfg.Hkv, cfg.d, cfg.rope_theta, cfg.rope_sections, cfg.G, cfg.Hg, cfg.Wg,
                         cfg.tau, cfg.W)
    pages = synth.gen_page_ids(16, cfg.n_chunks + 2, 0)
    sK, sV = synth.gen_sink_kv(cfg)
    st.add_sink(int(pages[0]), sK, sV)
    for t in range(cfg.n_chunks):
        def qkv(idx, n, t=t):
            X = Z[t].reshape(cfg.T, cfg.D)[idx].astype(np.float64)
            return ((X @ Wq).reshape(n, cfg.Hq, cfg.d), (X @ Wk).reshape(n, cfg.Hkv, cfg.d),
                    (X @ Wv).reshape(n, cfg.Hkv, cfg.d))
        r = st.ingest_chunk(Z[t], int(pages[t + 1]), qkv)
        assert r["visible"] == [int(pages[0])] + [int(p) for p in pages[1 + max(0, t - cfg.W):1 + t]]
        assert r["O"].shape == (r["n"], cfg.Hq, cfg.d) and np.isfinite(r["O"]).all()
        assert r["pos3"][0].tolist() == [cfg.sink + 4 * t] * 3    # base advances by max(G, Hg, Wg) = 4
    Q, K, V = synth.gen_query(cfg, 5)
    q = st.query(Q, K, V, int(pages[cfg.n_chunks + 1]), k=2, recent=2)
    assert len(set(q["visible"])) == len(q["visible"]) == 1 + 2 + 2   # no duplicates (D21)
    assert set(q["visible"][1:3]) == {int(pages[5]), int(pages[6])}


def test_oracle_stream_mode1_carries_previous_chunks_last_group_by_hand():
    """Frame-level dropping across a chunk boundary ("the current frame and the previous frame ...
    without a multi-frame chunk anchor"): group 0 of chunk t is compared with the LAST group of chunk t-1.  Three
    chunks of G = 2 groups x 3 positions built from orthonormal vectors, so every similarity is exactly 0 or 1 and
    the kept lists below are worked out by hand.  Each wrong carry gives another list: no carry (group 0 as anchor)
    keeps 0, 1, 2 everywhere; the FIRST group of chunk t-1 drops position 1 of chunk 1 and keeps all of chunk 2's
    group 0; a stale carry (chunk t-2) keeps 0 and 2 of chunk 2 and drops its 1."""
    e = np.eye(8)
    e1, e2, e3, e4 = e[0], e[1], e[2], e[3]
    chunks = [np.array([[e1, e2, e3], [e1, e4, e3]]),
              np.array([[e1, e2, e3], [e2, e2, e1]]),
              np.array([[e2, e4, e1], [e3, e3, e3]])]
    #            chunk 0: no previous frame, group 0 kept; group 1 repeats positions 0 and 2
    #            chunk 1: carry (e1, e4, e3) drops 0 and 2 of group 0; group 1 repeats position 1
    #            chunk 2: carry (e2, e2, e1) drops 0 and 2 of group 0; group 1 is new everywhere
    by_hand = [[0, 1, 2, 4], [1, 3, 5], [1, 3, 4, 5]]
    st = vo.OracleStream(2, 1, 8, 10000.0, (2, 1, 1), 2, 1, 3, 0.9, W=2, mode=1)
    for t, Z in enumerate(chunks):
        r = st.ingest_chunk(Z, 10 + t, lambda idx, n: (np.ones((n, 2, 8)), np.ones((n, 1, 8)), np.ones((n, 1, 8))),
                            attend=False)
        assert r["kept_idx"].tolist() == by_hand[t], (t, r["kept_idx"].tolist())
        assert r["n"] == len(by_hand[t]) == st.pool.page_len(10 + t)
        # positions of the kept tokens: (base + g, base + 0, base + column), base advancing by max(G, Hg, Wg) = 3
        assert r["pos3"].tolist() == [[3 * t + i // 3, 3 * t, 3 * t + i % 3] for i in by_hand[t]]
    # the same chunks under the chunk-level rule (mode 0) ignore the boundary: group 0 is always the anchor
    st0 = vo.OracleStream(2, 1, 8, 10000.0, (2, 1, 1), 2, 1, 3, 0.9, W=2, mode=0)
    for t, Z in enumerate(chunks):
        r = st0.ingest_chunk(Z, 10 + t, lambda idx, n: (np.ones((n, 2, 8)), np.ones((n, 1, 8)), np.ones((n, 1, 8))),
                             attend=False)
        assert r["kept_idx"].tolist()[:3] == [0, 1, 2]


def test_query_side_page_table_equals_eq4_qry_mask():
    """Query side of Eq. 4: a query token sees chunk j iff j is in V_qry (the
    retrieved set; BASELINE config 5 adds the recent window, reading D21), plus the sink (D14) and,
    causally, its own text tokens (D27).  The page-table construction of OracleStream.query must
    equal dense attention under eq4_mask with kind = "qry" rows over the WHOLE stream laid out in
    sequence order -- for top-k retrieval with a recent window, with no recent window, and with k
    larger than the number of eligible chunks."""
    cfg = synth.get_config("tiny")
    Z = synth.gen_hidden_tiny(cfg)
    Wq, Wk, Wv = synth.gen_proj_weights_tiny(cfg, std=0.4)            # sharp logits: a wrong mask entry shows
    for k, recent in [(2, 2), (3, 0), (9, 1)]:
        st = vo.OracleStream(cfg.Hq, cfg.Hkv, cfg.d, cfg.rope_theta, cfg.rope_sections, cfg.G, cfg.Hg, cfg.Wg,
                             cfg.tau, cfg.W)
        pages = [int(p) for p in synth.gen_page_ids(16, cfg.n_chunks + 2, 1)]
        sK, sV = synth.gen_sink_kv(cfg)
        st.add_sink(pages[0], sK, sV)
        Ks, Vs, Ps = [np.asarray(sK, float)], [np.asarray(sV, float)], [vo.text_positions(0, cfg.sink)]
        chunk_of, kind = [-1] * cfg.sink, ["sink"] * cfg.sink
        for t in range(cfg.n_chunks):
            rec = {}

            def qkv(idx, n, t=t, rec=rec):
                X = Z[t].reshape(cfg.T, cfg.D)[idx].astype(np.float64)
                rec["K"], rec["V"] = (X @ Wk).reshape(n, cfg.Hkv, cfg.d), (X @ Wv).reshape(n, cfg.Hkv, cfg.d)
                return (X @ Wq).reshape(n, cfg.Hq, cfg.d), rec["K"], rec["V"]
            r = st.ingest_chunk(Z[t], pages[t + 1], qkv, attend=False)
            Ks.append(rec["K"]); Vs.append(rec["V"]); Ps.append(r["pos3"])
            chunk_of += [t] * r["n"]; kind += ["vis"] * r["n"]
        Q, K, V = synth.gen_query(cfg, 5)
        Q = 6.0 * Q
        q = st.query(Q, K, V, pages[cfg.n_chunks + 1], k=k, recent=recent)
        page_chunk = {pages[t + 1]: t for t in range(cfg.n_chunks)}
        top_chunks = [page_chunk[int(p)] for p in q["topk"] if p >= 0]
        recent_chunks = list(range(cfg.n_chunks - recent, cfg.n_chunks))
        assert len(top_chunks) == min(k, cfg.n_chunks - recent) and not set(top_chunks) & set(recent_chunks)
        v_qry = set(top_chunks) | set(recent_chunks)
        assert q["visible"] == [pages[0]] + [pages[c + 1] for c in recent_chunks] + [pages[c + 1] for c in top_chunks]
        # the whole stream in sequence order, the query's own tokens last (their chunk id = n_chunks)
        nq = Q.shape[0]
        Ks.append(np.asarray(K, float)); Vs.append(np.asarray(V, float)); Ps.append(q["pos3"])
        chunk_of += [cfg.n_chunks] * nq; kind += ["qry"] * nq
        M = vo.eq4_mask(chunk_of, kind, cfg.W, retrieved=v_qry)
        n_all = len(chunk_of)
        rows = M[n_all - nq:]
        for j in range(n_all - nq):                                    # chunk-granular staircase of the query rows
            want = kind[j] == "sink" or chunk_of[j] in v_qry
            assert rows[:, j].all() == want and rows[:, j].any() == want
        assert np.array_equal(rows[:, n_all - nq:], np.tril(np.ones((nq, nq), bool)))
        Kall = vo.mrope_rotate(np.concatenate(Ks), np.concatenate(Ps), cfg.rope_theta, cfg.rope_sections)
        Vall = np.concatenate(Vs)
        Qr = vo.mrope_rotate(np.asarray(Q, float), q["pos3"], cfg.rope_theta, cfg.rope_sections)
        g = cfg.Hq // cfg.Hkv
        for h in range(cfg.Hq):
            ref = vo.masked_attention_dense(Qr[:, h], Kall[:, h // g], Vall[:, h // g], rows, 1.0 / np.sqrt(cfg.d))
            assert np.max(np.abs(q["O"][:, h] - ref)) < 1e-12


# ------------------------------------------------------------------ throughput formula --------
def test_golden_table2_fps():
    for ret, c, vp, vit, drop, llm, fps in _rows("table2_fps.txt"):
        got = vo.fps_max(int(c), [float(vp), float(vit), float(drop), float(llm)])
        tol = 1.0 if (ret, c) == ("50", "4") else 0.5
        assert abs(got - float(fps)) <= tol, (ret, c, got, fps)
    assert abs(vo.fps_max(16, [113, 119, 44, 42]) - 134.45) < 0.01   # abstract: 134 FPS
    assert 317 + 236 + 87 + 124 == 764                               # serial sum


# ---- O1b entropy-based spatial selection ---------------------------------------
def test_entropy_closed_forms_and_library():
    from scipy.stats import entropy as sp_entropy
    from scipy.special import softmax
    D = 64
    assert abs(vo.feature_entropy(np.zeros((1, D)))[0] - np.log(D)) < 1e-12          # uniform -> log D
    x = np.zeros((1, D)); x[0, 7] = 1e3
    assert vo.feature_entropy(x)[0] < 1e-12                                          # one dominant feature -> 0
    # two-level distribution: a features at logit t, D - a at 0 -> closed form
    a, t = 5, 2.0
    x = np.zeros((1, D)); x[0, :a] = t
    Zp = a * np.exp(t) + (D - a)
    want = np.log(Zp) - a * t * np.exp(t) / Zp
    assert abs(vo.feature_entropy(x)[0] - want) < 1e-12
    rng = np.random.default_rng(3)
    X = rng.standard_normal((9, 50)) * rng.uniform(0.2, 4.0, size=(9, 1))
    H = vo.feature_entropy(X)
    assert np.allclose(H, [sp_entropy(softmax(r)) for r in X], rtol=1e-12)           # library routine
    assert np.allclose(H, vo.feature_entropy(X + 123.0), rtol=1e-10)                 # shift invariance of softmax
    assert np.allclose(H, vo.feature_entropy(X[:, rng.permutation(50)]), rtol=1e-12) # feature permutation
    assert np.all(np.diff(vo.feature_entropy(np.outer([0.5, 1.0, 2.0, 4.0], X[0]))) < 0)   # sharper -> lower entropy


def test_entropy_topk_selection_rules():
    s = np.array([0.3, 0.9, 0.9, 0.1, 0.5])
    assert vo.topk_by_score(s, 2).tolist() == [1, 2]
    assert vo.topk_by_score(s, 1).tolist() == [1]                                     # tie -> lower index
    assert vo.topk_by_score(s, 3).tolist() == [1, 2, 4]                               # ascending index order
    assert vo.topk_by_score(s, 0).tolist() == [] and vo.topk_by_score(s, 9).tolist() == [0, 1, 2, 3, 4]
    rng = np.random.default_rng(5)
    v = rng.standard_normal(200)
    K = 37
    assert vo.topk_by_score(v, K).tolist() == sorted(np.argsort(-v, kind="stable")[:K].tolist())   # library argsort
    Z = rng.standard_normal((3, 20, 16)) * rng.uniform(0.3, 3.0, size=(3, 20, 1))
    H, idx, n = vo.spatial_entropy_select(Z, 8)
    assert n == 24 and np.all(np.diff(idx) > 0)
    for g in range(3):                                                                # per frame, independently
        mine = idx[(idx >= g * 20) & (idx < (g + 1) * 20)] - g * 20
        assert len(mine) == 8 and np.min(H[g][mine]) >= np.max(np.delete(H[g], mine))
    assert vo.spatial_entropy_select(Z, 20)[2] == 60                                  # K = P keeps everything
