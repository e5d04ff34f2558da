"""CPU checks of the boundary: the C-ABI library builds, loads, and exports every symbol that
include/vcs.h declares; host-side argument validation answers without a GPU; the product path
has no CPU fallback; the oracle and the product share no code."""
import ctypes as C
import os
import re

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2606_19849_b200 import build, vcs
    build.build_library()
    return vcs.lib()


def _declared_symbols():
    hdr = open(os.path.join(ROOT, "include", "vcs.h")).read()
    return sorted(set(re.findall(r"VCS_API[^;(]*?\b(vcs_[a-z0-9_]+)\s*\(", hdr)))


def test_header_symbols_exported(lib):
    from paper_2606_19849_b200 import vcs
    declared = _declared_symbols()
    assert len(declared) >= 13
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in vcs.h but not exported by libvcs.so"
    assert sorted(vcs.API_SYMBOLS) == declared
    for name in ("vcs_temporal_drop", "vcs_kv_append_pages", "vcs_bounded_prefill_attn", "vcs_retrieval_score"):
        assert name in declared and callable(getattr(vcs, name))
    assert lib.vcs_version() == vcs.VERSION == 101
    hdr = open(os.path.join(ROOT, "include", "vcs.h")).read()
    assert re.search(r"#define VCS_VERSION (\d+)", hdr).group(1) == "101"
    # the ctypes mirrors of the call structs have the size the library was compiled with
    assert lib.vcs_sizeof_chunk_call() == C.sizeof(vcs._ChunkCall)
    assert lib.vcs_sizeof_multi_call() == C.sizeof(vcs._MultiCall)


def test_library_is_sm100a_with_tcgen05_and_tma():
    import subprocess
    from paper_2606_19849_b200 import vcs
    out = subprocess.run(["cuobjdump", "-lelf", vcs.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    sass = subprocess.run(["cuobjdump", "-sass", vcs.LIB_PATH], capture_output=True, text=True).stdout
    assert "UTCHMMA" in sass, "tcgen05.mma (UTCHMMA) missing from the attention kernel"
    assert "UTMALDG" in sass, "TMA loads (UTMALDG) missing"
    assert "LDTM" in sass, "tcgen05.ld (LDTM) missing"


def test_host_side_errors_without_gpu(lib):
    from paper_2606_19849_b200 import vcs
    # every argument error below is detected before anything would be enqueued
    rc = lib.vcs_temporal_drop(None, None, 1, 4, 16, 64, vcs.BF16, 0.9, 0, None, None, None, None, 0, 0, 1, None,
                               None, 0, None)
    assert rc == vcs.EINVAL and b"NULL" in lib.vcs_last_error()
    rc = lib.vcs_temporal_drop(16, None, 1, 0, 16, 64, vcs.BF16, 0.9, 0, 16, 16, None, None, 0, 0, 1, None, 16, 1 << 20, None)
    assert rc == vcs.EINVAL
    rc = lib.vcs_temporal_drop(16, None, 1, 4, 16, 64, 7, 0.9, 0, 16, 16, None, None, 0, 0, 1, None, 16, 1 << 20, None)
    assert rc == vcs.EUNSUPPORTED
    rc = lib.vcs_temporal_drop(24, None, 1, 4, 16, 64, vcs.BF16, 0.9, 0, 16, 16, None, None, 0, 0, 1, None, 16, 1 << 20, None)
    assert rc == vcs.EALIGN                                     # z not 16-byte aligned
    rc = lib.vcs_temporal_drop(16, None, 1, 4, 16, 60, vcs.BF16, 0.9, 0, 16, 16, None, None, 0, 0, 1, None, 16, 1 << 20, None)
    assert rc == vcs.EALIGN                                     # D*2 not a multiple of 16
    rc = lib.vcs_temporal_drop(16, None, 1, 4, 16, 64, vcs.BF16, 0.9, 0, 16, 16, None, None, 0, 0, 1, None, 16, 8, None)
    assert rc == vcs.ECAP                                       # workspace too small
    rc = lib.vcs_temporal_drop(16, None, 1, 4, 16, 64, vcs.BF16, 0.9, 0, 16, 16, None, None, 0, 0, 1, None, 24, 1 << 20, None)
    assert rc == vcs.EALIGN and b"workspace" in lib.vcs_last_error()   # the flag rows are read with 128-bit loads
    rc = lib.vcs_temporal_drop(16, None, 1, 4, 16, 64, vcs.BF16, 0.9, 0, 16, 16, None, 16, 3, 5, 1, None, 16, 1 << 20, None)
    assert rc == vcs.EINVAL                                     # Hg*Wg != P with pos3 requested
    assert lib.vcs_temporal_drop_workspace_bytes(2, 4, 464) >= 2 * 4 * 464
    # pool validation
    pool = vcs._Pool(16, 16, 16, 16, 4, 128, 2, 16, 128, vcs.BF16, 1e6, (C.c_int32 * 3)(16, 24, 24), None)
    assert lib.vcs_kv_append_pages(C.byref(pool), 16, 16, 256, 256, 16, None, 8, 0, 0, None, 16, 1 << 20, None) == vcs.EINVAL
    assert b"opaque" in lib.vcs_last_error()
    bad = vcs._Pool(16, 16, 16, 16, 4, 128, 3, 16, 128, vcs.BF16, 1e6, (C.c_int32 * 3)(16, 24, 24), None)
    assert lib.vcs_pool_init(C.byref(bad)) == vcs.EINVAL        # Hq % Hkv
    bad = vcs._Pool(16, 16, 16, 16, 4, 128, 2, 16, 96, vcs.BF16, 1e6, (C.c_int32 * 3)(16, 16, 16), None)
    assert lib.vcs_pool_init(C.byref(bad)) == vcs.EUNSUPPORTED  # head_dim
    bad = vcs._Pool(16, 16, 16, 16, 4, 128, 2, 16, 128, vcs.BF16, 1e6, (C.c_int32 * 3)(16, 24, 23), None)
    assert lib.vcs_pool_init(C.byref(bad)) == vcs.EINVAL        # sections do not sum to d/2


def test_pool_init_and_call_validation_with_fake_pointers(lib):
    """fp32 pools need no TMA maps, so vcs_pool_init works on the CPU box; the later calls must
    still reject bad arguments before touching the (fake) device pointers."""
    from paper_2606_19849_b200 import vcs
    buf = C.create_string_buffer(lib.vcs_pool_opaque_bytes() + 64)
    op = (C.addressof(buf) + 63) // 64 * 64
    pool = vcs._Pool(4096, 8192, 256, 512, 4, 32, 1, 2, 64, vcs.F32, 1e6, (C.c_int32 * 3)(8, 12, 12), op)
    assert lib.vcs_pool_init(C.byref(pool)) == vcs.OK
    ws = 1 << 20
    P = C.byref(pool)
    assert lib.vcs_kv_append_pages(P, 4096, 4096, 64, 64, 4096, None, 8, 9, 0, None, 4096, ws, None) == vcs.ECAP   # page id
    assert lib.vcs_kv_append_pages(P, 4096, 4096, 64, 64, 4096, None, 8, 0, 33, None, 4096, ws, None) == vcs.ECAP  # offset
    assert lib.vcs_kv_append_pages(P, 4096, 4096, 32, 64, 4096, None, 8, 0, 0, None, 4096, ws, None) == vcs.EINVAL  # stride
    assert lib.vcs_kv_append_pages(P, 4100, 4096, 64, 64, 4096, None, 8, 0, 0, None, 4096, ws, None) == vcs.EALIGN
    assert lib.vcs_kv_append_pages(P, 4096, 4096, 64, 64, 4096, None, 8, 0, 0, None, 4096, 16, None) == vcs.ECAP   # workspace
    a = lib.vcs_bounded_prefill_attn
    assert a(P, 4096, 128, 4096, None, 8, 4096, None, 2, 4, 0, 0.0, 4096, 128, None, 0, None, 4096, ws, None) == vcs.ECAP
    assert a(P, 4096, 64, 4096, None, 8, 4096, None, 2, -1, 0, 0.0, 4096, 128, None, 0, None, 4096, ws, None) == vcs.EINVAL
    assert a(P, 4096, 128, 4096, None, 8, 4096, None, 2, -1, 0, 0.0, 4096, 128, None, 9, None, 4096, ws, None) == vcs.EINVAL
    assert a(P, 4096, 128, 4096, None, 8, 4096, None, 2, -1, 0, 0.0, 4096, 128, None, vcs.ATTN_TC, None, 4096, ws,
             None) == vcs.EUNSUPPORTED                          # tcgen05 path needs bf16 / d = 128
    assert a(P, 4096, 128, 4096, None, 0, 4096, None, 2, -1, 0, 0.0, 4096, 128, None, 0, None, 4096, ws, None) == vcs.OK
    r = lib.vcs_retrieval_score
    assert r(P, 4096, 128, None, 4, 4096, 8, None, 0, 0, 4096, 2, 4096, 4096, 16, None) == vcs.ECAP
    assert r(P, 4096, 128, None, 4, None, 8, None, 0, 0, 4096, 2, 4096, 4096, ws, None) == vcs.EINVAL


def test_new_entry_points_reject_bad_arguments(lib):
    """Batched append, threshold visibility, entropy top-K, upload / download: host-side errors only."""
    from paper_2606_19849_b200 import vcs
    buf = C.create_string_buffer(lib.vcs_pool_opaque_bytes() + 64)
    op = (C.addressof(buf) + 63) // 64 * 64
    pool = vcs._Pool(4096, 8192, 256, 512, 4, 32, 1, 2, 64, vcs.F32, 1e6, (C.c_int32 * 3)(8, 12, 12), op)
    assert lib.vcs_pool_init(C.byref(pool)) == vcs.OK
    P, ws = C.byref(pool), 1 << 22
    b = lib.vcs_kv_append_pages_batched
    assert b(P, 4096, 4096, 512, 512, 64, 64, 4096, None, 8, None, 2, None, 4096, ws, None) == vcs.EINVAL   # no page ids
    assert b(P, 4096, 4096, 512, 512, 64, 64, 4096, None, 8, 4096, 70000, None, 4096, ws, None) == vcs.EINVAL  # B
    assert b(P, 4096, 4096, 510, 512, 64, 64, 4096, None, 8, 4096, 2, None, 4096, ws, None) == vcs.EALIGN   # batch stride
    assert b(P, 4096, 4096, 512, 512, 64, 64, 4096, None, 8, 4096, 2, None, 4096, 64, None) == vcs.ECAP     # workspace
    assert b(P, 4096, 4096, 512, 512, 64, 64, 4096, None, 8, 4096, 0, None, 4096, ws, None) == vcs.OK       # B = 0
    assert lib.vcs_kv_append_batched_workspace_bytes(P, 8, 3) == 3 * lib.vcs_kv_append_workspace_bytes(P, 8)
    t = lib.vcs_retrieval_threshold
    assert t(P, 4096, 4096, 8, None, 0, 0.5, 4096, 8, None, None) == vcs.EINVAL                             # no count
    assert t(P, None, 4096, 8, None, 0, 0.5, 4096, 8, 4096, None) == vcs.EINVAL                             # no scores
    assert t(P, 4096, 4096, 8, None, 2, 0.5, 4096, 8, 4096, None) == vcs.EINVAL                             # no exclude list
    assert t(P, 4096, 4096, 8, None, 0, float("nan"), 4096, 8, 4096, None) == vcs.EINVAL
    e = lib.vcs_spatial_entropy_topk
    assert e(None, 1, 4, 16, 64, vcs.BF16, 4, 16, 16, None, None, 0, 0, 1, None, 16, ws, None) == vcs.EINVAL
    assert e(16, 1, 4, 16, 64, 5, 4, 16, 16, None, None, 0, 0, 1, None, 16, ws, None) == vcs.EUNSUPPORTED
    assert e(16, 1, 4, 16, 60, vcs.BF16, 4, 16, 16, None, None, 0, 0, 1, None, 16, ws, None) == vcs.EALIGN
    assert e(16, 1, 4, 16, 64, vcs.BF16, 4, 16, 16, None, None, 0, 0, 1, None, 16, 8, None) == vcs.ECAP
    assert e(16, 1, 4, 16, 64, vcs.BF16, 4, 16, 16, None, 16, 3, 5, 1, None, 16, ws, None) == vcs.EINVAL    # Hg*Wg != P
    assert e(16, 1, 4, 16, 64, vcs.BF16, -1, 16, 16, None, None, 0, 0, 1, None, 16, ws, None) == vcs.EINVAL
    assert lib.vcs_spatial_entropy_topk_workspace_bytes(2, 4, 464) >= 2 * 4 * 464 * 4
    assert lib.vcs_chunk_upload(P, None, 16, 16, 16, 16, None) == vcs.EINVAL
    assert lib.vcs_chunk_download(P, None, 16, 16, 16, None) == vcs.EINVAL


def test_no_cpu_fallback_in_binding():
    from paper_2606_19849_b200 import vcs
    z = torch.zeros((1, 2, 4, 8))
    with pytest.raises(vcs.VcsError):
        vcs.vcs_temporal_drop(z, 0.9, torch.zeros(1, 8, dtype=torch.int32), torch.zeros(1, dtype=torch.int32),
                              torch.zeros(1024, dtype=torch.uint8))


def test_oracle_and_product_are_independent():
    """Neither side imports the other; only `synth` (inputs, no arithmetic) is common."""
    pkg = os.path.join(ROOT, "paper_2606_19849_b200")
    for base, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(base, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, re.M), f
                assert "oracle/" not in src and "import synth" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_2606_19849_b200", src, re.M), f
            assert "ctypes" not in src and "torch" not in src, f
    for f in os.listdir(os.path.join(ROOT, "synth")):
        if f.endswith(".py"):
            src = open(os.path.join(ROOT, "synth", f)).read()
            assert not re.search(r"^\s*(from|import)\s+(oracle|paper_2606_19849_b200)", src, re.M), f


def test_visible_set_matches_eq4_at_chunk_granularity(lib):
    """Step a6 behind the C ABI: vcs_visible_set lists exactly the key pages that the oracle's Eq. 4
    predicate (readings D12 / D14) exposes to a vision token of chunk t besides its own
    chunk: sink first, then chunks t-W .. t-1 in stream order, clipped at the stream start."""
    import oracle as vo
    from paper_2606_19849_b200 import vcs
    pages = [40, 3, 17, 8, 29, 5, 11, 2, 36, 21]
    for W in (0, 1, 3, 8, 64, -1):
        acn = W if W >= 0 else 10 ** 9
        for t in range(len(pages) + 1):
            table, n = vcs.vcs_visible_set(t, W, 7, pages, 16)
            want = [7] + [pages[j] for j in range(t) if vo.eq4_visible(t, "vis", j, "vis", acn)]
            assert n == len(want) and table[:n] == want and all(x == -1 for x in table[n:]), (W, t, table)
            st = vo.OracleStream(4, 2, 128, 1e6, (16, 24, 24), 2, 2, 2, 0.9, W)
            st.sink_page, st.chunk_pages = 7, list(pages)
            assert st.visible_pages(t) == want
    table, n = vcs.vcs_visible_set(4, 2, -1, pages, 4)                      # no sink page
    assert n == 2 and table == [17, 8, -1, -1]
    with pytest.raises(RuntimeError):
        vcs.vcs_visible_set(9, -1, 7, pages, 4)                             # ECAP: 10 entries, 4 slots
    with pytest.raises(RuntimeError):
        vcs.vcs_visible_set(11, 2, 7, pages, 16)                            # EINVAL: t beyond the stream


def test_one_call_forms_reject_bad_workspaces_before_anything_is_enqueued(lib):
    """vcs_chunk_ingest / vcs_ingest_layers look at everything the host can see (B, page table, size and alignment of
    all three workspaces, pool geometry) before the first launch, so an error cannot leave a chunk half ingested.
    No GPU here: reaching the first launch would answer VCS_ECUDA, the argument errors must come first."""
    from paper_2606_19849_b200 import vcs

    def pool(page_cap=128, theta=1e6):
        buf = C.create_string_buffer(lib.vcs_pool_opaque_bytes() + 64)
        p = vcs._Pool(16, 16, 16, 16, 4, page_cap, 2, 16, 64, vcs.F32, theta, (C.c_int32 * 3)(8, 12, 12),
                      (C.addressof(buf) + 63) // 64 * 64)
        assert lib.vcs_pool_init(C.byref(p)) == vcs.OK
        return p, buf
    p0, _b0 = pool()
    big = 1 << 24

    def chunk(**kw):
        c = vcs._ChunkCall(G=2, P=8, D=64, Hg=2, Wg=4, t_stride=1, z_dtype=vcs.BF16, mode=0, tau=0.9, page_id=1, n_vis_cap=2,
                           attn_flags=0, host_rows=0, z_d=16, q_d=16, k_d=16, v_d=16, out_d=16, kept_idx_d=16, kept_count_d=16,
                           pos3_d=16, pos_base_d=16, page_table_d=16, n_vis_d=16, prev_last_group_d=None, status_d=16,
                           ws_drop=16, ws_append=16, ws_attn=16, ws_drop_bytes=big, ws_append_bytes=big, ws_attn_bytes=big)
        for k, v in kw.items():
            setattr(c, k, v)
        return c
    for kw, code in ((dict(ws_drop=24), vcs.EALIGN), (dict(ws_attn=8), vcs.EALIGN), (dict(ws_drop_bytes=8), vcs.ECAP),
                     (dict(ws_append_bytes=8), vcs.ECAP), (dict(ws_attn_bytes=8), vcs.ECAP), (dict(page_table_d=None), vcs.EINVAL)):
        assert lib.vcs_chunk_ingest(C.byref(p0), C.byref(chunk(**kw)), None) == code, kw

    def multi(**kw):
        m = vcs._MultiCall(B=2, L=2, G=2, P=8, D=64, Hg=2, Wg=4, t_stride=1, z_dtype=vcs.BF16, mode=0, tau=0.9, n_vis_cap=2,
                           attn_flags=0, q_layer_stride=0, kv_layer_stride=0, out_layer_stride=0, z_d=16, q_d=16, k_d=16, v_d=16,
                           out_d=16, prev_last_group_d=None, kept_idx_d=16, kept_count_d=16, pos3_d=16, pos_base_d=16,
                           page_ids_d=16, page_tables_d=16, n_vis_d=16, status_d=16, ws_drop=16, ws_append=16, ws_attn=16,
                           ws_drop_bytes=big, ws_append_bytes=big, ws_attn_bytes=big)
        for k, v in kw.items():
            setattr(m, k, v)
        return m
    PP = C.POINTER(vcs._Pool)
    p1, _b1 = pool()
    same = (PP * 2)(C.pointer(p0), C.pointer(p1))
    for kw, code in ((dict(B=65), vcs.ECAP), (dict(page_tables_d=None), vcs.EINVAL), (dict(ws_attn=40), vcs.EALIGN),
                     (dict(ws_drop_bytes=8), vcs.ECAP), (dict(ws_append_bytes=8), vcs.ECAP), (dict(ws_attn_bytes=8), vcs.ECAP)):
        assert lib.vcs_ingest_layers(same, C.byref(multi(**kw)), None) == code, kw
    for other in (pool(page_cap=64), pool(theta=1e4)):          # page_cap and rope belong to "identical geometry"
        mixed = (PP * 2)(C.pointer(p0), C.pointer(other[0]))
        assert lib.vcs_ingest_layers(mixed, C.byref(multi()), None) == vcs.EINVAL
        assert b"geometry" in lib.vcs_last_error()


def test_positions_and_query_visible_set_match_the_oracle(lib):
    """The last pieces of the method's arithmetic that lived in the Python drivers, now behind the C ABI and pinned
    against the oracle: the position-base advance and the text positions (reading D18, oracle O2) and the query-side
    visible list sink + recent + retrieved (reading D21: OracleStream.query builds the same list)."""
    import numpy as np
    import oracle as vo
    from paper_2606_19849_b200 import vcs
    for G, Hg, Wg, ts in ((4, 26, 46, 1), (4, 16, 29, 1), (8, 2, 3, 1), (4, 2, 3, 5), (1, 1, 1, 1), (16, 40, 9, 2)):
        b_ref, b = 128, 128
        for _ in range(5):
            b_ref = vo.next_position_base(G, Hg, Wg, b_ref, ts)
            b = vcs.vcs_next_position_base(G, Hg, Wg, b, ts)
            assert b == b_ref
    for start, n in ((0, 128), (100000, 48), (7, 0), (5, 1)):
        assert np.array_equal(vcs.vcs_text_positions(start, n, "cpu").numpy().reshape(-1, 3), vo.text_positions(start, n))
    with pytest.raises(vcs.VcsError):
        vcs.vcs_next_position_base(4, 0, 3, 10)
    with pytest.raises(vcs.VcsError):
        vcs.vcs_text_positions(2 ** 31 - 4, 8, "cpu")           # ECAP: overflows int32
    # query side: a real oracle stream tells which pages a query sees; the table must list them in the same order
    st = vo.OracleStream(2, 1, 8, 10000.0, (2, 1, 1), 2, 1, 3, 0.5, W=2)
    rng = np.random.default_rng(0)
    st.add_sink(40, rng.standard_normal((3, 1, 8)), rng.standard_normal((3, 1, 8)))
    pages = [31, 7, 19, 3, 25, 11]
    for pg in pages:
        st.ingest_chunk(rng.standard_normal((2, 3, 8)), pg, lambda idx, n: (rng.standard_normal((n, 2, 8)),
                        rng.standard_normal((n, 1, 8)), rng.standard_normal((n, 1, 8))), attend=False)
    for k, recent in ((2, 2), (3, 0), (9, 1)):
        q = st.query(rng.standard_normal((4, 2, 8)), rng.standard_normal((4, 1, 8)), rng.standard_normal((4, 1, 8)),
                     text_page=99, k=k, recent=recent)
        table, n_fixed = vcs.vcs_visible_set_query(40, pages[len(pages) - recent:] if recent else [], k)
        assert n_fixed == 1 + recent and table[n_fixed:] == [-1] * k
        table[n_fixed:] = [int(p) for p in q["topk"]]               # what vcs_retrieval_score writes on the device
        assert [p for p in table if p >= 0] == q["visible"]
    table, n_fixed = vcs.vcs_visible_set_query(-1, [5, 6], 2, table_cap=6)      # no sink page, padded table
    assert (table, n_fixed) == ([5, 6, -1, -1, -1, -1], 2)
    with pytest.raises(vcs.VcsError):
        vcs.vcs_visible_set_query(40, [5, 6], 2, table_cap=4)                   # ECAP


def test_graft_entry_builds_and_checks_the_current_version():
    """`__graft_entry__.build()` is the driver's build check: it must run through, and it must compare the library's
    version with the binding's constant, not with a literal (a literal went stale when VCS_VERSION moved to 101)."""
    import inspect
    import __graft_entry__ as g
    g.build()                                                   # raises if the version check or the load fails
    src = inspect.getsource(g.build)
    assert "vcs.VERSION" in src and "== 100" not in src
