"""Thin ctypes binding of libvcs.so (include/vcs.h): argument marshalling only -- every step of
the path runs in the CUDA kernels behind the C ABI.  torch is used for device memory and streams.

There is NO CPU fallback: importing works without a GPU (so that CPU tests can check the exported
symbols), but every compute call needs CUDA tensors and raises otherwise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libvcs.so")

VERSION = 101          # VCS_VERSION of include/vcs.h this binding was written against
OK, EINVAL, EALIGN, ECAP, EUNSUPPORTED, ECUDA = 0, -1, -2, -3, -4, -5
F32, BF16 = 0, 1
FLAG_COUNT_CLAMPED, FLAG_PAGE_OVERFLOW, FLAG_BAD_PAGE = 1, 2, 4
DROP_CHUNK_ALLPAIRS, DROP_CONSECUTIVE = 0, 1
ATTN_AUTO, ATTN_SIMT, ATTN_TC = 0, 1, 2

API_SYMBOLS = [
    "vcs_version", "vcs_sizeof_chunk_call", "vcs_sizeof_multi_call", "vcs_last_error", "vcs_device_info", "vcs_visible_set", "vcs_visible_set_query",
    "vcs_next_position_base", "vcs_text_positions", "vcs_pool_opaque_bytes", "vcs_pool_init",
    "vcs_temporal_drop_workspace_bytes", "vcs_temporal_drop", "vcs_temporal_drop_static",
    "vcs_spatial_entropy_topk_workspace_bytes", "vcs_spatial_entropy_topk",
    "vcs_kv_append_workspace_bytes", "vcs_kv_append_pages",
    "vcs_kv_append_batched_workspace_bytes", "vcs_kv_append_pages_batched",
    "vcs_bounded_prefill_attn_workspace_bytes", "vcs_bounded_prefill_attn", "vcs_bounded_prefill_attn_batched",
    "vcs_retrieval_score_workspace_bytes", "vcs_retrieval_score", "vcs_retrieval_threshold",
    "vcs_chunk_ingest", "vcs_chunk_ingest_host", "vcs_chunk_upload", "vcs_chunk_download",
    "vcs_selftest_exp2_poly", "vcs_selftest_rope_sincos",
    "vcs_ingest_layers", "vcs_graph_begin", "vcs_graph_end", "vcs_graph_launch", "vcs_graph_destroy",
]


class VcsError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"vcs error {code}: {msg}")
        self.code = code


class _Pool(C.Structure):
    _fields_ = [
        ("k_pages", C.c_void_p), ("v_pages", C.c_void_p), ("page_len", C.c_void_p), ("k_sum", C.c_void_p),
        ("n_pages", C.c_int32), ("page_cap", C.c_int32), ("Hkv", C.c_int32), ("Hq", C.c_int32),
        ("d", C.c_int32), ("dtype", C.c_int32), ("rope_theta", C.c_float), ("rope_sections", C.c_int32 * 3),
        ("opaque_h", C.c_void_p),
    ]


class _ChunkCall(C.Structure):
    _fields_ = [
        ("G", C.c_int32), ("P", C.c_int32), ("D", C.c_int32), ("Hg", C.c_int32), ("Wg", C.c_int32),
        ("t_stride", C.c_int32), ("z_dtype", C.c_int32), ("mode", C.c_int32), ("tau", C.c_float),
        ("page_id", C.c_int32), ("n_vis_cap", C.c_int32), ("attn_flags", C.c_int32), ("host_rows", C.c_int32),
        ("z_d", C.c_void_p), ("q_d", C.c_void_p), ("k_d", C.c_void_p), ("v_d", C.c_void_p), ("out_d", C.c_void_p),
        ("kept_idx_d", C.c_void_p), ("kept_count_d", C.c_void_p), ("pos3_d", C.c_void_p),
        ("pos_base_d", C.c_void_p), ("page_table_d", C.c_void_p), ("n_vis_d", C.c_void_p),
        ("prev_last_group_d", C.c_void_p), ("status_d", C.c_void_p),
        ("ws_drop", C.c_void_p), ("ws_append", C.c_void_p), ("ws_attn", C.c_void_p),
        ("ws_drop_bytes", C.c_size_t), ("ws_append_bytes", C.c_size_t), ("ws_attn_bytes", C.c_size_t),
    ]


class _MultiCall(C.Structure):
    _fields_ = [
        ("B", C.c_int32), ("L", C.c_int32),
        ("G", C.c_int32), ("P", C.c_int32), ("D", C.c_int32), ("Hg", C.c_int32), ("Wg", C.c_int32),
        ("t_stride", C.c_int32), ("z_dtype", C.c_int32), ("mode", C.c_int32), ("tau", C.c_float),
        ("n_vis_cap", C.c_int32), ("attn_flags", C.c_int32),
        ("q_layer_stride", C.c_int64), ("kv_layer_stride", C.c_int64), ("out_layer_stride", C.c_int64),
        ("z_d", C.c_void_p), ("q_d", C.c_void_p), ("k_d", C.c_void_p), ("v_d", C.c_void_p), ("out_d", C.c_void_p),
        ("prev_last_group_d", C.c_void_p),
        ("kept_idx_d", C.c_void_p), ("kept_count_d", C.c_void_p), ("pos3_d", C.c_void_p),
        ("pos_base_d", C.c_void_p), ("page_ids_d", C.c_void_p), ("page_tables_d", C.c_void_p), ("n_vis_d", C.c_void_p),
        ("status_d", C.c_void_p),
        ("ws_drop", C.c_void_p), ("ws_append", C.c_void_p), ("ws_attn", C.c_void_p),
        ("ws_drop_bytes", C.c_size_t), ("ws_append_bytes", C.c_size_t), ("ws_attn_bytes", C.c_size_t),
    ]


_lib = None


def lib() -> C.CDLL:
    """Load libvcs.so (fails loudly if it has not been built: no fallback path exists)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2606_19849_b200.build` "
                           "(or __graft_entry__.build()); the vcs CUDA library has no fallback")
    L = C.CDLL(LIB_PATH)
    i32, i64, f32, vp, sz = C.c_int, C.c_int64, C.c_float, C.c_void_p, C.c_size_t
    pp = C.POINTER(_Pool)
    L.vcs_version.restype = i32
    L.vcs_last_error.restype = C.c_char_p
    L.vcs_device_info.argtypes = [C.POINTER(i32), C.POINTER(i32), C.POINTER(i32), C.c_char_p, sz]
    L.vcs_visible_set.argtypes = [C.c_int32, C.c_int32, C.c_int32, C.POINTER(C.c_int32), C.c_int32, C.POINTER(C.c_int32), C.c_int32]
    L.vcs_visible_set_query.argtypes = [C.c_int32, C.POINTER(C.c_int32), C.c_int32, C.c_int32, C.POINTER(C.c_int32), C.c_int32]
    L.vcs_next_position_base.argtypes = [C.c_int32] * 5 + [C.POINTER(C.c_int32)]
    L.vcs_text_positions.argtypes = [C.c_int32, C.c_int32, C.POINTER(C.c_int32)]
    L.vcs_pool_opaque_bytes.restype = sz
    L.vcs_pool_init.argtypes = [pp]
    L.vcs_temporal_drop_workspace_bytes.restype = sz
    L.vcs_temporal_drop_workspace_bytes.argtypes = [i32, i32, i32]
    L.vcs_temporal_drop.argtypes = [vp, vp, i32, i32, i32, i32, i32, f32, i32, vp, vp, vp, vp, i32, i32, i32, vp,
                                    vp, sz, vp]
    L.vcs_temporal_drop_static.argtypes = [vp, vp, i32, i32, i32, i32, i32, f32, i32, vp, vp, vp, vp, i32, i32, i32, vp, vp]
    L.vcs_spatial_entropy_topk_workspace_bytes.restype = sz
    L.vcs_spatial_entropy_topk_workspace_bytes.argtypes = [i32, i32, i32]
    L.vcs_spatial_entropy_topk.argtypes = [vp, i32, i32, i32, i32, i32, i32, vp, vp, vp, vp, i32, i32, i32, vp, vp, sz, vp]
    L.vcs_kv_append_workspace_bytes.restype = sz
    L.vcs_kv_append_workspace_bytes.argtypes = [pp, i32]
    L.vcs_kv_append_pages.argtypes = [pp, vp, vp, i64, i64, vp, vp, i32, C.c_int32, C.c_int32, vp, vp, sz, vp]
    L.vcs_kv_append_batched_workspace_bytes.restype = sz
    L.vcs_kv_append_batched_workspace_bytes.argtypes = [pp, i32, i32]
    L.vcs_kv_append_pages_batched.argtypes = [pp, vp, vp, i64, i64, i64, i64, vp, vp, i32, vp, i32, vp, vp, sz, vp]
    L.vcs_bounded_prefill_attn_workspace_bytes.restype = sz
    L.vcs_bounded_prefill_attn_workspace_bytes.argtypes = [pp, i32, i32]
    L.vcs_bounded_prefill_attn.argtypes = [pp, vp, i64, vp, vp, i32, vp, vp, i32, C.c_int32, C.c_int32, f32, vp,
                                           i64, vp, i32, vp, vp, sz, vp]
    L.vcs_bounded_prefill_attn_batched.argtypes = [pp, vp, i64, i64, vp, vp, i32, vp, vp, i32, vp, C.c_int32, f32, vp,
                                                   i64, i64, vp, i32, i32, vp, vp, sz, vp]
    L.vcs_retrieval_score_workspace_bytes.restype = sz
    L.vcs_retrieval_score_workspace_bytes.argtypes = [pp, i32]
    L.vcs_retrieval_score.argtypes = [pp, vp, i64, vp, i32, vp, i32, vp, i32, i32, vp, i32, vp, vp, sz, vp]
    L.vcs_retrieval_threshold.argtypes = [pp, vp, vp, i32, vp, i32, f32, vp, i32, vp, vp]
    L.vcs_chunk_ingest.argtypes = [pp, C.POINTER(_ChunkCall), vp]
    L.vcs_chunk_ingest_host.argtypes = [pp, C.POINTER(_ChunkCall), vp, vp, vp, vp, vp, vp, vp, vp]
    L.vcs_chunk_upload.argtypes = [pp, C.POINTER(_ChunkCall), vp, vp, vp, vp, vp]
    L.vcs_chunk_download.argtypes = [pp, C.POINTER(_ChunkCall), vp, vp, vp, vp]
    L.vcs_ingest_layers.argtypes = [C.POINTER(pp), C.POINTER(_MultiCall), vp]
    L.vcs_graph_begin.argtypes = [vp]
    L.vcs_graph_end.argtypes = [vp, C.POINTER(vp)]
    L.vcs_graph_launch.argtypes = [vp, vp]
    L.vcs_graph_destroy.argtypes = [vp]
    L.vcs_sizeof_chunk_call.restype = sz
    L.vcs_selftest_exp2_poly.argtypes = [vp, vp, i32, vp]
    L.vcs_selftest_rope_sincos.argtypes = [vp, i32, C.c_double, vp, vp, vp]
    L.vcs_sizeof_multi_call.restype = sz
    # the structs above mirror include/vcs.h by hand: refuse a library built from another header
    if L.vcs_version() != VERSION or L.vcs_sizeof_chunk_call() != C.sizeof(_ChunkCall) or \
            L.vcs_sizeof_multi_call() != C.sizeof(_MultiCall):
        raise RuntimeError(f"{LIB_PATH} (version {L.vcs_version()}, vcs_chunk_call {L.vcs_sizeof_chunk_call()} B, vcs_multi_call "
                           f"{L.vcs_sizeof_multi_call()} B) does not match this binding (version {VERSION}, "
                           f"{C.sizeof(_ChunkCall)} B, {C.sizeof(_MultiCall)} B): rebuild with `python -m paper_2606_19849_b200.build`")
    _lib = L
    return L


def _check(rc: int):
    if rc != OK:
        raise VcsError(rc, lib().vcs_last_error().decode(errors="replace"))


def _ptr(t: Optional[torch.Tensor]) -> Optional[int]:
    if t is None:
        return None
    if not t.is_cuda:
        raise VcsError(ECUDA, "vcs calls need CUDA tensors (there is no CPU path)")
    return t.data_ptr()


def _stream(stream=None) -> int:
    s = torch.cuda.current_stream() if stream is None else stream
    return s.cuda_stream


def _dtype_code(dt: torch.dtype) -> int:
    if dt == torch.bfloat16:
        return BF16
    if dt == torch.float32:
        return F32
    raise VcsError(EUNSUPPORTED, f"dtype {dt}")


def vcs_version() -> int:
    return lib().vcs_version()


def vcs_device_info():
    sm, ma, mi = C.c_int(), C.c_int(), C.c_int()
    name = C.create_string_buffer(256)
    _check(lib().vcs_device_info(C.byref(sm), C.byref(ma), C.byref(mi), name, 256))
    return dict(sm_count=sm.value, cc=(ma.value, mi.value), name=name.value.decode())


def vcs_visible_set(t: int, W: int, sink_page: int, chunk_pages, table_cap: int):
    """Step a6 (include/vcs.h): (table padded with -1 to table_cap, n_vis) of chunk t; host lists."""
    n = len(chunk_pages)
    pages = (C.c_int32 * max(n, 1))(*chunk_pages)
    out = (C.c_int32 * max(table_cap, 1))()
    rc = lib().vcs_visible_set(t, W, sink_page, pages, n, out, table_cap)
    if rc < 0:
        _check(rc)
    return list(out[:table_cap]), rc


def vcs_visible_set_query(sink_page: int, recent_pages, k: int, table_cap: Optional[int] = None):
    """Query side of step a6 (include/vcs.h): (table with k empty slots padded with -1, index of the first slot)."""
    n = len(recent_pages)
    cap = (1 if sink_page >= 0 else 0) + n + k if table_cap is None else table_cap
    rec = (C.c_int32 * max(n, 1))(*recent_pages)
    out = (C.c_int32 * max(cap, 1))()
    rc = lib().vcs_visible_set_query(sink_page, rec, n, k, out, cap)
    if rc < 0:
        _check(rc)
    return list(out[:cap]), rc


def vcs_next_position_base(G: int, Hg: int, Wg: int, base: int, t_stride: int = 1) -> int:
    out = C.c_int32(0)
    _check(lib().vcs_next_position_base(G, Hg, Wg, t_stride, base, C.byref(out)))
    return out.value


def vcs_text_positions(start: int, n: int, device="cuda") -> torch.Tensor:
    """[n][3] int32 positions of sink / text tokens, computed behind the C ABI and copied to `device`."""
    buf = (C.c_int32 * max(3 * n, 1))()
    _check(lib().vcs_text_positions(start, n, buf))
    return torch.tensor(list(buf[:3 * n]), dtype=torch.int32).view(n, 3).to(device)


class KVPool:
    """Caller-side owner of the paged KV cache buffers (torch) + the vcs_kv_pool descriptor."""

    def __init__(self, n_pages: int, page_cap: int, Hq: int, Hkv: int, d: int, dtype: torch.dtype,
                 rope_theta: float, rope_sections, device="cuda"):
        self.n_pages, self.page_cap, self.Hq, self.Hkv, self.d, self.dtype = n_pages, page_cap, Hq, Hkv, d, dtype
        self.k_pages = torch.zeros((n_pages, Hkv, page_cap, d), dtype=dtype, device=device)
        self.v_pages = torch.zeros((n_pages, Hkv, page_cap, d), dtype=dtype, device=device)
        self.page_len = torch.zeros((n_pages,), dtype=torch.int32, device=device)
        self.k_sum = torch.zeros((n_pages, Hkv, d), dtype=torch.float32, device=device)
        nbytes = lib().vcs_pool_opaque_bytes()
        self._opaque = C.create_string_buffer(nbytes + 64)
        base = C.addressof(self._opaque)
        self.c = _Pool(self.k_pages.data_ptr(), self.v_pages.data_ptr(), self.page_len.data_ptr(),
                       self.k_sum.data_ptr(), n_pages, page_cap, Hkv, Hq, d, _dtype_code(dtype),
                       float(rope_theta), (C.c_int32 * 3)(*rope_sections), (base + 63) // 64 * 64)
        _check(lib().vcs_pool_init(C.byref(self.c)))

    @property
    def ref(self):
        return C.byref(self.c)


def workspace(nbytes: int, device="cuda") -> torch.Tensor:
    """Zeroed scratch buffer (the C ABI wants workspaces zeroed once before first use)."""
    return torch.zeros((max(int(nbytes), 256),), dtype=torch.uint8, device=device)


def vcs_temporal_drop_workspace_bytes(B: int, G: int, P: int) -> int:
    return lib().vcs_temporal_drop_workspace_bytes(B, G, P)


def vcs_temporal_drop(z: torch.Tensor, tau: float, kept_idx: torch.Tensor, kept_count: torch.Tensor,
                      workspace: torch.Tensor, mode: int = DROP_CHUNK_ALLPAIRS,
                      prev_last_group: Optional[torch.Tensor] = None, keep_mask: Optional[torch.Tensor] = None,
                      pos3: Optional[torch.Tensor] = None, Hg: int = 0, Wg: int = 0, t_stride: int = 1,
                      pos_base: Optional[torch.Tensor] = None, stream=None):
    """z: [B][G][P][D] contiguous CUDA tensor (bf16 / fp32).  See include/vcs.h."""
    B, G, P, D = z.shape
    if not z.is_contiguous():
        raise VcsError(EINVAL, "z must be contiguous [B][G][P][D]")
    _check(lib().vcs_temporal_drop(_ptr(z), _ptr(prev_last_group), B, G, P, D, _dtype_code(z.dtype), float(tau), mode,
                                   _ptr(kept_idx), _ptr(kept_count), _ptr(keep_mask), _ptr(pos3), Hg, Wg, t_stride,
                                   _ptr(pos_base), _ptr(workspace), workspace.numel(), _stream(stream)))


DROP_STATIC_SCRATCH_BYTES = 1 << 20


def vcs_temporal_drop_static(z: torch.Tensor, tau: float, kept_idx: torch.Tensor, kept_count: torch.Tensor,
                             mode: int = DROP_CHUNK_ALLPAIRS, prev_last_group: Optional[torch.Tensor] = None,
                             keep_mask: Optional[torch.Tensor] = None, pos3: Optional[torch.Tensor] = None,
                             Hg: int = 0, Wg: int = 0, t_stride: int = 1, pos_base: Optional[torch.Tensor] = None,
                             stream=None):
    """vcs_temporal_drop without a workspace argument, for callers that cannot allocate one (a server whose
    pool owns all device memory, a loop that must not call cudaMalloc, a plug-in without an allocator).  The
    scratch is a fixed DROP_STATIC_SCRATCH_BYTES array inside libvcs.so, one per GPU and shared by every call:
    shapes that need more raise VcsError(ECAP), and calls that may overlap on the GPU must be ordered by the
    caller.  The first call on a device looks the array up; make it before any stream capture.  See include/vcs.h."""
    B, G, P, D = z.shape
    if not z.is_contiguous():
        raise VcsError(EINVAL, "z must be contiguous [B][G][P][D]")
    _check(lib().vcs_temporal_drop_static(_ptr(z), _ptr(prev_last_group), B, G, P, D, _dtype_code(z.dtype), float(tau),
                                          mode, _ptr(kept_idx), _ptr(kept_count), _ptr(keep_mask), _ptr(pos3), Hg, Wg,
                                          t_stride, _ptr(pos_base), _stream(stream)))


def vcs_spatial_entropy_topk(z: torch.Tensor, K: int, kept_idx: torch.Tensor, kept_count: torch.Tensor,
                             workspace: Optional[torch.Tensor] = None, entropy: Optional[torch.Tensor] = None,
                             pos3: Optional[torch.Tensor] = None, Hg: int = 0, Wg: int = 0, t_stride: int = 1,
                             pos_base: Optional[torch.Tensor] = None, stream=None):
    """Entropy-based spatial top-K selection; z: [B][G][P][D] contiguous CUDA tensor."""
    B, G, P, D = z.shape
    if not z.is_contiguous():
        raise VcsError(EINVAL, "z must be contiguous [B][G][P][D]")
    _check(lib().vcs_spatial_entropy_topk(_ptr(z), B, G, P, D, _dtype_code(z.dtype), K, _ptr(kept_idx), _ptr(kept_count),
                                          _ptr(entropy), _ptr(pos3), Hg, Wg, t_stride, _ptr(pos_base), _ptr(workspace),
                                          0 if workspace is None else workspace.numel(), _stream(stream)))


def vcs_kv_append_workspace_bytes(pool: KVPool, n_cap: int) -> int:
    return lib().vcs_kv_append_workspace_bytes(pool.ref, n_cap)


def vcs_kv_append_pages(pool: KVPool, k: torch.Tensor, v: torch.Tensor, pos3: torch.Tensor,
                        n_d: Optional[torch.Tensor], n_cap: int, page_id: int, page_offset: int,
                        workspace: torch.Tensor, status: Optional[torch.Tensor] = None, stream=None):
    """k, v: [>=n_cap][Hkv][d] with arbitrary row stride (last two dims contiguous)."""
    _check(lib().vcs_kv_append_pages(pool.ref, _ptr(k), _ptr(v), k.stride(0) if k.dim() == 3 else 0,
                                     v.stride(0) if v.dim() == 3 else 0, _ptr(pos3), _ptr(n_d), n_cap, page_id,
                                     page_offset, _ptr(status), _ptr(workspace), workspace.numel(), _stream(stream)))


def vcs_kv_append_batched_workspace_bytes(pool: KVPool, n_cap: int, B: int) -> int:
    return lib().vcs_kv_append_batched_workspace_bytes(pool.ref, n_cap, B)


def vcs_kv_append_pages_batched(pool: KVPool, k: torch.Tensor, v: torch.Tensor, pos3: torch.Tensor,
                                n_d: Optional[torch.Tensor], n_cap: int, page_ids: torch.Tensor,
                                workspace: torch.Tensor, status: Optional[torch.Tensor] = None, stream=None):
    """k, v: [B][>=n_cap][Hkv][d]; pos3: [B][n_cap][3]; n_d: int32 [B] or None; page_ids: int32 [B] (device)."""
    B = k.shape[0]
    _check(lib().vcs_kv_append_pages_batched(pool.ref, _ptr(k), _ptr(v), k.stride(0), v.stride(0), k.stride(1),
                                             v.stride(1), _ptr(pos3), _ptr(n_d), n_cap, _ptr(page_ids), B,
                                             _ptr(status), _ptr(workspace), workspace.numel(), _stream(stream)))


def vcs_bounded_prefill_attn_workspace_bytes(pool: KVPool, nq_cap: int, n_vis_cap: int) -> int:
    return lib().vcs_bounded_prefill_attn_workspace_bytes(pool.ref, nq_cap, n_vis_cap)


def vcs_bounded_prefill_attn(pool: KVPool, q: torch.Tensor, q_pos3: torch.Tensor, nq_d: Optional[torch.Tensor],
                             nq_cap: int, page_table: Optional[torch.Tensor], n_vis_d: Optional[torch.Tensor],
                             n_vis_cap: int, self_page: int, self_offset: int, out: torch.Tensor,
                             workspace: torch.Tensor, lse: Optional[torch.Tensor] = None, softmax_scale: float = 0.0,
                             flags: int = ATTN_AUTO, status: Optional[torch.Tensor] = None, stream=None):
    """q, out: [>=nq_cap][Hq][d] (row stride free); page_table: int32 [>=n_vis_cap]."""
    _check(lib().vcs_bounded_prefill_attn(pool.ref, _ptr(q), q.stride(0), _ptr(q_pos3), _ptr(nq_d), nq_cap,
                                          _ptr(page_table), _ptr(n_vis_d), n_vis_cap, self_page, self_offset,
                                          float(softmax_scale), _ptr(out), out.stride(0), _ptr(lse), flags,
                                          _ptr(status), _ptr(workspace), workspace.numel(), _stream(stream)))


def vcs_bounded_prefill_attn_batched(pool: KVPool, q: torch.Tensor, q_pos3: torch.Tensor, nq_d: Optional[torch.Tensor],
                                     nq_cap: int, page_tables: torch.Tensor, n_vis_d: Optional[torch.Tensor],
                                     self_pages: Optional[torch.Tensor], self_offset: int, out: torch.Tensor,
                                     workspace: torch.Tensor, lse: Optional[torch.Tensor] = None,
                                     softmax_scale: float = 0.0, flags: int = ATTN_AUTO,
                                     status: Optional[torch.Tensor] = None, stream=None):
    """q, out: [B][>=nq_cap][Hq][d]; q_pos3: [B][nq_cap][3]; page_tables: int32 [B][n_vis_cap]; nq_d, n_vis_d,
    self_pages: int32 [B] (device); lse: [B][Hq][nq_cap]."""
    B, n_vis_cap = page_tables.shape
    _check(lib().vcs_bounded_prefill_attn_batched(pool.ref, _ptr(q), q.stride(0), q.stride(1), _ptr(q_pos3), _ptr(nq_d),
                                                  nq_cap, _ptr(page_tables), _ptr(n_vis_d), n_vis_cap, _ptr(self_pages),
                                                  self_offset, float(softmax_scale), _ptr(out), out.stride(0),
                                                  out.stride(1), _ptr(lse), B, flags, _ptr(status), _ptr(workspace),
                                                  workspace.numel(), _stream(stream)))


def vcs_retrieval_score_workspace_bytes(pool: KVPool, n_cand: int) -> int:
    return lib().vcs_retrieval_score_workspace_bytes(pool.ref, n_cand)


def vcs_retrieval_score(pool: KVPool, q: torch.Tensor, nq_d: Optional[torch.Tensor], nq_cap: int,
                        cand_pages: torch.Tensor, scores: torch.Tensor, workspace: torch.Tensor,
                        k: int = 0, topk_pages: Optional[torch.Tensor] = None,
                        exclude_pages: Optional[torch.Tensor] = None, normalize: bool = False, stream=None):
    n_excl = 0 if exclude_pages is None else exclude_pages.numel()
    _check(lib().vcs_retrieval_score(pool.ref, _ptr(q), q.stride(0), _ptr(nq_d), nq_cap, _ptr(cand_pages),
                                     cand_pages.numel(), _ptr(exclude_pages), n_excl, 1 if normalize else 0,
                                     _ptr(scores), k, _ptr(topk_pages), _ptr(workspace), workspace.numel(),
                                     _stream(stream)))


def vcs_retrieval_threshold(pool: KVPool, scores: torch.Tensor, cand_pages: torch.Tensor, tau_q: float,
                            vis_pages: torch.Tensor, vis_count: torch.Tensor,
                            exclude_pages: Optional[torch.Tensor] = None, stream=None):
    """V_qry = {j : s_j >= tau_q} from scores of vcs_retrieval_score; see include/vcs.h."""
    n_excl = 0 if exclude_pages is None else exclude_pages.numel()
    _check(lib().vcs_retrieval_threshold(pool.ref, _ptr(scores), _ptr(cand_pages), cand_pages.numel(),
                                         _ptr(exclude_pages), n_excl, float(tau_q), _ptr(vis_pages), vis_pages.numel(),
                                         _ptr(vis_count), _stream(stream)))


def vcs_selftest_exp2_poly(x: torch.Tensor, stream=None) -> torch.Tensor:
    """The softmax's polynomial 2^x evaluated on the device at the fp32 points x (include/vcs.h, self-test hooks)."""
    x = x.contiguous().float()
    y = torch.empty_like(x)
    _check(lib().vcs_selftest_exp2_poly(_ptr(x), _ptr(y), x.numel(), _stream(stream)))
    return y


def vcs_selftest_rope_sincos(pos: torch.Tensor, inv_freq: float, stream=None):
    """(sin, cos) of pos * inv_freq as the kernels compute them (Q0.64 turn fraction + MUFU); pos: int32 CUDA tensor."""
    pos = pos.contiguous().to(torch.int32)
    s = torch.empty(pos.shape, dtype=torch.float32, device=pos.device)
    c = torch.empty_like(s)
    _check(lib().vcs_selftest_rope_sincos(_ptr(pos), pos.numel(), float(inv_freq), _ptr(s), _ptr(c), _stream(stream)))
    return s, c


def make_chunk_call(pool: KVPool, z: torch.Tensor, q: torch.Tensor, k: torch.Tensor, v: torch.Tensor,
                    out: torch.Tensor, kept_idx: torch.Tensor, kept_count: torch.Tensor, pos3: torch.Tensor,
                    pos_base: torch.Tensor, page_table: torch.Tensor, n_vis: torch.Tensor, page_id: int,
                    Hg: int, Wg: int, tau: float, ws_drop: torch.Tensor, ws_append: torch.Tensor,
                    ws_attn: torch.Tensor, status: Optional[torch.Tensor] = None, t_stride: int = 1,
                    mode: int = DROP_CHUNK_ALLPAIRS, attn_flags: int = ATTN_AUTO,
                    prev_last_group: Optional[torch.Tensor] = None, host_rows: int = 0) -> _ChunkCall:
    """Fill a vcs_chunk_call (include/vcs.h) from device tensors; z: [G][P][D]."""
    G, P, D = z.shape
    return _ChunkCall(G, P, D, Hg, Wg, t_stride, _dtype_code(z.dtype), mode, float(tau), page_id,
                      page_table.numel(), attn_flags, int(host_rows), _ptr(z), _ptr(q), _ptr(k), _ptr(v), _ptr(out),
                      _ptr(kept_idx), _ptr(kept_count), _ptr(pos3), _ptr(pos_base), _ptr(page_table), _ptr(n_vis),
                      _ptr(prev_last_group), _ptr(status), _ptr(ws_drop), _ptr(ws_append), _ptr(ws_attn), ws_drop.numel(),
                      ws_append.numel(), ws_attn.numel())


def vcs_chunk_ingest(pool: KVPool, call: _ChunkCall, stream=None):
    _check(lib().vcs_chunk_ingest(pool.ref, C.byref(call), _stream(stream)))


def vcs_chunk_ingest_host(pool: KVPool, call: _ChunkCall, z_h: torch.Tensor, q_h: torch.Tensor, k_h: torch.Tensor,
                          v_h: torch.Tensor, out_h: torch.Tensor, kept_idx_h: torch.Tensor,
                          kept_count_h: torch.Tensor, stream=None):
    """Host (pinned) tensors in and out; copies and kernels are only enqueued on the stream."""
    for t in (z_h, q_h, k_h, v_h, out_h, kept_idx_h, kept_count_h):
        if t.is_cuda or not t.is_contiguous():
            raise VcsError(EINVAL, "vcs_chunk_ingest_host takes contiguous HOST tensors")
    _check(lib().vcs_chunk_ingest_host(pool.ref, C.byref(call), z_h.data_ptr(), q_h.data_ptr(), k_h.data_ptr(),
                                       v_h.data_ptr(), out_h.data_ptr(), kept_idx_h.data_ptr(),
                                       kept_count_h.data_ptr(), _stream(stream)))


def make_multi_call(pools, z: torch.Tensor, q: torch.Tensor, k: torch.Tensor, v: torch.Tensor, out: torch.Tensor,
                    kept_idx: torch.Tensor, kept_count: torch.Tensor, pos3: torch.Tensor, pos_base: torch.Tensor,
                    page_ids: torch.Tensor, page_tables: torch.Tensor, n_vis: torch.Tensor, Hg: int, Wg: int, tau: float,
                    ws_drop: torch.Tensor, ws_append: torch.Tensor, ws_attn: torch.Tensor,
                    status: Optional[torch.Tensor] = None, t_stride: int = 1, mode: int = DROP_CHUNK_ALLPAIRS,
                    attn_flags: int = ATTN_AUTO, prev_last_group: Optional[torch.Tensor] = None,
                    share_qkv_across_layers: bool = False) -> _MultiCall:
    """Fill a vcs_multi_call (include/vcs.h).  z: [B][G][P][D]; q, out: [L][B][T][Hq][d]; k, v: [L][B][T][Hkv][d]
    (or [B][T][..] with share_qkv_across_layers: layer stride 0); page_tables: int32 [B][n_vis_cap]."""
    B, G, P, D = z.shape
    L = len(pools)
    qs = 0 if share_qkv_across_layers else q.stride(0)
    ks = 0 if share_qkv_across_layers else k.stride(0)
    return _MultiCall(B, L, G, P, D, Hg, Wg, t_stride, _dtype_code(z.dtype), mode, float(tau), page_tables.shape[1],
                      attn_flags, qs, ks, out.stride(0), _ptr(z), _ptr(q), _ptr(k), _ptr(v), _ptr(out),
                      _ptr(prev_last_group), _ptr(kept_idx), _ptr(kept_count), _ptr(pos3), _ptr(pos_base), _ptr(page_ids),
                      _ptr(page_tables), _ptr(n_vis), _ptr(status), _ptr(ws_drop), _ptr(ws_append), _ptr(ws_attn),
                      ws_drop.numel(), ws_append.numel(), ws_attn.numel())


def vcs_ingest_layers(pools, call: _MultiCall, stream=None):
    """One token drop for the B streams, then per layer one batched KV append and one batched bounded prefill."""
    arr = (C.POINTER(_Pool) * len(pools))(*[C.pointer(p.c) for p in pools])
    _check(lib().vcs_ingest_layers(arr, C.byref(call), _stream(stream)))


class Graph:
    """CUDA graph of a chain of vcs calls: `with Graph.capture(stream) as g: ...calls...`, then g.launch()."""

    def __init__(self):
        self.handle = C.c_void_p()
        self.stream = None

    @classmethod
    def capture(cls, stream=None):
        g = cls()
        g.stream = torch.cuda.current_stream() if stream is None else stream
        return g

    def __enter__(self):
        _check(lib().vcs_graph_begin(self.stream.cuda_stream))
        return self

    def __exit__(self, exc_type, exc, tb):
        rc = lib().vcs_graph_end(self.stream.cuda_stream, C.byref(self.handle))
        if exc_type is None:
            _check(rc)
        return False

    def launch(self, stream=None):
        _check(lib().vcs_graph_launch(self.handle, _stream(stream)))

    def __del__(self):
        if self.handle and _lib is not None:
            _lib.vcs_graph_destroy(self.handle)
            self.handle = C.c_void_p()
