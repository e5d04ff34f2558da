"""Seeded synthetic input generators (numpy, CPU).  No method arithmetic lives here.

All floating-point outputs are float32 arrays whose values are exactly representable in the
config's storage type (bf16 for configs 2-5, fp32 for Tiny), so the fp64 oracle and the CUDA
path consume identical bits.  `to_torch` converts to the torch dtype the binding wants.

Recipe: BASELINE.json `configs` + SURVEY.md section 8(d); stated again in DESIGN.md.
  * Tiny (config 1): literal BASELINE text -- group 0 of chunk 0 is fresh N(0,1); every later
    group's token is the previous group's token + N(0, std 0.01) with p = 0.5, else fresh N(0,1);
    the chain runs across chunks; seed 0.
  * Configs 2-4: per (chunk, position) a static flag ~ Bernoulli(rho).  A static position gets
    base(p) + N(0, std 0.05) in each of the G groups, a dynamic one gets G fresh N(0,1) vectors.
    By construction every pairwise cosine at a static position is ~0.9975 and at a dynamic one
    ~N(0, 1/D), i.e. at least 1e-2 away from tau = 0.95 (tests assert the 1e-4 margin with the
    oracle; the generator itself never evaluates a similarity).
  * Q/K/V for configs 2-5: N(0,1) per kept token and head.  Sink K/V ~ N(0,1).
"""
from __future__ import annotations

import numpy as np

from .configs import StreamConfig


def bf16_round(x: np.ndarray) -> np.ndarray:
    """Round float32 -> nearest bf16 (ties to even), returned as float32.  Storage format only."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    u = x.view(np.uint32)
    r = ((u >> np.uint32(16)) & np.uint32(1)) + np.uint32(0x7FFF)
    out = ((u + r) & np.uint32(0xFFFF0000)).view(np.float32)
    return out.reshape(x.shape)


def bf16_bits(x: np.ndarray) -> np.ndarray:
    """Upper 16 bits of bf16-representable float32 values (uint16)."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    return (x.view(np.uint32) >> np.uint32(16)).astype(np.uint16).reshape(x.shape)


def _store(cfg: StreamConfig, x: np.ndarray) -> np.ndarray:
    x = x.astype(np.float32)
    return bf16_round(x) if cfg.dtype == "bf16" else x


def to_torch(x: np.ndarray, dtype: str):
    """numpy float32 (storage-exact) -> torch CPU tensor of the storage dtype."""
    import torch
    t = torch.from_numpy(np.ascontiguousarray(x, dtype=np.float32))
    return t.to(torch.bfloat16) if dtype == "bf16" else t


def _rng(cfg: StreamConfig, *key: int) -> np.random.Generator:
    return np.random.default_rng([cfg.config_id, cfg.seed, *key])


def gen_hidden_tiny(cfg: StreamConfig) -> np.ndarray:
    """Tiny config hidden tokens Z[n_chunks][G][P][D] (fp32), BASELINE.json config 1 recipe."""
    rng = np.random.default_rng(cfg.seed)
    Z = np.empty((cfg.n_chunks, cfg.G, cfg.P, cfg.D), dtype=np.float32)
    prev = None
    for t in range(cfg.n_chunks):
        for g in range(cfg.G):
            fresh = rng.standard_normal((cfg.P, cfg.D)).astype(np.float32)
            if prev is None:
                cur = fresh
            else:
                copy = rng.random(cfg.P) < 0.5
                noise = (0.01 * rng.standard_normal((cfg.P, cfg.D))).astype(np.float32)
                cur = np.where(copy[:, None], prev + noise, fresh).astype(np.float32)
            Z[t, g] = cur
            prev = cur
    return Z


def gen_hidden_chunk(cfg: StreamConfig, chunk_idx: int, stream_idx: int = 0):
    """Configs 2-4 hidden tokens of one chunk: (Z[G][P][D] storage-exact float32, static[P] bool)."""
    rng = _rng(cfg, 1, chunk_idx, stream_idx)
    static = rng.random(cfg.P) < cfg.rho
    Z = rng.standard_normal((cfg.G, cfg.P, cfg.D)).astype(np.float32)
    base = rng.standard_normal((cfg.P, cfg.D)).astype(np.float32)
    jitter = (0.05 * rng.standard_normal((cfg.G, cfg.P, cfg.D))).astype(np.float32)
    Z = np.where(static[None, :, None], base[None] + jitter, Z)
    return _store(cfg, Z), static


def gen_qkv(cfg: StreamConfig, chunk_idx: int, n_rows: int, stream_idx: int = 0, q_std: float = 1.0):
    """Direct synthetic Q[n][Hq][d], K[n][Hkv][d], V[n][Hkv][d] ~ N(0,1) (configs 2-5)."""
    rng = _rng(cfg, 2, chunk_idx, stream_idx)
    Q = q_std * rng.standard_normal((n_rows, cfg.Hq, cfg.d))
    K = rng.standard_normal((n_rows, cfg.Hkv, cfg.d))
    V = rng.standard_normal((n_rows, cfg.Hkv, cfg.d))
    return _store(cfg, Q), _store(cfg, K), _store(cfg, V)


def gen_sink_kv(cfg: StreamConfig):
    """Sink / system prefix K, V [S][Hkv][d] ~ N(0,1)."""
    rng = _rng(cfg, 3)
    K = rng.standard_normal((cfg.sink, cfg.Hkv, cfg.d))
    V = rng.standard_normal((cfg.sink, cfg.Hkv, cfg.d))
    return _store(cfg, K), _store(cfg, V)


def gen_proj_weights_tiny(cfg: StreamConfig, std: float = 0.02):
    """Tiny config projection matrices Wq[D][Hq*d], Wk[D][Hkv*d], Wv[D][Hkv*d] ~ N(0, std)."""
    rng = _rng(cfg, 4)
    Wq = (std * rng.standard_normal((cfg.D, cfg.Hq * cfg.d))).astype(np.float32)
    Wk = (std * rng.standard_normal((cfg.D, cfg.Hkv * cfg.d))).astype(np.float32)
    Wv = (std * rng.standard_normal((cfg.D, cfg.Hkv * cfg.d))).astype(np.float32)
    return Wq, Wk, Wv


def gen_page_ids(n_pool_pages: int, n_needed: int, seed: int) -> np.ndarray:
    """Scattered, non-contiguous physical page ids: a seeded permutation of the pool."""
    rng = np.random.default_rng([77, seed])
    return rng.permutation(n_pool_pages)[:n_needed].astype(np.int32)


def gen_bank(cfg: StreamConfig, n_bank: int, len_lo: int, len_hi: int):
    """Config-5 KV bank: per-page lengths in [len_lo, len_hi] and a seeded generator of page K/V.

    Returns (lens[n_bank] int32, page_kv) where page_kv(i) -> (K[len_i][Hkv][d], V[len_i][Hkv][d]).
    """
    rng = _rng(cfg, 5)
    lens = rng.integers(len_lo, len_hi + 1, size=n_bank).astype(np.int32)

    def page_kv(i: int):
        r = _rng(cfg, 6, i)
        K = r.standard_normal((int(lens[i]), cfg.Hkv, cfg.d))
        V = r.standard_normal((int(lens[i]), cfg.Hkv, cfg.d))
        return _store(cfg, K), _store(cfg, V)

    return lens, page_kv


def gen_query(cfg: StreamConfig, nq: int, draw: int = 0):
    """Config-5 text query tokens: Q[nq][Hq][d], K[nq][Hkv][d], V[nq][Hkv][d] ~ N(0,1)."""
    rng = _rng(cfg, 7, draw)
    Q = rng.standard_normal((nq, cfg.Hq, cfg.d))
    K = rng.standard_normal((nq, cfg.Hkv, cfg.d))
    V = rng.standard_normal((nq, cfg.Hkv, cfg.d))
    return _store(cfg, Q), _store(cfg, K), _store(cfg, V)
