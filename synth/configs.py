"""The five BASELINE.json workload configurations as plain data (no arithmetic).

Symbols follow SURVEY.md section 8: G temporal groups per chunk, grid Hg x Wg (P = Hg*Wg tokens
per group, T = G*P per chunk), D hidden size, Hq/Hkv heads, d head_dim, S sink length,
W window in chunks (paper `acn`), tau threshold (paper Eq. 2).
"""
from __future__ import annotations

from dataclasses import dataclass, replace
from typing import Tuple


@dataclass(frozen=True)
class StreamConfig:
    name: str
    config_id: int
    dtype: str                 # "f32" | "bf16" -- storage type of tokens / Q / K / V
    Hq: int
    Hkv: int
    d: int
    D: int
    G: int
    Hg: int
    Wg: int
    rho: float                 # static-position probability of the generator
    tau: float
    sink: int
    W: int                     # window in chunks; <0 means unbounded (full history)
    n_chunks: int
    rope_theta: float = 1.0e6
    t_stride: int = 1
    seed: int = 0

    @property
    def P(self) -> int:
        return self.Hg * self.Wg

    @property
    def T(self) -> int:
        return self.G * self.P

    @property
    def group(self) -> int:
        return self.Hq // self.Hkv

    @property
    def rope_sections(self) -> Tuple[int, int, int]:
        # pairs per (t, h, w) axis; sum == d/2 (reading D17)
        return {128: (16, 24, 24), 64: (8, 12, 12)}[self.d]

    @property
    def page_cap(self) -> int:
        # one page holds one chunk; rounded up to the attention kernel's 128-token tile
        return max(128, -(-max(self.T, self.sink) // 128) * 128)

    def with_(self, **kw) -> "StreamConfig":
        return replace(self, **kw)


CONFIGS = {
    # config 1: Tiny, fp32, 6 chunks of 2 groups x 16 tokens, hidden 128
    "tiny": StreamConfig("tiny", 1, "f32", Hq=2, Hkv=1, d=64, D=128, G=2, Hg=4, Wg=4,
                         rho=0.5, tau=0.9, sink=8, W=2, n_chunks=6, seed=0),
    # config 2: Qwen2.5-VL-3B-shaped layer, chunk = 4 groups x (16x29) merged tokens
    "vl3b": StreamConfig("vl3b", 2, "bf16", Hq=16, Hkv=2, d=128, D=2048, G=4, Hg=16, Wg=29,
                         rho=0.6, tau=0.95, sink=64, W=4, n_chunks=8, seed=2),
    # config 3: Qwen2.5-VL-7B-shaped layer, 720p chunk = 4 groups x (26x46), 32 chunks
    "vl7b": StreamConfig("vl7b", 3, "bf16", Hq=28, Hkv=4, d=128, D=3584, G=4, Hg=26, Wg=46,
                         rho=0.75, tau=0.95, sink=128, W=8, n_chunks=32, seed=3),
    # config 4: history sweep on the config-2 shape, chunk index 1..64, W=inf vs W=8
    "sweep": StreamConfig("sweep", 4, "bf16", Hq=16, Hkv=2, d=128, D=2048, G=4, Hg=16, Wg=29,
                          rho=0.6, tau=0.95, sink=64, W=8, n_chunks=64, seed=4),
    # config 5: query-time TTFT path on the 7B shape (48 query tokens, 256-page bank, top-8)
    "ttft": StreamConfig("ttft", 5, "bf16", Hq=28, Hkv=4, d=128, D=3584, G=4, Hg=26, Wg=46,
                         rho=0.75, tau=0.95, sink=128, W=4, n_chunks=256, seed=5),
}

TTFT_NQ = 48        # text query tokens (BASELINE.json config 5)
TTFT_TOPK = 8       # retrieved chunks
TTFT_BANK = 256     # pages in the bank


def get_config(name: str) -> StreamConfig:
    return CONFIGS[name]
