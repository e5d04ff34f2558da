"""Seeded synthetic inputs shared by the oracle-side tests and the CUDA-side tests/bench.

This package holds NONE of the method's arithmetic (no similarity, no RoPE, no softmax):
only shapes, seeds, random draws and the bf16 storage format.  The recipe is stated in
DESIGN.md ("Input recipe") and follows BASELINE.json `configs` / SURVEY.md section 8(d).
"""
from .configs import CONFIGS, StreamConfig, get_config  # noqa: F401
from .generators import (  # noqa: F401
    bf16_round, bf16_bits, gen_hidden_tiny, gen_hidden_chunk, gen_qkv, gen_sink_kv,
    gen_proj_weights_tiny, gen_page_ids, gen_bank, gen_query, to_torch,
)
