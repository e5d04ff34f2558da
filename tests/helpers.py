"""Shared helpers of the GPU parity tests: upload seeded inputs, read pools back."""
import numpy as np
import torch

import synth


def dev(x: np.ndarray, dtype: str):
    return synth.to_torch(x, dtype).cuda()


def i32(x):
    return torch.as_tensor(np.asarray(x), dtype=torch.int32).cuda()


def f64(t: torch.Tensor) -> np.ndarray:
    return t.detach().float().cpu().numpy().astype(np.float64)


def tdtype(dtype: str):
    return torch.bfloat16 if dtype == "bf16" else torch.float32


def attn_errors(got: np.ndarray, ref: np.ndarray):
    """(max-abs error, relative L2 error) of an attention output against the oracle."""
    diff = got - ref
    return float(np.max(np.abs(diff))) if diff.size else 0.0, \
        float(np.linalg.norm(diff) / max(np.linalg.norm(ref), 1e-30))


# north_star tolerances for bf16-in / fp32-accumulate attention, and the Tiny fp32 path
ATTN_MAX_ABS, ATTN_REL_L2 = 1e-2, 5e-3
F32_MAX_ABS = 1e-5
