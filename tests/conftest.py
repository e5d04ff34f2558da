import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on the B200 box)")


def pytest_collection_modifyitems(config, items):
    import torch
    if torch.cuda.is_available():
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)


def pytest_terminal_summary(terminalreporter):
    """Measured attention errors of the run beside their bars (reading D32 scales the max-abs bar only where the
    oracle's |O|_inf exceeds 1): the worst cases, and every comparison that NEEDED the scaled bar."""
    try:
        from helpers import ATTN_MAX_ABS, ATTN_REL_L2, PARITY_LOG
    except ImportError:
        return
    if not PARITY_LOG:
        return
    w_ma = max(PARITY_LOG, key=lambda r: r["ma"] / r["bar"])
    w_rl = max(PARITY_LOG, key=lambda r: r["rl"])
    scaled = [r for r in PARITY_LOG if r["bar"] > ATTN_MAX_ABS]
    needed = [r for r in PARITY_LOG if r["ma"] > ATTN_MAX_ABS]
    tr = terminalreporter
    tr.write_line(f"attention parity: {len(PARITY_LOG)} comparisons; worst max-abs {w_ma['ma']:.3e} of bar {w_ma['bar']:.3e} "
                  f"(|O|inf {w_ma['omax']:.2f}, {w_ma['test']}); worst rel-L2 {w_rl['rl']:.3e} of {ATTN_REL_L2:.0e} ({w_rl['test']})")
    tr.write_line(f"attention parity: {len(scaled)} comparisons had |O|inf > 1 (D32 bar applies), {len(needed)} of them exceeded the "
                  f"flat {ATTN_MAX_ABS:.0e}" + "".join(f"; {r['test']} {r['ma']:.3e} <= {r['bar']:.3e}" for r in needed[:6]))
