"""Multi-GPU = independent replicas: the path has no exchange step, so N ranks
run N independent streams and the only collective is the reduction of the TIMING (max over ranks).
Host logic only; used by bench.py and covered on CPU by a world_size-2 gloo test."""
from __future__ import annotations

from typing import Sequence, Tuple

import torch


def rank_stream_ids(rank: int, world: int, n_streams: int) -> Sequence[int]:
    """Streams (independent videos) are dealt round-robin to ranks; no stream is split across ranks."""
    return list(range(rank, n_streams, world))


def aggregate_throughput(times_ms: Sequence[float], units_this_rank: Sequence[float], world: int,
                         device="cpu") -> Tuple[list, list]:
    """times_ms[i]: this rank's device time of timed region i; units_this_rank[i]: work units this
    rank processed in it.  Returns (max-over-ranks times, whole-job units/s): every rank waits for
    the slowest one, so the job's throughput is the sum of all ranks' units over the MAX time."""
    t = torch.tensor(list(times_ms), dtype=torch.float64, device=device)
    u = torch.tensor(list(units_this_rank), dtype=torch.float64, device=device)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(u, op=dist.ReduceOp.SUM)
    t_l, u_l = t.tolist(), u.tolist()
    return t_l, [uu / (tt * 1e-3) if tt > 0 else 0.0 for tt, uu in zip(t_l, u_l)]
