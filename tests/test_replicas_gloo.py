"""N > 1 path on CPU: two gloo ranks (127.0.0.1) run the replica host logic of bench.py --
stream dealing without overlap and the max-over-ranks timing / summed throughput reduction."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    from paper_2606_19849_b200.replicas import aggregate_throughput, rank_stream_ids
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        times = [10.0 + 5.0 * rank, 100.0 - 20.0 * rank]          # rank 1 slower on region 0, rank 0 on region 1
        units = [1000.0 * (rank + 1), 500.0]
        t, v = aggregate_throughput(times, units, world, "cpu")
        dist.barrier()
        q.put((rank, t, v, list(rank_stream_ids(rank, world, 7))))
    finally:
        dist.destroy_process_group()


def test_two_rank_replicas_max_time_and_summed_throughput():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, t, v, _ in res:
        assert t == [15.0, 100.0]                                  # MAX over ranks, identical on every rank
        assert abs(v[0] - 3000.0 / 15e-3) < 1e-6 and abs(v[1] - 1000.0 / 100e-3) < 1e-6
    s0, s1 = res[0][3], res[1][3]
    assert sorted(s0 + s1) == list(range(7)) and not set(s0) & set(s1)


def test_single_rank_is_identity():
    from paper_2606_19849_b200.replicas import aggregate_throughput
    t, v = aggregate_throughput([2.0], [4000.0], 1)
    assert t == [2.0] and v == [2.0e6]
