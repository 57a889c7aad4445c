"""N > 1 host logic of bench.py on CPU (gloo, world_size 2): the path does not shard under
north_star (one GPU per simulation, replicas only -- DESIGN.md Sec. 8), so the only cross-rank
steps are the barrier and the max-over-ranks of the device times."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        mine = [100.0 + 7.0 * rank, 90.0 - 5.0 * rank]          # rank 1 slower overall, rank 0 slower on sweeps
        dist.barrier()
        total_ms, sweep_ms = bench.max_over_ranks(mine, dist, torch.device("cpu"))
        value = bench.whole_job_updates_per_ns(world, 256, 10, 4, total_ms)
        out.put((rank, total_ms, sweep_ms, value, bench.replica_seed(1, rank)))
    finally:
        dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, total_ms, sweep_ms, value, seed in res:
        assert total_ms == 107.0 and sweep_ms == 90.0            # element-wise max, same on both ranks
        assert value == pytest.approx(2 * 256 * 256 * 10 * 4 / (107.0 * 1e6), rel=1e-15)
        assert seed == 1 + rank                                  # independent replicas


def test_single_process_passthrough():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks([3.5, 2], None, None) == [3.5, 2.0]
    assert bench.whole_job_updates_per_ns(1, 1 << 18, 10, 10, 1000.0) == (1 << 36) * 100 / 1e9
