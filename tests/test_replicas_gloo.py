"""N > 1 host logic of bench.py on CPU (gloo, world_size 2).  Default: replicas (north_star: one GPU per
simulation), where the only cross-rank steps are the barrier and the max-over-ranks of the device times.
--parallel slabs (NEXT-4): one lattice cut into row slabs, rank k owning slab k; its host logic --
which rows a rank owns, the exchange of the IPC handles and who is whose neighbour, the partition, the whole-job value
-- is checked here, the device side (IPC mapping, halo loads, phase protocol) by tests/test_gpu_parts.py."""
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
        heights = [130, 126]
        plan = bench.rank_plan(rank, world, "slabs", heights)
        got = {}

        class FakePart:                                        # the exchange of attach_neighbours over gloo, no GPU
            def part_export(self):
                return bytes([rank]) * 64

            def part_attach(self, up, rows_up, dn, rows_dn):
                got["attach"] = (up[0], rows_up, dn[0], rows_dn)

        bench.attach_neighbours(FakePart(), rank, world, heights, dist.all_gather_object)
        plan = (plan, got["attach"])
        sharded = bench.whole_job_updates_per_ns(world, 256, 10, 4, total_ms, "slabs")
        out.put((rank, total_ms, sweep_ms, value, bench.replica_seed(1, rank), plan, sharded))
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
    for rank, total_ms, sweep_ms, value, seed, plan, sharded in res:
        assert total_ms == 107.0 and sweep_ms == 90.0            # element-wise max, same on both ranks
        assert value == pytest.approx(2 * 256 * 256 * 10 * 4 / (107.0 * 1e6), rel=1e-15)
        assert seed == 1 + rank                                  # independent replicas
        # --parallel slabs: one lattice, the same seed on both ranks, rank k owns slab k; with two parts the other rank is
        # the neighbour above and below; the whole-job value counts one lattice's updates
        other = 1 - rank
        assert plan == ((0, ((0, 130) if rank == 0 else (130, 126))), (other, [130, 126][other], other, [130, 126][other]))
        assert sharded == pytest.approx(256 * 256 * 10 * 4 / (107.0 * 1e6), rel=1e-15)


def test_single_process_passthrough():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks([3.5, 2], None, None) == [3.5, 2.0]
    assert bench.whole_job_updates_per_ns(1, 1 << 18, 10, 10, 1000.0) == (1 << 36) * 100 / 1e9
    assert bench.rank_plan(0, 1, "slabs", None) == (0, None) and bench.rank_plan(3, 8, "replicas", None) == (3, None)


def test_slab_partition_for_every_rank_count():
    """The slab heights --parallel slabs hands to the GPUs at the paper's strong-scaling sizes (Table 3:
    L = 2^19 and 2^20 on 1..64 GPUs): equal, even, adding up to L (host arithmetic of the C ABI, no GPU)."""
    sys.path.insert(0, ROOT)
    from paper_2502_18624_b200 import build as b
    b.build()
    import paper_2502_18624_b200 as eng
    for L in (1 << 18, 1 << 19, 1 << 20):
        for n in (1, 2, 4, 8, 16, 32, 64):
            rows = eng.slab_partition(L, n)
            assert (rows == L // n).all()
