"""One process per GPU (-m gpu): every rank owns ONE slab of the lattice (ising_create_part), the ranks exchange
CUDA IPC handles of their slab allocations and read the two halo rows from the neighbours' memory.
This box has one GPU, so the ranks are separate PROCESSES on device 0 -- the IPC mapping, the halo pointers and the
phase-by-phase protocol are the ones a multi-GPU run uses; only the barrier differs (a host barrier after ising_sync
here, so that no kernel ever waits for another process; a stream-ordered NCCL all-reduce across GPUs, bench.py).
The contract is PAPER.md:193: the parts together are the unsharded lattice, bit for bit."""
import os
import socket
import sys

import numpy as np
import pytest

import oracle
import workloads as wl

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CASES = [(wl.ISING, 256, wl.BETA_C, 0.0), (wl.BLUME_CAPEL, 192, 1 / 1.4, 1.0), (wl.ISING_LUT, 512, wl.BETA_C / 0.9, 0.0),
         (wl.BLUME_CAPEL_2BIT, 192, 1 / 1.4, 1.0)]


@pytest.fixture(scope="module")
def eng():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2502_18624_b200 as e
    e.load_library()
    return e


def _oracle_run(model, L, beta, D, seed, n):
    if model == wl.ISING_LUT:
        s = oracle.lut_init(L, seed)
        tl = oracle.observables(s)
        for t in range(n):
            tl = oracle.lut_sweep(s, beta, seed, t, tl)
    else:
        om = wl.BLUME_CAPEL if model == wl.BLUME_CAPEL_2BIT else model
        s = oracle.init(om, L, seed)
        tl = oracle.observables(s)
        for t in range(n):
            tl = oracle.sweep(om, s, beta, D, seed, t, tl)
    return s, tl


@pytest.mark.parametrize("model,L,beta,D", CASES)
def test_single_part_is_the_whole_lattice(eng, model, L, beta, D):
    """rows == L: the part is its own neighbour; phase-by-phase sweeps and ising_sweep give the oracle's lattice."""
    s, tl = _oracle_run(model, L, beta, D, 3, 6)
    with eng.IsingSim(model, L, beta, D, 3, part=(0, L)) as sim:
        for _ in range(4):
            sim.sweep_phase(0)
            with pytest.raises(eng.IsingError):
                sim.sweep_phase(0)                                   # colour 0, then colour 1
            sim.sweep_phase(1)
        sim.sweep(2)
        assert (sim.read_lattice() == s).all()
        o = sim.observables()
        assert (o.bond_sum, o.M, o.Q) == tl and o.n_sites == L * L and o.sweeps_done == 6
    with eng.IsingSim(model, L, beta, D, 3, part=(L // 2, L // 2)) as half:    # a real part without neighbours
        for bad in (lambda: half.sweep_phase(0), lambda: half.observables(), lambda: half.sweep(1), lambda: half.correlation(4),
                    lambda: half.read_lattice(0, 4)):
            with pytest.raises(eng.IsingError):
                bad()
        assert (half.read_lattice(L // 2, L // 2) == (oracle.lut_init(L, 3) if model == wl.ISING_LUT else
                                                      oracle.init(wl.BLUME_CAPEL if model == wl.BLUME_CAPEL_2BIT else model, L, 3))[L // 2:]).all()
        assert len(half.part_export()) == 64
    for y0, rows in [(1, 64), (0, 63), (L - 62, 64), (0, 0)]:
        with pytest.raises(eng.IsingError):
            eng.IsingSim(model, L, beta, D, 3, part=(y0, rows))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, heights, n_sweeps, out):
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist
    import paper_2502_18624_b200 as eng
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    res = []
    try:
        for model, L, beta, D in CASES:
            if all(h == 0 for h in heights):
                rows = [L // world] * world                                                      # equal parts
            else:
                rows = [h if h > 0 else L - sum(x for x in heights if x > 0) for h in heights]  # one entry is "the rest"
            y0 = sum(rows[:rank])
            sim = eng.IsingSim(model, L, beta, D, 3, part=(y0, rows[rank]))
            handles = [None] * world
            dist.all_gather_object(handles, sim.part_export())                                 # 64 bytes per rank
            up, dn = (rank - 1) % world, (rank + 1) % world
            sim.part_attach(handles[up], rows[up], handles[dn], rows[dn])
            dist.barrier()
            for _ in range(n_sweeps):
                for c in (0, 1):
                    sim.sweep_phase(c)
                    sim.sync()                      # one GPU, several processes: order the phases on the host,
                    dist.barrier()                  # no kernel of one process ever waits for another process
            o = sim.observables()
            v, hist = sim.schwinger_dyson()
            sums = torch.tensor([o.bond_sum, o.M, o.Q, o.n_sites] + [int(x) for x in hist], dtype=torch.int64)
            dist.all_reduce(sums)                   # the int64 reduction of the partial sums
            res.append((model, y0, rows[rank], sim.read_lattice(y0, rows[rank]), [int(x) for x in sums], o.sweeps_done))
            dist.barrier()                          # nobody unmaps a slab a neighbour still reads
            sim.close()
        out.put((rank, res))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("heights", [(0, 0), (6, -1, 10)], ids=["two equal parts", "three ragged parts"])
def test_parts_in_separate_processes_equal_the_oracle(eng, heights):
    """2 and 3 processes, one part each, all four model ids: every part's rows, the summed B, M, Q and the summed
    Schwinger-Dyson histogram equal the oracle's full-lattice run."""
    import torch.multiprocessing as mp
    n = 5
    world = len(heights)
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, heights, n, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = dict(q.get(timeout=600) for _ in procs)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    for i, (model, L, beta, D) in enumerate(CASES):
        s, tl = _oracle_run(model, L, beta, D, 3, n)
        _, ohist = oracle.schwinger_dyson(s, beta)
        covered = 0
        for rank in range(world):
            m, y0, rows, lat, sums, t = got[rank][i]
            assert m == model and t == n and (lat == s[y0:y0 + rows]).all(), (model, rank)
            assert tuple(sums[:3]) == tl and sums[3] == L * L and sums[4:] == [int(x) for x in ohist], (model, rank)
            covered += rows
        assert covered == L


@pytest.mark.parametrize("parallel", ["slabs", "replicas"])
def test_bench_two_ranks_on_one_gpu(eng, parallel):
    """bench.py --gpus 2 under torchrun, both ranks on the one GPU of the box (test hook: gloo instead of NCCL).
    --parallel slabs: the sharded step -- part handles, IPC exchange, a collective between colour phases, int64
    reduction of the parts' sums -- must print one JSON line whose observables are the oracle's after
    (warmup + steps) * S sweeps, and count ONE lattice's updates.  --parallel replicas (the default): two independent
    lattices (seed + rank), rank 0's observables are the oracle's for the base seed, the value counts both."""
    import json
    import subprocess
    L, S, K, W = 2048, 3, 2, 1
    env = dict(os.environ, ISING_BENCH_RANKS_ON_ONE_GPU="1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"), "--gpus", "2", "--parallel", parallel, "--L", str(L),
           "--sweeps-per-step", str(S), "--steps", str(K), "--warmup", str(W), "--no-cpu", "--no-e2e"]
    r = subprocess.run(cmd, env=env, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-3000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1                                             # rank 0 alone prints
    d = json.loads(lines[0])
    sharded = parallel == "slabs"
    assert d["n_gpus"] == 2 and d["scaling"] == ("strong" if sharded else "weak")
    assert d["config"]["launch"]["slabs"] == (2 if sharded else 1)
    if sharded:
        assert d["gpu_launches"] == 2 * S * K + K
    cfg = wl.config(2)
    n = (W + K) * S
    s, tl = _oracle_run(cfg.model, L, cfg.beta, cfg.D, cfg.seed, n)
    assert (d["last_observables"]["bond_sum"], d["last_observables"]["M"], d["last_observables"]["sweeps_done"]) == (tl[0], tl[1], n)
    lattices = 1 if sharded else 2
    assert d["value"] == pytest.approx(lattices * L * L * S / (d["ms_per_step"] * 1e6), rel=1e-9)
