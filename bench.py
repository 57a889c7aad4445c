#!/usr/bin/env python
"""bench.py -- spin updates/ns of the checkerboard Metropolis hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--config 0..4] [--L L] [--sweeps-per-step S] [--model ising|bc|lut|bc2]
                    [--slabs S] [--parallel replicas|slabs] [--tally] [--workload sweep|corr]

A "step" = S full sweeps (black + white update kernels)
followed by one observables pass (A8: E, M every S sweeps as in BASELINE.json
configs[1..3]).  Default workload = configs[2], the one the metric is quoted on:
Ising L = 2^18, T = 0.9 Tc, seed 1 (32 GiB packed, far larger than L2, so no L2
flush is needed between iterations).  Prints ONE JSON line (rank 0).

value     = L^2 * S * K / (device time of the K steps), lattice resident in HBM
e2e       = same through the C ABI with HOST buffers: every step uploads the lattice from
            pinned host memory in the compact transport format (ising_write_bits: 1 bit per
            Ising spin, 2 per Blume-Capel spin, expanded on the device), runs S sweeps and
            reads the observables back; two handles on two streams alternate so that the
            next step's upload overlaps this step's sweeps (serial figure beside it); the
            observables of every e2e step are asserted equal to a device-resident run's
roofline  = the update kernel against the bound that actually limits it: the integer
            ALU ("one Philox4x32-10 number per site" = 9.25 dispatch slots per site,
            DESIGN.md Sec. 5.1); peak derived from unit counts and the max SM clock, with
            the live pipe-probe rates and the Philox-only kernel's rate beside it
roofline_hbm = the same kernel against the measured HBM copy rate (MEASURED_PEAKS.json),
            algorithmic bytes 1.5 B per updated site (own nibble read + written, opposite
            nibble read once); `traffic` = dram bytes per launch from the committed ncu
            capture (profiles/update_kernel_dram.csv) when it was taken at this L
cpu_baseline = the oracle, as it stands, timed on the host cores on a bounded sample

N > 1 (torchrun): by default N independent replicas (seed + rank), weak scaling, no
collective on the data path (north_star: "one GPU, no sharding"); barrier + max-over-
ranks timing only.  --parallel slabs runs ONE lattice cut into N row slabs, rank k owning
slab k (NEXT-4, ising_create_part): halo rows by peer loads through CUDA
IPC, one NCCL all-reduce of a word between colour phases, strong scaling.  Unmeasured across
GPUs: this run's boxes have one (tests/test_gpu_parts.py runs the same protocol with 2 and
3 processes on one GPU; --slabs S cuts the lattice into S slabs inside one process).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as wl  # noqa: E402

BYTES_PER_SITE_LAUNCH = 1.5    # per UPDATED site: own nibble read + written, opposite nibble read once (3 x 4 bit)
PHILOX_SLOTS_PER_SITE = 9.25   # (18 IMAD.WIDE + 19 LOP3) / 4 sites, rounds 1-2 partly hoisted
# BASELINE.md Sec. 1 (the paper's single-GPU maxima, GB200, other machine: context): the 1-bit LUT Ising kernel
# at L = 2^20 and the 4-bit Blume-Capel kernel at L = 2^19.  No published number exists for the north_star
# contract (4-bit Ising, one number per spin), so the default workload reports vs_baseline = null.
MODEL_IDS = {"ising": wl.ISING, "bc": wl.BLUME_CAPEL, "lut": wl.ISING_LUT, "bc2": wl.BLUME_CAPEL_2BIT}
BITS_PER_SITE = {wl.ISING: 4, wl.BLUME_CAPEL: 4, wl.ISING_LUT: 1, wl.BLUME_CAPEL_2BIT: 2}
PAPER_UPDATES_PER_NS = {("lut", 1 << 20): 1802.0, ("bc", 1 << 19): 948.0}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--L", type=int, default=0, help="override the lattice size (default: configs[2], 2^18)")
    ap.add_argument("--config", type=int, default=-1, choices=[-1, 0, 1, 2, 3, 4],
                    help="time BASELINE.json configs[i] (model, L, beta, D, seed of that config); -1: --model / --workload decide")
    ap.add_argument("--model", default="ising", choices=["ising", "bc", "lut", "bc2"],
                    help="ising / bc: the north_star kernels (configs[2] / [3]); lut: NEXT-2, the paper's 1-bit look-up-table kernel on configs[2]'s parameters")
    ap.add_argument("--sweeps-per-step", type=int, default=10)
    ap.add_argument("--workload", default="sweep", choices=["sweep", "corr"],
                    help="sweep: S sweeps + observables (configs[2]/[3]); corr: configs[4], S sweeps + the paper's "
                         "correlation protocol (A10/A11) per step")
    ap.add_argument("--rows-per-thread", type=int, default=0, help="update-kernel launch geometry (0 = library default)")
    ap.add_argument("--block", type=int, default=0, help="update-kernel threads per block (0 = library default)")
    ap.add_argument("--variant", type=int, default=0, help="update-kernel variant (0 = default carry form)")
    ap.add_argument("--corr-path", type=int, default=0, help="ising_set_corr_path: 0 auto (fp4 tensor cores, path 4, for wide bands), 1 bit planes, 2 int8 tensor cores one CTA per tile, 3 int8 CTA pairs, 4 fp4 CTA pairs")
    ap.add_argument("--slabs", type=int, default=0, help="NEXT-4: cut the lattice into this many row slabs (allocations of their own, halo rows "
                                                          "read from the neighbours; all on this GPU unless --gpus-as-slabs)")
    ap.add_argument("--parallel", default="replicas", choices=["replicas", "slabs"],
                    help="N > 1: replicas = N independent lattices, one per rank (weak scaling; the default, north_star's "
                         "'no sharding'); slabs = ONE lattice cut into N row slabs, rank k owns slab k (ising_create_part), halo "
                         "rows read from the neighbouring ranks' memory through CUDA IPC, one NCCL all-reduce of a word between "
                         "colour phases (NEXT-4, PAPER.md:69-89; strong scaling at fixed L)")
    ap.add_argument("--sweep-mode", type=int, default=0, help="ising_set_sweep_mode for launch-bound lattices: 0 auto, 1 CUDA graph, 2 plain launches, 3 persistent cooperative kernel, 4 cluster kernel (lattice in DSMEM)")
    ap.add_argument("--tally", action="store_true", help="A7: keep E, M by the fused tally of the update kernels instead of the observables pass")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    return ap.parse_args()


def pick_workload(args):
    if getattr(args, "config", -1) >= 0:
        base = wl.config(args.config)
        args.model = "bc" if base.model == wl.BLUME_CAPEL else "ising"
        if args.config == 4:
            args.workload = "corr"
        return base, base.L, base.name
    base = wl.config(3) if args.model in ("bc", "bc2") else wl.config(2)
    if getattr(args, "workload", "sweep") == "corr":
        base = wl.config(4)
    L = args.L or base.L
    name = base.name if L == base.L else f"{base.name.split('_L')[0]}_L{L}_override"
    if args.model == "lut":          # NEXT-2: the paper's 1-bit kernel on config 2's temperature and seed
        name = f"ising_1bit_lut_L{L}_0.9Tc" + ("_paper_single_gpu_max" if L == (1 << 20) else "")
    if args.model == "bc" and L == (1 << 19):
        name = "bc_L524288_D1_paper_single_gpu_max"
    if args.model == "bc2":          # NEXT-3: the same Blume-Capel run stored at 2 bits per spin
        name = f"bc_2bit_L{L}_D1"
    return base, L, name


# ------------------------------------------------------------------ clocks ---
class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except ValueError:
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------- oracle on the host ---
def time_oracle(model: int, beta: float, D: float, seed: int, seconds: float, L: int = 4096):
    """The oracle as it stands (oracle/ising_oracle.c, OpenMP over rows) on a bounded
    sample of the workload: same model / beta / seed, lattice cut to L x L, as many
    full sweeps as fit in `seconds` (at least 2).  Returns (updates/ns, cores, text)."""
    import oracle
    if model == wl.BLUME_CAPEL_2BIT:                           # storage format only: the trajectory contract is model 1's
        model = wl.BLUME_CAPEL
    if model == wl.ISING_LUT:
        init = lambda: oracle.lut_init(L, seed)
        sweep = lambda s, t, tl: oracle.lut_sweep(s, beta, seed, t, tl)
    else:
        init = lambda: oracle.init(model, L, seed)
        sweep = lambda s, t, tl: oracle.sweep(model, s, beta, D, seed, t, tl)
    s = init()
    tl = oracle.observables(s)
    tl = sweep(s, 0, tl)                                       # untimed first touch
    n, t0 = 0, time.perf_counter()
    while True:
        tl = sweep(s, 1 + n, tl)
        n += 1
        dt = time.perf_counter() - t0
        if (dt >= seconds and n >= 2) or n >= 100000:
            break
    cores = oracle.threads()
    return L * L * n / (dt * 1e9), cores, f"{n} sweeps of the same model/beta/seed on an L={L} lattice ({dt:.1f} s)"


def run_reference(args):
    """--impl reference: this tier's reference arm is the oracle on the host cores."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    base, L, name = pick_workload(args)
    model = MODEL_IDS[args.model]
    per_step = max(1.0, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    vals, info, cores = [], "", 0
    for i in range(args.warmup + args.steps):
        v, cores, info = time_oracle(model, base.beta, base.D, base.seed, per_step)
        if i >= args.warmup:
            vals.append(v)
    value = sum(vals) / len(vals)
    line = {
        "impl": "reference", "metric": "spin updates/ns", "value": value, "unit": "updates/ns",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": per_step * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int8 spins, u32 Philox, f64 thresholds", "data": "synthetic (seeded random start)",
        "config": {"workload": name, "L": L, "sample": info},
        "cpu_baseline": {"value": value, "unit": "updates/ns", "cores": cores, "kind": "oracle", "sample": info},
        "e2e": {"value": value, "unit": "updates/ns", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------- the CUDA path ---
def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy rate)", d
    except (OSError, KeyError, ValueError):
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)", {}


def ncu_traffic(model: str, L: int):
    """dram__bytes_read.sum + dram__bytes_write.sum per update launch from the committed
    ncu --set full capture (a number measured under the profiler: reported, never timed)."""
    try:
        with open(os.path.join(ROOT, "profiles", "update_kernel_dram.csv")) as f:
            import csv
            rows = list(csv.reader(ln for ln in f if ln.strip() and not ln.startswith("#")))
        hdr = rows[0]
        vals = [float(r[hdr.index("dram_read_bytes")]) + float(r[hdr.index("dram_write_bytes")])
                for r in rows[1:] if r[hdr.index("model")] == model and int(r[hdr.index("L")]) == L]
        return sum(vals) / len(vals) if vals else None
    except (OSError, ValueError, IndexError):
        return None


def mem_available_bytes() -> int:
    try:
        with open("/proc/meminfo") as f:
            for line in f:
                if line.startswith("MemAvailable:"):
                    return int(line.split()[1]) * 1024
    except OSError:
        pass
    return 0


def run_e2e(eng, torch, model, L, beta, D, seed, S, steps, device):
    """End to end through the C ABI with HOST buffers: per step upload the lattice from pinned host memory in
    the compact transport format (ising_write_bits: 1 bit per Ising spin, 2 per Blume-Capel spin, expanded to
    the nibble layout on the device), run S sweeps, read the observables back."""
    row_words = L // 64 if model in (wl.BLUME_CAPEL, wl.BLUME_CAPEL_2BIT) else L // 128
    colour_bytes = L * row_words * 8
    need_dev = 2 * (L * L * BITS_PER_SITE[model] // 16)
    note = ""
    if mem_available_bytes() < 2 * colour_bytes + (8 << 30):
        while L > 4096 and mem_available_bytes() < 2 * (L * (L // 64) * 8) + (8 << 30):
            L //= 2
        row_words = L // 64 if model in (wl.BLUME_CAPEL, wl.BLUME_CAPEL_2BIT) else L // 128
        colour_bytes = L * row_words * 8
        need_dev = 2 * (L * L * BITS_PER_SITE[model] // 16)
        note = f"host memory too small for the full lattice; e2e measured at L={L}"
    words = colour_bytes // 8
    host = [torch.empty(words, dtype=torch.int64).pin_memory() for _ in range(2)]

    def enqueue(sim):                               # one step: the uploads block the host, the sweeps are asynchronous
        for c in range(2):
            sim.write_bits(c, host[c], 0, L)
        sim.set_sweeps_done(2)
        sim.sweep(S)

    # serial: upload, sweeps, observables, one after the other on one handle
    with eng.IsingSim(model, L, beta, D, seed, device=device) as sim:
        sim.sweep(2)
        for c in range(2):
            sim.read_bits(c, 0, L, out=host[c])
        times = []
        for i in range(3 + steps):                  # three untimed steps first, like the main timed region (one-time set-up:
            torch.cuda.synchronize(device)          # staging buffer, priority stream, the graph of S sweeps)
            t0 = time.perf_counter()
            enqueue(sim)
            o = sim.observables()                  # synchronises; D2H of B, M, Q
            torch.cuda.synchronize(device)
            if i >= 3:
                times.append(time.perf_counter() - t0)
        assert o.n_sites == L * L
        ref = (o.bond_sum, o.M, o.Q)
    with eng.IsingSim(model, L, beta, D, seed, device=device) as sim:   # the same S sweeps on a lattice that never left the device
        sim.sweep(2 + S)
        o = sim.observables()
        assert (o.bond_sum, o.M, o.Q) == ref, "the transport format is lossless: same observables as the resident run"
    dt = sum(times) / len(times)
    out = {"value": L * L * S / (dt * 1e9), "unit": "updates/ns", "h2d_bytes_per_step": 2 * colour_bytes,
           "d2h_bytes_per_step": 24, "L": L, "sweeps_per_step": S, "steps": steps, "ms_per_step": dt * 1e3,
           "what": "ising_write_bits(both colours, pinned host, compact transport format) + ising_sweep(S) + ising_observables"}
    # pipelined: the steps are independent inputs, so two handles on two streams alternate and the upload of
    # step i + 1 (copy engine) overlaps the sweeps of step i; fill and drain are inside the timed region
    free_b, _ = torch.cuda.mem_get_info(device)
    if free_b > 2 * need_dev + (8 << 30):
        streams = [torch.cuda.Stream(device=device) for _ in range(2)]
        sims = []
        for st in streams:
            with torch.cuda.stream(st):
                sims.append(eng.IsingSim(model, L, beta, D, seed, device=device))
        n_pipe = max(6 * steps, 18)                 # the fill (one upload that overlaps nothing) is inside the timed region
        for sim in sims:                            # warm-up: one step each
            enqueue(sim)
            sim.observables()
        torch.cuda.synchronize(device)
        t0 = time.perf_counter()
        pending = None
        for i in range(n_pipe):
            sim = sims[i % 2]
            enqueue(sim)
            if pending is not None:
                po = pending.observables()          # waits for step i - 1 while step i uploads
                assert (po.bond_sum, po.M, po.Q) == ref
            pending = sim
        po = pending.observables()
        torch.cuda.synchronize(device)
        dtp = (time.perf_counter() - t0) / n_pipe
        assert (po.bond_sum, po.M, po.Q) == ref
        for sim in sims:
            sim.close()
        out.update({"serial_value": out["value"], "serial_ms_per_step": out["ms_per_step"],
                    "value": L * L * S / (dtp * 1e9), "ms_per_step": dtp * 1e3, "steps": n_pipe,
                    "what": out["what"] + "; two handles on two streams, the upload of step i + 1 overlaps the sweeps "
                            "of step i (wall clock over all steps incl. pipeline fill and drain)"})
    if note:
        out["note"] = note
    return out


def max_over_ranks(values, dist, device):
    """Element-wise MAX over all ranks of a list of floats (device times in ms); the only
    cross-rank step of the replicas-only N > 1 run.  dist = None: single process."""
    if dist is None:
        return [float(v) for v in values]
    import torch
    t = torch.tensor([float(v) for v in values], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def whole_job_updates_per_ns(world: int, L: int, sweeps: int, steps: int, total_ms: float, parallel: str = "replicas") -> float:
    """replicas: N independent lattices of the same size, every rank does L^2 * sweeps * steps updates.
    slabs: one lattice shared by the N GPUs, L^2 * sweeps * steps updates in all."""
    lattices = world if parallel == "replicas" else 1
    return lattices * L * L * sweeps * steps / (total_ms * 1e6)


def rank_plan(rank: int, world: int, parallel: str, heights):
    """(seed offset, (y0, rows) or None) of one rank.  replicas: every rank its own unsharded lattice (seed + rank).
    slabs (N > 1): ONE lattice, the same seed everywhere; rank k owns the k-th slab of `heights` (ising_slab_partition)
    as a part handle (ising_create_part)."""
    if parallel == "slabs" and world > 1:
        return 0, (int(sum(heights[:rank])), int(heights[rank]))
    return rank, None


def attach_neighbours(sim, rank: int, world: int, heights, all_gather_object):
    """--parallel slabs: exchange the 64-byte CUDA IPC handles of the slab allocations (an all-gather through
    torch.distributed) and map the slab above and the slab below (periodic)."""
    handles = [None] * world
    all_gather_object(handles, sim.part_export())
    up, dn = (rank - 1) % world, (rank + 1) % world
    sim.part_attach(handles[up], int(heights[up]), handles[dn], int(heights[dn]))


def replica_seed(base_seed: int, rank: int) -> int:
    return base_seed + rank


def run_ours(args):
    import torch
    import paper_2502_18624_b200 as eng
    eng.load_library()                                     # raises if the CUDA library is missing
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device and no CPU fallback (use --impl reference for the oracle)")
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        if os.environ.get("ISING_BENCH_RANKS_ON_ONE_GPU") == "1":
            # test hook (tests/test_gpu_parts.py): a box with one GPU runs all ranks on cuda:0 over gloo, whose
            # collectives order the ranks on the host -- NCCL refuses two ranks on one GPU, and kernels of different
            # processes must not wait for one another there.  Not a measurement mode.
            local = 0
            dist.init_process_group("gloo")
        else:
            dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    device = torch.device(f"cuda:{local}")
    torch.cuda.set_device(device)

    base, L, name = pick_workload(args)
    model = MODEL_IDS[args.model]
    S, K, W = args.sweeps_per_step, args.steps, max(args.warmup, 0)
    sharded = args.parallel == "slabs" and world > 1
    heights = eng.slab_partition(L, world) if sharded else None
    seed_offset, part = rank_plan(rank, world, args.parallel, heights)
    n_slabs = args.slabs if (args.slabs > 1 and not sharded) else 0       # several slabs on this rank's own GPU
    sim = eng.IsingSim(model, L, base.beta, base.D, base.seed + seed_offset, device=device,
                       slabs=n_slabs if n_slabs > 1 else None, part=part)
    if sharded:
        attach_neighbours(sim, rank, world, heights, dist.all_gather_object)
        phase_flag = torch.zeros(1, dtype=torch.int32, device=device)
        sums = torch.zeros(3, dtype=torch.int64, device=device)
    if args.rows_per_thread or args.block:
        sim.set_launch(args.rows_per_thread, args.block)
    if args.variant:
        sim.set_variant(args.variant)
    if args.tally:
        sim.set_tally(True)
    if args.sweep_mode:
        sim.set_sweep_mode(args.sweep_mode)
    if args.corr_path:
        sim.set_corr_path(args.corr_path)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize(device)

    done = [0]

    def step(ev=None):
        if ev:
            ev[0].record()
        if sharded:
            # one lattice on N GPUs: a colour phase may start when the previous phase of both neighbours is done; the
            # NCCL all-reduce of one word is enqueued behind this rank's phase and ahead of its next one (stream-ordered,
            # no host synchronisation) and completes only when every rank has reached it
            for _ in range(S):
                for c in (0, 1):
                    sim.sweep_phase(c)
                    dist.all_reduce(phase_flag)
        else:
            sim.sweep(S)
        done[0] += S
        if ev:
            ev[1].record()
        if sharded:                                # the parts' integer sums, added up across the ranks in int64
            o = sim.tally() if args.tally else sim.observables()
            sums.copy_(torch.tensor([o.bond_sum, o.M, o.Q], dtype=torch.int64))
            dist.all_reduce(sums)
            b, m, q = (int(v) for v in sums)
            return eng.Observables(b, m, q, L * L, o.sweeps_done, float("nan"), float("nan"), m / float(L * L), float("nan"))
        if args.workload == "corr":                # A11: the protocol at this time, one native call (no sweeps left to do):
            _, obs = sim.run_protocol_schedule([done[0]])      # r <= 32 all sources + stride-16 sources up to L/2, and B, M, Q
            return obs[0]
        return sim.tally() if args.tally else sim.observables()

    for _ in range(W):
        step()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    e_start, e_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(local)
    launches0 = sim.launch_count()
    barrier()
    sampler.start()
    e_start.record()
    for k in range(K):
        obs = step(evs[k])
    e_end.record()
    barrier()
    clocks = sampler.stop()
    launches = sim.launch_count() - launches0
    total_ms = e_start.elapsed_time(e_end)
    sweep_ms = sum(a.elapsed_time(b) for a, b in evs)
    total_ms, sweep_ms = max_over_ranks([total_ms, sweep_ms], dist, device)

    # roofs, measured in the same process right after the timed region (rank 0 only matters)
    n_roof = 2 * S
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    lut = model == wl.ISING_LUT
    philox_ms = copy_ms = None
    if not lut and n_slabs <= 1 and not sharded:           # the roof helpers work on the 4-bit layout of an unsharded lattice
        sim.bench_philox_only(2); sim.bench_copy(2); torch.cuda.synchronize(device)
        ev[0].record(); sim.bench_philox_only(n_roof); ev[1].record(); sim.bench_copy(n_roof); ev[2].record()
        torch.cuda.synchronize(device)
        philox_ms = ev[0].elapsed_time(ev[1]) / n_roof
        copy_ms = ev[1].elapsed_time(ev[2]) / n_roof
    bytes_per_site = BYTES_PER_SITE_LAUNCH * BITS_PER_SITE[model] / 4   # 3 x (bits per site) per updated site
    slots_per_site = PHILOX_SLOTS_PER_SITE / 2 if lut else PHILOX_SLOTS_PER_SITE   # LUT: half a number per site
    tensor_roof = None
    if args.workload == "corr" and rank == 0:
        # full-range correlation (A9) on the tensor cores: whole ising_correlation(L/2) call, i.e.
        # bit planes + transposes + int8 expansion + the two Gram launches + the D2H of the sums
        sim.correlation(L // 2)
        ev2 = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        torch.cuda.synchronize(device)
        ev2[0].record(); sim.correlation(L // 2); ev2[1].record()
        torch.cuda.synchronize(device)
        full_ms = ev2[0].elapsed_time(ev2[1])
        fp4 = args.corr_path in (0, 4)
        tn = 224 if fp4 else 256                                # gram4_kernel: 256 x 224 tiles; gram2_kernel: 256 x 256
        n_jk = (L // 2 + 256 + tn - 1) // tn                    # columns I0 .. I0 + 255 + rmax
        macs = 2.0 * (L // 256) * n_jk * 256 * tn * L           # both axes, tiles actually multiplied
        ratio, nominal = (4.0, 9000.0) if fp4 else (2.0, 4500.0)   # guide: dense fp4 / int8 : bf16
        peak_t = ratio * float(measured_peaks()[2].get("bf16_tflops", 0.0)) or None
        tops = 2.0 * macs / (full_ms * 1e-3) / 1e12
        tensor_roof = {"bound": "tensor", "kernel": ("gram4_kernel (tcgen05 kind::mxf4, cta_group::2)" if fp4 else "gram2_kernel (tcgen05 kind::i8, cta_group::2)") + ", whole ising_correlation(L/2) call",
                       "achieved": tops, "peak": peak_t, "unit": "TOP/s (fp4)" if fp4 else "TOP/s (int8)",
                       "frac": (tops / peak_t) if peak_t else None, "frac_of_nominal": tops / nominal, "nominal_peak": nominal,
                       "traffic": None, "ms_per_call": full_ms,
                       "peak_source": f"{ratio:g} x MEASURED_PEAKS.json bf16_tflops (nominal ratio to bf16)",
                       "note": "frac > 1 is possible: the driver's bf16 figure is a power-limited cuBLAS run (SM clock about 1350 MHz "
                               "under load), this kernel multiplies -1/0/+1 and holds 1965 MHz; frac_of_nominal is against the datasheet rate",
                       "useful_pair_products": 2.0 * (L // 2) * L * L}
    sim.close()
    pipes = eng.bench_pipes(float(measured_peaks()[2].get("sm_max_mhz", 0.0))) if rank == 0 else {}

    sites_per_launch = L * L // 2
    kern_ms = sweep_ms / (2 * S * K)
    peak, peak_src, peaks = measured_peaks()
    achieved = bytes_per_site * sites_per_launch / (kern_ms * 1e-3) / 1e9
    traffic = ncu_traffic(args.model, L)
    # ALU roofline: one Philox4x32-10 call = 18 IMAD.WIDE + 19 LOP3 for 4 sites =
    # 9.25 dispatch slots per site; a slot is 2 clocks of a 16-lane pipe (0.5 warp-instructions per
    # sub-partition per clock, a wide multiply also taking one); 4 sub-partitions per SM.
    sm_ghz = float(peaks.get("sm_max_mhz", 1965.0)) / 1e3
    n_sm = torch.cuda.get_device_properties(device).multi_processor_count
    alu_peak = n_sm * 4 * sm_ghz * 32 * 0.5 / slots_per_site
    kern_upd = sites_per_launch / (kern_ms * 1e6)
    alu_roof = {"bound": "alu", "kernel": "update_kernel (one colour phase)", "achieved": kern_upd, "peak": alu_peak,
                "unit": "updates/ns", "frac": kern_upd / alu_peak, "traffic": traffic,
                "peak_source": f"derived: {n_sm} SMs x 4 sub-partitions x {sm_ghz} GHz x 32 lanes x 0.5 slots/clk / "
                               f"{slots_per_site} slots per site (Philox4x32-10 alone)",
                "avg_launch_ms": kern_ms,
                "philox_only_kernel_updates_per_ns": sites_per_launch / (philox_ms * 1e6) if philox_ms else None,
                "frac_of_philox_only_kernel": philox_ms / kern_ms if philox_ms else None,
                "pipe_rates_warp_instr_per_subpartition_clk": pipes}
    value = whole_job_updates_per_ns(world, L, S, K, total_ms, args.parallel)
    line = {
        "metric": "spin updates/ns", "value": value, "unit": "updates/ns", "n_gpus": world, "steps": K,
        "warmup": W, "ms_per_step": total_ms / K, "higher_is_better": True,
        "scaling": "strong" if (args.parallel == "slabs" and world > 1) else "weak",
        "vs_baseline": None,                      # BASELINE.json publishes no number for this metric on B200
        "vs_paper_gb200_context": (value / PAPER_UPDATES_PER_NS[(args.model, L)]) if (args.model, L) in PAPER_UPDATES_PER_NS and args.workload == "sweep" else None,
        "dtype": "u32 (Philox4x32-10, SWAR on 4-bit spins, integer compare)",
        "data": "synthetic (seeded random-start quench, the paper's own workload)",
        "config": {"workload": name, "hamiltonian": args.model, "L": L, "beta": base.beta, "D": base.D,
                   "seed": base.seed, "sweeps_per_step": S, "observables_every": S,
                   "step": "S sweeps + observables" if args.workload == "sweep" else "S sweeps + correlation protocol + observables",
                   "launch": {"rows_per_thread": args.rows_per_thread or "default", "block": args.block or "default",
                              "variant": args.variant, "fused_tally": bool(args.tally), "corr_path": args.corr_path, "sweep_mode": args.sweep_mode,
                              "slabs": world if sharded else max(1, n_slabs)},
                   "lattice_bytes": L * L * BITS_PER_SITE[model] // 8, "l2": "inputs larger than L2 (no flush needed)" if L * L // 2 > (256 << 20)
                   else "lattice fits L2: DRAM figures not meaningful",
                   "parallelism": f"slabs x{world} (one lattice, rank k owns slab k, halo rows by peer loads through CUDA IPC, one NCCL all-reduce of a word per colour phase)" if sharded else f"replicas x{world}"},
        "measurement_ms_per_step": (total_ms - sweep_ms) / K,
        "sweep_only_updates_per_ns": whole_job_updates_per_ns(world, L, S, K, sweep_ms, args.parallel),
        "roofline": alu_roof,
        "roofline_hbm": {"bound": "hbm", "kernel": "update_kernel (one colour phase)", "achieved": achieved,
                         "peak": peak, "unit": "GB/s", "frac": achieved / peak, "frac_of_nominal_8000_gbs": achieved / 8000.0,
                         "traffic": traffic,
                         "peak_source": peak_src, "algorithmic_bytes_per_launch": bytes_per_site * sites_per_launch,
                         "avg_launch_ms": kern_ms,
                         "copy_kernel_gbs": bytes_per_site * sites_per_launch / (copy_ms * 1e-3) / 1e9 if copy_ms else None},
        "roofline_tensor": tensor_roof,
        "clocks": clocks, "gpu_launches": launches,
        "last_observables": {"bond_sum": obs.bond_sum, "M": obs.M, "sweeps_done": obs.sweeps_done},
        "paper_context": "GB200: 1802 upd/ns (1-bit Ising, 1/2 RNG per spin), 948 upd/ns (Blume-Capel, 1 RNG per spin) -- other hardware/contract",
    }
    if rank == 0:
        if not args.no_e2e and not sharded:
            line["e2e"] = run_e2e(eng, torch, model, L, base.beta, base.D, base.seed, S, min(K, 3), device)
        if not args.no_cpu and world == 1:
            v, cores, info = time_oracle(model, base.beta, base.D, base.seed, args.cpu_seconds)
            import oracle
            oracle.set_threads(1)                                   # also on one core
            v1, _, info1 = time_oracle(model, base.beta, base.D, base.seed, min(4.0, args.cpu_seconds), L=1024)
            oracle.set_threads(cores)
            line["cpu_baseline"] = {"value": v, "unit": "updates/ns", "cores": cores, "kind": "oracle", "sample": info,
                                    "one_core": {"value": v1, "unit": "updates/ns", "cores": 1, "sample": info1}}
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
