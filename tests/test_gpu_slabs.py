"""NEXT-4 (-m gpu): the lattice cut into row slabs, each an allocation of its own whose kernels
read the two halo rows from the neighbouring slabs.  The contract is PAPER.md:193 -- "identical numerical
results ... regardless of the number of GPUs used": every result of a sharded handle must equal the
unsharded handle's and the oracle's bit for bit, for every model id and every partition.  This box has one
GPU, so all slabs live on device 0 (the same code path: streams per slab, events between neighbours)."""
import numpy as np
import pytest

import oracle
import workloads as wl

pytestmark = pytest.mark.gpu

ISING, BC, LUT, BC2 = wl.ISING, wl.BLUME_CAPEL, wl.ISING_LUT, wl.BLUME_CAPEL_2BIT


@pytest.fixture(scope="module")
def eng():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2502_18624_b200 as e
    e.load_library()
    return e


def _oracle_run(model, L, beta, D, seed, n):
    if model == LUT:
        s = oracle.lut_init(L, seed)
        tl = oracle.observables(s)
        for t in range(n):
            tl = oracle.lut_sweep(s, beta, seed, t, tl)
    else:
        om = BC if model == BC2 else model
        s = oracle.init(om, L, seed)
        tl = oracle.observables(s)
        for t in range(n):
            tl = oracle.sweep(om, s, beta, D, seed, t, tl)
    return s, tl


CASES = [(ISING, 256, wl.BETA_C, 0.0), (BC, 256, 1 / 1.4, 1.0), (LUT, 512, wl.BETA_C / 0.9, 0.0), (BC2, 256, 1 / 1.4, 1.0)]


@pytest.mark.parametrize("model,L,beta,D", CASES)
@pytest.mark.parametrize("slabs", [1, 2, 3, 8, "ragged"])
def test_sharded_lattice_equals_unsharded_and_oracle(eng, model, L, beta, D, slabs):
    """S in {1, 2, 3, 8} and a ragged partition whose heights are not multiples of the rows walked per thread:
    initial lattice, lattice after n sweeps, B, M, Q (full pass and fused tally), Schwinger-Dyson histogram,
    C(r) and the packed arrays equal the unsharded handle's; lattice and sums equal the oracle's."""
    seed, n = 13, 7
    part = [2, L // 2 - 6, 10, L // 2 - 6] if slabs == "ragged" else slabs
    s, tl = _oracle_run(model, L, beta, D, seed, n)
    with eng.IsingSim(model, L, beta, D, seed) as ref, eng.IsingSim(model, L, beta, D, seed, slabs=part) as sim:
        lay = sim.slab_layout()
        assert len(lay) == (4 if slabs == "ragged" else slabs) and lay[0][0] == 0 and sum(r for _, r, _ in lay) == L
        assert all(r % 2 == 0 and y % 2 == 0 for y, r, _ in lay)
        if slabs == "ragged":
            assert [r for _, r, _ in lay] == part
        assert (sim.read_lattice() == ref.read_lattice()).all()           # init is keyed by the global index
        sim.set_launch(4, 64)                                             # 4 rows per thread: 2- and 10-row slabs are ragged
        ref.set_launch(4, 64)
        sim.set_tally(True)
        sim.sweep(n)
        ref.sweep(n)
        lat = sim.read_lattice()
        assert (lat == ref.read_lattice()).all() and (lat == s).all()
        o, r_, tly = sim.observables(), ref.observables(), sim.tally()
        assert (o.bond_sum, o.M, o.Q) == (r_.bond_sum, r_.M, r_.Q) == tl == (tly.bond_sum, tly.M, tly.Q)
        assert o.E == r_.E and o.sweeps_done == n
        assert (sim.schwinger_dyson()[1] == ref.schwinger_dyson()[1]).all()
        assert (sim.schwinger_dyson()[1] == oracle.schwinger_dyson(s, beta)[1]).all()
        for a, b in zip(sim.correlation(L // 2), ref.correlation(L // 2)):
            assert (a == b).all()
        for c in range(2):
            assert (sim.read_packed(c) == ref.read_packed(c)).all()
        w = sim.read_window(L - 9, lay[1][0] - 3 if len(lay) > 1 else L - 3, 20, 11)     # a window across a slab seam
        assert (w == ref.read_window(L - 9, lay[1][0] - 3 if len(lay) > 1 else L - 3, 20, 11)).all()


@pytest.mark.parametrize("model,L,beta,D", CASES)
def test_sharded_io_and_resume(eng, model, L, beta, D):
    """write_lattice / write_packed across slab seams, checkpoint of a sharded handle resumed on an unsharded one."""
    seed = 3
    rng = np.random.default_rng(2)
    vals = np.array([-1, 0, 1] if model in (BC, BC2) else [-1, 1], dtype=np.int8)
    with eng.IsingSim(model, L, beta, D, seed, slabs=[6, L - 16, 10]) as sim, eng.IsingSim(model, L, beta, D, seed) as ref:
        a = rng.choice(vals, size=(L, L)).astype(np.int8)
        sim.write_lattice(a)
        assert (sim.read_lattice() == a).all()
        assert (sim.read_lattice(3, 9) == a[3:12]).all()                   # rows on both sides of the first seam
        b = rng.choice(vals, size=(8, L)).astype(np.int8)
        sim.write_lattice(b, y0=L - 14)                                    # rows across the second seam
        a[L - 14:L - 6] = b
        assert (sim.read_lattice() == a).all()
        o = sim.observables()
        assert (o.bond_sum, o.M, o.Q) == oracle.observables(a)
        sim.sweep(5)
        blk, wht = sim.read_packed(0), sim.read_packed(1)
        sim.sweep(4)
        ref.write_packed(0, blk)
        ref.write_packed(1, wht)
        ref.set_sweeps_done(5)
        ref.sweep(4)
        assert (sim.read_lattice() == ref.read_lattice()).all()
        nw = len(blk)
        part = sim.read_packed(1, nw // 3, nw // 2)                        # a word range that spans slabs
        assert (part == sim.read_packed(1)[nw // 3: nw // 3 + nw // 2]).all()
        sim.write_packed(0, blk[nw // 5: nw // 5 + nw // 2], word0=nw // 5)
        got = sim.read_packed(0)
        assert (got[nw // 5: nw // 5 + nw // 2] == blk[nw // 5: nw // 5 + nw // 2]).all()


def test_sharded_schedule_protocol_and_long_run(eng):
    """A longer sharded run through the native schedule calls: observables at every time equal the oracle's,
    the Sec. 3.3 protocol rows equal the unsharded handle's."""
    L, beta, seed = 512, wl.BETA_C / 0.5, 4
    times = [int(t) for t in eng.time_grid(40)]
    s = oracle.init(ISING, L, seed)
    tl = oracle.observables(s)
    want, t = [], 0
    for tt in times:
        while t < tt:
            tl = oracle.sweep(ISING, s, beta, 0.0, seed, t, tl)
            t += 1
        want.append(tl)
    with eng.IsingSim(ISING, L, beta, 0.0, seed, slabs=8) as sim, eng.IsingSim(ISING, L, beta, 0.0, seed) as ref:
        got = sim.run_schedule(times)
        assert [(o.bond_sum, o.M, o.Q) for o in got] == want
        ref.sweep(times[-1])
        rows, obs = sim.run_protocol_schedule([times[-1] + 3, times[-1] + 8])
        for k, tt in enumerate([times[-1] + 3, times[-1] + 8]):
            ref.sweep(tt - ref.observables().sweeps_done)
            for a, b in zip(rows[k], ref.correlation_protocol()):
                assert (a == b).all()
            o = ref.observables()
            assert (obs[k].bond_sum, obs[k].M) == (o.bond_sum, o.M)


def test_slab_argument_errors(eng):
    for bad in ([3, 253], [0, 256], [128, 126], [100, 100, 100]):
        with pytest.raises(eng.IsingError):
            eng.IsingSim(ISING, 256, 0.4, slabs=bad)
    with pytest.raises(eng.IsingError):
        eng.IsingSim(ISING, 64, 0.4, slabs=33)                             # fewer than two rows per slab
    with pytest.raises(eng.IsingError):
        eng.IsingSim(ISING, 256, 0.4, slabs=2, slab_devices=[0, 99])
    with eng.IsingSim(ISING, 256, 0.4, slabs=2) as sim:
        with pytest.raises(eng.IsingError):
            sim.bench_copy(1)                                              # measurement helpers: unsharded only
        sim.sweep(40)                                                      # no graph replay for sharded lattices
        s, _ = _oracle_run(ISING, 256, 0.4, 0.0, 1, 40)
        assert (sim.read_lattice() == s).all()


@pytest.mark.parametrize("model,L,beta,D,n", [(ISING, 1 << 16, wl.BETA_C / 0.5, 0.0, 20), (BC, 1 << 15, 1 / 1.4, 1.0, 12),
                                              (LUT, 1 << 16, wl.BETA_C / 0.9, 0.0, 12), (BC2, 1 << 15, 1 / 1.4, 1.0, 12)])
def test_light_cone_windows_across_slab_seams(eng, model, L, beta, D, n):
    """Large lattices in the launch configuration bench.py --slabs 8 times: 64 x 64 windows centred on slab seams
    (incl. the periodic seam between the last and the first slab) against the oracle's light-cone patches, and
    B, M, Q against the unsharded handle."""
    W = 64
    with eng.IsingSim(model, L, beta, D, 1, slabs=8) as sim:
        sim.sweep(n)
        lay = sim.slab_layout()
        for k, (x0, y0) in enumerate([(L // 3, lay[1][0] - W // 2), (L - W // 2, lay[5][0] - W // 2), (7, -W // 2), (L // 2, lay[7][0] - 2)]):
            if model == LUT:
                want = oracle.lut_window_after(L, beta, 1, n, x0, y0, W, W)
            else:
                want = oracle.window_after(BC if model == BC2 else model, L, beta, D, 1, n, x0, y0, W, W)
            assert (sim.read_window(x0, y0, W, W) == want).all(), (k, x0, y0)
        o = sim.observables()
    with eng.IsingSim(model, L, beta, D, 1) as ref:
        ref.sweep(n)
        r = ref.observables()
    assert (o.bond_sum, o.M, o.Q) == (r.bond_sum, r.M, r.Q)
