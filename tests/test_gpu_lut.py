"""GPU parity (-m gpu) of NEXT-2, the paper's one-bit look-up-table Ising kernel
(ISING_MODEL_ISING_LUT), against oracle section O7: table, initial lattice,
lattice after every sweep, B / M, Schwinger-Dyson histogram, correlation, lattice IO, and
light-cone windows at L = 2^16 and 2^18."""
import numpy as np
import pytest

import oracle
import workloads as wl

pytestmark = pytest.mark.gpu

LUT = wl.ISING_LUT
W = 64


@pytest.fixture(scope="module")
def eng():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2502_18624_b200 as e
    e.load_library()
    return e


@pytest.mark.parametrize("beta", [wl.BETA_C, wl.BETA_C / 0.5, wl.BETA_C / 0.9, 0.05, 2.5, 40.0])
def test_table_equals_oracle(eng, beta):
    with eng.IsingSim(LUT, 256, beta, 0.0, 1) as sim:
        assert (sim.thresholds() == oracle.lut_table(beta)).all()


def test_beta_outside_table_range_is_rejected(eng):
    for beta in (0.0, 1e-4):                                     # reading L7: a table entry above index 0 is 0
        with pytest.raises(eng.IsingError):
            eng.IsingSim(LUT, 256, beta, 0.0, 1)
    with pytest.raises(eng.IsingError):
        eng.IsingSim(LUT, 192, 0.4, 0.0, 1)                      # L must be a multiple of 256


@pytest.mark.parametrize("L,beta,seed,n", [(256, wl.BETA_C, 1, 12), (512, wl.BETA_C / 0.5, 7, 6), (768, 0.3, 3, 4),
                                           (1024, wl.BETA_C / 0.9, 11, 4), (256, 2.5, 2, 4), (256, 0.01, 2, 3)])
def test_lattice_and_observables_every_sweep(eng, L, beta, seed, n):
    s = oracle.lut_init(L, seed)
    tl = oracle.observables(s)
    with eng.IsingSim(LUT, L, beta, 0.0, seed) as sim:
        sim.set_variant(2)                                   # the bucket-table kernel (automatic from L = 6144)
        assert (sim.read_lattice() == s).all()
        for t in range(n):
            sim.sweep(1)
            tl = oracle.lut_sweep(s, beta, seed, t, tl)
            assert (sim.read_lattice() == s).all(), t
            o = sim.observables()
            assert (o.bond_sum, o.M, o.Q) == tl and o.E == -float(tl[0]) and o.sweeps_done == t + 1
        v, hist = sim.schwinger_dyson()
        ov, ohist = oracle.schwinger_dyson(s, beta)
        assert (hist == ohist).all() and abs(v - ov) <= 1e-12 * abs(ov)
        sx, sy = sim.correlation(L // 2)
        ox, oy = oracle.correlation(s, L // 2)
        assert (sx == ox).all() and (sy == oy).all()
        r = np.array([1, 5, 33, L // 2])
        lx, ly = sim.correlation_list(16, r)
        olx, oly = oracle.correlation_list(s, 16, r)
        assert (lx == olx).all() and (ly == oly).all()


@pytest.mark.parametrize("beta", [wl.BETA_C / 0.9, wl.BETA_C / 0.5, 1.2, 2.5, 0.01])
def test_bucket_table_and_binary_search_variants_agree(eng, beta):
    """Variant 2 (bucket table + rare binary-search fallback; low temperatures have buckets with several
    thresholds), variant 1 (binary search only) and the automatic choice against the oracle."""
    L, seed, n = 512, 13, 5
    s = oracle.lut_init(L, seed)
    for t in range(n):
        oracle.lut_sweep(s, beta, seed, t)
    for variant in (2, 1, 0):
        with eng.IsingSim(LUT, L, beta, 0.0, seed) as sim:
            sim.set_variant(variant)
            sim.sweep(n)
            assert (sim.read_lattice() == s).all(), variant


def test_launch_geometry_and_io_roundtrip(eng):
    L, beta, seed = 512, wl.BETA_C / 0.9, 5
    ref = None
    for rows, block in [(0, 0), (2, 32), (6, 96), (64, 256)]:
        with eng.IsingSim(LUT, L, beta, 0.0, seed) as sim:
            sim.set_launch(rows, block)
            sim.sweep(5)
            lat = sim.read_lattice()
        ref = lat if ref is None else ref
        assert (lat == ref).all(), (rows, block)
    with eng.IsingSim(LUT, L, beta, 0.0, seed) as sim:
        rng = np.random.default_rng(0)
        a = (2 * rng.integers(0, 2, size=(L, L)) - 1).astype(np.int8)
        sim.write_lattice(a)
        assert (sim.read_lattice() == a).all()
        assert (sim.read_window(-5, L - 3, 40, 17) == np.roll(a, (3, 5), axis=(0, 1))[:17, :40]).all()
        o = sim.observables()
        assert (o.bond_sum, o.M, o.Q) == oracle.observables(a)
        sim.set_sweeps_done(3)
        sim.sweep(2)
        s = a.copy()
        for t in (3, 4):
            oracle.lut_sweep(s, beta, seed, t)
        assert (sim.read_lattice() == s).all()
        bad = a.copy(); bad[7, 9] = 0
        with pytest.raises(eng.IsingError):
            sim.write_lattice(bad)
        sim.write_lattice(np.ones((L, L), np.int8))              # closed forms: all +1
        o = sim.observables()
        assert (o.bond_sum, o.M) == (2 * L * L, L * L)


@pytest.mark.parametrize("L,n", [(1 << 16, 20), (1 << 18, 10)])
def test_light_cone_windows_large(eng, L, n):
    """Large lattices (2^18: 8.6 GB at one bit per spin): windows on the wraps, the corner and across
    thread-column (256 sites) and row-chunk boundaries; M by popcount of the packed arrays; B = S(1)."""
    beta, seed = wl.BETA_C / 0.9, 1
    with eng.IsingSim(LUT, L, beta, 0.0, seed) as sim:
        sim.sweep(n)
        for (x0, y0) in [(-W // 2, -W // 2), (L - W // 2, L // 3 + 5), (L // 5 + 3, L - W // 2),
                         (256 * (L // 768) - W // 2, 32 * (L // 96) - W // 2), (L // 2 + 7, L // 2 - 13)]:
            want = oracle.lut_window_after(L, beta, seed, n, x0, y0, W, W)
            assert (sim.read_window(x0, y0, W, W) == want).all(), (x0, y0)
        o = sim.observables()
        words = L * L // 128
        up = 0
        for c in range(2):
            for w0 in range(0, words, 1 << 26):
                up += int(np.bitwise_count(sim.read_packed(c, w0, min(1 << 26, words - w0))).sum(dtype=np.int64))
        assert o.M == 2 * up - L * L and o.Q == L * L
        sx, sy = sim.correlation_list(1, [1])
        assert int(sx[0]) + int(sy[0]) == o.bond_sum
