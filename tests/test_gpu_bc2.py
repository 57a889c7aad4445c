"""GPU parity (-m gpu) of NEXT-3: Blume-Capel stored at 2 bits per spin,
ISING_MODEL_BLUME_CAPEL_2BIT.  The trajectory contract is the 4-bit model's (same keying,
thresholds and rule), so the oracle is the Blume-Capel oracle (model 1) unchanged: lattices
and integer observables bit-exact, doubles to rel 1e-12."""
import numpy as np
import pytest

import oracle
import workloads as wl

pytestmark = pytest.mark.gpu

BC, BC2 = 1, 3


@pytest.fixture(scope="module")
def eng():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2502_18624_b200 as e
    e.load_library()
    return e


def _close(a, b):
    return a == b or abs(a - b) <= 1e-12 * max(abs(a), abs(b))


def _check_obs(L, D, obs, bmq):
    assert (obs.bond_sum, obs.M, obs.Q) == tuple(bmq)
    E, e, m, z = oracle.normalised(BC, L, D, bmq)
    assert _close(obs.E, E) and _close(obs.e_per_site, e) and _close(obs.m_per_site, m) and _close(obs.zero_density, z)


def _pack2(s, colour):
    """The documented 2-bit layout (include/ising.h) written out in numpy: colour array =
    L rows x L/64 uint64, site k of a row at bits 2 (k % 32) of word k // 32, code = spin + 1."""
    L = s.shape[0]
    out = np.zeros((L, L // 64), dtype=np.uint64)
    for y in range(L):
        par = (y + colour) & 1
        codes = (s[y, par::2].astype(np.int64) + 1).astype(np.uint64)
        for j in range(32):
            out[y] |= codes[j::32] << np.uint64(2 * j)
    return out.reshape(-1)


@pytest.mark.parametrize("L", [64, 192, 1024])
def test_init_and_packed_layout(eng, L):
    s = oracle.init(BC, L, 7)
    with eng.IsingSim(BC2, L, 1 / 1.4, 1.0, 7) as sim:
        assert (sim.read_lattice() == s).all()
        for c in range(2):
            assert (sim.read_packed(c) == _pack2(s, c)).all()
        assert eng.workspace_bytes(BC2, L) - eng.workspace_bytes(BC, L) == -(L * L // 4)


@pytest.mark.parametrize("L,beta,D,seed,n", [(128, 1 / 1.4, 1.0, 1, 50), (320, 0.9, 1.9, 5, 20), (64, 0.3, -1.0, 2, 30)])
def test_every_sweep(eng, L, beta, D, seed, n):
    s = oracle.init(BC, L, seed)
    with eng.IsingSim(BC2, L, beta, D, seed) as sim:
        for t in range(n):
            oracle.sweep(BC, s, beta, D, seed, t)
            sim.sweep(1)
            assert (sim.read_lattice() == s).all(), f"lattice differs after sweep {t + 1}"
            _check_obs(L, D, sim.observables(), oracle.observables(s))


@pytest.mark.parametrize("variant", [0, 1])
@pytest.mark.parametrize("beta,D", [(0.0, 1.0), (1 / 1.4, 1.0), (0.4, -1.5), (2.0, 1.966), (12.0, 0.5), (30.0, 3.0)])
def test_kernel_variants_and_threshold_edge_cases(eng, variant, beta, D):
    """Carry-table and compare/select kernels; beta = 0 (every threshold 2^32) and large beta
    (thresholds exactly 0: the carry form falls back) included."""
    L, seed, n = 192, 11, 6
    s = oracle.init(BC, L, seed)
    for t in range(n):
        oracle.sweep(BC, s, beta, D, seed, t)
    with eng.IsingSim(BC2, L, beta, D, seed) as sim:
        sim.set_variant(variant)
        sim.sweep(n)
        assert (sim.read_lattice() == s).all()
        _check_obs(L, D, sim.observables(), oracle.observables(s))


def test_several_tiles_ragged_tail_and_launch_geometry(eng):
    L, beta, D, seed, n = 1088, 1 / 1.4, 1.0, 3, 4          # 17 columns: blocks end mid-row, last chunk ragged
    s = oracle.init(BC, L, seed)
    for t in range(n):
        oracle.sweep(BC, s, beta, D, seed, t)
    for rows, block in [(None, None), (2, 64), (6, 256), (30, 128), (32, 96)]:
        with eng.IsingSim(BC2, L, beta, D, seed) as sim:
            if rows:
                sim.set_launch(rows, block)
            sim.sweep(n)
            assert (sim.read_lattice() == s).all(), (rows, block)


def test_same_trajectory_as_the_4_bit_model(eng):
    """Config 3 parameters at L = 4096: the 2-bit and the 4-bit kernels give the same lattice."""
    w = wl.config(3)
    L, n = 4096, 12
    with eng.IsingSim(BC, L, w.beta, w.D, w.seed) as a, eng.IsingSim(BC2, L, w.beta, w.D, w.seed) as b:
        a.sweep(n); b.sweep(n)
        oa, ob = a.observables(), b.observables()
        assert (oa.bond_sum, oa.M, oa.Q) == (ob.bond_sum, ob.M, ob.Q)
        assert (a.read_lattice(0, 64) == b.read_lattice(0, 64)).all()
        assert (a.read_lattice(L - 64, 64) == b.read_lattice(L - 64, 64)).all()
        # a light-cone window of the oracle, straddling the periodic corner
        x0, y0, wdt, hgt = L - 20, L - 12, 48, 40
        ref = oracle.window_after(BC, L, w.beta, w.D, w.seed, n, x0, y0, wdt, hgt)
        assert (b.read_window(x0, y0, wdt, hgt) == ref).all()


def test_write_read_roundtrip_and_resume(eng):
    L, beta, D, seed = 256, 0.8, 1.2, 9
    rng = np.random.default_rng(5)
    s = rng.integers(-1, 2, size=(L, L)).astype(np.int8)
    with eng.IsingSim(BC2, L, beta, D, seed) as sim:
        sim.write_lattice(s)
        assert (sim.read_lattice() == s).all()
        _check_obs(L, D, sim.observables(), oracle.observables(s))
        bad = s.copy(); bad[3, 5] = 2
        with pytest.raises(eng.IsingError):
            sim.write_lattice(bad)
        assert (sim.read_lattice() == s).all()                       # a rejected write leaves the lattice alone
        sim.set_sweeps_done(4)
        sim.sweep(3)
        for t in range(4, 7):
            oracle.sweep(BC, s, beta, D, seed, t)
        assert (sim.read_lattice() == s).all()
        packed = [sim.read_packed(c) for c in range(2)]
    with eng.IsingSim(BC2, L, beta, D, seed) as sim:               # resume from the packed checkpoint
        for c in range(2):
            sim.write_packed(c, packed[c])
        sim.set_sweeps_done(7)
        sim.sweep(2)
        for t in range(7, 9):
            oracle.sweep(BC, s, beta, D, seed, t)
        assert (sim.read_lattice() == s).all()


def test_fused_tally_graph_replay_and_schwinger_dyson(eng):
    L, beta, D, seed = 320, 1 / 1.4, 1.0, 4
    s = oracle.init(BC, L, seed)
    with eng.IsingSim(BC2, L, beta, D, seed) as sim:
        sim.set_tally(True)
        for t in range(8):
            oracle.sweep(BC, s, beta, D, seed, t)
            sim.sweep(1)
            ta = sim.tally()
            assert (ta.bond_sum, ta.M, ta.Q) == tuple(oracle.observables(s))
        sim.sweep(40)                                                 # n >= 32 at small L: CUDA-graph replay
        for t in range(8, 48):
            oracle.sweep(BC, s, beta, D, seed, t)
        assert (sim.read_lattice() == s).all()
        ta, ob = sim.tally(), sim.observables()
        assert (ta.bond_sum, ta.M, ta.Q) == (ob.bond_sum, ob.M, ob.Q) == tuple(oracle.observables(s))
        sd_o, hist_o = oracle.schwinger_dyson(s, beta)
        sd, hist = sim.schwinger_dyson()
        assert (np.asarray(hist) == np.asarray(hist_o)).all() and _close(sd, sd_o)


@pytest.mark.parametrize("L,path", [(192, 1), (512, 1), (512, 4), (768, 3), (512, 2)])
def test_correlation(eng, L, path):
    beta, D, seed = 1 / 1.4, 1.0, 6
    s = oracle.init(BC, L, seed)
    for t in range(3):
        oracle.sweep(BC, s, beta, D, seed, t)
    sx_o, sy_o = oracle.correlation(s, L // 2)
    with eng.IsingSim(BC2, L, beta, D, seed) as sim:
        sim.sweep(3)
        sim.set_corr_path(path)
        sx, sy = sim.correlation(L // 2)
        assert (sx == sx_o).all() and (sy == sy_o).all()
        rows = sim.correlation_protocol()
        ref = oracle.correlation_protocol(s, 3)
        assert all((np.asarray(a) == np.asarray(b)).all() for a, b in zip(rows, ref))
