"""GPU parity (-m gpu): the CUDA path, called through the C ABI binding, against
the CPU oracle on the same seeded inputs.  Integer results are compared
bit-exactly; doubles to rel 1e-12 (north_star)."""
import numpy as np
import pytest

import oracle
import workloads as wl

pytestmark = pytest.mark.gpu

ISING, BC = 0, 1


@pytest.fixture(scope="module")
def eng():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2502_18624_b200 as e
    e.load_library()           # must fail loudly if the extension is missing
    return e


def _close(a, b):
    return a == b or abs(a - b) <= 1e-12 * max(abs(a), abs(b))


def _check_obs(model, L, D, obs, bmq):
    assert (obs.bond_sum, obs.M, obs.Q) == tuple(bmq)
    E, e, m, z = oracle.normalised(model, L, D, bmq)
    assert _close(obs.E, E) and _close(obs.e_per_site, e) and _close(obs.m_per_site, m) and _close(obs.zero_density, z)
    assert obs.n_sites == L * L


# ------------------------------------------------------------------ Philox ---
def test_device_philox_matches_oracle_and_curand(eng):
    rng = np.random.default_rng(0)
    n = 4096
    ctr = rng.integers(0, 2**32, size=(n, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2**32, size=(n, 2), dtype=np.uint64).astype(np.uint32)
    ctr[:4] = [[0, 0, 0, 0], [0xFFFFFFFF] * 4, [0x243F6A88, 0x85A308D3, 0x13198A2E, 0x03707344], [5, 0, 7, 1]]
    key[:4] = [[0, 0], [0xFFFFFFFF] * 2, [0xA4093822, 0x299F31D0], [1, 0]]
    ours = eng.debug_philox(ctr, key, with_curand=False)      # even rows generic, odd rows specialised path
    lib = eng.debug_philox(ctr, key, with_curand=True)        # the toolkit's curand_Philox4x32_10
    assert (ours == lib).all()
    for i in list(range(8)) + list(range(100, 164)):
        assert (ours[i] == oracle.philox4x32_10(ctr[i], key[i])).all()
    assert [hex(int(v)) for v in ours[0]] == ["0x6627e8d5", "0xe169c58d", "0xbc57ac4c", "0x9b00dbd8"]


# -------------------------------------------------------------- thresholds ---
@pytest.mark.parametrize("i", range(5))
def test_threshold_tables_equal(eng, i):
    """north_star: both sides compute the table independently in double and assert equality."""
    w = wl.config(i)
    with eng.IsingSim(w.model, 64, w.beta, w.D, w.seed) as sim:
        assert (sim.thresholds() == oracle.thresholds(w.model, w.beta, w.D)).all()


@pytest.mark.parametrize("beta,D", [(0.0, 0.0), (0.3, -2.0), (1.7, 1.966), (25.0, 3.0), (0.5, 0.0)])
def test_threshold_tables_equal_other_parameters(eng, beta, D):
    for model in (ISING, BC):
        with eng.IsingSim(model, 64, beta, D, 3) as sim:
            assert (sim.thresholds() == oracle.thresholds(model, beta, D)).all()


# -------------------------------------------------------------------- init ---
@pytest.mark.parametrize("model", [ISING, BC])
@pytest.mark.parametrize("L", [64, 192, 256, 1024])
def test_init_lattice(eng, model, L):
    with eng.IsingSim(model, L, 0.4, 0.5, 7) as sim:
        assert (sim.read_lattice() == oracle.init(model, L, 7)).all()


# ------------------------------------------------------------- full parity ---
def test_config0_ising_L256_every_sweep(eng):
    """configs[0]: final lattice and E, M after every one of 100 sweeps."""
    w = wl.config(0)
    s = oracle.init(w.model, w.L, w.seed)
    tl = oracle.observables(s)
    with eng.IsingSim(w.model, w.L, w.beta, w.D, w.seed) as sim:
        _check_obs(w.model, w.L, w.D, sim.observables(), tl)
        for t in range(w.sweeps):
            sim.sweep(1)
            tl = oracle.sweep(w.model, s, w.beta, w.D, w.seed, t, tl)
            _check_obs(w.model, w.L, w.D, sim.observables(), tl)
            if t % 10 == 9:
                assert (sim.read_lattice() == s).all(), t
        assert (sim.read_lattice() == s).all()
        assert sim.observables().sweeps_done == w.sweeps


@pytest.mark.parametrize("L,beta,D,seed,n", [(128, 1 / 1.4, 1.0, 1, 50), (320, 0.9, 1.9, 5, 20), (64, 0.3, -1.0, 2, 30)])
def test_blume_capel_every_sweep(eng, L, beta, D, seed, n):
    s = oracle.init(BC, L, seed)
    tl = oracle.observables(s)
    with eng.IsingSim(BC, L, beta, D, seed) as sim:
        _check_obs(BC, L, D, sim.observables(), tl)
        for t in range(n):
            sim.sweep(1)
            tl = oracle.sweep(BC, s, beta, D, seed, t, tl)
            _check_obs(BC, L, D, sim.observables(), tl)
            assert (sim.read_lattice() == s).all(), t


@pytest.mark.parametrize("model,L,beta,D", [(ISING, 2048, wl.BETA_C / 0.9, 0.0), (BC, 1024, 1 / 1.4, 1.0),
                                            (ISING, 1088, 0.2, 0.0), (ISING, 64, wl.BETA_C, 0.0)])
def test_several_tiles_and_ragged_tail(eng, model, L, beta, D):
    """Sizes that span several blocks / row chunks, a non-power-of-two L whose last
    chunk is ragged, and the minimum L (one 128-bit vector per row)."""
    seed, n = 11, 6
    s = oracle.init(model, L, seed)
    tl = oracle.observables(s)
    with eng.IsingSim(model, L, beta, D, seed) as sim:
        sim.sweep(n)
        for t in range(n):
            tl = oracle.sweep(model, s, beta, D, seed, t, tl)
        assert (sim.read_lattice() == s).all()
        _check_obs(model, L, D, sim.observables(), tl)


@pytest.mark.parametrize("model", [ISING, BC])
def test_result_independent_of_launch_geometry(eng, model):
    """Analogue of PAPER.md:193 ('identical numerical results regardless of the number of GPUs')."""
    L, beta, D, seed, n = 512, 0.45, 0.7, 4, 5
    ref = None
    for rows, block in [(0, 0), (2, 32), (6, 96), (64, 256), (512, 64), (10, 128)]:
        with eng.IsingSim(model, L, beta, D, seed) as sim:
            sim.set_launch(rows, block)
            sim.sweep(n)
            lat = sim.read_lattice()
        if ref is None:
            ref = lat
            s = oracle.init(model, L, seed)
            for t in range(n):
                oracle.sweep(model, s, beta, D, seed, t)
            assert (ref == s).all()
        assert (lat == ref).all(), (rows, block)


def test_beta_zero_flips_everything(eng):
    """R21: beta = 0 -> every threshold is 2^32 -> every spin flips every half sweep."""
    L = 128
    with eng.IsingSim(ISING, L, 0.0, 0.0, 3) as sim:
        a = sim.read_lattice()
        sim.sweep(1)
        assert (sim.read_lattice() == -a).all()
        s = oracle.init(ISING, L, 3)
        oracle.sweep(ISING, s, 0.0, 0.0, 3, 0)
        assert (sim.read_lattice() == s).all()


def test_large_beta_never_accepts_uphill(eng):
    L, beta = 128, 40.0
    s = oracle.init(ISING, L, 8)
    with eng.IsingSim(ISING, L, beta, 0.0, 8) as sim:
        for t in range(4):
            sim.sweep(1)
            oracle.sweep(ISING, s, beta, 0.0, 8, t)
        assert (sim.read_lattice() == s).all()


@pytest.mark.parametrize("variant", [0, 1])
@pytest.mark.parametrize("beta", [0.0, 0.1, wl.BETA_C, wl.BETA_C / 0.5, 3.0, 5.5, 5.6, 40.0])
def test_ising_kernel_variants_and_threshold_edge_cases(eng, variant, beta):
    """Both implementations of the flip rule (carry chain = default, compare/select) against the
    oracle, over thresholds that are 2^32 (beta = 0), ordinary, T8 = 0 < T4 (beta = 3: e^-24 2^32 < 1),
    T4 = 1 (beta = 5.5) and both 0 (beta = 5.6, 40)."""
    L, seed, n = 256, 21, 8
    s = oracle.init(ISING, L, seed)
    tl = oracle.observables(s)
    with eng.IsingSim(ISING, L, beta, 0.0, seed) as sim:
        sim.set_variant(variant)
        assert (sim.thresholds() == oracle.thresholds(ISING, beta)).all()
        for t in range(n):
            sim.sweep(1)
            tl = oracle.sweep(ISING, s, beta, 0.0, seed, t, tl)
            assert (sim.read_lattice() == s).all(), (variant, beta, t)
        _check_obs(ISING, L, 0.0, sim.observables(), tl)


@pytest.mark.parametrize("variant", [0, 1])
@pytest.mark.parametrize("beta,D", [(0.0, 1.0), (1 / 1.4, 1.0), (0.4, -1.5), (2.0, 1.966), (12.0, 0.5), (30.0, 3.0)])
def test_blume_capel_kernel_variants_and_threshold_edge_cases(eng, variant, beta, D):
    """Carry-table kernel (default) and compare/select kernel against the oracle: all thresholds
    2^32 (beta = 0), ordinary tables, negative D, and tables holding exact zeros (beta = 12, 30:
    the default variant must fall back, see launch_update)."""
    L, seed, n = 192, 33, 6
    s = oracle.init(BC, L, seed)
    tl = oracle.observables(s)
    with eng.IsingSim(BC, L, beta, D, seed) as sim:
        sim.set_variant(variant)
        assert (sim.thresholds() == oracle.thresholds(BC, beta, D)).all()
        for t in range(n):
            sim.sweep(1)
            tl = oracle.sweep(BC, s, beta, D, seed, t, tl)
            assert (sim.read_lattice() == s).all(), (variant, beta, D, t)
        _check_obs(BC, L, D, sim.observables(), tl)


def test_resume_from_packed_checkpoint(eng):
    """state = (lattice, t): restoring both reproduces the trajectory exactly."""
    L, beta = 256, 0.5
    with eng.IsingSim(ISING, L, beta, 0.0, 5) as a, eng.IsingSim(ISING, L, beta, 0.0, 5) as b:
        a.sweep(7)
        blk, wht = a.read_packed(0), a.read_packed(1)
        a.sweep(5)
        b.write_packed(0, blk)
        b.write_packed(1, wht)
        b.set_sweeps_done(7)
        b.sweep(5)
        assert (a.read_lattice() == b.read_lattice()).all()
        assert blk.dtype == np.uint64 and len(blk) == L * L // 32
        assert ((blk & np.uint64(0xEEEEEEEEEEEEEEEE)) == 0).all()       # Ising nibbles are 0/1


# ----------------------------------------------------------- lattice IO ------
@pytest.mark.parametrize("model", [ISING, BC])
def test_write_read_roundtrip_and_closed_forms(eng, model):
    L = 128
    N = L * L
    rng = np.random.default_rng(1)
    vals = np.array([-1, 1] if model == ISING else [-1, 0, 1], dtype=np.int8)
    with eng.IsingSim(model, L, 0.4, 1.0, 1) as sim:
        a = rng.choice(vals, size=(L, L)).astype(np.int8)
        sim.write_lattice(a)
        assert (sim.read_lattice() == a).all()
        _check_obs(model, L, 1.0, sim.observables(), oracle.observables(a))
        assert (sim.read_window(L - 5, L - 3, 11, 9) == np.roll(a, (3, 5), axis=(0, 1))[:9, :11]).all()
        assert (sim.read_lattice(17, 3) == a[17:20]).all()
        b = a.copy()
        b[40:44] = rng.choice(vals, size=(4, L))
        sim.write_lattice(b[40:44], y0=40)
        assert (sim.read_lattice() == b).all()
        up = np.ones((L, L), np.int8)
        sim.write_lattice(up)
        o = sim.observables()
        assert (o.bond_sum, o.M, o.Q) == (2 * N, N, N)
        yy, xx = np.mgrid[0:L, 0:L]
        sim.write_lattice(np.where((xx + yy) % 2 == 0, 1, -1).astype(np.int8))
        o = sim.observables()
        assert (o.bond_sum, o.M, o.Q) == (-2 * N, 0, N)
        one = up.copy()
        one[3, 5] = -1
        sim.write_lattice(one)
        o = sim.observables()
        assert (o.bond_sum, o.M, o.Q) == (2 * N - 8, N - 2, N)
        if model == BC:
            sim.write_lattice(np.zeros((L, L), np.int8))
            o = sim.observables()
            assert (o.bond_sum, o.M, o.Q, o.zero_density) == (0, 0, 0, 1.0)
        bad = up.copy()
        bad[7, 9] = 2 if model == BC else 0
        with pytest.raises(eng.IsingError):
            sim.write_lattice(bad)
        assert (sim.read_lattice() == (np.zeros((L, L), np.int8) if model == BC else one)).all()


def test_argument_errors(eng):
    with pytest.raises(eng.IsingError):
        eng.IsingSim(ISING, 100, 0.4)              # L not a multiple of 64
    with pytest.raises(eng.IsingError):
        eng.IsingSim(2, 64, 0.4)                   # the 1-bit model needs L % 256 == 0
    with pytest.raises(eng.IsingError):
        eng.IsingSim(7, 256, 0.4)                  # unknown model
    with pytest.raises(eng.IsingError):
        eng.IsingSim(ISING, 64, -0.1)              # beta < 0
    with pytest.raises(eng.IsingError):
        eng.IsingSim(ISING, 64, float("nan"))
    with pytest.raises(eng.IsingError):
        eng.IsingSim(BC, 64, 0.5, float("inf"))
    with eng.IsingSim(ISING, 64, 0.4) as sim:
        for bad in (lambda: sim.sweep(-1), lambda: sim.correlation(0), lambda: sim.correlation(33),
                    lambda: sim.read_lattice(60, 8), lambda: sim.set_launch(3, 0), lambda: sim.set_launch(0, 100),
                    lambda: sim.correlation_list(3, [1]), lambda: sim.correlation_list(1, [40])):
            with pytest.raises(eng.IsingError):
                bad()
        sim.sweep(0)
        assert sim.observables().sweeps_done == 0
    import ctypes as C                                                # a host pointer is not a lattice buffer
    lib, n = eng.load_library(), eng.workspace_bytes(ISING, 64)
    host = np.zeros(n + 256, dtype=np.uint8)
    hp = (host.ctypes.data + 255) & ~255
    handle = C.c_void_p()
    assert lib.ising_create(ISING, 64, 0.4, 0.0, 1, hp, n, None, C.byref(handle)) == -1
    assert b"not device memory" in lib.ising_last_error()
    sim2 = eng.IsingSim(ISING, 64, 0.4, use_torch_memory=False)     # library-owned memory
    sim2.sweep(2)
    s = oracle.init(ISING, 64, 1)
    for t in range(2):
        oracle.sweep(ISING, s, 0.4, 0.0, 1, t)
    assert (sim2.read_lattice() == s).all()
    sim2.close()


# ------------------------------------------------------------- correlation ---
@pytest.mark.parametrize("model,L", [(ISING, 256), (BC, 256), (ISING, 64), (BC, 192), (ISING, 576)])
def test_correlation_full_range(eng, model, L):
    beta, D, seed = (wl.BETA_C / 0.5, 0.0, 1) if model == ISING else (1 / 1.4, 1.0, 1)
    with eng.IsingSim(model, L, beta, D, seed) as sim:
        sim.sweep(8)
        lat = sim.read_lattice()
        sx, sy = sim.correlation(L // 2)
        ox, oy = oracle.correlation(lat, L // 2)
        assert (sx == ox).all() and (sy == oy).all()
        o = sim.observables()
        assert sx[0] + sy[0] == o.bond_sum
        sx3, sy3 = sim.correlation(3)
        assert (sx3 == ox[:3]).all() and (sy3 == oy[:3]).all()


@pytest.mark.parametrize("model", [ISING, BC])
def test_correlation_list_and_protocol(eng, model):
    L = 1024
    beta, D = (wl.BETA_C / 0.5, 0.0) if model == ISING else (1 / 1.4, 1.0)
    with eng.IsingSim(model, L, beta, D, 2) as sim:
        sim.sweep(5)
        lat = sim.read_lattice()
        r = np.array([1, 2, 31, 32, 33, 100, 257, 511, 512])
        for stride in (1, 16, 4, 64):
            sx, sy = sim.correlation_list(stride, r)
            ox, oy = oracle.correlation_list(lat, stride, r)
            assert (sx == ox).all() and (sy == oy).all(), stride
        pr, px, py, pn = sim.correlation_protocol()
        orr, ox, oy, on = oracle.correlation_protocol(lat, 5)
        assert (pr == orr).all() and (pn == on).all() and (px == ox).all() and (py == oy).all()


@pytest.mark.parametrize("model,L", [(ISING, 512), (BC, 512), (ISING, 768), (BC, 1280), (ISING, 2048)])
def test_correlation_tensor_core_path(eng, model, L):
    """The int8 tcgen05 Gram kernel (path 2) against the oracle's plain sums and against the
    XOR + POPC kernels (path 1): full band, a band that ends inside a tile, a single distance;
    L = 768 and 1280 make the 256-row B tile wrap around the lattice edge."""
    beta, D = (wl.BETA_C / 0.5, 0.0) if model == ISING else (1 / 1.4, 1.0)
    with eng.IsingSim(model, L, beta, D, 5) as sim:
        sim.sweep(4)
        lat = sim.read_lattice()
        ox, oy = oracle.correlation(lat, L // 2)
        for rmax in (L // 2, L // 2 - 37, 129, 1):
            sim.set_corr_path(3)                             # CTA-pair kernel (cta_group::2), the automatic choice
            px, py = sim.correlation(rmax)
            assert (px == ox[:rmax]).all() and (py == oy[:rmax]).all(), rmax
            sim.set_corr_path(2)                             # single-CTA kernel
            tx, ty = sim.correlation(rmax)
            assert (tx == ox[:rmax]).all() and (ty == oy[:rmax]).all(), rmax
            sim.set_corr_path(4)                             # fp4 (kind::mxf4, unit block scales), CTA pairs
            fx, fy = sim.correlation(rmax)
            assert (fx == ox[:rmax]).all() and (fy == oy[:rmax]).all(), rmax
            sim.set_corr_path(1)
            bx, by = sim.correlation(rmax)
            assert (bx == tx).all() and (by == ty).all(), rmax
        sim.set_corr_path(0)
        ax, ay = sim.correlation(L // 2)                     # automatic choice
        assert (ax == ox).all() and (ay == oy).all()
        # closed form at the largest accumulator magnitude: all +1 -> every Gram entry is L, S(r) = N
        sim.write_lattice(np.ones((L, L), dtype=np.int8))
        for path in (2, 3, 4):
            sim.set_corr_path(path)
            tx, ty = sim.correlation(L // 2)
            assert (tx == L * L).all() and (ty == L * L).all(), path
    with eng.IsingSim(model, 192, beta, D, 5) as sim:        # L % 256 != 0: tensor path refuses, auto falls back
        sim.set_corr_path(2)
        with pytest.raises(eng.IsingError):
            sim.correlation(96)
        sim.set_corr_path(0)
        lat = sim.read_lattice()
        ax, ay = sim.correlation(96)
        ox, oy = oracle.correlation(lat, 96)
        assert (ax == ox).all() and (ay == oy).all()


@pytest.mark.parametrize("model", [ISING, BC])
@pytest.mark.parametrize("L", [64, 192, 320])
def test_correlation_list_small_and_ragged_comb(eng, model, L):
    """Every stride at sizes where the comb row is a fraction of a 64-bit word (L = 64, stride 64:
    one bit per row) or a ragged number of words (L = 192, 320)."""
    beta, D = (0.3, 0.0) if model == ISING else (0.5, 0.4)
    with eng.IsingSim(model, L, beta, D, 9) as sim:
        sim.sweep(3)
        lat = sim.read_lattice()
        r = np.array(sorted({1, 2, 3, L // 4, L // 2 - 1, L // 2}))
        for stride in (1, 2, 4, 8, 16, 32, 64):
            sx, sy = sim.correlation_list(stride, r)
            ox, oy = oracle.correlation_list(lat, stride, r)
            assert (sx == ox).all() and (sy == oy).all(), stride


def test_protocol_distance_lists_match_oracle(eng):
    """Host logic of Sec. 3.3 at sizes where the log grid is non-trivial (lists only)."""
    for L, t in [(4096, 1), (4096, 3000)]:
        with eng.IsingSim(ISING, L, 0.5, 0.0, 1) as sim:
            sim.set_sweeps_done(t)
            pr, px, py, pn = sim.correlation_protocol()
            orr, ost = oracle.protocol_list(L, t)
            assert (pr == orr).all()
            assert (pn == np.where(ost == 1, L * L, (L // 16) ** 2)).all()


@pytest.mark.parametrize("model,L,beta,D", [(ISING, 256, wl.BETA_C, 0.0), (ISING, 1088, wl.BETA_C / 0.5, 0.0), (BC, 320, 1 / 1.4, 1.0),
                                            (BC, 192, 12.0, 0.5), (wl.ISING_LUT, 512, wl.BETA_C / 0.9, 0.0)])
def test_fused_tally_equals_recompute_and_oracle(eng, model, L, beta, D):
    """A7 / north_star: the incremental tally kept by the update kernels equals a full recompute of
    B, M, Q after every sweep, and the oracle's own incremental tally."""
    seed = 17
    if model == wl.ISING_LUT:
        s = oracle.lut_init(L, seed)
        osweep = lambda t, tl: oracle.lut_sweep(s, beta, seed, t, tl)
    else:
        s = oracle.init(model, L, seed)
        osweep = lambda t, tl: oracle.sweep(model, s, beta, D, seed, t, tl)
    tl = oracle.observables(s)
    with eng.IsingSim(model, L, beta, D, seed) as sim:
        with pytest.raises(eng.IsingError):
            sim.tally()                                      # off by default
        sim.set_tally(True)
        a = sim.tally()
        assert (a.bond_sum, a.M, a.Q) == tl
        for t in range(6):
            sim.sweep(1)
            tl = osweep(t, tl)
            a, b = sim.tally(), sim.observables()
            assert (a.bond_sum, a.M, a.Q) == tl == (b.bond_sum, b.M, b.Q), t
            assert a.E == b.E and a.m_per_site == b.m_per_site and a.sweeps_done == t + 1
        assert (sim.read_lattice() == s).all()               # the tally kernels give the same trajectory
        ones = np.ones((L, L), dtype=np.int8)
        sim.write_lattice(ones)                              # a lattice write re-synchronises the tally
        a = sim.tally()
        assert (a.bond_sum, a.M) == (2 * L * L, L * L)
        sim.set_tally(False)
        sim.sweep(1)
        with pytest.raises(eng.IsingError):
            sim.tally()


@pytest.mark.parametrize("model,L,beta,D", [(ISING, 256, wl.BETA_C, 0.0), (BC, 192, 1 / 1.4, 1.0), (wl.ISING_LUT, 512, wl.BETA_C / 0.9, 0.0)])
def test_graph_replayed_sweeps_equal_plain_launches(eng, model, L, beta, D):
    """Small lattices replay the sweep loop from a CUDA graph (16 sweeps per replay, base sweep number in
    device memory): 75 sweeps in one call (4 replays + 11 plain sweeps) must equal the oracle's 75 sweeps and
    a sweep-by-sweep run; changing the launch geometry or the tally in between rebuilds the graph."""
    seed, n = 23, 75
    if model == wl.ISING_LUT:
        s = oracle.lut_init(L, seed)
        for t in range(n + 40):
            oracle.lut_sweep(s, beta, seed, t)
    else:
        s = oracle.init(model, L, seed)
        for t in range(n + 40):
            oracle.sweep(model, s, beta, D, seed, t)
    with eng.IsingSim(model, L, beta, D, seed) as sim:
        sim.sweep(n)                                         # graph path (the automatic mode)
        sim.set_launch(4, 64)
        sim.set_tally(True)
        sim.sweep(40)                                        # rebuilt graph (2 replays + 8 plain), tally kernels
        assert (sim.read_lattice() == s).all()
        a, b = sim.tally(), sim.observables()
        assert (a.bond_sum, a.M, a.Q) == (b.bond_sum, b.M, b.Q) == oracle.observables(s)
        assert b.sweeps_done == n + 40
    with eng.IsingSim(model, L, beta, D, seed) as sim:
        for _ in range(n + 40):
            sim.sweep(1)                                     # plain launches only
        assert (sim.read_lattice() == s).all()


@pytest.mark.parametrize("model,L,beta,D", [(ISING, 256, wl.BETA_C, 0.0), (ISING, 64, wl.BETA_C / 0.9, 0.0), (ISING, 1088, wl.BETA_C / 0.5, 0.0),
                                            (ISING, 2048, wl.BETA_C, 0.0), (BC, 192, 1 / 1.4, 1.0), (BC, 1024, 12.0, 0.5),
                                            (wl.BLUME_CAPEL_2BIT, 320, 1 / 1.4, 1.0)])
def test_persistent_sweep_kernel_equals_plain_launches_and_oracle(eng, model, L, beta, D):
    """Launch-bound lattices.  Sweep mode 4 (automatic for L <= 512): ONE cluster of 16 CTAs keeps the lattice in
    distributed shared memory for all n sweeps, colour phases separated by the hardware cluster barrier.  Sweep mode 3:
    ising_sweep(n) runs all n sweeps in ONE cooperative launch with a grid barrier per colour phase.  Lattice, fused tally and observables must equal those of one launch per colour phase (mode 2), of
    the CUDA graph (mode 1, the automatic choice) and of the oracle; mixing the modes in one trajectory changes nothing."""
    seed, n = 29, 37
    om = BC if model == wl.BLUME_CAPEL_2BIT else model
    s = oracle.init(om, L, seed)
    tl = oracle.observables(s)
    for t in range(n):
        tl = oracle.sweep(om, s, beta, D, seed, t, tl)
    lats = []
    for mode in (4, 3, 2, 1):                                    # 4: one cluster, lattice in distributed shared memory
        with eng.IsingSim(model, L, beta, D, seed) as sim:
            sim.set_sweep_mode(mode)
            sim.set_tally(True)
            k0 = sim.launch_count()
            sim.sweep(n)
            launches = sim.launch_count() - k0
            a, b = sim.tally(), sim.observables()
            assert (a.bond_sum, a.M, a.Q) == (b.bond_sum, b.M, b.Q) == tl and b.sweeps_done == n, mode
            lats.append(sim.read_lattice())
            if mode in (3, 4):
                assert launches == 1                                # one kernel for the 37 sweeps
                sim.sweep(1)                                        # n = 1: a plain pair of launches
                sim.set_sweep_mode(2)
                sim.sweep(2)
                sim.set_sweep_mode(mode)
                sim.sweep(5)
                s2 = s.copy()
                for t in range(n, n + 8):
                    oracle.sweep(om, s2, beta, D, seed, t)
                assert (sim.read_lattice() == s2).all()
    assert all((lat == s).all() for lat in lats)


def test_run_schedule_matches_stepwise_run(eng):
    """A11: one native call over the paper's time grid gives the same observables as sweeping step by step
    (and as the oracle), with and without the fused tally."""
    L, beta, seed = 256, wl.BETA_C / 0.5, 4
    times = eng.time_grid(40)
    assert (times == oracle.time_grid(40)).all()
    s = oracle.init(ISING, L, seed)
    tl = oracle.observables(s)
    want, t = [], 0
    for tt in times:
        while t < tt:
            tl = oracle.sweep(ISING, s, beta, 0.0, seed, t, tl)
            t += 1
        want.append(tl)
    for tally in (False, True):
        with eng.IsingSim(ISING, L, beta, 0.0, seed) as sim:
            sim.set_tally(tally)
            got = sim.run_schedule(times)
            assert [(o.bond_sum, o.M, o.Q) for o in got] == want
            assert [o.sweeps_done for o in got] == [int(x) for x in times]
            with pytest.raises(eng.IsingError):
                sim.run_schedule([3])                        # earlier than sweeps_done


def test_pipe_probe_rates_are_sane(eng):
    """ising_bench_pipes (measurement helper behind the ALU roofline): rates are positive, no pipe
    issues more than one warp-instruction per sub-partition per clock, the 16-lane pipes sit near
    0.5 and a wide multiply is slower than a 32-bit one."""
    r = eng.bench_pipes()
    assert set(r) == set(eng.PIPE_PROBES)
    assert all(0.05 < v < 1.1 for v in r.values()), r
    assert 0.35 < r["LOP3"] < 0.6 and 0.35 < r["IMAD"] < 0.6
    assert r["IMAD.WIDE"] < 0.8 * r["IMAD"]


# --------------------------------------------------------- Schwinger-Dyson ---
@pytest.mark.parametrize("model", [ISING, BC])
def test_schwinger_dyson_histogram(eng, model):
    L, beta, D = 256, 0.4, 0.8
    with eng.IsingSim(model, L, beta, D, 6) as sim:
        sim.sweep(12)
        v, hist = sim.schwinger_dyson()
        ov, ohist = oracle.schwinger_dyson(sim.read_lattice(), beta)
        assert (hist == ohist).all() and _close(v, ov)


# ------------------------------------------- memory safety without a sanitizer ---
@pytest.mark.parametrize("model,L", [(ISING, 320), (BC, 192), (wl.ISING_LUT, 512), (wl.BLUME_CAPEL_2BIT, 192), (ISING, 64)])
def test_no_write_outside_the_lattice_buffer(eng, model, L):
    """compute-sanitizer is closed on this pool (profiles/r02_sanitizer.md), so out-of-bounds WRITES are looked for
    with guard bands: the caller-owned buffer sits in the middle of a larger torch allocation filled with a canary
    pattern; after every kind of call (sweeps in several launch geometries incl. threads past the lattice, fused
    tally, observables, histogram, IO, bit planes and all correlation paths) the bands must be untouched and the
    results still equal the oracle's."""
    import ctypes as C
    import torch
    lib = eng.load_library()
    need = eng.workspace_bytes(model, L)
    guard = 1 << 20
    buf = torch.full((need + 2 * guard,), 0xA5, dtype=torch.uint8, device="cuda:0")
    handle = C.c_void_p()
    stream = torch.cuda.current_stream().cuda_stream
    beta, D, seed = (1 / 1.4, 1.0, 9) if model in (BC, wl.BLUME_CAPEL_2BIT) else (wl.BETA_C / 0.9, 0.0, 9)
    assert (buf.data_ptr() + guard) % 256 == 0
    assert lib.ising_create(model, L, beta, D, seed, buf.data_ptr() + guard, need, stream, C.byref(handle)) == 0
    sim = eng.IsingSim.__new__(eng.IsingSim)                     # wrap the raw handle in the binding's class
    sim._lib, sim._h, sim._buf, sim.model, sim.L = lib, handle, buf, model, L
    try:
        for rows, block in [(0, 0), (2, 32), (6, 96), (14, 256)]:
            sim.set_launch(rows, block)
            sim.sweep(2)
        sim.set_tally(True)
        sim.sweep(3)
        o, tly = sim.observables(), sim.tally()
        sim.schwinger_dyson()
        lat = sim.read_lattice()
        sim.write_lattice(lat)
        sim.read_window(L - 3, L - 5, 17, 9)
        for path in ((1,) if L % 256 else (1, 2, 3, 4)):
            sim.set_corr_path(path)
            sim.correlation(L // 2)
        sim.correlation_protocol()
        sim.sweep(40)                                            # CUDA-graph replay on small lattices
        sim.sync()
        assert bool((buf[:guard] == 0xA5).all()) and bool((buf[guard + need:] == 0xA5).all())
        n = 11
        if model == wl.ISING_LUT:
            s = oracle.lut_init(L, seed)
            for t in range(n):
                oracle.lut_sweep(s, beta, seed, t)
        else:
            om = BC if model == wl.BLUME_CAPEL_2BIT else model
            s = oracle.init(om, L, seed)
            for t in range(n):
                oracle.sweep(om, s, beta, D, seed, t)
        assert (lat == s).all() and (o.bond_sum, o.M, o.Q) == oracle.observables(s) == (tly.bond_sum, tly.M, tly.Q)
    finally:
        sim.close()


@pytest.mark.parametrize("model", [ISING, BC])
def test_tensor_core_correlation_is_deterministic(eng, model):
    """The tcgen05 kernels synchronise through mbarriers, TMA transaction counts, remote arrives and a cluster
    multicast commit; a race there would show as run-to-run differences.  40 repeats of each path on one lattice
    (L = 768: wrapping B tiles, ragged band) must give identical integers, equal to the oracle's."""
    L = 768
    beta, D = (wl.BETA_C / 0.5, 0.0) if model == ISING else (1 / 1.4, 1.0)
    with eng.IsingSim(model, L, beta, D, 5) as sim:
        sim.sweep(4)
        ox, oy = oracle.correlation(sim.read_lattice(), L // 2)
        for path in (2, 3, 4):
            sim.set_corr_path(path)
            for rep in range(40):
                sx, sy = sim.correlation(L // 2 - (rep % 3) * 37)
                n = len(sx)
                assert (sx == ox[:n]).all() and (sy == oy[:n]).all(), (path, rep)


# ------------------------------------------------------- compact transport format ---
def _numpy_bits(lat, model, colour):
    """The documented layout restated with numpy: colour row y holds the sites x = 2k + ((y + colour) & 1),
    k = 0..L/2-1; Ising: bit k & 63 of word k >> 6 is 1 for spin +1; Blume-Capel: bits 2 (k & 31) .. +1 of word
    k >> 5 hold spin + 1."""
    L = lat.shape[0]
    rows = []
    for y in range(L):
        v = lat[y, (y + colour) & 1::2].astype(np.int64)
        if model in (BC, wl.BLUME_CAPEL_2BIT):
            codes = (v + 1).astype(np.uint64).reshape(-1, 32)
            rows.append((codes << (2 * np.arange(32, dtype=np.uint64))).sum(axis=1, dtype=np.uint64))
        else:
            bits = (v > 0).astype(np.uint64).reshape(-1, 64)
            rows.append((bits << np.arange(64, dtype=np.uint64)).sum(axis=1, dtype=np.uint64))
    return np.concatenate(rows)


@pytest.mark.parametrize("model,L", [(ISING, 256), (BC, 192), (wl.ISING_LUT, 512), (wl.BLUME_CAPEL_2BIT, 192), (ISING, 128), (BC, 64)])
@pytest.mark.parametrize("slabs", [None, 3])
def test_bit_transport_format(eng, model, L, slabs):
    """ising_read_bits / ising_write_bits: the documented layout (numpy restatement), lossless round trip
    through another handle incl. row ranges, resume of the trajectory, rejection of the 2-bit code 3."""
    beta, D = (1 / 1.4, 1.0) if model in (BC, wl.BLUME_CAPEL_2BIT) else (wl.BETA_C / 0.9, 0.0)
    part = None if slabs is None else [2, L - 12, 10]
    with eng.IsingSim(model, L, beta, D, 5, slabs=part) as a, eng.IsingSim(model, L, beta, D, 5) as b:
        a.sweep(3)
        b.sweep(1)                                                      # some other lattice, overwritten below
        lat = a.read_lattice()
        assert not (b.read_lattice() == lat).all()
        rw = a.bits_row_words()
        for c in range(2):
            bits = a.read_bits(c)
            assert len(bits) == L * rw and (bits == _numpy_bits(lat, model, c)).all()
            assert (a.read_bits(c, 5, 9) == bits[5 * rw: 14 * rw]).all()
            b.write_bits(c, bits[: 7 * rw], 0, 7)                       # in two pieces
            b.write_bits(c, bits[7 * rw:], 7)
        assert (b.read_lattice() == lat).all()
        b.set_sweeps_done(3)
        a.sweep(4)
        b.sweep(4)
        assert (a.read_lattice() == b.read_lattice()).all()
        oa, ob = a.observables(), b.observables()
        assert (oa.bond_sum, oa.M, oa.Q) == (ob.bond_sum, ob.M, ob.Q)
        if model in (BC, wl.BLUME_CAPEL_2BIT):
            before = b.read_lattice()
            bad = b.read_bits(0)
            bad[len(bad) // 2] |= np.uint64(3 << 10)
            with pytest.raises(eng.IsingError):
                b.write_bits(0, bad)
            assert (b.read_lattice() == before).all()
        for fn in (lambda: a.read_bits(2), lambda: a.read_bits(0, L - 2, 5), lambda: a.write_bits(0, np.zeros(rw, np.uint64), L, 1)):
            with pytest.raises(eng.IsingError):
                fn()
    if model == ISING:                                                  # half a word per colour row: refused
        with eng.IsingSim(ISING, 192, beta) as c:
            with pytest.raises(eng.IsingError):
                c.read_bits(0, 0, 1)


@pytest.mark.parametrize("model", [ISING, BC, wl.ISING_LUT])
def test_run_protocol_schedule_matches_oracle(eng, model):
    """A11 with the correlation measurement in one native call: at every time of the schedule the
    rows (r, S_x, S_y, n_src) and B, M, Q equal the oracle's protocol and observables on the oracle's own trajectory."""
    L, seed = 1024, 6
    beta, D = (1 / 1.4, 1.0) if model == BC else (wl.BETA_C / 0.5, 0.0)
    times = [1, 2, 5, 9]
    if model == wl.ISING_LUT:
        s = oracle.lut_init(L, seed)
        step = lambda t: oracle.lut_sweep(s, beta, seed, t)
    else:
        s = oracle.init(model, L, seed)
        step = lambda t: oracle.sweep(model, s, beta, D, seed, t)
    with eng.IsingSim(model, L, beta, D, seed) as sim:
        rows, obs = sim.run_protocol_schedule(times)
        t = 0
        for k, tt in enumerate(times):
            while t < tt:
                step(t)
                t += 1
            orr, ox, oy, on = oracle.correlation_protocol(s, tt)
            r, sx, sy, ns = rows[k]
            assert (r == orr).all() and (sx == ox).all() and (sy == oy).all() and (ns == on).all(), tt
            assert (obs[k].bond_sum, obs[k].M, obs[k].Q) == oracle.observables(s) and obs[k].sweeps_done == tt
        with pytest.raises(eng.IsingError):
            sim.run_protocol_schedule([3])                       # earlier than sweeps_done
        lib, n = eng.load_library(), __import__("ctypes").c_int64(0)
        tm = np.array([20], dtype=np.uint64)
        buf = [np.zeros(8, dtype=np.int64) for _ in range(5)]
        assert lib.ising_run_protocol_schedule(sim._h, 1, tm.ctypes.data, 8, *(b.ctypes.data for b in buf), None) == -1   # cap too small
        assert sim.observables().sweeps_done == 9                # nothing was swept


@pytest.mark.parametrize("model,L,tally", [(ISING, 4096, False), (BC, 2048, True), (wl.BLUME_CAPEL_2BIT, 2048, False), (wl.ISING_LUT, 4096, False)])
def test_protocol_schedule_equals_one_call_per_time(eng, model, L, tally):
    """ising_run_protocol_schedule over many closely spaced times, a repeated time (no sweep in between), a second call
    with a longer list, with and without the observables, all four layouts -- every row equals what one sweep call + one
    ising_correlation_protocol call per time give on a twin handle, and the empty schedule is a no-op."""
    beta, D = (1 / 1.4, 1.0) if model in (BC, wl.BLUME_CAPEL_2BIT) else (wl.BETA_C / 0.5, 0.0)
    first, second = [1, 2, 2, 3, 5, 6, 40], [41, 43, 44, 44, 45, 47, 50, 51, 52, 90]
    with eng.IsingSim(model, L, beta, D, 8) as sim, eng.IsingSim(model, L, beta, D, 8) as twin:
        if tally:
            sim.set_tally(True)
        for times, with_obs in ((first, True), (second, False)):
            rows, obs = sim.run_protocol_schedule(times, with_observables=with_obs)
            assert len(rows) == len(times) and (obs is None) == (not with_obs)
            for k, t in enumerate(times):
                twin.sweep(t - twin.observables().sweeps_done)
                r, sx, sy, ns = twin.correlation_protocol()
                assert all((a == b).all() for a, b in zip(rows[k], (r, sx, sy, ns))), (t, k)
                assert len(rows[k][0]) == len(eng.protocol_distances(L, t)[0])
                if with_obs:
                    o = twin.observables()
                    assert (obs[k].bond_sum, obs[k].M, obs[k].Q, obs[k].sweeps_done) == (o.bond_sum, o.M, o.Q, t)
        assert (sim.read_lattice(0, 64) == twin.read_lattice(0, 64)).all()
        assert sim.run_protocol_schedule([]) == ([], [])


@pytest.mark.parametrize("variant", [0, 1])
@pytest.mark.parametrize("model,L,beta,D", [(ISING, 192, 0.0, 0.0), (ISING, 384, wl.BETA_C, 0.0), (ISING, 128, 3.0, 0.0), (ISING, 64, 40.0, 0.0),
                                            (BC, 128, 1 / 1.4, 1.0), (BC, 448, 0.0, 1.0), (BC, 192, 12.0, 0.5), (BC, 512, 1 / 1.4, 1.0)])
def test_cluster_kernel_half_granularity_variants_and_edge_thresholds(eng, variant, model, L, beta, D):
    """The cluster kernel below L = 512 gives every 32-bit half a thread (cluster_phase_halves; L = 512: a thread per
    vector): both flip-rule variants, thresholds that are 2^32 (beta = 0), exactly 0 (beta = 3, 12, 40: the carry forms fold
    or fall back) and ordinary, with the fused tally, sizes whose halves do not fill the block -- against the oracle."""
    seed, n = 31, 9
    s = oracle.init(model, L, seed)
    tl = oracle.observables(s)
    for t in range(n):
        tl = oracle.sweep(model, s, beta, D, seed, t, tl)
    with eng.IsingSim(model, L, beta, D, seed) as sim:
        sim.set_variant(variant)
        sim.set_tally(True)
        k0 = sim.launch_count()
        sim.sweep(n)                                             # automatic mode: one cluster launch
        assert sim.launch_count() - k0 == 1
        assert (sim.read_lattice() == s).all()
        a, b = sim.tally(), sim.observables()
        assert (a.bond_sum, a.M, a.Q) == (b.bond_sum, b.M, b.Q) == tl


@pytest.mark.parametrize("model,L,beta,D", [(ISING, 1024, wl.BETA_C / 0.5, 0.0), (BC, 576, 1 / 1.4, 1.0), (wl.ISING_LUT, 512, wl.BETA_C / 0.9, 0.0),
                                            (ISING, 4096, wl.BETA_C / 0.9, 0.0)])
def test_short_repeated_sweep_counts_replay_a_graph_of_their_own(eng, model, L, beta, D):
    """"E, M every 10 sweeps": the second call in a row with the same short count runs from a graph of exactly that many
    sweeps (one set-base kernel + 2n update kernels per call, the same launch count as plain launches + 1).  Changing the
    count, the launch geometry or the tally in between must rebuild it; the trajectory is the oracle's throughout."""
    seed = 19
    if model == wl.ISING_LUT:
        s = oracle.lut_init(L, seed)
        step = lambda t, tl: oracle.lut_sweep(s, beta, seed, t, tl)
    else:
        s = oracle.init(model, L, seed)
        step = lambda t, tl: oracle.sweep(model, s, beta, D, seed, t, tl)
    tl = oracle.observables(s)
    plan = [10, 10, 10, 7, 7, 10, 10, 5, 5, 5]                  # counts per call
    with eng.IsingSim(model, L, beta, D, seed) as sim:
        t = 0
        for i, n in enumerate(plan):
            if i == 5:
                sim.set_launch(4, 64)                            # another key: the graph of 10 is rebuilt
            if i == 7:
                sim.set_tally(True)
            k0 = sim.launch_count()
            sim.sweep(n)
            replayed = i > 0 and plan[i - 1] == n
            assert sim.launch_count() - k0 == 2 * n + (1 if replayed else 0), (i, n)
            for _ in range(n):
                tl = step(t, tl)
                t += 1
            o = sim.observables()
            assert (o.bond_sum, o.M, o.Q) == tl and o.sweeps_done == t, (i, n)
        a = sim.tally()
        assert (a.bond_sum, a.M, a.Q) == tl
        assert (sim.read_lattice() == s).all()
        times = list(range(t + 10, t + 60, 10))                  # the native schedule call: every 10 sweeps
        got = sim.run_schedule(times)
        for o in got:
            for _ in range(10):
                tl = step(t, tl)
                t += 1
            assert (o.bond_sum, o.M, o.Q) == tl
