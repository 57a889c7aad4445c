"""GPU parity at BASELINE.json's full sizes (-m gpu), in the launch configuration
bench.py times (default rows-per-thread / block size, default kernel variant).

The oracle cannot hold a 69 GB lattice nor do 1.4e13 updates, so:
  * light-cone windows: the w x h window after n sweeps depends only on the initial
    spins within 2n sites of it; oracle.window_after simulates that patch with global
    coordinates mod L and its centre must equal ising_read_window byte for byte.
    Windows sit on the x wrap, the y wrap, the corner, across thread-column (64 sites),
    row-chunk (32 rows) and block boundaries;
  * integer observables: the oracle's O5 / Schwinger-Dyson routines applied to the GPU lattice
    streamed out in row bands (oracle.observables_rows / sd_hist_rows, pinned by "the bands
    add up to the full-lattice routine"), plain definitions evaluated with numpy on the packed
    lattice (M = 2 popcount - N), the oracle's O5/O6 routines on the whole lattice read back
    where it fits the host, and identities that hold at any size (S_x(1) + S_y(1) = B).
Every config runs to the length BASELINE.json states (200 / 1000 / 500 / 2000 sweeps).
"""
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

import oracle
import workloads as wl

pytestmark = pytest.mark.gpu

ISING, BC = 0, 1
W = 64   # window edge


@pytest.fixture(scope="module")
def eng():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2502_18624_b200 as e
    e.load_library()
    return e


def window_origins(L):
    """(x0, y0) of W x W windows: corner wrap, x wrap, y wrap, thread-column boundary
    (x multiple of 64), row-chunk boundary (y multiple of 32), block boundary, interior."""
    return [(-W // 2, -W // 2), (L - W // 2, L // 3 + 5), (L // 5 + 3, L - W // 2),
            (64 * (L // 192) - W // 2, 32 * (L // 96) - W // 2), (L // 2 + 7, L // 2 - 13),
            (128 * 64 % L - 20, 7 * 32 - 40)]


def check_windows(sim, cfg, n, origins):
    got = [sim.read_window(x0, y0, W, W) for (x0, y0) in origins]
    with ThreadPoolExecutor(max_workers=len(origins)) as pool:       # the oracle patches are independent (ctypes drops the GIL)
        want = list(pool.map(lambda o: oracle.window_after(cfg.model, cfg.L, cfg.beta, cfg.D, cfg.seed, n, o[0], o[1], W, W), origins))
    for (x0, y0), g, w in zip(origins, got, want):
        assert (g == w).all(), (cfg.name, n, x0, y0, int((g != w).sum()))


def streamed_oracle_sums(sim, L, band_rows, with_hist=True):
    """The oracle's O5 routine (and the Schwinger-Dyson histogram) applied to the GPU lattice streamed out
    in row bands: band = rows y0 - 1 .. y0 + ny (one halo row on each side, wrapping), read through
    ising_read_window.  Returns ((B, M, Q), hist)."""
    tot, hist = np.zeros(3, dtype=np.int64), np.zeros(9, dtype=np.int64)
    for y0 in range(0, L, band_rows):
        ny = min(band_rows, L - y0)
        band = sim.read_window(0, y0 - 1, L, ny + 2)
        tot += np.array(oracle.observables_rows(L, band[1:]))
        if with_hist:
            hist += oracle.sd_hist_rows(L, band)
        del band
    return tuple(int(v) for v in tot), hist


def packed_sums(sim, model, L, chunk_words=1 << 26):
    """M and Q from the packed colour arrays by the plain definition (numpy popcount):
    Ising nibble 1 = +1, 0 = -1; Blume-Capel nibble = s + 1."""
    words = L * L // 32
    M = Q = 0
    for c in range(2):
        for w0 in range(0, words, chunk_words):
            nw = min(chunk_words, words - w0)
            a = sim.read_packed(c, w0, nw).view(np.uint64)
            if model == ISING:
                up = int(np.bitwise_count(a).sum(dtype=np.int64))
                M += 2 * up - 16 * nw
                Q += 16 * nw
            else:
                two = int(np.bitwise_count(a & np.uint64(0x2222222222222222)).sum(dtype=np.int64))   # s = +1
                one = int(np.bitwise_count(a & np.uint64(0x1111111111111111)).sum(dtype=np.int64))   # s = 0
                zero = 16 * nw - two - one                                                            # s = -1
                M += two - zero
                Q += two + zero
    return M, Q


# ---------------------------------------------------------------- configs[2] ---
def test_config2_ising_L2p18_windows_and_observables(eng):
    """Headline workload: Ising L = 2^18, T = 0.9 Tc, seed 1, 200 sweeps (34 GB packed)."""
    cfg = wl.config(2)
    L = cfg.L
    with eng.IsingSim(cfg.model, L, cfg.beta, cfg.D, cfg.seed) as sim:
        assert (sim.thresholds() == oracle.thresholds(cfg.model, cfg.beta)).all()
        check_windows(sim, cfg, 0, window_origins(L)[:3])          # the init kernel at full size
        done = 0
        for n, origins in [(10, window_origins(L)), (50, window_origins(L)), (200, window_origins(L)[:2])]:
            sim.sweep(n - done)
            done = n
            check_windows(sim, cfg, n, origins)
        o = sim.observables()
        assert o.sweeps_done == 200 and o.n_sites == L * L and o.Q == L * L
        M, _ = packed_sums(sim, cfg.model, L)
        assert o.M == M
        # B, M, Q and the Schwinger-Dyson histogram anchored to the ORACLE at the headline size (the only size
        # where byte offsets inside a colour array pass 2^32): 69 GB of int8 streamed back in 64 bands
        bmq, hist = streamed_oracle_sums(sim, L, 4096)
        assert (o.bond_sum, o.M, o.Q) == bmq
        v, ghist = sim.schwinger_dyson()
        assert (ghist == hist).all() and int(hist.sum()) == L * L
        want_v = sum(float(hist[k + 4]) * np.exp(-2.0 * cfg.beta * k) for k in range(-4, 5)) / float(L * L)
        assert abs(v - want_v) <= 1e-12 * abs(want_v)
        sx, sy = sim.correlation_list(1, [1, 2])                   # independent kernels (bit planes)
        assert int(sx[0]) + int(sy[0]) == o.bond_sum               # S_x(1) + S_y(1) = B
        sim.set_corr_path(4)                                       # tensor cores at L = 2^18 (34 GB e2m1 matrix)
        tx, ty = sim.correlation(1024)
        sim.set_corr_path(3)                                       # int8 CTA pairs (69 GB int8 matrix)
        ix, iy = sim.correlation(1024)
        assert (tx == ix).all() and (ty == iy).all()
        sim.set_corr_path(1)                                       # XOR + POPC kernels
        bx, by = sim.correlation(1024)
        assert (tx == bx).all() and (ty == by).all()
        assert int(tx[0]) + int(ty[0]) == o.bond_sum and (int(tx[1]), int(ty[1])) == (int(sx[1]), int(sy[1]))
        assert o.E == -float(o.bond_sum) and o.e_per_site == o.E / float(L * L)
        assert o.m_per_site == float(o.M) / float(L * L)


# ---------------------------------------------------------------- configs[1] ---
def test_config1_ising_L2p14_1000_sweeps(eng):
    """Ising L = 2^14, T = 0.5 Tc, 1000 sweeps, E and M every 10 sweeps (BASELINE.json configs[1]).
    The oracle runs the first 100 sweeps on the full lattice (B, M every 10, lattice at 20 and 100); from there to
    1000 every measurement of ising_run_schedule is compared with the oracle's O5 routine on the lattice read back
    (B, M, Q -- the kernels that produced the trajectory are anchored by the light-cone windows at 200 and 500)."""
    cfg = wl.config(1)
    L = cfg.L
    s = oracle.init(cfg.model, L, cfg.seed)
    tl = oracle.observables(s)
    with eng.IsingSim(cfg.model, L, cfg.beta, cfg.D, cfg.seed) as sim:
        assert (sim.read_lattice() == s).all()
        for k in range(10):
            for t in range(10 * k, 10 * k + 10):
                tl = oracle.sweep(cfg.model, s, cfg.beta, cfg.D, cfg.seed, t, tl)
            (o,) = sim.run_schedule([10 * k + 10])
            assert (o.bond_sum, o.M, o.Q) == tl and o.sweeps_done == 10 * k + 10, k
            if k in (1, 9):
                assert (sim.read_lattice() == s).all(), k
        assert oracle.observables(s) == tl                          # tally == recompute
        b100 = tl[0]
        del s
        for k in range(10, 100):                                    # E, M every 10 sweeps up to 1000
            (o,) = sim.run_schedule([10 * k + 10])
            lat = sim.read_lattice()
            assert (o.bond_sum, o.M, o.Q) == oracle.observables(lat), k
            del lat
            if 10 * k + 10 in (200, 500):
                check_windows(sim, cfg, 10 * k + 10, window_origins(L)[:3] if k == 19 else window_origins(L)[:2])
        assert o.sweeps_done == 1000
        assert packed_sums(sim, cfg.model, L) == (o.M, o.Q)
        v, hist = sim.schwinger_dyson()
        ov, ohist = oracle.schwinger_dyson(sim.read_lattice(), cfg.beta)
        assert (hist == ohist).all() and abs(v - ov) <= 1e-12 * abs(ov)
        assert o.bond_sum > b100                                    # a deep quench keeps lowering the energy


# ---------------------------------------------------------------- configs[3] ---
def test_config3_blume_capel_L2p15_500_sweeps(eng):
    """Blume-Capel L = 2^15, D = 1, beta = 1/1.4, 500 sweeps; E, M and the density of zeros every 10 sweeps
    (BASELINE.json configs[3]): full lattice vs the oracle for 5 sweeps, then every one of the 50 measurements of
    ising_run_schedule against the oracle's O5 routine on the lattice read back, light-cone windows at 50, 100
    and 500 sweeps, normalised doubles to rel 1e-12."""
    cfg = wl.config(3)
    L = cfg.L
    s = oracle.init(cfg.model, L, cfg.seed)
    tl = oracle.observables(s)
    with eng.IsingSim(cfg.model, L, cfg.beta, cfg.D, cfg.seed) as sim:
        assert (sim.thresholds() == oracle.thresholds(cfg.model, cfg.beta, cfg.D)).all()
        for t in range(5):
            tl = oracle.sweep(cfg.model, s, cfg.beta, cfg.D, cfg.seed, t, tl)
        sim.sweep(5)
        o = sim.observables()
        assert (o.bond_sum, o.M, o.Q) == tl
        assert (sim.read_lattice() == s).all()
        del s
        for n in range(10, 501, 10):
            (o,) = sim.run_schedule([n])
            lat = sim.read_lattice()
            bmq = oracle.observables(lat)
            del lat
            assert (o.bond_sum, o.M, o.Q) == bmq and o.sweeps_done == n, n
            E, e, m, z = oracle.normalised(cfg.model, L, cfg.D, bmq)
            for a, b in [(o.E, E), (o.e_per_site, e), (o.m_per_site, m), (o.zero_density, z)]:
                assert a == b or abs(a - b) <= 1e-12 * max(abs(a), abs(b))
            if n in (50, 100, 500):
                check_windows(sim, cfg, n, window_origins(L)[:4] if n == 50 else window_origins(L)[:2])
        assert packed_sums(sim, cfg.model, L) == (o.M, o.Q)
        v, hist = sim.schwinger_dyson()
        ov, ohist = oracle.schwinger_dyson(sim.read_lattice(), cfg.beta)
        assert (hist == ohist).all() and abs(v - ov) <= 1e-12 * abs(ov)


# ---------------------------------------------------------------- configs[4] ---
def test_config4_ising_L2p16_correlation_protocol_2000_sweeps(eng, golden_dir):
    """Ising L = 2^16, T = 0.5 Tc, 2000 sweeps, C(r) interleaved with the updates at t = 2^k (eleven times) and
    at t = 2000 (BASELINE.json configs[4]; A10/A11).  One native call (ising_run_protocol_schedule) per stretch.
    At every time: the distance list against the pins of tests/golden/protocol_pins.txt (480 distances and
    r_c = 256 up to t = 1024; 490, r_c = 268, grid from 273 at t = 2000) and the oracle's list, S(1) identity, B, M
    against O5 of the oracle at t = 1, 64, 2000.  Full range r = 1..L/2 at t = 1, 64 and 2000 (tensor cores; XOR + POPC
    kernels at t = 1): sampled r against the oracle's O6 routine on the lattice read back, all-source and
    block-source protocol rows likewise.  Light-cone windows at t = 64 and 256 anchor the trajectory (a window
    at t = 2000 would need 1.3e11 oracle site updates)."""
    cfg = wl.config(4)
    L = cfg.L
    pins = {}
    import os
    with open(os.path.join(golden_dir, "protocol_pins.txt")) as f:
        for ln in f:
            if ln.strip() and not ln.startswith("#"):
                kind, pl, pt, want = ln.split()
                if int(pl) == L:
                    pins[(kind, int(pt))] = int(want)
    assert pins[("count", 2000)] == 490 and pins[("rc", 2000)] == 268 and pins[("first_log", 2000)] == 273
    sample_r = np.array([1, 2, 3, 31, 32, 33, 63, 64, 65, 1000, 4097, L // 4, L // 2 - 1, L // 2], dtype=np.int64)
    times = wl.pow2_times(cfg.sweeps) + [cfg.sweeps]
    assert len(times) == 12 and times[-2:] == [1024, 2000]
    with eng.IsingSim(cfg.model, L, cfg.beta, cfg.D, cfg.seed) as sim:
        for t in times:
            rows, obs = sim.run_protocol_schedule([t])
            (r, sx, sy, nsrc), o = rows[0], obs[0]
            assert o.sweeps_done == t
            pr, pstride = oracle.protocol_list(L, t)
            assert (r == pr).all() and (nsrc == (L // pstride) ** 2).all()
            dense = pstride == 1
            rc = 268 if t == 2000 else 256                          # protocol_pins.txt: rc 65536 1820 256 / 2000 268
            assert len(r) == (490 if t == 2000 else 480) and int(r[-1]) == pins[("last", 100)]
            assert (r[:rc] == np.arange(1, rc + 1)).all() and int(r[rc]) == (273 if t == 2000 else 261)
            assert int(sx[0]) + int(sy[0]) == o.bond_sum            # r[0] = 1, all sources
            if t in (64, 256):
                check_windows(sim, cfg, t, window_origins(L)[:3] if t == 64 else window_origins(L)[:2])
            if t in (1, 64, 2000):
                fx, fy = sim.correlation(L // 2)                    # automatic path: tensor cores at this size
                if t == 1:
                    sim.set_corr_path(1)                            # XOR + POPC kernels: identical integers
                    bx, by = sim.correlation(L // 2)
                    sim.set_corr_path(0)
                    assert (bx == fx).all() and (by == fy).all()
                assert (sx[dense] == fx[r[dense] - 1]).all() and (sy[dense] == fy[r[dense] - 1]).all()
                lat = sim.read_lattice()
                assert (o.bond_sum, o.M, o.Q) == oracle.observables(lat)
                ox, oy = oracle.correlation_list(lat, 1, sample_r)
                assert (fx[sample_r - 1] == ox).all() and (fy[sample_r - 1] == oy).all()
                sparse_r = r[~dense][:: max(1, (~dense).sum() // 12)]
                if t == 2000:                                       # the rows only the r_c = 268 list has
                    sparse_r = np.unique(np.concatenate([sparse_r, [257, 262, 268, 273]]))
                bx, by = oracle.correlation_list(lat, 16, sparse_r)
                sel = np.isin(r, sparse_r) & ~dense
                assert (sx[sel] == bx).all() and (sy[sel] == by).all()
                del lat
        assert sim.observables().sweeps_done == 2000


# ------------------------------------------------------------ maximum sizes ---
@pytest.mark.parametrize("model,L,beta,D", [(wl.ISING_LUT, 1 << 20, wl.BETA_C / 0.9, 0.0),
                                            (ISING, 1 << 19, wl.BETA_C / 0.9, 0.0), (BC, 1 << 19, 1 / 1.4, 1.0),
                                            (wl.BLUME_CAPEL_2BIT, 3 << 18, 1 / 1.4, 1.0)])
def test_maximum_lattice_sizes(eng, model, L, beta, D):
    """The largest lattices one B200 holds -- the paper's single-GPU maxima: 2^40 spins at
    one bit (137 GB) and 2^38 at four bits (137 GB); Blume-Capel at two bits per spin (NEXT-3) reaches
    L = 3 * 2^18 (6.2e11 spins, 155 GB) against the 4-bit oracle.  Light-cone windows on the wraps and in the
    last rows (64-bit offsets), Q and n_sites at 2^40."""
    n = 3
    with eng.IsingSim(model, L, beta, D, 1) as sim:
        sim.sweep(n)
        for (x0, y0) in [(-W // 2, -W // 2), (L - W // 2, L // 3 + 5), (L // 5 + 3, L - W // 2), (L // 2 + 7, L - 40)]:
            if model == wl.ISING_LUT:
                want = oracle.lut_window_after(L, beta, 1, n, x0, y0, W, W)
            else:
                want = oracle.window_after(BC if model == wl.BLUME_CAPEL_2BIT else model, L, beta, D, 1, n, x0, y0, W, W)
            assert (sim.read_window(x0, y0, W, W) == want).all(), (x0, y0)
        o = sim.observables()
        assert o.n_sites == L * L and o.sweeps_done == n and abs(o.M) < L * L // 1000
        assert o.Q == L * L if model not in (BC, wl.BLUME_CAPEL_2BIT) else 0 < o.Q < L * L
        # no room left for the bit planes of the correlation pass: a clean ISING_ENOMEM, and the handle stays usable
        with pytest.raises(eng.IsingError) as err:
            sim.correlation(4)
        assert err.value.code == -2
        sim.sweep(1)
        x0, y0 = L - W // 2, L - W // 2
        omodel = BC if model == wl.BLUME_CAPEL_2BIT else model
        want = (oracle.lut_window_after(L, beta, 1, n + 1, x0, y0, W, W) if model == wl.ISING_LUT
                else oracle.window_after(omodel, L, beta, D, 1, n + 1, x0, y0, W, W))
        assert (sim.read_window(x0, y0, W, W) == want).all()
