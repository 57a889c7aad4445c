"""GPU parity at BASELINE.json's full sizes (-m gpu), in the launch configuration
bench.py times (default rows-per-thread / block size, default kernel variant).

The oracle cannot hold a 69 GB lattice nor do 1.4e13 updates, so:
  * light-cone windows: the w x h window after n sweeps depends only on the initial
    spins within 2n sites of it; oracle.window_after simulates that patch with global
    coordinates mod L and its centre must equal ising_read_window byte for byte.
    Windows sit on the x wrap, the y wrap, the corner, across thread-column (64 sites),
    row-chunk (32 rows) and block boundaries;
  * integer observables: plain definitions evaluated with numpy on the packed lattice
    streamed back (M = 2 popcount - N), the oracle's O5/O6 routines on the lattice read
    back where it fits the host, and identities that hold at any size
    (S_x(1) + S_y(1) = B).
"""
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
    for (x0, y0) in origins:
        want = oracle.window_after(cfg.model, cfg.L, cfg.beta, cfg.D, cfg.seed, n, x0, y0, W, W)
        got = sim.read_window(x0, y0, W, W)
        assert (got == want).all(), (cfg.name, n, x0, y0, int((got != want).sum()))


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
def test_config1_ising_L2p14_full_lattice_then_windows(eng):
    """Ising L = 2^14, T = 0.5 Tc: full lattice + B, M against the oracle for the first 20
    sweeps (B, M every 10), then E, M every 10 sweeps to 1000 checked by the definition on
    the packed lattice / the identity, and light-cone windows at 200 sweeps."""
    cfg = wl.config(1)
    L = cfg.L
    s = oracle.init(cfg.model, L, cfg.seed)
    tl = oracle.observables(s)
    with eng.IsingSim(cfg.model, L, cfg.beta, cfg.D, cfg.seed) as sim:
        assert (sim.read_lattice() == s).all()
        for t in range(20):
            tl = oracle.sweep(cfg.model, s, cfg.beta, cfg.D, cfg.seed, t, tl)
            if (t + 1) % 10 == 0:
                sim.sweep(10)
                o = sim.observables()
                assert (o.bond_sum, o.M, o.Q) == tl, t
        assert (sim.read_lattice() == s).all()
        assert oracle.observables(s) == tl                          # tally == recompute
        sim.sweep(180)
        check_windows(sim, cfg, 200, window_origins(L)[:3])
        for k in range(20, 100):                                    # E, M every 10 sweeps up to 1000
            sim.sweep(10)
            o = sim.observables()
            assert o.Q == L * L and abs(o.M) <= L * L and -2 * L * L <= o.bond_sum <= 2 * L * L
        assert o.sweeps_done == 1000
        lat = sim.read_lattice()
        assert (o.bond_sum, o.M, o.Q) == oracle.observables(lat)    # O5 on the GPU lattice
        assert packed_sums(sim, cfg.model, L) == (o.M, o.Q)
        # deep quench at 0.5 Tc coarsens: the energy must have dropped well below the t = 20 value
        assert o.bond_sum > tl[0]


# ---------------------------------------------------------------- configs[3] ---
def test_config3_blume_capel_L2p15(eng):
    """Blume-Capel L = 2^15, D = 1, beta = 1/1.4: full lattice vs oracle for 5 sweeps, windows at
    50 and 100 sweeps, B, M, Q (-> E, zero density) every 10 sweeps, O5 on the final lattice."""
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
        done = 5
        for n in (50, 100):
            while done < n:
                step = min(10 - done % 10, n - done)
                sim.sweep(step)
                done += step
                o = sim.observables()
                assert 0 <= o.Q <= L * L and abs(o.M) <= o.Q
            check_windows(sim, cfg, n, window_origins(L)[:4] if n == 50 else window_origins(L)[:2])
        lat = sim.read_lattice()
        bmq = oracle.observables(lat)
        assert (o.bond_sum, o.M, o.Q) == bmq
        E, e, m, z = oracle.normalised(cfg.model, L, cfg.D, bmq)
        for a, b in [(o.E, E), (o.e_per_site, e), (o.m_per_site, m), (o.zero_density, z)]:
            assert a == b or abs(a - b) <= 1e-12 * max(abs(a), abs(b))
        assert packed_sums(sim, cfg.model, L) == (o.M, o.Q)


# ---------------------------------------------------------------- configs[4] ---
def test_config4_ising_L2p16_correlation_protocol(eng):
    """Ising L = 2^16, T = 0.5 Tc, correlation interleaved with updates at t = 2^k (A11).
    Full range r = 1..L/2 at t = 1 and t = 64; the paper's protocol at every t.  Checks:
    the oracle's O6 routine on the GPU lattice for sampled r, S(1) identity, all-source and
    block-source protocol rows against the full-range sums / the oracle."""
    cfg = wl.config(4)
    L = cfg.L
    sample_r = np.array([1, 2, 3, 31, 32, 33, 63, 64, 65, 1000, 4097, L // 4, L // 2 - 1, L // 2], dtype=np.int64)
    with eng.IsingSim(cfg.model, L, cfg.beta, cfg.D, cfg.seed) as sim:
        done = 0
        for t in wl.pow2_times(64):
            sim.sweep(t - done)
            done = t
            o = sim.observables()
            r, sx, sy, nsrc = sim.correlation_protocol()
            pr, pstride = oracle.protocol_list(L, t)
            assert (r == pr).all() and (nsrc == (L // pstride) ** 2).all()
            assert int(sx[0]) + int(sy[0]) == o.bond_sum            # r[0] = 1, all sources
            if t in (1, 64):
                fx, fy = sim.correlation(L // 2)                    # automatic path: tensor cores at this size
                if t == 1:
                    sim.set_corr_path(1)                            # XOR + POPC kernels: identical integers
                    bx, by = sim.correlation(L // 2)
                    sim.set_corr_path(0)
                    assert (bx == fx).all() and (by == fy).all()
                dense = pstride == 1
                assert (sx[dense] == fx[r[dense] - 1]).all() and (sy[dense] == fy[r[dense] - 1]).all()
                lat = sim.read_lattice()
                ox, oy = oracle.correlation_list(lat, 1, sample_r)
                assert (fx[sample_r - 1] == ox).all() and (fy[sample_r - 1] == oy).all()
                sparse_r = r[~dense][:: max(1, (~dense).sum() // 12)]
                bx, by = oracle.correlation_list(lat, 16, sparse_r)
                sel = np.isin(r, sparse_r) & ~dense
                assert (sx[sel] == bx).all() and (sy[sel] == by).all()
                del lat
        assert done == 64


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
