"""Pins for the oracle's correlation sums, the Sec. 3.3 protocol lists and the
light-cone window helper (-m "not gpu")."""
import os

import numpy as np
import pytest

import oracle
import workloads as wl

ISING, BC = oracle.ISING, oracle.BLUME_CAPEL


def _lattice(model, L, seed, sweeps=3):
    s = oracle.init(model, L, seed)
    for t in range(sweeps):
        oracle.sweep(model, s, 0.6, 0.5, seed, t)
    return s


@pytest.mark.parametrize("model", [ISING, BC])
def test_correlation_bruteforce_python(model):
    """PAPER.md:65 'from each lattice site at multiple distances along the two
    lattice dimensions' (R13): python-int double loop on a tiny lattice."""
    L = 12
    s = _lattice(model, L, 4)
    sx, sy = oracle.correlation(s, L // 2)
    a = s.astype(int).tolist()
    for r in range(1, L // 2 + 1):
        ex = sum(a[y][x] * a[y][(x + r) % L] for y in range(L) for x in range(L))
        ey = sum(a[y][x] * a[(y + r) % L][x] for y in range(L) for x in range(L))
        assert (sx[r - 1], sy[r - 1]) == (ex, ey)


@pytest.mark.parametrize("model", [ISING, BC])
def test_correlation_identities(model):
    """Exact integer identities: S_x(1)+S_y(1) = B; sum_{r=0}^{L-1} S_x(r) =
    sum_y (row magnetisation)^2 with S(0) = Q and S(r) = S(L-r)."""
    L = 64
    s = _lattice(model, L, 7)
    B, M, Q = oracle.observables(s)
    sx, sy = oracle.correlation(s, L // 2)
    assert sx[0] + sy[0] == B
    g = s.astype(np.int64)
    # r = 1..L/2-1 appear twice in a full circle, r = L/2 once
    assert Q + 2 * sx[:-1].sum() + sx[-1] == (g.sum(axis=1) ** 2).sum()
    assert Q + 2 * sy[:-1].sum() + sy[-1] == (g.sum(axis=0) ** 2).sum()


def test_correlation_crafted():
    L = 32
    up = np.ones((L, L), np.int8)
    sx, sy = oracle.correlation(up, L // 2)
    assert (sx == L * L).all() and (sy == L * L).all()
    yy, xx = np.mgrid[0:L, 0:L]
    w = 4
    stripes = np.where((xx // w) % 2 == 0, 1, -1).astype(np.int8)
    sx, sy = oracle.correlation(stripes, L // 2)
    assert (sy == L * L).all()
    for r in range(1, L // 2 + 1):                     # triangle wave of period 2w
        q = r % (2 * w)
        per_site = (w - 2 * q) / w if q <= w else (2 * q - 3 * w) / w
        assert sx[r - 1] == int(round(per_site * L * L))
    # x and y are not transposed: horizontal stripes give the mirrored result
    sx2, sy2 = oracle.correlation(np.ascontiguousarray(stripes.T), L // 2)
    assert (sx2 == sy).all() and (sy2 == sx).all()


def test_correlation_list_matches_definition():
    L = 64
    s = _lattice(ISING, L, 3)
    a = s.astype(np.int64)
    r = np.array([1, 5, 17, 32])
    sx, sy = oracle.correlation_list(s, 16, r)
    for i, d in enumerate(r):
        src = a[::16, ::16]
        assert sx[i] == (src * np.roll(a, -d, axis=1)[::16, ::16]).sum()
        assert sy[i] == (src * np.roll(a, -d, axis=0)[::16, ::16]).sum()
    fx, fy = oracle.correlation(s, 32)
    lx, ly = oracle.correlation_list(s, 1, np.arange(1, 33))
    assert (fx == lx).all() and (fy == ly).all()


def test_protocol_lists(golden_dir):
    """PAPER.md:163-174 with readings R15-R17; expected numbers from SURVEY.md Sec. 8(c)."""
    with open(os.path.join(golden_dir, "protocol_pins.txt")) as f:
        rows = [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]
    for kind, L, t, want in rows:
        L, t, want = int(L), int(t), int(want)
        if kind == "rc":
            assert oracle.protocol_rc(L, t) == want
        elif kind == "timegrid":
            assert len(oracle.time_grid(t)) == want
        else:
            r, st = oracle.protocol_list(L, t)
            if kind == "count":
                assert len(r) == want
            elif kind == "last":
                assert r[-1] == want
            elif kind == "first_log":
                rc = oracle.protocol_rc(L, t)
                assert r[r > rc][0] == want


def test_time_grid_and_log_grid_exact_integer_criteria():
    """Pins that need no floating point: t = nearest integer to 2^(x/8) <=> (2t - 1)^8 <= 2^(x+8) < (2t + 1)^8, and
    d = floor(2^(x/32)) <=> d^32 <= 2^x < (d + 1)^32, in Python integers."""
    tg = [int(t) for t in oracle.time_grid(1 << 20)]
    x, want = 1, []
    while True:
        t = max(1, round(2.0 ** (x / 8.0)))
        while (2 * t + 1) ** 8 <= 2 ** (x + 8):
            t += 1
        while (2 * t - 1) ** 8 > 2 ** (x + 8):
            t -= 1
        if t > 1 << 20:
            break
        if not want or want[-1] != t:
            want.append(t)
        x += 1
    assert tg == want
    L = 1 << 20
    r, st = oracle.protocol_list(L, 1)
    rc = oracle.protocol_rc(L, 1)
    grid, x = [], 0
    while 2 ** x <= (L // 2) ** 32:
        d = int(2.0 ** (x / 32.0))
        while (d + 1) ** 32 <= 2 ** x:
            d += 1
        while d ** 32 > 2 ** x:
            d -= 1
        if d > rc and (not grid or grid[-1] != d):
            grid.append(d)
        x += 1
    assert [int(v) for v in r[r > rc]] == grid


def test_protocol_structure():
    L, t = 1 << 16, 100
    r, st = oracle.protocol_list(L, t)
    assert (np.diff(r) > 0).all()
    assert (r[:32] == np.arange(1, 33)).all() and (st[:32] == 1).all()          # all sources, r <= 2R
    assert (r[32:256] == np.arange(33, 257)).all() and (st[32:] == 16).all()   # one per RxR block
    assert len(r) == 32 + 224 + 224
    # "32 values of r for each power of two" once floor() stops colliding
    for k in range(9, 15):
        assert ((r > 2**k) & (r <= 2**(k + 1))).sum() == 32
    tg = oracle.time_grid(2000)
    assert list(tg[:12]) == list(range(1, 13)) and list(tg[-4:]) == [1448, 1579, 1722, 1878]
    assert set(wl.pow2_times(2000)) <= set(int(x) for x in tg)               # config 5's grid = x = 8k
    # small lattices: everything clipped to L/2
    r, st = oracle.protocol_list(256, 7)
    assert r[-1] == 128 and (r == np.arange(1, 129)).all()
    rr, sx, sy, ns = oracle.correlation_protocol(_lattice(ISING, 256, 2), 7)
    assert (ns[:32] == 256 * 256).all() and (ns[32:] == 16 * 16).all()


@pytest.mark.parametrize("model,beta,D", [(ISING, wl.BETA_C, 0.0), (BC, 1 / 1.4, 1.0)])
def test_light_cone_window_equals_full_lattice(model, beta, D):
    """The window helper (used for L = 2^18 parity) against the full-lattice sweep,
    including windows that straddle the periodic wrap; and margin 2n is tight."""
    L, n, seed = 64, 5, 6
    s = oracle.init(model, L, seed)
    for t in range(n):
        oracle.sweep(model, s, beta, D, seed, t)
    for (x0, y0, w, h) in [(10, 12, 16, 8), (L - 7, 20, 14, 9), (30, L - 5, 12, 10), (L - 3, L - 3, 6, 6)]:
        win = oracle.window_after(model, L, beta, D, seed, n, x0, y0, w, h)
        ys = [(y0 + j) % L for j in range(h)]
        xs = [(x0 + i) % L for i in range(w)]
        assert (win == s[np.ix_(ys, xs)]).all()
    # a margin far inside the light cone must fail somewhere (the helper is not vacuous)
    m = 1
    p = oracle.init_patch(model, L, seed, 10 - m, 12 - m, 16 + 2 * m, 8 + 2 * m)
    for t in range(n):
        oracle.sweep_patch(model, L, p, beta, D, seed, t, 10 - m, 12 - m)
    ys = [(12 + j) % L for j in range(8)]
    xs = [(10 + i) % L for i in range(16)]
    assert not (p[m:m + 8, m:m + 16] == s[np.ix_(ys, xs)]).all()
