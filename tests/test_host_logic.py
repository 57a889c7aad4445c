"""-m "not gpu": the PRODUCT's host arithmetic, called through the C ABI without a GPU, pinned
directly to what the paper and the mathematics fix -- not to the oracle:

  ising_time_grid            t = floor(2^(x/8) + 1/2): exact integer criterion
                             (2t - 1)^8 <= 2^(x+8) < (2t + 1)^8 with Python integers, and the
                             counts / end points of tests/golden/protocol_pins.txt
  ising_protocol_distances   PAPER.md:163-170: tests/golden/protocol_pins.txt (r_c, counts, first
                             and last grid value incl. the L = 2^22, t = 524288 rows), the exact
                             criterion d^32 <= 2^x < (d + 1)^32 for every grid value, structure
  ising_threshold_table      PAPER.md:93 / Eq. 2: closed forms at beta_c (integer square roots),
                             60-digit decimals; the 1-bit model's table: marginals
                             and pairwise independence of the four bits

The same pins are applied to the oracle in tests/test_oracle_*.py; that the two sides then agree with
each other is checked last, as a consequence.
"""
import ctypes as C
import math
import os
from decimal import Decimal, getcontext
from math import isqrt

import numpy as np
import pytest

import workloads as wl

TWO32 = 1 << 32


@pytest.fixture(scope="module")
def eng():
    from paper_2502_18624_b200 import build as b
    b.build()
    import paper_2502_18624_b200 as e
    e.load_library()
    return e


def _pins(golden_dir):
    with open(os.path.join(golden_dir, "protocol_pins.txt")) as f:
        return [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]


# ------------------------------------------------------------------ time grid ---
def _exact_time_grid(tmax):
    """t_x = nearest integer to 2^(x/8), by integers only: t - 1/2 <= 2^(x/8) < t + 1/2
    <=> (2t - 1)^8 <= 2^(x + 8) < (2t + 1)^8."""
    out, x = [], 1
    while True:
        t = max(1, int(round(2.0 ** (x / 8.0))))
        while (2 * t + 1) ** 8 <= 2 ** (x + 8):
            t += 1
        while (2 * t - 1) ** 8 > 2 ** (x + 8):
            t -= 1
        if t > tmax:
            return out
        if not out or out[-1] != t:
            out.append(t)
        x += 1


@pytest.mark.parametrize("tmax", [1, 12, 13, 2000, 524288, 2**31 - 1])
def test_time_grid_is_the_exact_rounding(eng, tmax):
    got = [int(t) for t in eng.time_grid(tmax)]
    assert got == _exact_time_grid(tmax)


def test_time_grid_golden_pins(eng, golden_dir):
    for kind, L, t, want in _pins(golden_dir):
        if kind == "timegrid":
            assert len(eng.time_grid(int(t))) == int(want)
    tg = [int(t) for t in eng.time_grid(2000)]
    assert tg[:12] == list(range(1, 13)) and tg[-4:] == [1448, 1579, 1722, 1878]
    assert set(wl.pow2_times(2000)) <= set(tg)                                         # config 4's grid is x = 8k
    assert len(eng.time_grid(0)) == 0


def test_time_grid_size_query_and_errors(eng):
    lib = eng.load_library()
    n = C.c_int64(-1)
    assert lib.ising_time_grid(2000, None, 0, C.addressof(n)) == 0 and n.value == 70     # size query
    buf = np.zeros(8, dtype=np.uint64)
    assert lib.ising_time_grid(2000, buf.ctypes.data, 8, C.addressof(n)) == -1 and n.value == 70
    assert (buf == 0).all()                                                                 # nothing written
    assert lib.ising_time_grid(2000, None, 0, None) == -1


# ------------------------------------------------------- Sec. 3.3 distance lists ---
def test_protocol_distances_golden_pins(eng, golden_dir):
    """r_c, list length, first / last value of the logarithmic grid: tests/golden/protocol_pins.txt
    (derived from PAPER.md:163-170 with readings R15, R16)."""
    seen = set()
    for kind, L, t, want in _pins(golden_dir):
        L, t, want = int(L), int(t), int(want)
        if kind == "timegrid":
            continue
        r, st = eng.protocol_distances(L, t)
        block = r[st == 16]
        # r_c = the end of the run of consecutive block-source distances that starts at 33
        run = 33
        for v in block:
            if v != run:
                break
            run += 1
        rc = run - 1
        if kind == "rc":
            assert rc == want, (L, t)
        elif kind == "count":
            assert len(r) == want, (L, t)
        elif kind == "last":
            assert int(r[-1]) == want, (L, t)
        elif kind == "first_log":
            assert int(r[r > rc][0]) == want, (L, t)
        seen.add(kind)
    assert seen == {"rc", "count", "last", "first_log"}


@pytest.mark.parametrize("L,t", [(1 << 16, 100), (1 << 16, 2000), (1 << 22, 524288), (4096, 1), (4096, 3000),
                                 (4160, 50), (256, 7), (64, 0), (1 << 20, 1 << 31)])
def test_protocol_distances_structure_and_exact_grid(eng, L, t):
    r, st = eng.protocol_distances(L, t)
    r, st = [int(v) for v in r], [int(v) for v in st]
    half = L // 2
    assert all(b > a for a, b in zip(r, r[1:])) and r[0] == 1 and r[-1] <= half
    n_all = min(32, half)
    assert r[:n_all] == list(range(1, n_all + 1)) and st[:n_all] == [1] * n_all      # every site a source, r <= 2R
    assert all(s == 16 for s in st[n_all:])                                          # one source per 16 x 16 block
    # r_c(t) = max{256, nearest integer to g(L) sqrt(t)}, g(L) = 6 sqrt(ln(L / 2^16) / 3.3^2 + 1): in 60-digit
    # decimals, with a guard against a value that sits on a rounding boundary
    getcontext().prec = 60
    g = 6 * (Decimal(L / 65536.0).ln() / (Decimal("3.3") ** 2) + 1).sqrt()
    v = g * Decimal(t).sqrt() + Decimal("0.5")
    assert abs(v - v.to_integral_value()) > Decimal("1e-9")
    rc = max(256, int(v.to_integral_value(rounding="ROUND_FLOOR")))
    dense_end = min(rc, half)
    assert r[: dense_end] == list(range(1, dense_end + 1))
    # the logarithmic grid: every d = floor(2^(x/32)) with 2^(x/32) <= L/2 and d > r_c, each once;
    # d = floor(2^(x/32)) <=> d^32 <= 2^x < (d + 1)^32, and 2^(x/32) <= L/2 <=> 2^x <= (L/2)^32
    grid, x = [], 0
    while 2 ** x <= half ** 32:
        d = int(2.0 ** (x / 32.0))
        while (d + 1) ** 32 <= 2 ** x:
            d += 1
        while d ** 32 > 2 ** x:
            d -= 1
        if d > max(rc, 32) and (not grid or grid[-1] != d):
            grid.append(d)
        x += 1
    assert r[dense_end:] == grid
    if L >= 1 << 16 and rc < 512:                      # "32 values of r for each power of two"
        for k in range(9, int(math.log2(half)) - 1):
            assert sum(1 for d in r if 2 ** k < d <= 2 ** (k + 1)) == 32


def test_protocol_distances_size_query_and_errors(eng):
    lib = eng.load_library()
    n = C.c_int64(-1)
    assert lib.ising_protocol_distances(1 << 16, 2000, 0, None, None, C.addressof(n)) == 0 and n.value == 490
    r = np.zeros(10, dtype=np.int64)
    st = np.zeros(10, dtype=np.int64)
    assert lib.ising_protocol_distances(1 << 16, 2000, 10, r.ctypes.data, st.ctypes.data, C.addressof(n)) == -1
    assert n.value == 490 and (r == 0).all()
    assert lib.ising_protocol_distances(65, 1, 0, None, None, C.addressof(n)) == -1           # odd L
    assert lib.ising_protocol_distances(64, 1, 0, None, None, None) == -1


# ------------------------------------------------------------------ thresholds ---
def _floor_sqrt_scaled(n, shift):
    """floor(sqrt(n) 2^shift) exactly."""
    return isqrt(n << (2 * shift))


def test_ising_thresholds_closed_forms_at_beta_c(eng):
    """e^{-4 beta_c} = 3 - 2 sqrt 2, e^{-8 beta_c} = 17 - 12 sqrt 2 (beta_c = ln(1 + sqrt 2) / 2):
    floor(p 2^32) by integer square roots; SURVEY.md Sec. 8(c) prints 736899888 and 126432032."""
    T = [int(v) for v in eng.threshold_table(wl.ISING, wl.BETA_C)]
    # floor((3 - 2 sqrt 2) 2^32) = 3 2^32 - ceil(sqrt(8) 2^32) = 3 2^32 - floor(sqrt(8) 2^32) - 1 (irrational)
    t4 = 3 * TWO32 - _floor_sqrt_scaled(8, 32) - 1
    t8 = 17 * TWO32 - _floor_sqrt_scaled(288, 32) - 1
    assert T == [TWO32, TWO32, TWO32, t4, t8] and (t4, t8) == (736899888, 126432032)


@pytest.mark.parametrize("tau,t4,t8", [(0.5, 126432032, 3721811), (0.9, 605825050, 85454432)])
def test_ising_thresholds_survey_values(eng, tau, t4, t8):
    T = [int(v) for v in eng.threshold_table(wl.ISING, wl.BETA_C / tau)]
    assert T[3:] == [t4, t8]


def test_blume_capel_thresholds_against_decimals(eng):
    """All 54 entries of config 3's table against exp(-beta dE) in 60-digit decimals (the decimal
    value of the double beta, so the only rounding left is libm's exp: every entry is >= 0.03 from an
    integer before the floor, reading R5), and the SURVEY.md Sec. 8(c) values by dE."""
    getcontext().prec = 60
    beta, D = 1.0 / 1.4, 1.0
    T = [int(v) for v in eng.threshold_table(wl.BLUME_CAPEL, beta, D)]
    assert T == [int(v) for v in eng.threshold_table(wl.BLUME_CAPEL_2BIT, beta, D)]
    by_dE = {1: 2102565417, 2: 1029293363, 3: 503881981, 4: 246671221, 5: 120755839, 6: 59115013, 8: 14166974}
    for s in (-1, 0, 1):
        for b in (0, 1):
            for h in range(-4, 5):
                sp = ((s + 1) + 1 + b) % 3 - 1
                dE = D * (sp * sp - s * s) - (sp - s) * h
                got = T[((s + 1) * 2 + b) * 9 + (h + 4)]
                if dE <= 0:
                    assert got == TWO32
                else:
                    p = (-(Decimal(beta) * Decimal(dE))).exp() * TWO32
                    assert got == int(p.to_integral_value(rounding="ROUND_FLOOR"))
                    assert abs(p - p.to_integral_value()) > Decimal("1e-3")
                    assert got == by_dE[int(dE)]
    assert T[((-1 + 1) * 2 + 0) * 9 + 0] == by_dE[3] and T[((1 + 1) * 2 + 0) * 9 + 8] == by_dE[8]      # SURVEY examples
    assert T[((0 + 1) * 2 + 1) * 9 + 8] == by_dE[5]


@pytest.mark.parametrize("beta", [wl.BETA_C, wl.BETA_C / 0.5, wl.BETA_C / 0.9, 0.1, 1.5])
def test_lut_table_marginals_and_independence(eng, beta):
    """four independent bits, each 1 with probability p = e^{-4 beta}; on the integer
    table of the PRODUCT, to the quantisation error (16 counts)."""
    p = math.exp(-4 * beta)
    t = [int(v) for v in eng.threshold_table(wl.ISING_LUT, beta)] + [TWO32]
    w = [t[i + 1] - t[i] for i in range(16)]
    assert t[0] == 0 and all(x >= 0 for x in w) and sum(w) == TWO32
    for k in range(4):
        assert abs(sum(w[i] for i in range(16) if (i >> k) & 1) - p * TWO32) <= 16
        for l in range(k + 1, 4):
            assert abs(sum(w[i] for i in range(16) if (i >> k) & 1 and (i >> l) & 1) - p * p * TWO32) <= 16
    assert abs(w[15] - p ** 4 * TWO32) <= 16 and abs(w[0] - (1 - p) ** 4 * TWO32) <= 16
    if beta == wl.BETA_C:                                   # p = 3 - 2 sqrt 2: patterns 0..7 have bit 3 clear
        p_c = 3 - 2 * math.sqrt(2)
        assert abs(t[8] - (1 - p_c) * TWO32) <= 2 and abs(t[1] - (1 - p_c) ** 4 * TWO32) <= 2


def test_lut_table_extremes_and_errors(eng):
    assert (eng.threshold_table(wl.ISING_LUT, 0.0) == 0).all()               # p = 1: always pattern 15
    t = eng.threshold_table(wl.ISING_LUT, 40.0)                              # p = e^-160: always pattern 0
    assert int(t[0]) == 0 and all(int(v) == TWO32 for v in t[1:])
    assert [int(v) for v in eng.threshold_table(wl.ISING, 0.0)] == [TWO32] * 5
    lib = eng.load_library()
    n = C.c_int(-1)
    assert lib.ising_threshold_table(1, 0.5, 1.0, None, 0, C.addressof(n)) == 0 and n.value == 54     # size query
    assert lib.ising_threshold_table(7, 0.5, 1.0, None, 0, C.addressof(n)) == -1
    assert lib.ising_threshold_table(0, -1.0, 0.0, None, 0, C.addressof(n)) == -1
    assert lib.ising_threshold_table(0, float("nan"), 0.0, None, 0, C.addressof(n)) == -1


# ------------------------------------------------------------- slab partition ---
def test_slab_partition(eng):
    """NEXT-4 host logic: even heights >= 2 that add up to L, as even as row pairs allow."""
    for L, n in [(256, 1), (256, 3), (256, 8), (1 << 18, 8), (1 << 20, 64), (64, 32), (192, 7), (1 << 19, 6)]:
        rows = [int(r) for r in eng.slab_partition(L, n)]
        assert len(rows) == n and sum(rows) == L and all(r >= 2 and r % 2 == 0 for r in rows)
        assert max(rows) - min(rows) <= 2
    assert [int(r) for r in eng.slab_partition(256, 3)] == [84, 86, 86]
    for L, n in [(256, 0), (256, 65), (64, 33), (255, 2)]:
        with pytest.raises(eng.IsingError):
            eng.slab_partition(L, n)


# ------------------------------------------------ and, as a consequence, == oracle ---
def test_host_logic_agrees_with_the_oracle(eng):
    import oracle
    for tmax in (1, 12, 2000, 524288):
        assert (eng.time_grid(tmax) == oracle.time_grid(tmax)).all()
    for L, t in [(1 << 16, 1), (1 << 16, 2000), (1 << 22, 524288), (4096, 3000), (256, 7), (4160, 50)]:
        r, st = eng.protocol_distances(L, t)
        orr, ost = oracle.protocol_list(L, t)
        assert (r == orr).all() and (st == ost).all()
    for i in range(5):
        w = wl.config(i)
        assert (eng.threshold_table(w.model, w.beta, w.D) == oracle.thresholds(w.model, w.beta, w.D)).all()
    for beta in (0.0, 0.05, wl.BETA_C, wl.BETA_C / 0.9, wl.BETA_C / 0.5, 1.5, 40.0):
        assert (eng.threshold_table(wl.ISING_LUT, beta) == oracle.lut_table(beta)).all()
        for D in (-2.0, 0.0, 1.966):
            assert (eng.threshold_table(wl.BLUME_CAPEL, beta, D) == oracle.thresholds(1, beta, D)).all()
