"""Pins of the NEXT-2 oracle (oracle/ising_oracle.c, section O7): the paper's one-bit Ising kernel
with look-up-table random bits.  The paper prints no worked example, so the pins
are properties the mathematics fixes: the table's marginals and independence, getMaxLE against a
library search, two independently written sweeps (per word / per site), the tally invariant, exact
enumeration of the 4x4 lattice and Onsager's closed forms."""
import ctypes as C
import math

import numpy as np
import pytest

import oracle
import workloads as wl

from test_oracle_pins import _blocked, _enumerate, _onsager_m0, _onsager_u, _pins  # noqa: F401  (shared exact values)

TWO32 = 1 << 32


def _widths(table):
    t = [int(v) for v in table] + [TWO32]
    return [t[i + 1] - t[i] for i in range(16)]


@pytest.mark.parametrize("beta", [wl.BETA_C, wl.BETA_C / 0.5, wl.BETA_C / 0.9, 0.1, 1.5])
def test_table_marginals_and_independence(beta):
    """Each of the four bits is 1 with probability p = e^{-4 beta} and the bits are independent
    (PAPER.md:133-135): checked on the integer table to the quantisation error (16 counts)."""
    p = math.exp(-4 * beta)
    t = oracle.lut_table(beta)
    w = _widths(t)
    assert int(t[0]) == 0 and all(x >= 0 for x in w) and sum(w) == TWO32
    for k in range(4):
        got = sum(w[i] for i in range(16) if (i >> k) & 1)
        assert abs(got - p * TWO32) <= 16, (k, got, p * TWO32)
        for l in range(k + 1, 4):
            both = sum(w[i] for i in range(16) if (i >> k) & 1 and (i >> l) & 1)
            assert abs(both - p * p * TWO32) <= 16
    assert abs(w[15] - p ** 4 * TWO32) <= 16 and abs(w[0] - (1 - p) ** 4 * TWO32) <= 16
    # closed forms at beta_c: p = 3 - 2 sqrt 2
    if beta == wl.BETA_C:
        p_c = 3 - 2 * math.sqrt(2)
        assert abs(int(t[8]) - (1 - p_c) * TWO32) <= 2          # patterns 0..7 have bit 3 clear
        assert abs(int(t[1]) - (1 - p_c) ** 4 * TWO32) <= 2


def test_table_extremes():
    assert (oracle.lut_table(0.0) == 0).all()                   # p = 1: every number maps to pattern 15
    t = oracle.lut_table(40.0)                                  # p = e^-160: pattern 0 always
    assert int(t[0]) == 0 and all(int(v) == TWO32 for v in t[1:])


def test_random_words_against_library_search_and_keying():
    """orc_lut_bits against numpy.searchsorted on the same table and the KAT-pinned Philox: nibble
    4 (q & 3) + u of the exp4 (q < 4) / exp8 (q >= 4) word comes from output word u of the call
    with counter (8 w + q, t, tag)."""
    beta, seed = wl.BETA_C / 0.9, 0x1234567890ABCDEF
    table = oracle.lut_table(beta)
    key = [seed & 0xFFFFFFFF, seed >> 32]
    for w, t, tag in [(0, 0, 0), (5, 7, 1), ((1 << 33) + 3, 199, 0)]:
        for which in (0, 1):
            want = 0
            for q4 in range(4):
                g = 8 * w + which * 4 + q4
                out = oracle.philox4x32_10([g & 0xFFFFFFFF, g >> 32, t, tag], key)
                idx = np.searchsorted(table, out.astype(np.uint64), side="right") - 1
                for u in range(4):
                    want |= int(idx[u]) << (16 * q4 + 4 * u)
            assert oracle.lut_bits(table, seed, w, t, tag, which) == want


def test_bit_frequencies_of_random_words():
    """Empirical rate of ones in 2^16 random bits = p within 5 sigma (catches a reversed table)."""
    beta = wl.BETA_C / 0.9
    p = math.exp(-4 * beta)
    table = oracle.lut_table(beta)
    ones = sum(bin(oracle.lut_bits(table, 3, w, 0, 0, 0)).count("1") for w in range(1024))
    n = 1024 * 64
    assert abs(ones - n * p) < 5 * math.sqrt(n * p * (1 - p))


@pytest.mark.parametrize("L,beta", [(64, wl.BETA_C), (96, 0.6), (256, wl.BETA_C / 0.5)])
def test_tally_equals_recompute_and_init_is_balanced(L, beta):
    s = oracle.lut_init(L, 7)
    assert abs(int(s.sum())) < 5 * L                            # +-1 with probability 1/2
    tl = oracle.observables(s)
    for t in range(6):
        tl = oracle.lut_sweep(s, beta, 7, t, tl)
        assert tl == oracle.observables(s)


def test_init_mapping_reading_L5():
    """Reading L5, site by site with the KAT-pinned Philox and Python integers: colour c = (x + y) & 1,
    compact index k = x >> 1, word w = y * ceil(L / 128) + (k >> 6) of colour c is (out[0] | out[1] << 32) of
    Philox(ctr = (w_lo, w_hi, 0, 2 + c), key = seed); bit k & 63 set <-> spin +1.  Covers both colours, both
    32-bit halves of a word, several words per row, the last row, and a patch that wraps."""
    seed = 0x0123456789ABCDEF
    key = [seed & 0xFFFFFFFF, seed >> 32]
    for L in (256, 640, 96):
        s = oracle.lut_init(L, seed)
        Wr = (L // 2 + 63) // 64
        sites = [(0, 0), (1, 0), (0, 1), (63, 0), (64, 0), (65, 1), (127, 5), (128, 5), (129, 6), (L - 1, L - 1),
                 (L - 2, L - 1), (L - 1, 0), (L // 2 + 1, L // 3)]
        for x, y in [(x, y) for x, y in sites if x < L and y < L]:
            c, k = (x + y) & 1, x >> 1
            w = y * Wr + (k >> 6)
            out = oracle.philox4x32_10([w & 0xFFFFFFFF, w >> 32, 0, 2 + c], key)
            bits = int(out[0]) | (int(out[1]) << 32)
            assert s[y, x] == (1 if (bits >> (k & 63)) & 1 else -1), (L, x, y)
        patch = oracle.lut_init_patch(L, seed, L - 3, L - 2, 7, 5)                     # wraps in x and y
        assert (patch == np.roll(s, (2, 3), axis=(0, 1))[:5, :7]).all()


def test_word_sweep_equals_per_site_patch_sweep():
    """The paper-order sweep (random words per 64 sites) and the per-site light-cone patch sweep are
    written independently; they must give the same spins where the patch is exact, including
    windows across the periodic wrap."""
    L, beta, seed, n = 128, wl.BETA_C / 0.9, 11, 5
    s = oracle.lut_init(L, seed)
    for t in range(n):
        oracle.lut_sweep(s, beta, seed, t)
    for (x0, y0) in [(40, 40), (-10, 50), (70, -12), (L - 16, L - 16)]:
        got = oracle.lut_window_after(L, beta, seed, n, x0, y0, 32, 32)
        ys = np.arange(y0, y0 + 32) % L
        xs = np.arange(x0, x0 + 32) % L
        assert (got == s[np.ix_(ys, xs)]).all(), (x0, y0)


def test_flip_rule_limits():
    """beta = 0: every spin flips in every half sweep; beta large: only eq <= 2 sites flip."""
    L = 64
    s = oracle.lut_init(L, 2)
    a = s.copy()
    oracle.lut_sweep(s, 0.0, 2, 0)
    assert (s == -a).all()
    s = np.ones((L, L), np.int8)
    oracle.lut_sweep(s, 40.0, 2, 0)
    assert (s == 1).all()                                       # all neighbours equal: needs exp8, never set
    s = np.ones((L, L), np.int8)
    s[::2, ::2] = -1                                            # isolated minority spins have eq = 0: flip back
    oracle.lut_sweep(s, 40.0, 2, 0)
    assert (s == 1).all()


def _lut_trace(s, beta, seed, n):
    tr = np.zeros(3 * n, dtype=np.int64)
    tl = np.asarray(oracle.observables(s), dtype=np.int64)
    oracle.lib().orc_lut_run(C.c_int64(s.shape[0]), C.c_double(beta), C.c_uint64(seed), C.c_uint32(0), C.c_int64(n),
                             s.ctypes.data_as(C.POINTER(C.c_int8)), tl.ctypes.data_as(C.POINTER(C.c_int64)),
                             tr.ctypes.data_as(C.POINTER(C.c_int64)))
    return tr.reshape(-1, 3)


@pytest.mark.parametrize("tau", [1.0, 0.9])
def test_lut_4x4_exact_enumeration(golden_dir, tau):
    """Long-run <E>, <|M|> of the LUT chain on the 4x4 lattice vs the exact partition function."""
    beta = wl.BETA_C / tau
    ex = _enumerate(4, (-1, 1), beta, 0.0)
    rows = []
    for seed in range(1, 513):
        s = oracle.lut_init(4, seed)
        tr = _lut_trace(s, beta, seed, 100 + 300)[100:]
        rows.append([(-tr[:, 0]).mean(), np.abs(tr[:, 1]).mean()])
    rows = np.asarray(rows)
    mean, se = rows.mean(axis=0), rows.std(axis=0, ddof=1) / math.sqrt(len(rows))
    assert abs(mean[0] - ex[0]) < 5 * se[0] and abs(mean[1] - ex[2]) < 5 * se[1], (mean, se, ex)
    assert se[0] < 0.08


def test_lut_onsager_ordered_phase():
    """L = 128 cold start at 0.9 Tc: u and <|m|> against Onsager / Yang (finite-size shift < 2e-3)."""
    L, beta = 128, wl.BETA_C / 0.9
    s = np.ones((L, L), np.int8)
    tr = _lut_trace(s, beta, 4, 300 + 1200)[300:]
    u, se_u = _blocked(-tr[:, 0] / (L * L))
    m, se_m = _blocked(np.abs(tr[:, 1]) / (L * L))
    assert abs(u - _onsager_u(beta)) < 5 * se_u + 2e-3, (u, se_u, _onsager_u(beta))
    assert abs(m - _onsager_m0(beta)) < 5 * se_m + 2e-3, (m, se_m, _onsager_m0(beta))
