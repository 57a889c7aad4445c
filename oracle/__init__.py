"""CPU oracle for the checkerboard Metropolis path -- TEST INFRASTRUCTURE ONLY.

Thin ctypes wrapper over ``oracle/ising_oracle.c`` (plain C, int8 per spin,
fp64 where floating point appears).  Only ``tests/``, ``__graft_entry__.smoke()``
and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this
package.  It imports nothing from ``paper_2502_18624_b200`` and shares no code
with the CUDA path.  See the header of ``ising_oracle.c`` for citations and
``DESIGN.md`` for the readings of the paper.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

ISING, BLUME_CAPEL = 0, 1
_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ising_oracle.c")
_LIB = os.path.join(_HERE, "libising_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, OpenMP, no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
             "-o", _LIB, _SRC, "-lm"])
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_draw.restype = C.c_uint32
        _lib.orc_draw.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32]
        _lib.orc_schwinger_dyson.restype = C.c_double
        _lib.orc_protocol_rc.restype = C.c_int64
        _lib.orc_protocol_list.restype = C.c_int64
        _lib.orc_time_grid.restype = C.c_int64
    return _lib


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(_p(c, C.c_uint32), _p(k, C.c_uint32), _p(out, C.c_uint32))
    return out


def draw(seed: int, n: int, t: int, tag: int) -> int:
    return int(lib().orc_draw(seed, n, t, tag))


def thresholds(model: int, beta: float, D: float = 0.0) -> np.ndarray:
    out = np.zeros(54, dtype=np.uint64)
    n = lib().orc_thresholds(C.c_int(model), C.c_double(beta), C.c_double(D), _p(out, C.c_uint64))
    return out[:n].copy()


def init(model: int, L: int, seed: int) -> np.ndarray:
    s = np.zeros((L, L), dtype=np.int8)
    lib().orc_init(C.c_int(model), C.c_int64(L), C.c_uint64(seed), _p(s, C.c_int8))
    return s


def init_patch(model, L, seed, x0, y0, w, h) -> np.ndarray:
    s = np.zeros((h, w), dtype=np.int8)
    lib().orc_init_patch(C.c_int(model), C.c_int64(L), C.c_uint64(seed), C.c_int64(x0),
                         C.c_int64(y0), C.c_int64(w), C.c_int64(h), _p(s, C.c_int8))
    return s


def observables(s: np.ndarray):
    """(B, M, Q) by full recompute."""
    s = np.ascontiguousarray(s, dtype=np.int8)
    out = np.zeros(3, dtype=np.int64)
    lib().orc_observables(C.c_int64(s.shape[0]), _p(s, C.c_int8), _p(out, C.c_int64))
    return int(out[0]), int(out[1]), int(out[2])


def observables_rows(L: int, band: np.ndarray):
    """(B, M, Q) of the first ny rows of ``band`` ((ny + 1) x L: the last row is only the lower neighbour)."""
    band = np.ascontiguousarray(band, dtype=np.int8)
    assert band.ndim == 2 and band.shape[1] == L and band.shape[0] >= 2
    out = np.zeros(3, dtype=np.int64)
    lib().orc_observables_rows(C.c_int64(L), C.c_int64(band.shape[0] - 1), _p(band, C.c_int8), _p(out, C.c_int64))
    return int(out[0]), int(out[1]), int(out[2])


def sd_hist_rows(L: int, band: np.ndarray) -> np.ndarray:
    """Schwinger-Dyson histogram of the inner rows of ``band`` ((ny + 2) x L: first and last row are halos)."""
    band = np.ascontiguousarray(band, dtype=np.int8)
    assert band.ndim == 2 and band.shape[1] == L and band.shape[0] >= 3
    hist = np.zeros(9, dtype=np.int64)
    lib().orc_sd_hist_rows(C.c_int64(L), C.c_int64(band.shape[0] - 2), _p(band, C.c_int8), _p(hist, C.c_int64))
    return hist


def normalised(model: int, L: int, D: float, bmq):
    """(E, E/N, M/N, zero density) in double from the integers."""
    b = np.asarray(bmq, dtype=np.int64).copy()
    out = np.zeros(4, dtype=np.float64)
    lib().orc_normalised(C.c_int(model), C.c_int64(L), C.c_double(D), _p(b, C.c_int64),
                         _p(out, C.c_double))
    return tuple(float(v) for v in out)


def sweep(model, s: np.ndarray, beta, D, seed, t, tallies=None):
    """One full sweep number ``t`` in place; returns the updated (B, M, Q)."""
    assert s.dtype == np.int8 and s.flags.c_contiguous and s.shape[0] == s.shape[1]
    tl = np.asarray(observables(s) if tallies is None else tallies, dtype=np.int64).copy()
    lib().orc_sweep(C.c_int(model), C.c_int64(s.shape[0]), C.c_double(beta), C.c_double(D),
                    C.c_uint64(seed), C.c_uint32(t), _p(s, C.c_int8), _p(tl, C.c_int64))
    return int(tl[0]), int(tl[1]), int(tl[2])


def sweep_patch(model, L, s: np.ndarray, beta, D, seed, t, x0, y0):
    assert s.dtype == np.int8 and s.flags.c_contiguous
    h, w = s.shape
    lib().orc_sweep_patch(C.c_int(model), C.c_int64(L), C.c_double(beta), C.c_double(D),
                          C.c_uint64(seed), C.c_uint32(t), C.c_int64(x0), C.c_int64(y0),
                          C.c_int64(w), C.c_int64(h), _p(s, C.c_int8))


def window_after(model, L, beta, D, seed, n_sweeps, x0, y0, w, h) -> np.ndarray:
    """Exact state of the w x h window at (x0, y0) after ``n_sweeps`` sweeps from
    the seeded initial lattice, by simulating the light-cone patch grown by 2n
    sites on every side (one site of influence per half sweep)."""
    m = 2 * n_sweeps
    assert w + 2 * m <= L and h + 2 * m <= L, "light cone wraps onto itself"
    s = init_patch(model, L, seed, x0 - m, y0 - m, w + 2 * m, h + 2 * m)
    for t in range(n_sweeps):
        sweep_patch(model, L, s, beta, D, seed, t, x0 - m, y0 - m)
    return s[m:m + h, m:m + w].copy()


def schwinger_dyson(s: np.ndarray, beta: float):
    s = np.ascontiguousarray(s, dtype=np.int8)
    hist = np.zeros(9, dtype=np.int64)
    v = lib().orc_schwinger_dyson(C.c_int64(s.shape[0]), C.c_double(beta), _p(s, C.c_int8),
                                  _p(hist, C.c_int64))
    return float(v), hist


def correlation(s: np.ndarray, rmax: int):
    s = np.ascontiguousarray(s, dtype=np.int8)
    sx = np.zeros(rmax, dtype=np.int64)
    sy = np.zeros(rmax, dtype=np.int64)
    lib().orc_correlation(C.c_int64(s.shape[0]), _p(s, C.c_int8), C.c_int64(rmax),
                          _p(sx, C.c_int64), _p(sy, C.c_int64))
    return sx, sy


def correlation_list(s: np.ndarray, stride: int, r):
    s = np.ascontiguousarray(s, dtype=np.int8)
    r = np.ascontiguousarray(r, dtype=np.int64)
    sx = np.zeros(len(r), dtype=np.int64)
    sy = np.zeros(len(r), dtype=np.int64)
    lib().orc_correlation_list(C.c_int64(s.shape[0]), _p(s, C.c_int8), C.c_int64(stride),
                               C.c_int64(len(r)), _p(r, C.c_int64), _p(sx, C.c_int64),
                               _p(sy, C.c_int64))
    return sx, sy


def protocol_rc(L: int, t: int) -> int:
    return int(lib().orc_protocol_rc(C.c_int64(L), C.c_uint64(t)))


def protocol_list(L: int, t: int):
    """(r, stride) arrays of the Sec. 3.3 protocol at time t."""
    cap = 64 + protocol_rc(L, t) + 32 * 64
    r = np.zeros(cap, dtype=np.int64)
    st = np.zeros(cap, dtype=np.int64)
    n = lib().orc_protocol_list(C.c_int64(L), C.c_uint64(t), C.c_int64(cap), _p(r, C.c_int64),
                                _p(st, C.c_int64))
    return r[:n].copy(), st[:n].copy()


def correlation_protocol(s: np.ndarray, t: int):
    """(r, S_x, S_y, n_sources) per protocol distance."""
    L = s.shape[0]
    r, st = protocol_list(L, t)
    sx = np.zeros(len(r), dtype=np.int64)
    sy = np.zeros(len(r), dtype=np.int64)
    nsrc = np.zeros(len(r), dtype=np.int64)
    for stride in (1, 16):
        sel = st == stride
        if sel.any():
            sx[sel], sy[sel] = correlation_list(s, stride, r[sel])
            nsrc[sel] = ((L + stride - 1) // stride) ** 2
    return r, sx, sy, nsrc


def time_grid(tmax: int) -> np.ndarray:
    out = np.zeros(8 * 64, dtype=np.uint64)
    n = lib().orc_time_grid(C.c_uint64(tmax), C.c_int64(len(out)), _p(out, C.c_uint64))
    return out[:n].copy()


# ------------------------------------------------------------ NEXT-2: 1-bit LUT kernel ---
def lut_table(beta: float) -> np.ndarray:
    out = np.zeros(16, dtype=np.uint64)
    lib().orc_lut_table(C.c_double(beta), _p(out, C.c_uint64))
    return out


def lut_bits(table: np.ndarray, seed: int, w: int, t: int, tag: int, which: int) -> int:
    table = np.ascontiguousarray(table, dtype=np.uint64)
    lib().orc_lut_bits.restype = C.c_uint64
    return int(lib().orc_lut_bits(_p(table, C.c_uint64), C.c_uint64(seed), C.c_uint64(w), C.c_uint32(t),
                                  C.c_uint32(tag), C.c_int(which)))


def lut_init(L: int, seed: int) -> np.ndarray:
    s = np.zeros((L, L), dtype=np.int8)
    lib().orc_lut_init(C.c_int64(L), C.c_uint64(seed), _p(s, C.c_int8))
    return s


def lut_init_patch(L, seed, x0, y0, w, h) -> np.ndarray:
    s = np.zeros((h, w), dtype=np.int8)
    lib().orc_lut_init_patch(C.c_int64(L), C.c_uint64(seed), C.c_int64(x0), C.c_int64(y0), C.c_int64(w),
                             C.c_int64(h), _p(s, C.c_int8))
    return s


def lut_sweep(s: np.ndarray, beta, seed, t, tallies=None):
    """One sweep number ``t`` of the 1-bit LUT kernel in place; returns the updated (B, M, Q)."""
    assert s.dtype == np.int8 and s.flags.c_contiguous and s.shape[0] == s.shape[1]
    tl = np.asarray(observables(s) if tallies is None else tallies, dtype=np.int64).copy()
    lib().orc_lut_sweep(C.c_int64(s.shape[0]), C.c_double(beta), C.c_uint64(seed), C.c_uint32(t),
                        _p(s, C.c_int8), _p(tl, C.c_int64))
    return int(tl[0]), int(tl[1]), int(tl[2])


def lut_sweep_patch(L, s: np.ndarray, beta, seed, t, x0, y0):
    assert s.dtype == np.int8 and s.flags.c_contiguous
    h, w = s.shape
    lib().orc_lut_sweep_patch(C.c_int64(L), C.c_double(beta), C.c_uint64(seed), C.c_uint32(t),
                              C.c_int64(x0), C.c_int64(y0), C.c_int64(w), C.c_int64(h), _p(s, C.c_int8))


def lut_window_after(L, beta, seed, n_sweeps, x0, y0, w, h) -> np.ndarray:
    m = 2 * n_sweeps
    assert w + 2 * m <= L and h + 2 * m <= L, "light cone wraps onto itself"
    s = lut_init_patch(L, seed, x0 - m, y0 - m, w + 2 * m, h + 2 * m)
    for t in range(n_sweeps):
        lut_sweep_patch(L, s, beta, seed, t, x0 - m, y0 - m)
    return s[m:m + h, m:m + w].copy()


def set_threads(n: int) -> None:
    """OpenMP thread count of the sweeps (timing only)."""
    lib().orc_set_threads(C.c_int(n))


def threads() -> int:
    return int(lib().orc_threads())
