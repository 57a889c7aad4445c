"""ctypes binding of include/ising.h.  Same names as the C ABI; no arithmetic of
the method lives here.  torch is used for device memory and streams only."""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np

ISING, BLUME_CAPEL, ISING_LUT, BLUME_CAPEL_2BIT = 0, 1, 2, 3
_HERE = os.path.dirname(os.path.abspath(__file__))
# ISING_B200_LIB: another build of the same library (build.py's `out` / `defines`), for A/B timing of kernel variants
_LIB_PATH = os.environ.get("ISING_B200_LIB") or os.path.join(_HERE, "libising_b200.so")
_lib = None

EXPORTS = [
    "ising_workspace_bytes", "ising_create", "ising_sweep", "ising_observables", "ising_correlation",
    "ising_correlation_protocol", "ising_correlation_list", "ising_schwinger_dyson", "ising_read_lattice",
    "ising_read_window", "ising_write_lattice", "ising_read_packed", "ising_write_packed",
    "ising_set_sweeps_done", "ising_thresholds", "ising_set_launch", "ising_set_variant", "ising_bench_pipes", "ising_set_corr_path", "ising_set_tally", "ising_tally", "ising_time_grid", "ising_run_schedule",
    "ising_launch_count", "ising_sync", "ising_destroy", "ising_last_error", "ising_bench_philox_only",
    "ising_bench_copy", "ising_debug_philox", "ising_protocol_distances", "ising_threshold_table",
    "ising_run_protocol_schedule", "ising_create_slabs", "ising_slab_count", "ising_slab_info",
    "ising_write_bits", "ising_read_bits", "ising_slab_partition",
    "ising_set_sweep_mode", "ising_create_part", "ising_part_export", "ising_part_attach", "ising_sweep_phase",
    "ising_correlation_noalloc",
]


class IsingError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"ising error {code}: {msg}")
        self.code = code


class _Obs(C.Structure):
    _fields_ = [("bond_sum", C.c_int64), ("M", C.c_int64), ("Q", C.c_int64), ("n_sites", C.c_int64),
                ("sweeps_done", C.c_uint64), ("E", C.c_double), ("e_per_site", C.c_double),
                ("m_per_site", C.c_double), ("zero_density", C.c_double)]


@dataclass(frozen=True)
class Observables:
    bond_sum: int
    M: int
    Q: int
    n_sites: int
    sweeps_done: int
    E: float
    e_per_site: float
    m_per_site: float
    zero_density: float


def lib_path() -> str:
    return _LIB_PATH


def load_library():
    """dlopen the CUDA library; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise IsingError(-3, f"{_LIB_PATH} is missing: run `python -m paper_2502_18624_b200.build` "
                             "(or __graft_entry__.build()); there is no CPU fallback")
    lib = C.CDLL(_LIB_PATH)
    i64, u64, vp, dbl = C.c_int64, C.c_uint64, C.c_void_p, C.c_double
    lib.ising_workspace_bytes.restype = C.c_size_t
    lib.ising_workspace_bytes.argtypes = [C.c_int, i64]
    lib.ising_create.argtypes = [C.c_int, i64, dbl, dbl, u64, vp, C.c_size_t, vp, C.POINTER(vp)]
    lib.ising_create_slabs.argtypes = [C.c_int, i64, dbl, dbl, u64, C.c_int, vp, vp, vp, C.POINTER(vp)]
    lib.ising_slab_count.argtypes = [vp]
    lib.ising_slab_info.argtypes = [vp, C.c_int, vp, vp, vp]
    lib.ising_create_part.argtypes = [C.c_int, i64, dbl, dbl, u64, i64, i64, vp, C.POINTER(vp)]
    lib.ising_part_export.argtypes = [vp, vp]
    lib.ising_part_attach.argtypes = [vp, vp, i64, vp, i64]
    lib.ising_sweep_phase.argtypes = [vp, C.c_int]
    lib.ising_sweep.argtypes = [vp, i64]
    lib.ising_observables.argtypes = [vp, C.POINTER(_Obs)]
    lib.ising_correlation.argtypes = [vp, i64, vp, vp]
    lib.ising_correlation_noalloc.argtypes = [vp, i64, vp, vp]
    lib.ising_correlation_protocol.argtypes = [vp, i64, vp, vp, vp, vp, C.POINTER(i64)]
    lib.ising_correlation_list.argtypes = [vp, i64, i64, vp, vp, vp]
    lib.ising_schwinger_dyson.argtypes = [vp, vp, C.POINTER(dbl)]
    lib.ising_read_lattice.argtypes = [vp, i64, i64, vp]
    lib.ising_read_window.argtypes = [vp, i64, i64, i64, i64, vp]
    lib.ising_write_lattice.argtypes = [vp, i64, i64, vp]
    lib.ising_read_packed.argtypes = [vp, C.c_int, i64, i64, vp]
    lib.ising_write_packed.argtypes = [vp, C.c_int, i64, i64, vp]
    lib.ising_write_bits.argtypes = [vp, C.c_int, i64, i64, vp]
    lib.ising_read_bits.argtypes = [vp, C.c_int, i64, i64, vp]
    lib.ising_set_sweeps_done.argtypes = [vp, u64]
    lib.ising_thresholds.argtypes = [vp, vp, C.c_int, C.POINTER(C.c_int)]
    lib.ising_set_launch.argtypes = [vp, C.c_int, C.c_int]
    lib.ising_set_variant.argtypes = [vp, C.c_int]
    lib.ising_launch_count.restype = i64
    lib.ising_launch_count.argtypes = [vp]
    lib.ising_sync.argtypes = [vp]
    lib.ising_destroy.argtypes = [vp]
    lib.ising_last_error.restype = C.c_char_p
    lib.ising_bench_philox_only.argtypes = [vp, C.c_int]
    lib.ising_bench_copy.argtypes = [vp, C.c_int]
    lib.ising_debug_philox.argtypes = [i64, vp, vp, vp, C.c_int]
    lib.ising_time_grid.argtypes = [u64, vp, i64, vp]
    lib.ising_protocol_distances.argtypes = [i64, u64, i64, vp, vp, vp]
    lib.ising_threshold_table.argtypes = [C.c_int, dbl, dbl, vp, C.c_int, vp]
    lib.ising_run_protocol_schedule.argtypes = [vp, i64, vp, i64, vp, vp, vp, vp, vp, vp]
    lib.ising_run_schedule.argtypes = [vp, i64, vp, vp]
    lib.ising_set_tally.argtypes = [vp, C.c_int]
    lib.ising_tally.argtypes = [vp, vp]
    lib.ising_set_corr_path.argtypes = [vp, C.c_int]
    lib.ising_bench_pipes.argtypes = [dbl, vp, C.c_int, vp]
    _lib = lib
    return lib


def _check(rc: int):
    if rc != 0:
        raise IsingError(rc, load_library().ising_last_error().decode())


def workspace_bytes(model: int, L: int) -> int:
    return int(load_library().ising_workspace_bytes(model, L))


PIPE_PROBES = ["IMAD.WIDE", "LOP3", "IMAD", "IMAD.WIDE+LOP3", "IMAD.WIDE+2LOP3", "IADD3(carry)+IMAD.X",
               "IMAD.WIDE+IMAD", "POPC+IADD"]


def bench_pipes(sm_mhz: float = 0.0) -> dict:
    """Issue rates (warp-instructions per SM sub-partition per clock) of the integer-pipe probes."""
    lib = load_library()
    rates = np.zeros(len(PIPE_PROBES), dtype=np.float64)
    n = C.c_int(0)
    _check(lib.ising_bench_pipes(float(sm_mhz), rates.ctypes.data, len(rates), C.addressof(n)))
    return {k: float(v) for k, v in zip(PIPE_PROBES, rates)}


def time_grid(tmax: int) -> np.ndarray:
    """The paper's measurement times up to tmax.  Host arithmetic: no GPU needed."""
    lib = load_library()
    n = C.c_int64(0)
    _check(lib.ising_time_grid(int(tmax), None, 0, C.addressof(n)))
    out = np.zeros(n.value, dtype=np.uint64)
    _check(lib.ising_time_grid(int(tmax), out.ctypes.data, len(out), C.addressof(n)))
    return out


def protocol_distances(L: int, t: int):
    """(r, stride) of the Sec. 3.3 protocol at time t.  Host arithmetic: no GPU needed."""
    lib = load_library()
    n = C.c_int64(0)
    _check(lib.ising_protocol_distances(int(L), int(t), 0, None, None, C.addressof(n)))
    r = np.zeros(n.value, dtype=np.int64)
    st = np.zeros(n.value, dtype=np.int64)
    _check(lib.ising_protocol_distances(int(L), int(t), len(r), r.ctypes.data, st.ctypes.data, C.addressof(n)))
    return r, st


def slab_partition(L: int, n_slabs: int) -> np.ndarray:
    """Default slab heights of ising_create_slabs.  Host arithmetic: no GPU needed."""
    lib = load_library()
    lib.ising_slab_partition.argtypes = [C.c_int64, C.c_int, C.c_void_p]
    rows = np.zeros(n_slabs, dtype=np.int64)
    _check(lib.ising_slab_partition(int(L), int(n_slabs), rows.ctypes.data))
    return rows


def threshold_table(model: int, beta: float, D: float = 0.0) -> np.ndarray:
    """The integer acceptance table of (model, beta, D) (A1; the 16-entry cumulative table for the 1-bit
    model).  Host arithmetic: no GPU needed."""
    lib = load_library()
    out = np.zeros(64, dtype=np.uint64)
    n = C.c_int(0)
    _check(lib.ising_threshold_table(int(model), float(beta), float(D), out.ctypes.data, 64, C.addressof(n)))
    return out[: n.value].copy()


def debug_philox(ctr: np.ndarray, key: np.ndarray, with_curand: bool = False) -> np.ndarray:
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32).reshape(-1, 4)
    key = np.ascontiguousarray(key, dtype=np.uint32).reshape(-1, 2)
    out = np.zeros_like(ctr)
    _check(load_library().ising_debug_philox(len(ctr), ctr.ctypes.data, key.ctypes.data, out.ctypes.data,
                                             int(with_curand)))
    return out


class IsingSim:
    """One lattice on one GPU.  Methods mirror the C ABI one to one."""

    def __init__(self, model: int, L: int, beta: float, D: float = 0.0, seed: int = 1, device="cuda:0",
                 use_torch_memory: bool = True, slabs=None, slab_devices=None, part=None):
        """slabs: None = one lattice (ising_create); an int S or a list of row counts = ising_create_slabs
        (row slabs in allocations of their own, optionally on the CUDA device indices slab_devices).
        part = (y0, rows): this handle is ONE slab of the lattice (ising_create_part; one process per GPU)."""
        import torch
        if not torch.cuda.is_available():
            raise IsingError(-3, "no CUDA device: the engine has no CPU fallback")
        self._lib = load_library()
        self._torch = torch
        self.device = torch.device(device)
        self.model, self.L, self.beta, self.D, self.seed = model, L, float(beta), float(D), seed
        nbytes = workspace_bytes(model, L)
        if nbytes == 0:
            raise IsingError(-1, "invalid (model, L): L must be a multiple of 64, >= 64 (256 for the LUT model)")
        self._h = C.c_void_p()
        with torch.cuda.device(self.device):
            self._stream = torch.cuda.current_stream(self.device)
            if part is not None:
                self._buf = None
                _check(self._lib.ising_create_part(model, L, beta, D, seed, int(part[0]), int(part[1]),
                                                   self._stream.cuda_stream, C.byref(self._h)))
                return
            if slabs is not None:
                rows = None if isinstance(slabs, int) else np.ascontiguousarray(slabs, dtype=np.int64)
                n = slabs if rows is None else len(rows)
                devs = None if slab_devices is None else np.ascontiguousarray(slab_devices, dtype=np.int32)
                self._buf = None
                _check(self._lib.ising_create_slabs(model, L, beta, D, seed, n, None if rows is None else rows.ctypes.data,
                                                    None if devs is None else devs.ctypes.data,
                                                    self._stream.cuda_stream, C.byref(self._h)))
                return
            if use_torch_memory:
                self._buf = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
                ptr, size = self._buf.data_ptr(), nbytes
            else:
                self._buf, ptr, size = None, None, 0
            _check(self._lib.ising_create(model, L, beta, D, seed, ptr, size, self._stream.cuda_stream,
                                          C.byref(self._h)))

    # -- lifetime
    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            self._lib.ising_destroy(self._h)
            self._h = None
            self._buf = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def slab_layout(self):
        """[(y0, rows, device)] of the row slabs (one entry for an unsharded lattice)."""
        out = []
        for k in range(self._lib.ising_slab_count(self._h)):
            y0, rows, dev = C.c_int64(0), C.c_int64(0), C.c_int(0)
            _check(self._lib.ising_slab_info(self._h, k, C.addressof(y0), C.addressof(rows), C.addressof(dev)))
            out.append((y0.value, rows.value, dev.value))
        return out

    def part_export(self) -> bytes:
        """The CUDA IPC handle of this part's allocation (64 bytes), for the neighbouring ranks."""
        buf = C.create_string_buffer(64)
        _check(self._lib.ising_part_export(self._h, buf))
        return buf.raw

    def part_attach(self, ipc_above: bytes, rows_above: int, ipc_below: bytes, rows_below: int):
        _check(self._lib.ising_part_attach(self._h, C.c_char_p(ipc_above), rows_above, C.c_char_p(ipc_below), rows_below))

    def sweep_phase(self, colour: int):
        _check(self._lib.ising_sweep_phase(self._h, colour))

    # -- the path
    def sweep(self, n: int = 1):
        _check(self._lib.ising_sweep(self._h, n))

    def sync(self):
        _check(self._lib.ising_sync(self._h))

    def observables(self) -> Observables:
        o = _Obs()
        _check(self._lib.ising_observables(self._h, C.byref(o)))
        return Observables(*(getattr(o, f[0]) for f in _Obs._fields_))

    def set_tally(self, on: bool = True):
        _check(self._lib.ising_set_tally(self._h, int(on)))

    def tally(self) -> Observables:
        o = _Obs()
        _check(self._lib.ising_tally(self._h, C.byref(o)))
        return Observables(*(getattr(o, f[0]) for f in _Obs._fields_))

    def run_schedule(self, times):
        """Sweep to every time of the ascending list and record the observables there (one native call)."""
        times = np.ascontiguousarray(times, dtype=np.uint64)
        arr = (_Obs * len(times))()
        _check(self._lib.ising_run_schedule(self._h, len(times), times.ctypes.data, C.addressof(arr)))
        return [Observables(*(getattr(o, f[0]) for f in _Obs._fields_)) for o in arr]

    def correlation(self, rmax: int):
        sx = np.zeros(rmax, dtype=np.int64)
        sy = np.zeros(rmax, dtype=np.int64)
        _check(self._lib.ising_correlation(self._h, rmax, sx.ctypes.data, sy.ctypes.data))
        return sx, sy

    def correlation_noalloc(self, rmax: int):
        """ising_correlation on a static device scratch array: no allocation, L <= 1024 (ISING_NOALLOC_MAX_L)."""
        sx = np.zeros(rmax, dtype=np.int64)
        sy = np.zeros(rmax, dtype=np.int64)
        _check(self._lib.ising_correlation_noalloc(self._h, rmax, sx.ctypes.data, sy.ctypes.data))
        return sx, sy

    def correlation_list(self, stride: int, r):
        r = np.ascontiguousarray(r, dtype=np.int64)
        sx = np.zeros(len(r), dtype=np.int64)
        sy = np.zeros(len(r), dtype=np.int64)
        _check(self._lib.ising_correlation_list(self._h, stride, len(r), r.ctypes.data, sx.ctypes.data,
                                                sy.ctypes.data))
        return sx, sy

    def run_protocol_schedule(self, times, with_observables: bool = True):
        """Sweep to every time of the ascending list and run the Sec. 3.3 protocol there (one native call).
        Returns a list of (r, sx, sy, n_src) per time and the list of observables (or None)."""
        times = np.ascontiguousarray(times, dtype=np.uint64)
        n = C.c_int64(0)
        _check(self._lib.ising_protocol_distances(self.L, int(times[-1]) if len(times) else 0, 0, None, None, C.byref(n)))
        cap = n.value
        arrs = [np.zeros((len(times), cap), dtype=np.int64) for _ in range(4)]
        counts = np.zeros(len(times), dtype=np.int64)
        obs = (_Obs * len(times))() if with_observables else None
        _check(self._lib.ising_run_protocol_schedule(self._h, len(times), times.ctypes.data, cap,
                                                     *(a.ctypes.data for a in arrs), counts.ctypes.data,
                                                     C.addressof(obs) if obs is not None else None))
        rows = [tuple(a[i, : counts[i]].copy() for a in arrs) for i in range(len(times))]
        o = [Observables(*(getattr(x, f[0]) for f in _Obs._fields_)) for x in obs] if obs is not None else None
        return rows, o

    def correlation_protocol(self):
        n = C.c_int64(0)
        _check(self._lib.ising_correlation_protocol(self._h, 0, None, None, None, None, C.byref(n)))
        cap = n.value
        arrs = [np.zeros(cap, dtype=np.int64) for _ in range(4)]
        _check(self._lib.ising_correlation_protocol(self._h, cap, *(a.ctypes.data for a in arrs), C.byref(n)))
        return tuple(arrs)

    def schwinger_dyson(self):
        hist = np.zeros(9, dtype=np.int64)
        v = C.c_double(0.0)
        _check(self._lib.ising_schwinger_dyson(self._h, hist.ctypes.data, C.byref(v)))
        return v.value, hist

    def read_lattice(self, y0: int = 0, ny: int | None = None) -> np.ndarray:
        ny = self.L - y0 if ny is None else ny
        out = np.empty((ny, self.L), dtype=np.int8)
        _check(self._lib.ising_read_lattice(self._h, y0, ny, out.ctypes.data))
        return out

    def read_window(self, x0: int, y0: int, w: int, h: int) -> np.ndarray:
        out = np.empty((h, w), dtype=np.int8)
        _check(self._lib.ising_read_window(self._h, x0, y0, w, h, out.ctypes.data))
        return out

    def write_lattice(self, spins: np.ndarray, y0: int = 0):
        spins = np.ascontiguousarray(spins, dtype=np.int8)
        assert spins.ndim == 2 and spins.shape[1] == self.L
        _check(self._lib.ising_write_lattice(self._h, y0, spins.shape[0], spins.ctypes.data))

    def read_packed(self, colour: int, word0: int = 0, nwords: int | None = None, out=None):
        total = self.L * (self.L // {ISING_LUT: 128, BLUME_CAPEL_2BIT: 64}.get(self.model, 32))
        nwords = total - word0 if nwords is None else nwords
        if out is None:
            out = np.empty(nwords, dtype=np.uint64)
            ptr = out.ctypes.data
        else:
            ptr = out.data_ptr() if hasattr(out, "data_ptr") else out.ctypes.data
        _check(self._lib.ising_read_packed(self._h, colour, word0, nwords, ptr))
        return out

    def write_packed(self, colour: int, words, word0: int = 0, nwords: int | None = None):
        if hasattr(words, "data_ptr"):
            ptr, n = words.data_ptr(), words.numel() * words.element_size() // 8
        else:
            words = np.ascontiguousarray(words, dtype=np.uint64)
            ptr, n = words.ctypes.data, len(words)
        _check(self._lib.ising_write_packed(self._h, colour, word0, n if nwords is None else nwords, ptr))

    def bits_row_words(self) -> int:
        """uint64 words per colour row of the compact transport format (ising_write_bits / ising_read_bits)."""
        return self.L // 64 if self.model in (BLUME_CAPEL, BLUME_CAPEL_2BIT) else self.L // 128

    def read_bits(self, colour: int, row0: int = 0, nrows: int | None = None, out=None):
        nrows = self.L - row0 if nrows is None else nrows
        if out is None:
            out = np.empty(nrows * self.bits_row_words(), dtype=np.uint64)
            ptr = out.ctypes.data
        else:
            ptr = out.data_ptr() if hasattr(out, "data_ptr") else out.ctypes.data
        _check(self._lib.ising_read_bits(self._h, colour, row0, nrows, ptr))
        return out

    def write_bits(self, colour: int, words, row0: int = 0, nrows: int | None = None):
        if hasattr(words, "data_ptr"):
            ptr, n = words.data_ptr(), words.numel() * words.element_size() // 8
        else:
            words = np.ascontiguousarray(words, dtype=np.uint64)
            ptr, n = words.ctypes.data, len(words)
        nrows = n // self.bits_row_words() if nrows is None else nrows
        _check(self._lib.ising_write_bits(self._h, colour, row0, nrows, ptr))

    def set_sweeps_done(self, t: int):
        _check(self._lib.ising_set_sweeps_done(self._h, t))

    def thresholds(self) -> np.ndarray:
        out = np.zeros(64, dtype=np.uint64)
        n = C.c_int(0)
        _check(self._lib.ising_thresholds(self._h, out.ctypes.data, 64, C.byref(n)))
        return out[: n.value].copy()

    def set_launch(self, rows_per_thread: int = 0, block_threads: int = 0):
        _check(self._lib.ising_set_launch(self._h, rows_per_thread, block_threads))

    def set_variant(self, variant: int):
        _check(self._lib.ising_set_variant(self._h, variant))

    def set_sweep_mode(self, mode: int):
        self._lib.ising_set_sweep_mode.argtypes = [C.c_void_p, C.c_int]
        _check(self._lib.ising_set_sweep_mode(self._h, mode))

    def set_corr_path(self, path: int):
        _check(self._lib.ising_set_corr_path(self._h, path))

    def launch_count(self) -> int:
        return int(self._lib.ising_launch_count(self._h))

    def bench_philox_only(self, n: int):
        _check(self._lib.ising_bench_philox_only(self._h, n))

    def bench_copy(self, n: int):
        _check(self._lib.ising_bench_copy(self._h, n))
