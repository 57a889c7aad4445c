"""-m "not gpu": the C-ABI library loads and exports every symbol include/ising.h
declares (no compute calls), and host-only argument checks."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2502_18624_b200 import build as b
    b.build()
    import paper_2502_18624_b200 as eng
    return eng.load_library()


def _declared():
    src = open(os.path.join(ROOT, "include", "ising.h")).read() + open(os.path.join(ROOT, "include", "ising_bench.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ising_[a-z_0-9]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    names = _declared()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), n
    from paper_2502_18624_b200.binding import EXPORTS
    assert sorted(EXPORTS) == names


def test_workspace_bytes_and_validation(lib):
    assert lib.ising_workspace_bytes(0, 256) == 256 * 256 // 2 + 4096
    assert lib.ising_workspace_bytes(1, 1 << 18) == (1 << 36) // 2 + 4096
    for bad_L in (0, 32, 100, 65, -64, (1 << 20) + 64):
        assert lib.ising_workspace_bytes(0, bad_L) == 0
    assert lib.ising_workspace_bytes(2, 256) == 256 * 256 // 8 + 4096      # LUT model: one bit per spin
    assert lib.ising_workspace_bytes(3, 256) == 256 * 256 // 4 + 4096      # Blume-Capel at 2 bits per spin
    assert lib.ising_workspace_bytes(2, 192) == 0 and lib.ising_workspace_bytes(4, 256) == 0


def test_null_handle_errors(lib):
    assert lib.ising_sweep(None, 1) == -1
    assert b"NULL" in lib.ising_last_error()
    assert lib.ising_observables(None, None) == -1
    assert lib.ising_destroy(None) == 0
    out = C.c_void_p()
    assert lib.ising_create(0, 100, 0.4, 0.0, 1, None, 0, None, C.byref(out)) == -1      # bad L, before any CUDA call
    assert lib.ising_create(0, 64, -1.0, 0.0, 1, None, 0, None, C.byref(out)) == -1
    assert lib.ising_create(0, 64, 0.4, 0.0, 1, None, 0, None, None) == -1
    assert lib.ising_create(2, 192, 0.4, 0.0, 1, None, 0, None, C.byref(out)) == -1      # LUT model: L % 256
    lib.ising_create_slabs.argtypes = [C.c_int, C.c_int64, C.c_double, C.c_double, C.c_uint64, C.c_int, C.c_void_p, C.c_void_p,
                                       C.c_void_p, C.POINTER(C.c_void_p)]
    assert lib.ising_create_slabs(0, 100, 0.4, 0.0, 1, 2, None, None, None, C.byref(out)) == -1   # bad L, before any CUDA call
    assert lib.ising_create_slabs(0, 256, 0.4, 0.0, 1, 0, None, None, None, C.byref(out)) == -1   # no slab
    assert lib.ising_create_slabs(0, 256, 0.4, 0.0, 1, 2, None, None, None, None) == -1
    assert lib.ising_slab_count(None) == 0
    for fn, args in [(lib.ising_set_tally, (None, 1)), (lib.ising_tally, (None, None)), (lib.ising_set_corr_path, (None, 1)),
                     (lib.ising_run_schedule, (None, 0, None, None)), (lib.ising_correlation, (None, 1, None, None)),
                     (lib.ising_set_variant, (None, 0)), (lib.ising_set_launch, (None, 0, 0)),
                     (lib.ising_time_grid, (10, None, 0, None)), (lib.ising_write_bits, (None, 0, 0, 1, None)),
                     (lib.ising_read_bits, (None, 0, 0, 1, None)), (lib.ising_set_sweep_mode, (None, 0)),
                     (lib.ising_run_protocol_schedule, (None, 0, None, 0, None, None, None, None, None, None)),
                     (lib.ising_slab_info, (None, 0, None, None, None)), (lib.ising_slab_partition, (256, 2, None)),
                     (lib.ising_protocol_distances, (256, 1, 0, None, None, None)),
                     (lib.ising_threshold_table, (0, 0.4, 0.0, None, 0, None))]:
        assert fn(*args) == -1, fn.__name__
        assert len(lib.ising_last_error()) > 0


def test_no_cpu_fallback():
    """The product path must fail loudly without a GPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import paper_2502_18624_b200 as eng
    with pytest.raises(eng.IsingError):
        eng.IsingSim(0, 64, 0.4)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2502_18624_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "ising_oracle" not in txt, f
    orc = open(os.path.join(ROOT, "oracle", "__init__.py")).read() + open(os.path.join(ROOT, "oracle", "ising_oracle.c")).read()
    assert "import paper_2502_18624_b200" not in orc and "ising.h" not in orc


def test_time_grid_host_logic_matches_oracle(lib):
    """A11 host logic through the C ABI (no GPU needed): the paper's measurement times."""
    import ctypes as C
    import numpy as np
    import oracle
    lib.ising_time_grid.argtypes = [C.c_uint64, C.c_void_p, C.c_int64, C.c_void_p]
    for tmax in (1, 12, 2000, 524288):
        n = C.c_int64(0)
        assert lib.ising_time_grid(tmax, None, 0, C.addressof(n)) == 0          # size query
        out = np.zeros(n.value, dtype=np.uint64)
        assert lib.ising_time_grid(tmax, out.ctypes.data, len(out), C.addressof(n)) == 0
        assert (out == oracle.time_grid(tmax)).all()
    assert n.value > 100 and out[-1] == 524288
