"""-m gpu, collected last: ising_correlation_noalloc -- the full-source pair sums on a static device scratch
array (no cudaMalloc; L <= ISING_NOALLOC_MAX_L = 1024) -- against the existing ising_correlation, which
allocates its scratch.  Integers, so the comparison is bit-exact like every other correlation test here.
Two calls in a row on a lattice that changes in between: the static array keeps the first call's planes and
accumulators, the second call must not see them.  Passes alone in a fresh process and after the other tests
(the array then holds whatever the last caller left)."""
import numpy as np
import pytest

import oracle
import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def eng():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2502_18624_b200 as e
    e.load_library()
    return e


@pytest.mark.parametrize("model,L,beta,D", [(wl.ISING, 1024, wl.BETA_C / 0.5, 0.0), (wl.BLUME_CAPEL, 320, 1 / 1.4, 1.0),
                                            (wl.ISING_LUT, 512, wl.BETA_C / 0.9, 0.0), (wl.BLUME_CAPEL_2BIT, 192, 1 / 1.4, 1.0)])
def test_noalloc_correlation_equals_the_allocating_path_twice_in_a_row(eng, model, L, beta, D):
    import torch
    with eng.IsingSim(model, L, beta, D, 11) as sim:
        sim.sweep(3)
        # first call: the whole band; nothing on the allocating path has run on this handle yet
        nx, ny = sim.correlation_noalloc(L // 2)
        sim.sweep(2)                                             # another lattice
        torch.cuda.synchronize()
        free_before, _ = torch.cuda.mem_get_info()
        mx, my = sim.correlation_noalloc(L // 2 - 5)             # second call in a row, narrower band: stale accumulators would show
        torch.cuda.synchronize()
        free_after, _ = torch.cuda.mem_get_info()
        assert free_after >= free_before                         # the call took no device memory
        ax, ay = sim.correlation(L // 2 - 5)                     # existing path (allocates planes and accumulators)
        assert (mx == ax).all() and (my == ay).all()
        lat = sim.read_lattice()
        if L <= 512:                                             # and the oracle's plain sums
            ox, oy = oracle.correlation(lat, L // 2 - 5)
            assert (mx == ox).all() and (my == oy).all()
        o = sim.observables()
        assert int(mx[0]) + int(my[0]) == o.bond_sum             # S_x(1) + S_y(1) = B
    with eng.IsingSim(model, L, beta, D, 11) as ref:             # the first call, against the existing path on a twin
        ref.sweep(3)
        rx, ry = ref.correlation(L // 2)
        assert (nx == rx).all() and (ny == ry).all()


def test_noalloc_rejects_what_the_static_array_cannot_hold(eng):
    with eng.IsingSim(wl.ISING, 2048, 0.4) as big:
        with pytest.raises(eng.IsingError) as err:
            big.correlation_noalloc(8)
        assert err.value.code == -1 and "ISING_NOALLOC_MAX_L" in str(err.value)
        sx, sy = big.correlation(8)                              # the handle stays usable
        assert len(sx) == 8
    with eng.IsingSim(wl.ISING, 256, 0.4) as sim:
        for bad in (0, 129):
            with pytest.raises(eng.IsingError):
                sim.correlation_noalloc(bad)
        a = sim.correlation_noalloc(128)
        b = sim.correlation(128)
        assert (a[0] == b[0]).all() and (a[1] == b[1]).all()
        c = sim.correlation_noalloc(1)                           # after the allocating path has run on the handle: its planes pointer is intact
        assert int(c[0][0]) == int(b[0][0]) and int(c[1][0]) == int(b[1][0])
        d = sim.correlation(128)
        assert (d[0] == b[0]).all() and (d[1] == b[1]).all()
