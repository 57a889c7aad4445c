"""Oracle-free physics checks of the CUDA path itself (-m gpu): the closed forms the paper's own
validation relies on -- Onsager's energy, Yang's spontaneous magnetisation and the
Schwinger-Dyson identity -- for the 4-bit and the 1-bit Ising kernels, and the Schwinger-Dyson identity for
Blume-Capel.  Long runs are cheap on the GPU: L = 512, thousands of sweeps, measured through the native
schedule runner and the fused tally."""
import math

import numpy as np
import pytest

import workloads as wl

from test_oracle_pins import _blocked, _onsager_m0, _onsager_u

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def eng():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2502_18624_b200 as e
    e.load_library()
    return e


@pytest.mark.parametrize("model", [wl.ISING, wl.ISING_LUT])
def test_onsager_ordered_phase_on_the_gpu(eng, model):
    """Cold start at 0.9 Tc, L = 512: u -> Onsager, <|m|> -> (1 - sinh^-4 2 beta)^(1/8); 5 standard errors
    (blocked) plus a finite-size allowance of 1e-3."""
    L, beta = 512, wl.BETA_C / 0.9
    with eng.IsingSim(model, L, beta, 0.0, 5) as sim:
        sim.write_lattice(np.ones((L, L), dtype=np.int8))
        sim.set_tally(True)
        sim.sweep(1000)
        obs = sim.run_schedule(np.arange(1001, 1001 + 4000, dtype=np.uint64))
        full = sim.observables()
        assert (obs[-1].bond_sum, obs[-1].M) == (full.bond_sum, full.M)      # tally == recompute after 5000 sweeps
    u, se_u = _blocked([o.e_per_site for o in obs])
    m, se_m = _blocked([abs(o.m_per_site) for o in obs])
    assert abs(u - _onsager_u(beta)) < 5 * se_u + 1e-3, (u, se_u, _onsager_u(beta))
    assert abs(m - _onsager_m0(beta)) < 5 * se_m + 1e-3, (m, se_m, _onsager_m0(beta))
    assert se_u < 1e-3 and se_m < 1e-3


@pytest.mark.parametrize("model,beta,D", [(wl.ISING, wl.BETA_C / 0.9, 0.0), (wl.ISING_LUT, wl.BETA_C / 0.9, 0.0),
                                          (wl.ISING, wl.BETA_C / 1.5, 0.0), (wl.BLUME_CAPEL, 1 / 1.4, 1.0)])
def test_schwinger_dyson_identity_on_the_gpu(eng, model, beta, D):
    """Eq. 3: (1/N) sum_x <exp(-2 beta s_x h_x)> = 1 in equilibrium, for any single-site
    heat-bath-compatible dynamics with these Boltzmann weights (Blume-Capel: the same identity over the
    sign-flip s -> -s, whose energy change is 2 s h)."""
    L = 1024
    with eng.IsingSim(model, L, beta, D, 9) as sim:
        if beta > wl.BETA_C and model != wl.BLUME_CAPEL:
            sim.write_lattice(np.ones((L, L), dtype=np.int8))                # ordered phase: skip the coarsening
        sim.sweep(2000)
        vals = []
        for _ in range(40):
            sim.sweep(25)
            v, hist = sim.schwinger_dyson()
            assert int(hist.sum()) == L * L
            vals.append(v)
    mean, se = np.mean(vals), np.std(vals, ddof=1) / math.sqrt(len(vals))
    assert abs(mean - 1.0) < 5 * se + 2e-3, (mean, se)
