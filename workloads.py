"""Seeded synthetic workloads (BASELINE.json configs) shared by tests, bench.py
and smoke().  Holds parameters only -- none of the method's arithmetic -- so
both the oracle and the CUDA path can be driven from the same inputs without
sharing code.  The paper uses no dataset: its workloads are random-start
quenches generated from a seed; these configs ARE those
workloads.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

ISING, BLUME_CAPEL, ISING_LUT, BLUME_CAPEL_2BIT = 0, 1, 2, 3   # ISING_LUT: the paper's 1-bit look-up-table kernel (NEXT-2)

# beta_c = ln(1 + sqrt(2)) / 2 (2D Ising, J = k_B = 1); the same double is
# handed to both sides (reading R6).
BETA_C = 0.5 * math.log(1.0 + math.sqrt(2.0))


@dataclass(frozen=True)
class Workload:
    name: str
    model: int
    L: int
    beta: float
    D: float
    seed: int
    sweeps: int
    note: str = ""


CONFIGS = [
    Workload("cfg0_ising_L256_Tc", ISING, 256, BETA_C, 0.0, 1, 100,
             "configs[0]: full-lattice + E, M after every sweep vs oracle"),
    Workload("cfg1_ising_L16384_0.5Tc", ISING, 1 << 14, BETA_C / 0.5, 0.0, 1, 1000,
             "configs[1]: quench at T = 0.5 Tc, E and M every 10 sweeps"),
    Workload("cfg2_ising_L262144_0.9Tc", ISING, 1 << 18, BETA_C / 0.9, 0.0, 1, 200,
             "configs[2]: headline updates/ns and HBM GB/s (34 GB packed)"),
    Workload("cfg3_bc_L32768_D1", BLUME_CAPEL, 1 << 15, 1.0 / 1.4, 1.0, 1, 500,
             "configs[3]: Blume-Capel, E, M, zero density every 10 sweeps"),
    Workload("cfg4_ising_L65536_corr", ISING, 1 << 16, BETA_C / 0.5, 0.0, 1, 2000,
             "configs[4]: coarsening with C(r), r = 1..L/2, every 2^k sweeps"),
]


def config(i: int) -> Workload:
    return CONFIGS[i]


def pow2_times(tmax: int):
    """config[4]'s measurement grid t = 1, 2, 4, ... <= tmax."""
    out, t = [], 1
    while t <= tmax:
        out.append(t)
        t *= 2
    return out
