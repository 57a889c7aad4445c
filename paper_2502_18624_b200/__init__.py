"""B200-native checkerboard Metropolis engine for the 2D Ising and Blume-Capel
models (hot path of arxiv 2502.18624).  The product is the CUDA library
``libising_b200.so`` behind the C ABI of ``include/ising.h``; this package is
the thin ctypes binding (argument marshalling only).  There is no CPU fallback:
creating a simulation without the library or without a CUDA device raises."""
from .binding import (ISING, BLUME_CAPEL, ISING_LUT, BLUME_CAPEL_2BIT, PIPE_PROBES, IsingError, IsingSim, Observables,  # noqa: F401
                      bench_pipes, debug_philox, time_grid, protocol_distances, threshold_table, slab_partition, lib_path, load_library,
                      workspace_bytes)
