/*
 * include/ising_bench.h -- measurement and debug entry points of libising_b200.so.
 * Not part of the method's surface (that is include/ising.h): kernels that bound the
 * update kernel's rooflines, the integer-pipe probe behind the ALU ceiling of DESIGN.md
 * Sec. 5.1, and a test hook for the device Philox4x32-10 (PAPER.md:149 names the generator).
 * Same conventions as ising.h: host pointers, int status codes, ising_last_error().
 */
#ifndef ISING_B200_BENCH_H
#define ISING_B200_BENCH_H

#include "ising.h"

#ifdef __cplusplus
extern "C" {
#endif

/* n calls of the Philox-only
 * kernel with the update kernel's grid (the ALU roof), and a plain
 * read+write pass over the colour arrays (the HBM roof).  Asynchronous.     */
int ising_bench_philox_only(ising_t *h, int n);
int ising_bench_copy(ising_t *h, int n);

/* Integer-pipe probe: issue rates, in warp-instructions per SM
 * sub-partition per clock at sm_mhz (<= 0: the device's maximum clock), of dependent chains of
 * [0] IMAD.WIDE  [1] LOP3  [2] IMAD  [3] IMAD.WIDE+LOP3  [4] IMAD.WIDE+2 LOP3
 * [5] IADD3(carry)+IMAD.X  [6] IMAD.WIDE+IMAD  [7] POPC+IADD (sum of both kinds per entry).
 * rates: host array of capacity cap; *count = 8.  Runs on the current device, default
 * stream, synchronises.  The ALU roofline of the update kernel is derived from these.     */
int ising_bench_pipes(double sm_mhz, double *rates, int cap, int *count);

/* Debug / test entry: evaluates this library's device Philox4x32-10 for count
 * (ctr, key) pairs (host arrays: ctr 4*count, key 2*count, out 4*count words).
 * with_curand != 0 evaluates the CUDA toolkit's curand_Philox4x32_10 instead.  */
int ising_debug_philox(int64_t count, const uint32_t *ctr, const uint32_t *key, uint32_t *out,
                       int with_curand);

#ifdef __cplusplus
}
#endif
#endif /* ISING_B200_BENCH_H */
