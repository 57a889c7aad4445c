/*
 * include/ising.h -- C ABI of the B200-native checkerboard Metropolis engine
 * (hot path of arxiv 2502.18624, Bisson et al.; citations are PAPER.md lines).
 *
 * One handle = one periodic L x L lattice resident in HBM, stored as two
 * colour arrays ("two separate buffers arranged in a checkerboard
 * pattern"), 4 bits per spin, 16 spins per 64-bit word (PAPER.md:57, 93
 * "Multiple Spin Coding ... four bits per spin"; the 4-bit store is what the
 * paper keeps for Blume-Capel).
 *
 *   site (x, y): x = column, y = row, 0 <= x, y < L, periodic
 *   colour c = (x + y) & 1; colour 0 ("black") is updated first in a sweep
 *   inside a colour: k = x >> 1, word m = k >> 4, nibble j = k & 15
 *   colour array = L rows x (L / 32) uint64 words, row-major
 *   nibble value: Ising 1 = spin +1, 0 = spin -1;  Blume-Capel s + 1 in {0,1,2}
 *   colour-site index n = y * (L/2) + k (64 bit) keys the random numbers:
 *   r(n) = word (n & 3) of Philox4x32-10(ctr = (g_lo, g_hi, t, tag), key = seed),
 *   g = n >> 2, t = sweep number, tag = colour (update) or 2 + colour (init).
 *
 * Pointers: every pointer argument is a HOST pointer unless its name starts
 * with dev_.  All calls return ISING_OK (0) or a negative error; outputs are
 * written only on ISING_OK, with one documented exception: calls that fill
 * caller arrays of a size only the library knows take a `count` pointer, which
 * is written whenever the arguments up to it are valid -- pass NULL for the
 * output arrays to ask for the size (returns ISING_OK), a too small `cap`
 * gives ISING_EINVAL with *count still set.  Nothing throws or aborts.  ising_last_error()
 * gives a thread-local message for the last non-OK return on this thread.
 * A handle is not thread-safe; distinct handles are independent.  Work is
 * enqueued on the stream given at create; calls documented as "synchronises"
 * block until that stream has drained.
 */
#ifndef ISING_B200_H
#define ISING_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ising_sim ising_t; /* opaque */

enum { ISING_MODEL_ISING = 0, ISING_MODEL_BLUME_CAPEL = 1,
       ISING_MODEL_ISING_LUT = 2, /* the paper's own kernel: 1 bit per spin, look-up-table random bits */
       ISING_MODEL_BLUME_CAPEL_2BIT = 3 /* Blume-Capel stored at 2 bits per spin, expanded to nibbles in
                                           registers: the same trajectory and results as ISING_MODEL_BLUME_CAPEL in half the memory */ };
enum { ISING_OK = 0, ISING_EINVAL = -1, ISING_ENOMEM = -2, ISING_ECUDA = -3 };

/* Integer observables are the bit-exact contract; the doubles are formed on
 * the host from them with one operation each (Eq. 1, Eq. 2):
 * E = -bond_sum (Ising) or -bond_sum + D*Q (Blume-Capel), J = 1.            */
typedef struct {
    int64_t bond_sum;     /* B = sum over the 2N nearest-neighbour bonds of s_x s_y */
    int64_t M;            /* sum of spins                                            */
    int64_t Q;            /* sum of squared spins (= N for Ising)                    */
    int64_t n_sites;      /* N = L*L                                                 */
    uint64_t sweeps_done; /* t                                                       */
    double E, e_per_site, m_per_site, zero_density;
} ising_obs_t;

/* Device bytes a caller-provided buffer must have for (model, L): the two
 * colour arrays (L*L/2 bytes at 4 bits per spin, L*L/4 at 2 bits, L*L/8 at 1 bit)
 * plus a small fixed scratch area.  0 if (model, L) is invalid.             */
size_t ising_workspace_bytes(int model, int64_t L);

/* Create a simulation (PAPER.md:25 problem statement; Eq. 1 / Eq. 2).
 *   model       ISING_MODEL_*
 *   L           linear size, multiple of 64, >= 64 (one 128-bit vector = 32
 *               same-colour sites of a row); ISING_MODEL_ISING_LUT stores one
 *               bit per spin (128 sites per vector): multiple of 256, >= 256,
 *               colour array = L rows x (L / 128) uint64 words, bit 1 = spin +1;
               ISING_MODEL_BLUME_CAPEL_2BIT: L rows x (L / 64) uint64 words, site j
               of a word at bits 2j..2j+1, code = spin + 1
 *   beta        1/(k_B T) >= 0, finite;  D = crystal field Delta of Eq. 2
 *               (finite; ignored for Ising);  seed = Philox key
 *   dev_buf     device memory of >= ising_workspace_bytes() bytes, 256-byte
 *               aligned, owned by the caller and alive until ising_destroy;
 *               NULL: the library allocates (cudaMalloc) and frees it.
 *               The simulation lives on dev_buf's device (the current device
 *               when dev_buf is NULL); every later call on the handle switches
 *               to that device and restores the caller's on return
 *   cuda_stream a cudaStream_t (e.g. torch's current stream); NULL = default
 * Builds the acceptance thresholds floor(min(1, exp(-beta dE)) 2^32) in double
 * (PAPER.md:93 for the Ising probabilities), fills the lattice from the seed
 * (Ising: top bit of r; Blume-Capel: (3 r) >> 32), sets t = 0.  Asynchronous. */
int ising_create(int model, int64_t L, double beta, double D, uint64_t seed,
                 void *dev_buf, size_t dev_bytes, void *cuda_stream, ising_t **out);

/* NEXT-4 of SURVEY.md Sec. 8(f): the same simulation with the lattice cut into n_slabs horizontal slabs
 * ("partitioning each buffer into horizontal slabs, which are stored in device memory ...
 * restricting [communication] to just two rows: the last row of the slab on the preceding GPU and the
 * first row of the slab on the next GPU"; the first and last slab are neighbours too).  Slab k holds
 * slab_rows[k] consecutive rows of both colour arrays (even, >= 2, adding up to L; NULL: an even split) in
 * an allocation of its own on CUDA device devices[k] (NULL: all on the current device).  The library
 * allocates; peer access between the devices involved is switched on, and the update / observables
 * kernels of a slab read its two halo rows from the neighbouring slabs' memory with plain loads
 * (PAPER.md:89).  Slabs of one colour phase run concurrently on streams of their own and wait only for
 * the previous phase of their two neighbours; integer observables are summed over the slabs in int64.
 * Random numbers are keyed by the global site index, so the trajectory is the unsharded lattice's bit for
 * bit whatever the partition ("identical numerical results ... regardless of the number of
 * GPUs used").  Every call of this header works on such a handle; cuda_stream is slab 0's stream.        */
int ising_create_slabs(int model, int64_t L, double beta, double D, uint64_t seed, int n_slabs,
                       const int64_t *slab_rows, const int *devices, void *cuda_stream, ising_t **out);
/* The default partition on its own (host arithmetic, no GPU): the L/2 row pairs dealt as evenly as possible
 * over n_slabs slabs, rows[k] = height of slab k (even, >= 2).                                             */
int ising_slab_partition(int64_t L, int n_slabs, int64_t *rows);
/* Number of slabs (1 for ising_create), and rows [y0, y0 + rows) / device of one of them (NULL: skip). */
int ising_slab_count(const ising_t *h);
int ising_slab_info(const ising_t *h, int slab, int64_t *y0, int64_t *rows, int *device);

/* One process per GPU (torch.distributed's arrangement): ONE slab of the lattice per handle.  ising_create_part
 * makes the handle of the rows [y0, y0 + rows) (both even, rows >= 2; the library allocates on the current device)
 * and fills them from the seed exactly as the whole lattice would be.  ising_part_export writes the
 * ISING_IPC_HANDLE_BYTES-byte CUDA IPC handle of the slab's allocation; the ranks exchange these (an all-gather) and
 * every rank calls ising_part_attach with the handles and heights of the slab above and the slab below (periodic; with
 * two parts both are the other part): the allocations are mapped (cudaIpcOpenMemHandle, peer access over NVLink) and
 * the kernels read their two halo rows from them with plain loads.  A part covering the whole
 * lattice (rows == L) needs no attach.  ising_sweep_phase launches ONE colour phase (0, then 1; after colour 1 the sweep
 * counter advances); between two phases the caller orders the ranks -- a stream-ordered collective on the handle's
 * stream (an NCCL all-reduce of one word) or a host barrier after ising_sync: a phase may start once the previous phase
 * of both neighbours has finished.  On a part handle the observables, the tally and the histogram are the sums over
 * its own rows (bonds counted at their black site; n_sites = rows * L): the ranks add them up (an int64 all-reduce).
 * Lattice IO addresses global rows inside the part; the correlation calls need the whole lattice and return
 * ISING_EINVAL.  Results are those of the unsharded lattice bit for bit.                          */
#define ISING_IPC_HANDLE_BYTES 64
int ising_create_part(int model, int64_t L, double beta, double D, uint64_t seed, int64_t y0, int64_t rows,
                      void *cuda_stream, ising_t **out);
int ising_part_export(ising_t *h, void *ipc_handle);
int ising_part_attach(ising_t *h, const void *ipc_above, int64_t rows_above, const void *ipc_below, int64_t rows_below);
int ising_sweep_phase(ising_t *h, int colour);

/* n >= 0 full sweeps: colour 0 then colour 1 ("two update phases"),
 * one Philox number per site, accept iff r < T.  Asynchronous:
 * 2n kernel launches on the handle's stream, no host synchronisation; small
 * lattices run in one cluster kernel (L <= 512) or replay a CUDA graph (L <= 2^14);
 * see ising_set_sweep_mode.                                                                  */
int ising_sweep(ising_t *h, int64_t n);

/* Full recompute of B, M, Q by warp-shuffle / block reduction over both colour
 * arrays.  Synchronises.                                                    */
int ising_observables(ising_t *h, ising_obs_t *out);

/* Fused tally (optional, A7 of SURVEY.md Sec. 8(a)): on != 0 makes the update kernels keep
 * running B, M, Q on the device -- the changes caused by every accepted move are added block
 * by block -- starting from a full recompute made by this call (and again after every lattice
 * write).  ising_tally returns the running values in the same struct as ising_observables
 * (they must always agree: north_star's "incremental dE tally equals a full recompute of H")
 * without a pass over the lattice.  Costs about 10 % of the update rate while on.
 * ising_tally synchronises.                                                          */
int ising_set_tally(ising_t *h, int on);
int ising_tally(ising_t *h, ising_obs_t *out);

/* Full-source pair sums: sx[r-1] = sum_{x,y} s(x,y) s(x+r,y),
 * sy[r-1] = sum_{x,y} s(x,y) s(x,y+r), periodic, r = 1..rmax, 1 <= rmax <= L/2.
 * Host arrays of length rmax.  Synchronises.                                */
int ising_correlation(ising_t *h, int64_t rmax, int64_t *sx, int64_t *sy);

/* The same sums for callers that may not allocate (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): ising_correlation keeps its scratch -- bit planes, transposed planes,
 * accumulators -- in buffers it cudaMallocs on first use; this entry point runs the same bit-plane kernels on
 * a static device array of 532480 bytes (held by every GPU that loads the library until exit) and calls no
 * cudaMalloc, cudaFree or allocating library routine.  Limit: L <= ISING_NOALLOC_MAX_L (ISING_EINVAL beyond
 * it).  Every call on a device shares the array, which keeps the last call's contents: what must start at
 * zero is cleared by the call itself, but two calls that OVERLAP on the GPU (two handles on two streams, two
 * host threads) race on it.  Same arguments, same integers as ising_correlation.  Synchronises.          */
#define ISING_NOALLOC_MAX_L 1024
int ising_correlation_noalloc(ising_t *h, int64_t rmax, int64_t *sx, int64_t *sy);

/* Which kernels ising_correlation uses: 0 = automatic (tensor cores at the fp4 rate, path 4, when
 * rmax >= 512 and L is a multiple of 256; bit planes otherwise), 1 = bit planes (XOR + POPC),
 * 2 = tensor cores, int8, one CTA per 128 x 256 tile, 3 = int8, CTA pairs (cta_group::2, 256 x 256
 * tiles), 4 = CTA pairs at the fp4 rate (e2m1 matrix, kind::mxf4 with unit block scales, 256 x 224
 * tiles, fp32 accumulation of exact integers).  Paths 2-4 need L % 256 == 0 and allocate the
 * spin matrix on first use (L*L bytes for int8, about L*L/2 for fp4).  The results are identical integers in every case.                    */
int ising_set_corr_path(ising_t *h, int path);

/* The paper's down-sampled protocol at t = sweeps_done:
 * all sources for r <= 32; sources {x % 16 == 0, y % 16 == 0} for 32 < r <=
 * r_c(t) and for r on the logarithmic grid up to L/2.  Arrays of capacity cap;
 * *count receives the number of distances (size query: all four arrays NULL).
 * The arrays are written only when every kernel has succeeded.  Synchronises. */
int ising_correlation_protocol(ising_t *h, int64_t cap, int64_t *r, int64_t *sx, int64_t *sy,
                               int64_t *n_src, int64_t *count);

/* The distance list of that protocol on its own (host arithmetic, no handle, no GPU):
 *   r = 1..2R, R = 16                                   every site a source   stride[i] = 1
 *   r = 2R+1..r_c(t), r_c = max{256, [g(L) sqrt(t)]},
 *       g(L) = 6 sqrt(ln(L / 2^16) / 3.3^2 + 1)         one source per R x R  stride[i] = 16
 *   r = floor(2^(x/32)) > r_c(t) while 2^(x/32) <= L/2   stride[i] = 16
 * ascending, clipped to L/2 (L even).  Size query: r == stride == NULL.          */
int ising_protocol_distances(int64_t L, uint64_t t, int64_t cap, int64_t *r, int64_t *stride, int64_t *count);

/* Same sums for an explicit strictly positive distance list (each <= L/2) and
 * a source stride (sources x % stride == 0 and y % stride == 0; stride 1 or a
 * power of two <= 64).  Synchronises.                                        */
int ising_correlation_list(ising_t *h, int64_t stride, int64_t count, const int64_t *r,
                           int64_t *sx, int64_t *sy);

/* Schwinger-Dyson check (Eq. 3): hist[k+4] = number of sites with
 * s_x h_x = k, k = -4..4; *value = (1/N) sum_k hist[k+4] exp(-2 beta k).
 * Synchronises.                                                             */
int ising_schwinger_dyson(ising_t *h, int64_t hist[9], double *value);

/* Unpack rows [y0, y0+ny) to int8 spins, row-major ny x L (host).  Synchronises. */
int ising_read_lattice(ising_t *h, int64_t y0, int64_t ny, int8_t *host_out);
/* Unpack the w x hgt window whose top-left site is (x0, y0); coordinates wrap
 * (any integer x0, y0; 1 <= w, hgt <= L).  Synchronises.                     */
int ising_read_window(ising_t *h, int64_t x0, int64_t y0, int64_t w, int64_t hgt, int8_t *host_out);
/* Overwrite rows [y0, y0+ny) from int8 spins (values outside the model's set
 * give ISING_EINVAL and leave the lattice unchanged).  Synchronises.         */
int ising_write_lattice(ising_t *h, int64_t y0, int64_t ny, const int8_t *host_in);

/* Raw packed colour array <-> host: words [word0, word0 + nwords) of colour
 * c (row-major L x L/32).  For checkpoints and the end-to-end benchmark.    */
int ising_read_packed(ising_t *h, int colour, int64_t word0, int64_t nwords, uint64_t *host_out);
int ising_write_packed(ising_t *h, int colour, int64_t word0, int64_t nwords, const uint64_t *host_in);
/* Compact transport format: the rows [row0, row0 + nrows) of colour array `colour` at the information content
 * of a spin instead of its storage size -- Ising: 1 bit per spin, bit j of word m of a row = compact site
 * k = 64 m + j, 1 = spin +1, L/128 words per colour row (the layout of ISING_MODEL_ISING_LUT);
 * Blume-Capel: 2 bits per spin, site j of a word at bits 2j..2j+1, code = spin + 1, L/64 words per colour row
 * (the layout of ISING_MODEL_BLUME_CAPEL_2BIT; a code equal to 3 gives ISING_EINVAL and leaves the lattice
 * unchanged).  The 4-bit models expand / gather on the device, so a whole-lattice upload moves L*L/8 bytes
 * for Ising (L*L/4 for Blume-Capel) instead of L*L/2; for the 1-bit and 2-bit models the format is the
 * packed layout itself.  Host arrays of nrows * (words per colour row) uint64, row-major; the Ising format
 * needs L to be a multiple of 128 (whole words per colour row).  Synchronises.                              */
int ising_write_bits(ising_t *h, int colour, int64_t row0, int64_t nrows, const uint64_t *host_in);
int ising_read_bits(ising_t *h, int colour, int64_t row0, int64_t nrows, uint64_t *host_out);

/* Schedule interleave (A11 of SURVEY.md Sec. 8(a)).  ising_time_grid: the paper's measurement
 * times t = floor(2^(x/8) + 0.5), x = 1, 2, ..., de-duplicated, t <= tmax, into the
 * host array out (capacity cap); *count = number of times (size query: out == NULL).  Host
 * arithmetic only: no handle, no GPU.  ising_run_schedule: sweeps to each time of the ascending host array times
 * (all >= sweeps_done) and records the integer observables there in out[i] (by the fused tally
 * if it is on, else by the observables pass).  Synchronises at every measurement.        */
int ising_time_grid(uint64_t tmax, uint64_t *out, int64_t cap, int64_t *count);
int ising_run_schedule(ising_t *h, int64_t n_times, const uint64_t *times, ising_obs_t *out);
/* The same interleave with the correlation measurement: sweeps to each time and runs
 * the Sec. 3.3 protocol there.  r, sx, sy, n_src are host arrays of n_times x cap int64, row-major: row i
 * receives counts[i] entries (as ising_correlation_protocol at times[i]); cap must hold the longest list
 * (ising_protocol_distances at the last time).  obs (may be NULL): the integer observables at the same
 * times.  Synchronises at every measurement.                                                  */
int ising_run_protocol_schedule(ising_t *h, int64_t n_times, const uint64_t *times, int64_t cap,
                                int64_t *r, int64_t *sx, int64_t *sy, int64_t *n_src, int64_t *counts,
                                ising_obs_t *obs);

/* Set the sweep counter t (exact resume: state = lattice + t).               */
int ising_set_sweeps_done(ising_t *h, uint64_t t);

/* Threshold table dump for the equality assert against the oracle: Ising 5
 * entries indexed (dE+8)/4; Blume-Capel 54 entries ((s+1)*2+b)*9 + (h+4); the
 * 1-bit look-up-table model 16 entries, entry i = floor(2^32 P(pattern < i)),
 * patterns of four independent bits that are 1 with probability e^{-4 beta}
 * (PAPER.md:133-149).  Values in [0, 2^32].  *count = entries (size query: out
 * == NULL).  ising_threshold_table computes the same table from (model, beta, D)
 * alone: host arithmetic, no handle, no GPU.                                */
int ising_thresholds(ising_t *h, uint64_t *out, int cap, int *count);
int ising_threshold_table(int model, double beta, double D, uint64_t *out, int cap, int *count);

/* Launch geometry of the update kernel (results never depend on it,
 * cf. PAPER.md:193): rows walked per thread and threads per block
 * (multiple of 32, <= 1024).  0 keeps the current value.                    */
int ising_set_launch(ising_t *h, int rows_per_thread, int block_threads);
/* Update kernel variant (0 = default: carry-chain compare; for the LUT model the
 * bucket table at L >= 8192 and the binary search below; 1 = compare/select,
 * binary search; 2 (LUT model only) = bucket table; equivalent implementations
 * kept for parity / performance comparison).                                */
int ising_set_variant(ising_t *h, int variant);

/* How ising_sweep runs launch-bound lattices (unsharded; results never depend on it): 0 = automatic
 * (4 for L <= 512, else 1), 1 = replay of a CUDA graph (L <= 2^14, where a launch gap of about 2.4 microseconds
 * still shows: a graph of 16 sweeps when n >= 32, a graph of exactly n sweeps when the same 4 <= n < 32 is asked
 * for twice in a row -- "E, M every 10 sweeps"), 2 = one launch per colour
 * phase, 3 = one cooperative launch for all n sweeps with a grid-wide barrier after every colour phase
 * (measured a little slower than the graph), 4 = one thread-block cluster of 16 CTAs that
 * keeps the lattice in distributed shared memory for all n sweeps, halo rows read from the neighbouring CTA's
 * shared memory, hardware cluster barrier between the colour phases.  3 and 4: 4-bit and 2-bit models; they
 * fall back to 1 when the device refuses the launch (4: also when the lattice does not fit the cluster).   */
int ising_set_sweep_mode(ising_t *h, int mode);

/* Number of kernels this handle has launched since create.                  */
int64_t ising_launch_count(const ising_t *h);
/* Block until the handle's stream is idle.                                  */
int ising_sync(ising_t *h);
int ising_destroy(ising_t *h);
const char *ising_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* ISING_B200_H */
