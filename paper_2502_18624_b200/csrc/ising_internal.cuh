// Internal declarations shared by the .cu files of libising_b200.so.
// Nothing here is shared with oracle/ (the CPU checker).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "ising.h"
#include "ising_bench.h"

// ----------------------------------------------------------------- handle ---
struct RoundKeys {  // Philox key schedule (PAPER.md:149 names the generator): k(i) = seed + i*W
    uint32_t k0[10], k1[10];
};

// NEXT-4 ("partitioning each buffer into horizontal slabs ... restricting [communication] to
// just two rows"): a slab = the consecutive rows [y0, y0 + rows) of both colour arrays in an allocation of
// its own, on a device of its own choice.  The kernels of a slab take its base pointers and, separately,
// pointers to the one row above and the one row below it in the neighbouring slabs (plain loads, peer
// memory when the neighbour lives on another device).  An unsharded lattice is one slab whose
// halo rows are its own last and first row.
struct Slab {
    int device = -1;
    cudaStream_t stream = nullptr;          // slab 0: the caller's stream; others: created by the library
    bool own_stream = false;
    int64_t y0 = 0, rows = 0;               // global rows [y0, y0 + rows); both even
    uint64_t *lat[2] = {nullptr, nullptr};  // black, white rows of this slab (device)
    void *owned = nullptr;                  // allocation made by the library (lattice + scratch), or NULL
    long long *d_acc = nullptr;             // 64 int64 accumulators in the slab's scratch area
    uint32_t *d_table = nullptr;            // Blume-Capel tables / LUT search tree on the slab's device
    void *lut_buckets = nullptr;            // LUT model: bucket table on the slab's device (cudaMalloc)
    cudaEvent_t done = nullptr;             // recorded after every colour phase (and every per-slab pass)
};

#define ISING_MAX_SLABS 64

// Row directory handed by value to the kernels that address the lattice by global row (IO, bit planes):
// slab k holds the rows [y_end[k-1], y_end[k]).
struct SlabDir {
    int n;
    long long y_first;                      // first row of slab 0 (0 unless the handle is one part of a lattice)
    long long y_end[ISING_MAX_SLABS];
    uint64_t *lat[2][ISING_MAX_SLABS];
};

struct ising_sim {
    std::vector<Slab> slabs;                // >= 1; lat / d_acc / d_bc_table / stream below are slab 0's (single-slab code paths)
    // One process per GPU (ising_create_part): the handle owns ONE slab of the lattice, the slabs above and below belong
    // to other handles -- other processes -- and their boundary rows are mapped through CUDA IPC (plain loads over NVLink).
    bool part = false;
    const uint64_t *part_halo[2][2] = {{nullptr, nullptr}, {nullptr, nullptr}};   // [above / below][colour]; NULL until attached
    void *part_ipc[2] = {nullptr, nullptr};                                        // mapped neighbour allocations (cudaIpcOpenMemHandle)
    int part_phase = 0;                                                            // colour the next ising_sweep_phase must update
    int model = 0;
    int64_t L = 0;
    double beta = 0, D = 0;
    uint64_t seed = 0;
    uint64_t t = 0;  // sweeps done
    cudaStream_t stream = nullptr;
    int device = -1;  // CUDA device of the lattice (the current device at ising_create, or dev_buf's)
    uint64_t *lat[2] = {nullptr, nullptr};  // black, white colour arrays (device)
    long long *d_acc = nullptr;             // 64 int64 accumulators inside the scratch area
    long long *h_acc = nullptr;             // pinned mirror
    uint64_t T[54] = {};                    // thresholds in [0, 2^32]
    int n_T = 0;
    uint32_t *d_bc_table = nullptr;         // Blume-Capel: 64-entry uint32 table + flags (scratch)
    RoundKeys rk;
    int rows_per_thread = 0, block_threads = 0, variant = 0;
    int64_t launches = 0;
    // lazily allocated (cudaMalloc, owned)
    void *io_stage = nullptr; size_t io_stage_bytes = 0;
    cudaStream_t io_stream = nullptr;                         // highest-priority stream of ising_write_bits (its small expansion
    cudaEvent_t io_event = nullptr;                           // kernels must not queue behind another handle's sweeps)
    uint64_t *planes = nullptr; size_t planes_bytes = 0;      // bit planes for the correlation
    uint64_t *comb = nullptr; size_t comb_bytes = 0;          // planes down-sampled to the source comb (stride >= 2)
    int8_t *gram = nullptr; size_t gram_bytes = 0;            // L x L int8 spin matrix for the tensor-core correlation
    // CUDA graph of K sweeps for launch-bound (small) lattices: kernels baked with t = 0..K-1, the base
    // sweep number lives in device memory (d_acc[48] as two uint32: [0] = 0 for plain launches, [1] = base)
    bool graph_capture = false;
    // two cached graphs: [0] of kGraphSweeps sweeps (long runs), [1] of a short sweep count that is asked for again and
    // again ("E, M every 10 sweeps": ising_run_schedule, the bench step)
    cudaGraphExec_t graph_exec[2] = {nullptr, nullptr};
    int graph_key[2][5] = {{0, 0, 0, 0, 0}, {0, 0, 0, 0, 0}};  // rows_per_thread, block_threads, variant, tally_on, sweeps in the graph
    int64_t last_short_n = 0;                                 // the previous call's n when it was too short for graph [0]
    bool tally_on = false;                                    // A7: update kernels keep running B, M, Q at d_acc[40..42]
    bool pdl_in_graph = false;                                // programmatic edges inside captured graphs (see launch_with_pdl)
    int sweep_mode = 0;                                       // small lattices (ising_set_sweep_mode): 0 auto, 1 graph, 2 plain, 3 persistent, 4 cluster
    int corr_path = 0;                                        // ising_set_corr_path: 0 auto, 1 bit planes, 2-4 tensor cores
    long long *d_corr = nullptr; size_t d_corr_bytes = 0;
    long long *d_rlist = nullptr; size_t d_rlist_bytes = 0;
};

static const size_t kScratchBytes = 4096;  // accumulators + BC table at the end of dev_buf

int set_error(int code, const std::string &msg);
int cuda_fail(cudaError_t e, const char *what);
#define CUDA_TRY(x)                                            \
    do {                                                       \
        cudaError_t e__ = (x);                                 \
        if (e__ != cudaSuccess) return cuda_fail(e__, #x);     \
    } while (0)

// Every entry point that takes a handle runs on the handle's device, whatever the caller's current
// device is, and puts the caller's device back on return.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(const ising_sim *h) { if (h) enter(h->device); }
    explicit DeviceGuard(int device) { enter(device); }
    void enter(int device)
    {
        if (device < 0 || cudaGetDevice(&prev) != cudaSuccess || prev == device) return;
        switched = cudaSetDevice(device) == cudaSuccess;
    }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

// Programmatic dependent launch (PTX griddepcontrol).  An update kernel loads its tables, then waits until the launch
// before it has completed and its writes are visible (griddepcontrol.wait: every lattice access comes after it), then
// lets the next launch of its stream be scheduled (griddepcontrol.launch_dependents): the next phase's blocks take the
// SM slots as they free up and sit ready, tables loaded, when the last block of this phase retires.  The trigger comes
// AFTER the wait: issued at the top, every kernel of a captured graph triggers the one after it at once and the
// whole chain piles up on the SMs, each generation waiting for the one before (L = 2048: 619 -> 328 updates/ns).
// Plain launches always carry the attribute (measured, profiles/r02_README.md: L = 4096 815 -> 967, 2^14 1291 ->
// 1316, Blume-Capel 2^15 1139 -> 1146).  Inside a captured graph the programmatic edges win where the launch latency
// or the table load dominates -- the 1-bit kernel at every size (+2..7 %), the 4-bit Ising kernel up to L = 3072
// (+4..7 %), everything up to L = 1536 (+5..14 %) -- and lose 7-11 % at L = 4096 / 8192 (the greedy placement of
// the early blocks packs a partial wave onto the SMs that free up first): ising_sim::pdl_in_graph, set at create.
#ifndef UPDATE_PDL
#define UPDATE_PDL 1
#endif
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_launch_dependents()
{
#if UPDATE_PDL
    asm volatile("griddepcontrol.launch_dependents;");
#endif
}
__device__ __forceinline__ void pdl_wait()
{
#if UPDATE_PDL
    asm volatile("griddepcontrol.wait;" ::: "memory");
#endif
}

template <typename Kernel, typename Params>
static inline cudaError_t launch_with_pdl(Kernel kernel, unsigned grid, int block, size_t smem, cudaStream_t stream, const Params &p,
                                          bool allow)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3((unsigned)block); cfg.dynamicSmemBytes = smem; cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = (UPDATE_PDL && allow) ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, p);
}
#endif

// host-only arithmetic (host_logic.cu)
int host_threshold_table(int model, double beta, double D, uint64_t *T);     // returns the number of entries (<= 54)
void host_time_grid(uint64_t tmax, std::vector<uint64_t> &times);
int64_t host_protocol_crossover(int64_t L, uint64_t t);
void host_protocol_lists(int64_t L, uint64_t t, std::vector<int64_t> &all_sources, std::vector<int64_t> &block_sources);

static inline int64_t words_per_row(int64_t L) { return L / 32; }              // uint64 per colour row
static inline int64_t words_per_colour(int64_t L) { return L * (L / 32); }
static inline bool is_blume_capel(int model) { return model == ISING_MODEL_BLUME_CAPEL || model == ISING_MODEL_BLUME_CAPEL_2BIT; }
// same-colour sites per uint64 word: 16 (4 bits each), 32 (2-bit Blume-Capel), 64 (1-bit LUT model)
static inline int64_t sites_per_word(int model)
{
    return model == ISING_MODEL_ISING_LUT ? 64 : model == ISING_MODEL_BLUME_CAPEL_2BIT ? 32 : 16;
}
// uint64 words of one colour array / of one colour row
static inline int64_t colour_words(const ising_sim *h) { return h->L * (h->L / (2 * sites_per_word(h->model))); }
static inline int64_t colour_row_words(const ising_sim *h) { return h->L / (2 * sites_per_word(h->model)); }
// Halo rows of slab k in colour array c: the last row of the slab above, the first row of the slab below (periodic).
static inline const uint64_t *halo_up(const ising_sim *h, int k, int c)
{
    if (h->part) return h->part_halo[0][c];
    const Slab &a = h->slabs[(k + (int)h->slabs.size() - 1) % (int)h->slabs.size()];
    return a.lat[c] + (a.rows - 1) * colour_row_words(h);
}
static inline const uint64_t *halo_down(const ising_sim *h, int k, int c)
{
    if (h->part) return h->part_halo[1][c];
    return h->slabs[(k + 1) % (int)h->slabs.size()].lat[c];
}
// 64-bit words per row of a plane down-sampled to the bits x % stride == 0 (zero padded)
static inline int64_t comb_words_per_row(int64_t L, int64_t stride) { return (L / stride + 63) / 64; }

// kernels' host launchers (each returns a cudaError_t from the launch)
// per-slab launchers run on the slab's stream (the caller has switched to the slab's device)
cudaError_t launch_init(ising_sim *h, int slab);
cudaError_t launch_update(ising_sim *h, int slab, int colour, uint32_t t);
int update_blocks_per_sm(const ising_sim *h, int block);         // occupancy of the update kernel this handle launches
int lut_blocks_per_sm(const ising_sim *h, int block);
cudaError_t launch_sweeps_persistent(ising_sim *h, uint32_t t0, int n_sweeps);   // unsharded small lattices, one cooperative launch
cudaError_t launch_sweeps_cluster(ising_sim *h, uint32_t t0, int n_sweeps);      // tiny lattices: one cluster, lattice in DSMEM
cudaError_t launch_observables(ising_sim *h, int slab);             // -> slab d_acc[0..2] = B, M, Q of the slab's rows
cudaError_t launch_sd_hist(ising_sim *h, int slab);                 // -> slab d_acc[8..16]
SlabDir slab_directory(const ising_sim *h);
cudaError_t launch_unpack(ising_sim *h, int64_t x0, int64_t y0, int64_t w, int64_t hgt, int8_t *dev_out);
cudaError_t launch_pack(ising_sim *h, int64_t y0, int64_t ny, const int8_t *dev_in, int *dev_bad, int write);
cudaError_t launch_bits(ising_sim *h, int colour, int64_t row0, int64_t nrows, uint32_t *dev_buf, int mode, int *dev_bad);
cudaError_t launch_planes(ising_sim *h);                            // lattice -> bit planes
cudaError_t launch_corr(ising_sim *h, int64_t stride, int64_t count, const long long *dev_r,
                        long long *dev_sx, long long *dev_sy);
bool corr_gram_supported(const ising_sim *h, int64_t rmax);
size_t corr_gram_bytes(const ising_sim *h);
cudaError_t launch_corr_gram(ising_sim *h, int64_t count, long long *dev_sx, long long *dev_sy);
cudaError_t launch_lut_init(ising_sim *h, int slab);
cudaError_t launch_lut_update(ising_sim *h, int slab, int colour, uint32_t t);
cudaError_t launch_lut_observables(ising_sim *h, int slab);         // -> slab d_acc[0..1] = B, M
cudaError_t launch_lut_sd_hist(ising_sim *h, int slab);             // -> slab d_acc[8..16]
cudaError_t launch_philox_only(ising_sim *h, uint32_t t);
cudaError_t launch_copy(ising_sim *h);
cudaError_t launch_debug_philox(int64_t count, const uint32_t *d_ctr, const uint32_t *d_key,
                                uint32_t *d_out, int with_curand, cudaStream_t s);

// ----------------------------------------------------------------- Philox ---
#ifdef __CUDACC__
#define PHILOX_M0 0xD2511F53u
#define PHILOX_M1 0xCD9E8D57u
#define PHILOX_W0 0x9E3779B9u
#define PHILOX_W1 0xBB67AE85u

// Row y of colour array c through the row directory (kernels that address the lattice by global row)
__device__ __forceinline__ uint64_t *slab_row(const SlabDir &d, int c, long long y, long long row_words)
{
    int k = 0;
    while (k + 1 < d.n && y >= d.y_end[k]) ++k;
    const long long first = k ? d.y_end[k - 1] : d.y_first;
    return d.lat[c][k] + (y - first) * row_words;
}

// Block-level sum of N per-thread ints into the int64 accumulators dst[0..N): warp
// reduction (warp sums must fit 32 bits), one shared-memory atomic per warp, ONE
// global atomic per block and quantity.  Same-address global atomics serialise in
// one L2 slice (about 1.3 ns each on B200): with one per warp the observables pass
// at L = 2^18 spent 4 of its 9 ms waiting for 3.1 M of them.  Every thread of the
// block must call this (it contains two block barriers): kernels keep threads past
// the lattice alive and let them add zeros.
template <int N>
__device__ __forceinline__ void block_accumulate(const int (&v)[N], long long *dst)
{
    __shared__ unsigned long long s_acc[N];
    if (threadIdx.x == 0) {
#pragma unroll
        for (int k = 0; k < N; ++k) s_acc[k] = 0;
    }
    __syncthreads();
    const unsigned m = 0xffffffffu;               // blocks are whole warps (ising_set_launch), all of them here
    const bool leader = (threadIdx.x & 31) == 0;
#pragma unroll
    for (int k = 0; k < N; ++k) {
        const int sum = __reduce_add_sync(m, v[k]);
        if (leader && sum) atomicAdd(&s_acc[k], (unsigned long long)(long long)sum);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int k = 0; k < N; ++k)
            if (s_acc[k]) atomicAdd(reinterpret_cast<unsigned long long *>(&dst[k]), s_acc[k]);
    }
}

// Generic Philox4x32-10: ten rounds of
//   (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0)).
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, const RoundKeys &rk)
{
#pragma unroll
    for (int i = 0; i < 10; ++i) {
        uint64_t p0 = (uint64_t)PHILOX_M0 * c.x;
        uint64_t p1 = (uint64_t)PHILOX_M1 * c.z;
        c = make_uint4((uint32_t)(p1 >> 32) ^ c.y ^ rk.k0[i], (uint32_t)p1,
                       (uint32_t)(p0 >> 32) ^ c.w ^ rk.k1[i], (uint32_t)p0);
    }
    return c;
}

// Per-(row, launch) constants of the counter (g_lo, g_hi, t, tag): everything in
// rounds 1-2 that does not depend on g_lo.  Saves 2 of the 20 multiplies per call.
struct PhiloxRow {
    uint32_t u2;   // tag ^ k1[0]
    uint32_t v0;   // lo(M1*t) ^ k0[1]
    uint32_t v1;   // hi(M0*U0) ^ k1[1],  U0 = hi(M1*t) ^ g_hi ^ k0[0]
    uint32_t v3;   // lo(M0*U0) ^ k1[2]
};

__device__ __forceinline__ PhiloxRow philox_row(uint32_t g_hi, uint32_t t, uint32_t tag, const RoundKeys &rk)
{
    uint64_t p1 = (uint64_t)PHILOX_M1 * t;
    uint32_t U0 = (uint32_t)(p1 >> 32) ^ g_hi ^ rk.k0[0];
    uint64_t q0 = (uint64_t)PHILOX_M0 * U0;
    PhiloxRow r;
    r.u2 = tag ^ rk.k1[0];
    r.v0 = (uint32_t)p1 ^ rk.k0[1];
    r.v1 = (uint32_t)(q0 >> 32) ^ rk.k1[1];
    r.v3 = (uint32_t)q0 ^ rk.k1[2];
    return r;
}

// The counter word g_lo = gl + q of the q-th call of a row, handed to the multiplier as an opaque value.  Left to
// itself the compiler rewrites M0 (gl | q) as M0 (gl & ~q) + M0 q: a masking LOP3, an IMAD.WIDE with a 64-bit constant
// addend that two IMAD.MOVs rebuild every time, and an add -- 0.25 to 0.4 dispatch slots per site more and 72 instead
// of 56 registers (measured: 1407 -> 1429 updates/ns for the 4-bit Ising kernel at L = 2^18).
__device__ __forceinline__ uint32_t philox_counter(uint32_t c)
{
    asm("" : "+r"(c));
    return c;
}

// Same function as philox4x32_10(make_uint4(g_lo, g_hi, t, tag)) with rounds 1-2 specialised.
__device__ __forceinline__ uint4 philox_site4(uint32_t g_lo, const PhiloxRow &pr, const RoundKeys &rk)
{
    // round 1: c = (U0, U1, hi0 ^ u2, lo0), U0/U1 folded into pr
    uint64_t p0 = (uint64_t)PHILOX_M0 * g_lo;
    uint32_t c2 = (uint32_t)(p0 >> 32) ^ pr.u2, c3 = (uint32_t)p0;
    // round 2: c = (hi(M1*c2) ^ U1 ^ k0[1], lo(M1*c2), hi(M0*U0) ^ c3 ^ k1[1], lo(M0*U0))
    uint64_t p1 = (uint64_t)PHILOX_M1 * c2;
    uint32_t d0 = (uint32_t)(p1 >> 32) ^ pr.v0, d1 = (uint32_t)p1, d2 = c3 ^ pr.v1;
    // round 3: c3 of round 2 is uniform and folded with k1[2] into v3
    p0 = (uint64_t)PHILOX_M0 * d0;
    p1 = (uint64_t)PHILOX_M1 * d2;
    uint4 c = make_uint4((uint32_t)(p1 >> 32) ^ d1 ^ rk.k0[2], (uint32_t)p1,
                         (uint32_t)(p0 >> 32) ^ pr.v3, (uint32_t)p0);
#pragma unroll
    for (int i = 3; i < 10; ++i) {
        p0 = (uint64_t)PHILOX_M0 * c.x;
        p1 = (uint64_t)PHILOX_M1 * c.z;
        c = make_uint4((uint32_t)(p1 >> 32) ^ c.y ^ rk.k0[i], (uint32_t)p1,
                       (uint32_t)(p0 >> 32) ^ c.w ^ rk.k1[i], (uint32_t)p0);
    }
    return c;
}
#endif  // __CUDACC__
