// C ABI of libising_b200.so (include/ising.h).  Host logic only: argument checks,
// threshold table (A1), launch sequencing (A11), integer -> double observables.
#include <math.h>
#include <string.h>

#include <algorithm>
#include <new>
#include <string>
#include <vector>

#include "ising_internal.cuh"

static thread_local std::string g_err;

int set_error(int code, const std::string &msg)
{
    g_err = msg;
    return code;
}

int cuda_fail(cudaError_t e, const char *what)
{
    return set_error(ISING_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

extern "C" const char *ising_last_error(void) { return g_err.c_str(); }

static void drop_graph(ising_sim *h);

static bool valid_model_L(int model, int64_t L)
{
    if (model == ISING_MODEL_ISING_LUT) return L >= 256 && (L % 256) == 0 && L <= (1ll << 20);   // 128-bit vector = 128 sites
    return (model == ISING_MODEL_ISING || is_blume_capel(model)) && L >= 64 && (L % 64) == 0 &&
           L <= (1ll << 20);
}

extern "C" size_t ising_workspace_bytes(int model, int64_t L)
{
    if (!valid_model_L(model, L)) return 0;
    return (size_t)L * (size_t)L / (size_t)sites_per_word(model) * 8 + kScratchBytes;   // both colour arrays
}

// A1 / L2: the tables themselves are host arithmetic (host_logic.cu)
static void build_thresholds(ising_sim *h)
{
    h->n_T = host_threshold_table(h->model, h->beta, h->D, h->T);
}

static void build_round_keys(ising_sim *h)
{
    uint32_t k0 = (uint32_t)(h->seed & 0xFFFFFFFFull), k1 = (uint32_t)(h->seed >> 32);
    for (int i = 0; i < 10; ++i) {
        h->rk.k0[i] = k0; h->rk.k1[i] = k1;
        k0 += PHILOX_W0; k1 += PHILOX_W1;
    }
}

// Rows per thread: as many as 32 (64 for the LUT model) to amortise the two halo rows of the sliding
// window, but never so many that the grid drops below ~1024 threads per SM: mid-size lattices
// (L = 4096: 64 columns) would otherwise run on a fraction of the 148 SMs.
static void default_launch(ising_sim *h)
{
    const bool lut = h->model == ISING_MODEL_ISING_LUT;
    const int64_t cols = lut ? h->L / 256 : h->L / 64;
    const int64_t target = 148 * 1024;
    int64_t r = 2 * ((h->L * cols) / (2 * target));
    const int64_t rmax = lut ? 64 : 32;
    if (r > rmax) r = rmax;
    if (r < 2) r = 2;
    h->rows_per_thread = (int)r;
    h->block_threads = lut ? 256 : 128;           // LUT: 32 KB bucket table per block, fewer and larger blocks
}

// Wave quantisation.  A colour phase of a mid-size lattice is a handful of waves of blocks (a wave = the blocks the
// GPU holds at once), and a last wave that is nearly empty costs as much as a full one: at L = 2^14 the first
// choice R = 26 gives 1262 blocks for 1184 places -- R = 28 (1172 blocks, one wave) runs 4.6 % faster, R = 14 (two
// full waves) the same.  So among the even R up to the first choice's ceiling the one with the least
// waves x (R + halo) is taken; lattices of many waves keep the first choice.
static void tune_rows_for_waves(ising_sim *h)
{
    const bool lut = h->model == ISING_MODEL_ISING_LUT;
    int n_sm = 0;
    if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, h->device) != cudaSuccess) { cudaGetLastError(); return; }
    const int block = h->block_threads;
    const int per_sm = lut ? lut_blocks_per_sm(h, block) : update_blocks_per_sm(h, block);
    if (per_sm <= 0 || n_sm <= 0) return;
    const int64_t capacity = (int64_t)per_sm * n_sm, cols = lut ? h->L / 256 : h->L / 64, rmax = lut ? 64 : 32;
    int64_t rows = 0;
    for (const Slab &sl : h->slabs) rows = std::max(rows, sl.rows);
    auto blocks = [&](int64_t r) { return (((rows + r - 1) / r) * cols + block - 1) / block; };
    if (blocks(rmax) > 16 * capacity) {                         // many waves: the tail is a few per cent at most
        // 4-bit Ising kernel: longer columns re-read fewer halo rows (2 per R) -- L = 2^18: R = 32 1450.9, 64 1454.5,
        // 128 1455.5, 512 1449.0 updates/ns (profiles/r02_README.md); the table kernels lose with long columns
        if (h->model == ISING_MODEL_ISING && blocks(128) > 16 * capacity) h->rows_per_thread = 128;
        return;
    }
    const double wave_slack = is_blume_capel(h->model) ? 0.5 : 0.0;
    double best = 0.0;
    int64_t best_r = h->rows_per_thread;
    for (int64_t r = 2; r <= rmax; r += 2) {
        const int64_t waves = (blocks(r) + capacity - 1) / capacity;
        // two halo rows cost about a third of a row each.  Blume-Capel: half a wave on top -- its blocks (random table
        // look-ups) finish unevenly, and one wave of long blocks loses to four waves of short ones (L = 2^14: R = 32
        // 990, R = 8 1100 updates/ns); the Ising kernels lose with that term (measured, profiles/r02_README.md)
        const double cost = ((double)waves + wave_slack) * ((double)r + 0.7);
        if (best == 0.0 || cost <= best) { best = cost; best_r = r; }
    }
    h->rows_per_thread = (int)best_r;
}

// ---------------------------------------------------------------- create ---
// Device tables derived from the integer thresholds: Blume-Capel compare / carry tables, or the search
// tree and bucket table of the 1-bit kernel's getMaxLE.  Built once on the host, copied to every slab's device.
struct HostTables {
    std::vector<uint32_t> table;     // -> Slab::d_table
    std::vector<uint32_t> buckets;   // -> Slab::lut_buckets (LUT model only)
};

static int build_host_tables(const ising_sim *h, HostTables &ht)
{
    if (is_blume_capel(h->model)) {
        // [0, 66): thresholds clamped to 2^32-1 + "always" bit mask (compare/select variant).
        // [80, 80 + 132): carry form for the default variant, two halves of 66 words (264 bytes):
        // C[b][16 code + S] = 2^32 - T, 0 for T = 2^32 (never a carry -> always accepted).  T = 0 has
        // no 32-bit carry constant: launch_update then uses the compare/select variant.
        ht.table.assign(80 + 132, 0u);
        uint64_t always = 0;
        for (int i = 0; i < 54; ++i) {
            if (h->T[i] >> 32) { always |= 1ull << i; ht.table[i] = 0xFFFFFFFFu; }
            else ht.table[i] = (uint32_t)h->T[i];
        }
        ht.table[64] = (uint32_t)always; ht.table[65] = (uint32_t)(always >> 32);
        for (int code = 0; code < 3; ++code)
            for (int S = 0; S <= 8; ++S)
                for (int b = 0; b < 2; ++b) {
                    const uint64_t T = h->T[(code * 2 + b) * 9 + S];
                    ht.table[80 + 66 * b + 16 * code + S] = (T >> 32) ? 0u : (uint32_t)((1ull << 32) - T);
                }
    }
    if (h->model == ISING_MODEL_ISING_LUT) {
        // heap-ordered carry constants of the binary search: node n at level l splits at table index
        // ((n - 2^l) << (4 - l)) | (1 << (3 - l));  rnd >= table[i]  <=>  rnd + (2^32 - table[i]) carries
        for (int i = 1; i < 16; ++i)
            if (h->T[i] == 0)        // "rnd >= 0" has no 32-bit carry constant (2^32 is fine: constant 0, never a carry)
                return set_error(ISING_EINVAL, "ising_create: beta too small for the look-up-table model "
                                               "(a table entry above index 0 is 0; needs beta > about 0.001)");
        ht.table.assign(16, 0u);
        for (int l = 0; l < 4; ++l)
            for (int n = 1 << l; n < (2 << l); ++n) {
                const int idx = ((n - (1 << l)) << (4 - l)) | (1 << (3 - l));
                ht.table[n] = (uint32_t)((1ull << 32) - h->T[idx]);
            }
        // bucket table of the default kernel variant: entry b covers rnd in [b 2^20, (b+1) 2^20):
        // {C, meta} with getMaxLE(rnd) = meta + carry(rnd + C) when the bucket holds at most one threshold,
        // meta = 256 (recompute by binary search) when it holds more
        ht.buckets.assign(2 * 4096, 0u);
        for (uint64_t b = 0; b < 4096; ++b) {
            const uint64_t lo = b << 20, hi = lo + (1ull << 20) - 1;
            int base = 0, inside = 0;
            for (int i = 1; i < 16; ++i) {
                if (h->T[i] <= lo) base = i;
                else if (h->T[i] <= hi) ++inside;
            }
            if (inside == 0) { ht.buckets[2 * b] = 0u; ht.buckets[2 * b + 1] = (uint32_t)base; }
            else if (inside == 1) { ht.buckets[2 * b] = (uint32_t)((1ull << 32) - h->T[base + 1]); ht.buckets[2 * b + 1] = (uint32_t)base; }
            else { ht.buckets[2 * b] = 0u; ht.buckets[2 * b + 1] = 256u; }
        }
    }
    return ISING_OK;
}

// Scratch, tables and the seeded lattice of one slab (its memory and stream are in place).
static int setup_slab(ising_sim *h, int k, const HostTables &ht)
{
    Slab &sl = h->slabs[k];
    DeviceGuard dev_guard(sl.device);
    CUDA_TRY(cudaEventCreateWithFlags(&sl.done, cudaEventDisableTiming));
    CUDA_TRY(cudaMemsetAsync(sl.d_acc, 0, 1024, sl.stream));              // accumulators, tally, t_base words
    if (!ht.table.empty())
        CUDA_TRY(cudaMemcpyAsync(sl.d_table, ht.table.data(), ht.table.size() * sizeof(uint32_t), cudaMemcpyHostToDevice, sl.stream));
    if (!ht.buckets.empty()) {
        CUDA_TRY(cudaMalloc(&sl.lut_buckets, ht.buckets.size() * sizeof(uint32_t)));
        CUDA_TRY(cudaMemcpyAsync(sl.lut_buckets, ht.buckets.data(), ht.buckets.size() * sizeof(uint32_t), cudaMemcpyHostToDevice, sl.stream));
    }
    cudaError_t e = (h->model == ISING_MODEL_ISING_LUT) ? launch_lut_init(h, k) : launch_init(h, k);
    if (e != cudaSuccess) return cuda_fail(e, "init kernel");
    CUDA_TRY(cudaStreamSynchronize(sl.stream));                           // the host tables go out of scope after create
    return ISING_OK;
}

static void carve_slab(ising_sim *h, Slab &sl, char *base)
{
    const size_t colour_bytes = (size_t)sl.rows * (size_t)colour_row_words(h) * 8;
    sl.lat[0] = (uint64_t *)base;
    sl.lat[1] = (uint64_t *)(base + colour_bytes);
    sl.d_acc = (long long *)(base + 2 * colour_bytes);                 // 64 int64 = 512 B (+ sink area)
    sl.d_table = (uint32_t *)(base + 2 * colour_bytes + 1024);         // 212 uint32 (two table forms)
}

static int check_create_args(const char *who, int model, int64_t L, double beta, double D, ising_t **out)
{
    if (!out) return set_error(ISING_EINVAL, std::string(who) + ": out is NULL");
    if (!valid_model_L(model, L))
        return set_error(ISING_EINVAL, std::string(who) + ": unknown model, or L not a multiple of 64 (256 for the LUT model) in [64, 2^20]");
    if (!(beta >= 0.0) || !isfinite(beta)) return set_error(ISING_EINVAL, std::string(who) + ": beta must be finite and >= 0");
    if (!isfinite(D)) return set_error(ISING_EINVAL, std::string(who) + ": D must be finite");
    return ISING_OK;
}

static ising_sim *new_handle(int model, int64_t L, double beta, double D, uint64_t seed, void *cuda_stream)
{
    ising_sim *h = new (std::nothrow) ising_sim();
    if (!h) return nullptr;
    h->model = model; h->L = L; h->beta = beta; h->D = is_blume_capel(model) ? D : 0.0; h->seed = seed;
    h->stream = (cudaStream_t)cuda_stream;
    build_thresholds(h);
    build_round_keys(h);
    default_launch(h);
    return h;
}

// common tail of both create calls: slabs carved, streams in place
static int finish_create(ising_sim *h, ising_t **out)
{
    HostTables ht;
    int rc = build_host_tables(h, ht);
    if (rc) { ising_destroy(h); return rc; }
    cudaError_t e = cudaMallocHost(&h->h_acc, (size_t)ISING_MAX_SLABS * 64 * sizeof(long long));
    if (e != cudaSuccess) { ising_destroy(h); return cuda_fail(e, "cudaMallocHost"); }
    for (int k = 0; k < (int)h->slabs.size(); ++k) {
        rc = setup_slab(h, k, ht);
        if (rc) { ising_destroy(h); return rc; }
    }
    {
        DeviceGuard g(h->device);
        tune_rows_for_waves(h);
    }
    h->pdl_in_graph = h->model == ISING_MODEL_ISING_LUT || h->L <= 1536 || (h->model == ISING_MODEL_ISING && h->L <= 3072);
    const Slab &s0 = h->slabs[0];
    h->lat[0] = s0.lat[0]; h->lat[1] = s0.lat[1]; h->d_acc = s0.d_acc; h->d_bc_table = s0.d_table;
    *out = h;
    return ISING_OK;
}

extern "C" int ising_create(int model, int64_t L, double beta, double D, uint64_t seed, void *dev_buf,
                            size_t dev_bytes, void *cuda_stream, ising_t **out)
{
    int rc = check_create_args("ising_create", model, L, beta, D, out);
    if (rc) return rc;
    const size_t need = ising_workspace_bytes(model, L);
    if (dev_buf && dev_bytes < need) return set_error(ISING_EINVAL, "ising_create: dev_bytes < ising_workspace_bytes()");
    if (dev_buf && ((uintptr_t)dev_buf & 255u)) return set_error(ISING_EINVAL, "ising_create: dev_buf must be 256-byte aligned");

    ising_sim *h = new_handle(model, L, beta, D, seed, cuda_stream);
    if (!h) return set_error(ISING_ENOMEM, "ising_create: host allocation failed");
    char *base = (char *)dev_buf;
    cudaGetDevice(&h->device);                       // NULL dev_buf: the caller's current device
    if (base) {
        cudaPointerAttributes attr;
        if (cudaPointerGetAttributes(&attr, base) != cudaSuccess || attr.type != cudaMemoryTypeDevice) {
            cudaGetLastError();
            delete h;
            return set_error(ISING_EINVAL, "ising_create: dev_buf is not device memory");
        }
        h->device = attr.device;
    }
    DeviceGuard dev_guard(h->device);
    Slab sl;                                         // the whole lattice is one slab; its halo rows are its own
    sl.device = h->device; sl.stream = h->stream; sl.y0 = 0; sl.rows = L;
    if (!base) {
        cudaError_t e = cudaMalloc(&sl.owned, need);
        if (e != cudaSuccess) {
            delete h;
            cudaGetLastError();
            return set_error(e == cudaErrorMemoryAllocation ? ISING_ENOMEM : ISING_ECUDA,
                             std::string("ising_create: cudaMalloc: ") + cudaGetErrorString(e));
        }
        base = (char *)sl.owned;
    }
    carve_slab(h, sl, base);
    h->slabs.push_back(sl);
    return finish_create(h, out);
}

// NEXT-4: the lattice as n_slabs row slabs, each an
// allocation of its own on the device the caller names, with the two halo rows of a slab read straight from
// its neighbours' memory (peer access between the devices involved is switched on here).
extern "C" int ising_create_slabs(int model, int64_t L, double beta, double D, uint64_t seed, int n_slabs,
                                  const int64_t *slab_rows, const int *devices, void *cuda_stream, ising_t **out)
{
    int rc = check_create_args("ising_create_slabs", model, L, beta, D, out);
    if (rc) return rc;
    if (n_slabs < 1 || n_slabs > ISING_MAX_SLABS || 2 * (int64_t)n_slabs > L)
        return set_error(ISING_EINVAL, "ising_create_slabs: n_slabs must be in [1, 64] and leave every slab two rows");
    std::vector<int64_t> rows(n_slabs);
    int64_t total = 0;
    if (!slab_rows) { rc = ising_slab_partition(L, n_slabs, rows.data()); if (rc) return rc; }
    for (int k = 0; k < n_slabs; ++k) {
        if (slab_rows) rows[k] = slab_rows[k];
        if (rows[k] < 2 || (rows[k] & 1)) return set_error(ISING_EINVAL, "ising_create_slabs: every slab needs an even number of rows >= 2");
        total += rows[k];
    }
    if (total != L) return set_error(ISING_EINVAL, "ising_create_slabs: slab_rows must add up to L");
    int n_dev = 0, cur = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev < 1 || cudaGetDevice(&cur) != cudaSuccess) {
        cudaGetLastError();
        return set_error(ISING_ECUDA, "ising_create_slabs: no CUDA device");
    }
    for (int k = 0; devices && k < n_slabs; ++k)
        if (devices[k] < 0 || devices[k] >= n_dev) return set_error(ISING_EINVAL, "ising_create_slabs: device index out of range");

    ising_sim *h = new_handle(model, L, beta, D, seed, cuda_stream);
    if (!h) return set_error(ISING_ENOMEM, "ising_create_slabs: host allocation failed");
    h->device = devices ? devices[0] : cur;
    // plain loads across devices: every device used maps every other one
    for (int a = 0; devices && a < n_slabs; ++a)
        for (int b = 0; b < n_slabs; ++b) {
            if (devices[a] == devices[b]) continue;
            DeviceGuard g(devices[a]);
            cudaError_t e = cudaDeviceEnablePeerAccess(devices[b], 0);
            if (e == cudaErrorPeerAccessAlreadyEnabled) { cudaGetLastError(); continue; }
            if (e != cudaSuccess) { delete h; return cuda_fail(e, "cudaDeviceEnablePeerAccess (slabs on devices without peer access)"); }
        }
    int64_t y0 = 0;
    for (int k = 0; k < n_slabs; ++k) {
        Slab sl;
        sl.device = devices ? devices[k] : cur;
        sl.y0 = y0; sl.rows = rows[k];
        y0 += rows[k];
        DeviceGuard g(sl.device);
        cudaError_t e = cudaSuccess;
        if (k == 0) sl.stream = h->stream;
        else { e = cudaStreamCreateWithFlags(&sl.stream, cudaStreamNonBlocking); sl.own_stream = e == cudaSuccess; }
        const size_t bytes = (size_t)sl.rows * (size_t)colour_row_words(h) * 16 + kScratchBytes;
        if (e == cudaSuccess) e = cudaMalloc(&sl.owned, bytes);
        h->slabs.push_back(sl);                      // before the error check: ising_destroy frees what exists
        if (e != cudaSuccess) {
            cudaGetLastError();
            ising_destroy(h);
            return set_error(e == cudaErrorMemoryAllocation ? ISING_ENOMEM : ISING_ECUDA,
                             std::string("ising_create_slabs: slab allocation: ") + cudaGetErrorString(e));
        }
        carve_slab(h, h->slabs.back(), (char *)sl.owned);
    }
    return finish_create(h, out);
}

extern "C" int ising_slab_count(const ising_t *h) { return h ? (int)h->slabs.size() : 0; }

extern "C" int ising_slab_info(const ising_t *h, int slab, int64_t *y0, int64_t *rows, int *device)
{
    if (!h || slab < 0 || slab >= (int)h->slabs.size()) return set_error(ISING_EINVAL, "ising_slab_info: bad handle or slab index");
    if (y0) *y0 = h->slabs[slab].y0;
    if (rows) *rows = h->slabs[slab].rows;
    if (device) *device = h->slabs[slab].device;
    return ISING_OK;
}

// ------------------------------------------------- one slab per process ---
// The torch.distributed arrangement (one process per GPU): every rank creates the handle of its own slab, the
// ranks exchange 64-byte CUDA IPC handles of the slab allocations (an all-gather), map the slabs above and below,
// and from then on the update / observables kernels read the two halo rows from the neighbours' memory with plain
// loads.  What has to be ordered across ranks is one thing only: a colour phase may start when the
// previous phase of both neighbours has finished -- ising_sweep_phase launches one phase, the caller puts a
// stream-ordered collective (e.g. an NCCL all-reduce of one word) or a host barrier between two phases.
extern "C" int ising_create_part(int model, int64_t L, double beta, double D, uint64_t seed, int64_t y0, int64_t rows,
                                 void *cuda_stream, ising_t **out)
{
    int rc = check_create_args("ising_create_part", model, L, beta, D, out);
    if (rc) return rc;
    if (y0 < 0 || rows < 2 || (y0 & 1) || (rows & 1) || y0 + rows > L)
        return set_error(ISING_EINVAL, "ising_create_part: y0 and rows must be even, rows >= 2, y0 + rows <= L");
    ising_sim *h = new_handle(model, L, beta, D, seed, cuda_stream);
    if (!h) return set_error(ISING_ENOMEM, "ising_create_part: host allocation failed");
    h->part = true;
    cudaGetDevice(&h->device);
    Slab sl;
    sl.device = h->device; sl.stream = h->stream; sl.y0 = y0; sl.rows = rows;
    const size_t bytes = (size_t)rows * (size_t)colour_row_words(h) * 16 + kScratchBytes;
    cudaError_t e = cudaMalloc(&sl.owned, bytes);
    if (e != cudaSuccess) {
        delete h;
        cudaGetLastError();
        return set_error(e == cudaErrorMemoryAllocation ? ISING_ENOMEM : ISING_ECUDA,
                         std::string("ising_create_part: cudaMalloc: ") + cudaGetErrorString(e));
    }
    carve_slab(h, sl, (char *)sl.owned);
    h->slabs.push_back(sl);
    if (rows == L) {                                  // the only part: its halo rows are its own last and first row
        for (int c = 0; c < 2; ++c) {
            h->part_halo[0][c] = sl.lat[c] + (rows - 1) * colour_row_words(h);
            h->part_halo[1][c] = sl.lat[c];
        }
    }
    return finish_create(h, out);
}

extern "C" int ising_part_export(ising_t *h, void *ipc_handle)
{
    DeviceGuard dev_guard(h);
    if (!h || !ipc_handle || !h->part) return set_error(ISING_EINVAL, "ising_part_export: needs a handle made by ising_create_part");
    static_assert(sizeof(cudaIpcMemHandle_t) == ISING_IPC_HANDLE_BYTES, "ISING_IPC_HANDLE_BYTES");
    cudaIpcMemHandle_t mh;
    CUDA_TRY(cudaIpcGetMemHandle(&mh, h->slabs[0].owned));
    memcpy(ipc_handle, &mh, sizeof(mh));
    return ISING_OK;
}

extern "C" int ising_part_attach(ising_t *h, const void *ipc_above, int64_t rows_above, const void *ipc_below, int64_t rows_below)
{
    DeviceGuard dev_guard(h);
    if (!h || !h->part || !ipc_above || !ipc_below) return set_error(ISING_EINVAL, "ising_part_attach: needs a part handle and both neighbours' IPC handles");
    if (rows_above < 2 || rows_below < 2 || (rows_above & 1) || (rows_below & 1))
        return set_error(ISING_EINVAL, "ising_part_attach: neighbour heights must be even and >= 2");
    if (h->part_ipc[0] || h->part_ipc[1] || h->part_halo[0][0]) return set_error(ISING_EINVAL, "ising_part_attach: neighbours already attached");
    const bool same = memcmp(ipc_above, ipc_below, ISING_IPC_HANDLE_BYTES) == 0;     // two parts: one neighbour on both sides
    const void *src[2] = {ipc_above, ipc_below};
    for (int k = 0; k < (same ? 1 : 2); ++k) {
        cudaIpcMemHandle_t mh;
        memcpy(&mh, src[k], sizeof(mh));
        cudaError_t e = cudaIpcOpenMemHandle(&h->part_ipc[k], mh, cudaIpcMemLazyEnablePeerAccess);
        if (e != cudaSuccess) { h->part_ipc[k] = nullptr; return cuda_fail(e, "cudaIpcOpenMemHandle (neighbour slab)"); }
    }
    // a part's allocation is [colour 0 rows | colour 1 rows | scratch] (carve_slab)
    const int64_t rw = colour_row_words(h);
    const uint64_t *above = (const uint64_t *)h->part_ipc[0], *below = (const uint64_t *)(same ? h->part_ipc[0] : h->part_ipc[1]);
    for (int c = 0; c < 2; ++c) {
        h->part_halo[0][c] = above + (int64_t)c * rows_above * rw + (rows_above - 1) * rw;     // last row of the slab above
        h->part_halo[1][c] = below + (int64_t)c * rows_below * rw;                             // first row of the slab below
    }
    return ISING_OK;
}

extern "C" int ising_sweep_phase(ising_t *h, int colour)
{
    DeviceGuard dev_guard(h);
    if (!h || (colour != 0 && colour != 1)) return set_error(ISING_EINVAL, "ising_sweep_phase: bad argument");
    if (!h->part || !h->part_halo[0][0]) return set_error(ISING_EINVAL, "ising_sweep_phase: needs a part handle with its neighbours attached");
    if (colour != h->part_phase) return set_error(ISING_EINVAL, "ising_sweep_phase: the phases of a sweep are colour 0, then colour 1");
    if (h->t >= 0xFFFFFFFFull) return set_error(ISING_EINVAL, "ising_sweep_phase: sweep counter would exceed 2^32-1");
    cudaError_t e = (h->model == ISING_MODEL_ISING_LUT) ? launch_lut_update(h, 0, colour, (uint32_t)h->t) : launch_update(h, 0, colour, (uint32_t)h->t);
    if (e != cudaSuccess) return cuda_fail(e, "update kernel");
    h->part_phase = 1 - colour;
    if (colour == 1) h->t++;
    return ISING_OK;
}

extern "C" int ising_destroy(ising_t *h)
{
    if (!h) return ISING_OK;
    for (Slab &sl : h->slabs) {
        DeviceGuard g(sl.device);
        cudaStreamSynchronize(sl.stream);
    }
    {
        DeviceGuard dev_guard(h);
        if (h->io_stage) cudaFree(h->io_stage);
        if (h->io_stream) cudaStreamDestroy(h->io_stream);
        if (h->io_event) cudaEventDestroy(h->io_event);
        if (h->planes) cudaFree(h->planes);
        if (h->comb) cudaFree(h->comb);
        if (h->gram) cudaFree(h->gram);
        drop_graph(h);
        if (h->d_corr) cudaFree(h->d_corr);
        if (h->d_rlist) cudaFree(h->d_rlist);
        if (h->h_acc) cudaFreeHost(h->h_acc);
    }
    for (int k = 0; k < 2; ++k)
        if (h->part_ipc[k]) { DeviceGuard g(h->device); cudaIpcCloseMemHandle(h->part_ipc[k]); }
    for (Slab &sl : h->slabs) {
        DeviceGuard g(sl.device);
        if (sl.lut_buckets) cudaFree(sl.lut_buckets);
        if (sl.done) cudaEventDestroy(sl.done);
        if (sl.own_stream) cudaStreamDestroy(sl.stream);
        if (sl.owned) cudaFree(sl.owned);
    }
    delete h;
    return ISING_OK;
}

// ------------------------------------------------------- slab sequencing ---
// Work that touches the whole lattice through one stream (IO, bit planes, copies) runs on the main stream
// = slab 0's; per-slab kernels run on the slab's own stream and device.  fan_out: every slab stream waits
// for what is queued on the main stream; fan_in: the main stream waits for every slab stream.  Both are
// no-ops for an unsharded lattice.
static int fan_out(ising_sim *h)
{
    if (h->slabs.size() < 2) return ISING_OK;
    {
        DeviceGuard g(h->slabs[0].device);
        CUDA_TRY(cudaEventRecord(h->slabs[0].done, h->slabs[0].stream));
    }
    for (size_t k = 1; k < h->slabs.size(); ++k) {
        DeviceGuard g(h->slabs[k].device);
        CUDA_TRY(cudaStreamWaitEvent(h->slabs[k].stream, h->slabs[0].done, 0));
    }
    return ISING_OK;
}

static int fan_in(ising_sim *h)
{
    for (size_t k = 1; k < h->slabs.size(); ++k) {
        {
            DeviceGuard g(h->slabs[k].device);
            CUDA_TRY(cudaEventRecord(h->slabs[k].done, h->slabs[k].stream));
        }
        DeviceGuard g(h->slabs[0].device);
        CUDA_TRY(cudaStreamWaitEvent(h->slabs[0].stream, h->slabs[k].done, 0));
    }
    return ISING_OK;
}

// One per-slab pass (observables, histogram): launch(k) on every slab between fan_out and fan_in.
template <typename F>
static int for_each_slab(ising_sim *h, const char *what, F launch)
{
    int rc = fan_out(h);
    if (rc) return rc;
    for (int k = 0; k < (int)h->slabs.size(); ++k) {
        DeviceGuard g(h->slabs[k].device);
        cudaError_t e = launch(k);
        if (e != cudaSuccess) return cuda_fail(e, what);
    }
    return fan_in(h);
}

// Mirror the accumulators [first, first + n) of every slab into h_acc[64 k + first ...] and add them up in int64.
static int sum_over_slabs(ising_sim *h, int first, int n, long long *total)
{
    for (int k = 0; k < (int)h->slabs.size(); ++k)
        CUDA_TRY(cudaMemcpyAsync(h->h_acc + 64 * k + first, h->slabs[k].d_acc + first, n * sizeof(long long),
                                 cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    for (int j = 0; j < n; ++j) {
        total[j] = 0;
        for (int k = 0; k < (int)h->slabs.size(); ++k) total[j] += h->h_acc[64 * k + first + j];
    }
    return ISING_OK;
}

extern "C" int ising_sync(ising_t *h)
{
    DeviceGuard dev_guard(h);
    if (!h) return set_error(ISING_EINVAL, "ising_sync: NULL handle");
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    return ISING_OK;
}

extern "C" int64_t ising_launch_count(const ising_t *h) { return h ? h->launches : 0; }

// ----------------------------------------------------------------- sweep ---
// Launch-bound lattices (a colour phase of a few microseconds): sweeps are replayed from a CUDA graph
// of kGraphSweeps sweeps whose kernels carry t = 0..K-1; the base sweep number is a device word that
// a one-thread kernel sets before every replay.  Same kernels, same numbers, fewer launch gaps.
static const int kGraphSweeps = 16;
#ifndef GRAPH_MAX_SITES
#define GRAPH_MAX_SITES (1ll << 28)
#endif
static const int64_t kGraphMaxSites = GRAPH_MAX_SITES;      // L <= 2^14

__global__ void set_t_base_kernel(uint32_t *t_base, uint32_t value) { *t_base = value; }

// One colour phase of sweep t on every slab.  A slab's kernel reads the boundary rows of its two neighbours
// (written by their previous phase) and overwrites rows they read in that phase, so it waits for the previous
// phase of both; slabs of the same phase run concurrently on their own streams.  Unsharded: one launch.
static cudaError_t launch_colour(ising_sim *h, int c, uint32_t t)
{
    const int S = (int)h->slabs.size();
    for (int k = 0; S > 1 && k < S; ++k) {
        DeviceGuard g(h->slabs[k].device);
        for (int nb : {(k + S - 1) % S, (k + 1) % S}) {
            if (nb == k) continue;
            cudaError_t e = cudaStreamWaitEvent(h->slabs[k].stream, h->slabs[nb].done, 0);
            if (e != cudaSuccess) return e;
        }
    }
    for (int k = 0; k < S; ++k) {
        DeviceGuard g(h->slabs[k].device);
        cudaError_t e = (h->model == ISING_MODEL_ISING_LUT) ? launch_lut_update(h, k, c, t) : launch_update(h, k, c, t);
        if (e != cudaSuccess) return e;
    }
    for (int k = 0; S > 1 && k < S; ++k) {
        DeviceGuard g(h->slabs[k].device);
        cudaError_t e = cudaEventRecord(h->slabs[k].done, h->slabs[k].stream);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

static void drop_graph(ising_sim *h)
{
    for (int k = 0; k < 2; ++k)
        if (h->graph_exec[k]) { cudaGraphExecDestroy(h->graph_exec[k]); h->graph_exec[k] = nullptr; }
}

// A dependent plain launch costs about 2.4 microseconds on B200; a colour phase takes 1.5 us at L = 1024, 10 us at
// L = 4096, 104 us at L = 2^14.  Replaying the sweeps from a graph removes that gap: +30 % at L = 4096, +9 % at 8192,
// +2.3 % at 2^14 (profiles/r02_README.md); above that it is below 1 % and the graph is not built.
static bool graph_allowed(const ising_sim *h)
{
    return h->L * h->L <= kGraphMaxSites && h->slabs.size() == 1 && !h->part && (h->sweep_mode <= 1 || h->sweep_mode >= 3);
}

// Graph `slot` holding `sweeps` sweeps whose kernels carry t = 0..sweeps-1 (the base sweep number is a device word).
static int ensure_graph(ising_sim *h, int slot, int sweeps)
{
    const int key[5] = {h->rows_per_thread, h->block_threads, h->variant, h->tally_on ? 1 : 0, sweeps};
    if (h->graph_exec[slot] && memcmp(key, h->graph_key[slot], sizeof(key)) == 0) return ISING_OK;
    if (h->graph_exec[slot]) { cudaGraphExecDestroy(h->graph_exec[slot]); h->graph_exec[slot] = nullptr; }
    // captured on a private stream (the caller's may be the legacy default stream, which cannot be
    // captured); the instantiated graph is then launched on the caller's stream
    cudaGraph_t graph = nullptr;
    cudaStream_t cap = nullptr, user = h->stream;
    CUDA_TRY(cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking));
    cudaError_t e = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal);
    if (e != cudaSuccess) { cudaStreamDestroy(cap); return cuda_fail(e, "cudaStreamBeginCapture"); }
    h->graph_capture = true;
    h->stream = h->slabs[0].stream = cap;
    const int64_t launches_before = h->launches;
    for (int j = 0; j < sweeps && e == cudaSuccess; ++j)
        for (int c = 0; c < 2 && e == cudaSuccess; ++c) e = launch_colour(h, c, (uint32_t)j);
    h->stream = h->slabs[0].stream = user;
    h->graph_capture = false;
    h->launches = launches_before;                              // counted when the graph is replayed
    cudaError_t e2 = cudaStreamEndCapture(cap, &graph);
    cudaStreamDestroy(cap);
    if (e != cudaSuccess || e2 != cudaSuccess) {
        if (graph) cudaGraphDestroy(graph);
        return cuda_fail(e != cudaSuccess ? e : e2, "CUDA graph capture of the sweep loop");
    }
    e = cudaGraphInstantiate(&h->graph_exec[slot], graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) { h->graph_exec[slot] = nullptr; return cuda_fail(e, "cudaGraphInstantiate"); }
    memcpy(h->graph_key[slot], key, sizeof(key));
    return ISING_OK;
}

static int replay_graph(ising_sim *h, int slot, int sweeps)
{
    uint32_t *t_base = reinterpret_cast<uint32_t *>(h->d_acc + 48) + 1;
    set_t_base_kernel<<<1, 1, 0, h->stream>>>(t_base, (uint32_t)h->t);
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaGraphLaunch(h->graph_exec[slot], h->stream));
    h->launches += 1 + 2 * sweeps;
    h->t += sweeps;
    return ISING_OK;
}

extern "C" int ising_sweep(ising_t *h, int64_t n)
{
    DeviceGuard dev_guard(h);
    if (!h) return set_error(ISING_EINVAL, "ising_sweep: NULL handle");
    if (n < 0) return set_error(ISING_EINVAL, "ising_sweep: n < 0");
    if (h->t + (uint64_t)n > 0xFFFFFFFFull) return set_error(ISING_EINVAL, "ising_sweep: sweep counter would exceed 2^32-1");
    if (h->part && (h->slabs[0].rows != h->L || h->part_phase != 0))
        return set_error(ISING_EINVAL, "ising_sweep: one part of a lattice is swept phase by phase (ising_sweep_phase), with the "
                                       "caller's barrier between the phases");
    const bool small = h->L * h->L <= (1ll << 22) && h->slabs.size() == 1 && !h->part;      // launch-bound: L <= 2048
    // Tiny lattices (L <= 512; mode 4: whatever fits): one cluster of 16 CTAs keeps the lattice in distributed shared
    // memory for all n sweeps, the colour phases separated by the hardware cluster barrier (update.cu).
    if (small && n >= 2 && h->model != ISING_MODEL_ISING_LUT && ((h->sweep_mode == 0 && h->L <= 512) || h->sweep_mode == 4)) {
        while (n > 0) {
            const int chunk = (int)std::min<int64_t>(n, 4096);          // bounds the 32-bit per-warp tally sums
            cudaError_t e = launch_sweeps_cluster(h, (uint32_t)h->t, chunk);
            if (e == cudaErrorNotSupported) break;
            if (e != cudaSuccess) return cuda_fail(e, "cluster sweep kernel");
            h->t += (uint64_t)chunk;
            n -= chunk;
        }
    }
    // On request (ising_set_sweep_mode 3): n sweeps in one cooperative launch with a grid barrier per colour phase
    // (update.cu).  Measured slower than the CUDA graph below (L = 256: 5.95 against 5.5 microseconds per sweep): a
    // barrier through L2 costs what a kernel boundary inside a graph costs.
    if (small && n >= 2 && h->sweep_mode == 3 && h->model != ISING_MODEL_ISING_LUT) {
        while (n > 0) {
            const int chunk = (int)std::min<int64_t>(n, 4096);          // bounds the 32-bit per-warp tally sums
            cudaError_t e = launch_sweeps_persistent(h, (uint32_t)h->t, chunk);
            if (e == cudaErrorNotSupported) break;
            if (e != cudaSuccess) return cuda_fail(e, "persistent sweep kernel");
            h->t += (uint64_t)chunk;
            n -= chunk;
        }
    }
    if (graph_allowed(h) && n >= 2 * kGraphSweeps) {
        int rc = ensure_graph(h, 0, kGraphSweeps);
        if (rc) return rc;
        while (n >= kGraphSweeps) {
            rc = replay_graph(h, 0, kGraphSweeps);
            if (rc) return rc;
            n -= kGraphSweeps;
        }
    } else if (graph_allowed(h) && n >= 4) {
        // a short count asked for a second time in a row gets a graph of exactly that many sweeps
        if (n == h->last_short_n) {
            int rc = ensure_graph(h, 1, (int)n);
            if (rc) return rc;
            rc = replay_graph(h, 1, (int)n);
            if (rc) return rc;
            n = 0;
        } else {
            h->last_short_n = n;
        }
    }
    if (n > 0) {
        int rc = fan_out(h);
        if (rc) return rc;
    }
    for (int64_t i = 0; i < n; ++i) {
        for (int c = 0; c < 2; ++c) {
            cudaError_t e = launch_colour(h, c, (uint32_t)h->t);
            if (e != cudaSuccess) return cuda_fail(e, "update kernel");
        }
        h->t++;
    }
    return n > 0 ? fan_in(h) : ISING_OK;
}

// A11: sweep to every time of an ascending schedule and record B, M, Q there (fused tally if it is on,
// else the observables pass).  One call for "E and M every k sweeps" (BASELINE.json configs 1-3).
extern "C" int ising_run_schedule(ising_t *h, int64_t n_times, const uint64_t *times, ising_obs_t *out)
{
    DeviceGuard dev_guard(h);
    if (!h || !times || !out || n_times < 0) return set_error(ISING_EINVAL, "ising_run_schedule: bad argument");
    uint64_t prev = h->t;
    for (int64_t i = 0; i < n_times; ++i) {
        if (times[i] < prev) return set_error(ISING_EINVAL, "ising_run_schedule: times must be ascending and >= sweeps_done");
        prev = times[i];
    }
    for (int64_t i = 0; i < n_times; ++i) {
        int rc = ising_sweep(h, (int64_t)(times[i] - h->t));
        if (rc) return rc;
        rc = h->tally_on ? ising_tally(h, &out[i]) : ising_observables(h, &out[i]);
        if (rc) return rc;
    }
    return ISING_OK;
}

extern "C" int ising_set_sweeps_done(ising_t *h, uint64_t t)
{
    DeviceGuard dev_guard(h);
    if (!h) return set_error(ISING_EINVAL, "ising_set_sweeps_done: NULL handle");
    if (t > 0xFFFFFFFFull) return set_error(ISING_EINVAL, "ising_set_sweeps_done: t > 2^32-1");
    h->t = t;
    return ISING_OK;
}

extern "C" int ising_set_launch(ising_t *h, int rows_per_thread, int block_threads)
{
    DeviceGuard dev_guard(h);
    if (!h) return set_error(ISING_EINVAL, "ising_set_launch: NULL handle");
    if (rows_per_thread < 0 || (rows_per_thread & 1) || rows_per_thread > 4096)
        return set_error(ISING_EINVAL, "ising_set_launch: rows_per_thread must be even, in [2, 4096] (0 = keep)");
    if (block_threads < 0 || (block_threads % 32) || block_threads > 256)
        return set_error(ISING_EINVAL, "ising_set_launch: block_threads must be a multiple of 32, <= 256 (0 = keep)");
    if (rows_per_thread) h->rows_per_thread = rows_per_thread;
    if (block_threads) h->block_threads = block_threads;
    return ISING_OK;
}

extern "C" int ising_set_sweep_mode(ising_t *h, int mode)
{
    DeviceGuard dev_guard(h);
    if (!h) return set_error(ISING_EINVAL, "ising_set_sweep_mode: NULL handle");
    if (mode < 0 || mode > 4) return set_error(ISING_EINVAL, "ising_set_sweep_mode: mode must be 0 (auto), 1 (CUDA graph), 2 (plain launches), 3 (persistent kernel) or 4 (cluster kernel)");
    h->sweep_mode = mode;
    return ISING_OK;
}

extern "C" int ising_set_variant(ising_t *h, int variant)
{
    DeviceGuard dev_guard(h);
    if (!h) return set_error(ISING_EINVAL, "ising_set_variant: NULL handle");
    if (variant < 0 || variant > (h->model == ISING_MODEL_ISING_LUT ? 2 : 1)) return set_error(ISING_EINVAL, "ising_set_variant: unknown variant");
    h->variant = variant;
    return ISING_OK;
}

// Rows a handle holds: all of them, or [y0, y0 + rows) for one part of a lattice (ising_create_part).
static int64_t local_sites(const ising_sim *h) { return (h->part ? h->slabs[0].rows : h->L) * h->L; }

static int check_local_rows(const ising_sim *h, const char *who, int64_t y0, int64_t ny)
{
    if (!h->part) return ISING_OK;
    const Slab &sl = h->slabs[0];
    if (y0 < sl.y0 || y0 + ny > sl.y0 + sl.rows)
        return set_error(ISING_EINVAL, std::string(who) + ": rows outside this part of the lattice (ising_slab_info gives its range)");
    return ISING_OK;
}

static int no_parts(const ising_sim *h, const char *who)
{
    if (h->part && h->slabs[0].rows != h->L)
        return set_error(ISING_EINVAL, std::string(who) + ": needs the whole lattice, this handle holds one part of it");
    return ISING_OK;
}

// ----------------------------------------------------------- observables ---
static int observe_all_slabs(ising_sim *h)                // -> d_acc[0..2] of every slab
{
    if (h->part && !h->part_halo[0][0]) return set_error(ISING_EINVAL, "observables of a part need its neighbours (ising_part_attach)");
    const bool lut = h->model == ISING_MODEL_ISING_LUT;
    return for_each_slab(h, "observables kernel", [&](int k) { return lut ? launch_lut_observables(h, k) : launch_observables(h, k); });
}

static void fill_obs(const ising_sim *h, const long long *bmq, ising_obs_t *o)
{
    const bool lut = h->model == ISING_MODEL_ISING_LUT;
    o->bond_sum = bmq[0]; o->M = bmq[1]; o->Q = (lut || h->model == ISING_MODEL_ISING) ? local_sites(h) : bmq[2];
    o->n_sites = local_sites(h); o->sweeps_done = h->t;       // one part of a lattice: the sums and N of its own rows
    const double N = (double)local_sites(h);
    o->E = !is_blume_capel(h->model) ? -(double)o->bond_sum : -(double)o->bond_sum + h->D * (double)o->Q;
    o->e_per_site = o->E / N;
    o->m_per_site = (double)o->M / N;
    o->zero_density = (double)(o->n_sites - o->Q) / N;
}

extern "C" int ising_observables(ising_t *h, ising_obs_t *out)
{
    DeviceGuard dev_guard(h);
    if (!h || !out) return set_error(ISING_EINVAL, "ising_observables: NULL argument");
    int rc = observe_all_slabs(h);
    if (rc) return rc;
    long long bmq[3];                                    // every slab's sums, added in int64
    rc = sum_over_slabs(h, 0, 3, bmq);
    if (rc) return rc;
    fill_obs(h, bmq, out);
    return ISING_OK;
}

// A7: fused tally.  d_acc[40..42] hold running B, M, Q; the update kernels add the changes.
static int tally_resync(ising_sim *h)
{
    int rc = observe_all_slabs(h);
    if (rc) return rc;
    for (const Slab &sl : h->slabs)                      // every slab keeps the running sums of its own rows
        CUDA_TRY(cudaMemcpyAsync(sl.d_acc + 40, sl.d_acc, 3 * sizeof(long long), cudaMemcpyDeviceToDevice, h->stream));
    return ISING_OK;
}

extern "C" int ising_set_tally(ising_t *h, int on)
{
    DeviceGuard dev_guard(h);
    if (!h) return set_error(ISING_EINVAL, "ising_set_tally: NULL handle");
    h->tally_on = on != 0;
    return h->tally_on ? tally_resync(h) : ISING_OK;
}

extern "C" int ising_tally(ising_t *h, ising_obs_t *out)
{
    DeviceGuard dev_guard(h);
    if (!h || !out) return set_error(ISING_EINVAL, "ising_tally: NULL argument");
    if (!h->tally_on) return set_error(ISING_EINVAL, "ising_tally: the tally is off (ising_set_tally)");
    long long bmq[3];
    int rc = sum_over_slabs(h, 40, 3, bmq);
    if (rc) return rc;
    fill_obs(h, bmq, out);
    return ISING_OK;
}

extern "C" int ising_schwinger_dyson(ising_t *h, int64_t hist[9], double *value)
{
    DeviceGuard dev_guard(h);
    if (!h || !hist || !value) return set_error(ISING_EINVAL, "ising_schwinger_dyson: NULL argument");
    const bool lut = h->model == ISING_MODEL_ISING_LUT;
    if (h->part && !h->part_halo[0][0]) return set_error(ISING_EINVAL, "ising_schwinger_dyson: a part needs its neighbours (ising_part_attach)");
    int rc = for_each_slab(h, "Schwinger-Dyson kernel", [&](int k) { return lut ? launch_lut_sd_hist(h, k) : launch_sd_hist(h, k); });
    if (rc) return rc;
    long long bins[9];
    rc = sum_over_slabs(h, 8, 9, bins);
    if (rc) return rc;
    double acc = 0.0;
    for (int k = -4; k <= 4; ++k) {
        hist[k + 4] = bins[k + 4];
        acc += (double)hist[k + 4] * exp(-2.0 * h->beta * (double)k);
    }
    *value = acc / (double)local_sites(h);
    return ISING_OK;
}

extern "C" int ising_thresholds(ising_t *h, uint64_t *out, int cap, int *count)
{
    DeviceGuard dev_guard(h);
    if (!h || !count) return set_error(ISING_EINVAL, "ising_thresholds: NULL argument");
    *count = h->n_T;
    if (!out) return ISING_OK;                                   // size query
    if (cap < h->n_T) return set_error(ISING_EINVAL, "ising_thresholds: cap too small");
    memcpy(out, h->T, h->n_T * sizeof(uint64_t));
    return ISING_OK;
}

// ------------------------------------------------------------ lattice IO ---
static int ensure_stage(ising_sim *h, size_t bytes)
{
    if (h->io_stage_bytes >= bytes) return ISING_OK;
    if (h->io_stage) { cudaFree(h->io_stage); h->io_stage = nullptr; h->io_stage_bytes = 0; }
    cudaError_t e = cudaMalloc(&h->io_stage, bytes);
    if (e != cudaSuccess) { cudaGetLastError(); return set_error(ISING_ENOMEM, "staging buffer: cudaMalloc failed"); }
    h->io_stage_bytes = bytes;
    return ISING_OK;
}

static const int64_t kStageBytes = 64ll << 20;

extern "C" int ising_read_window(ising_t *h, int64_t x0, int64_t y0, int64_t w, int64_t hgt, int8_t *host_out)
{
    DeviceGuard dev_guard(h);
    if (!h || !host_out) return set_error(ISING_EINVAL, "ising_read_window: NULL argument");
    if (w < 1 || hgt < 1 || w > h->L || hgt > h->L) return set_error(ISING_EINVAL, "ising_read_window: window size out of range");
    if (int rcp = check_local_rows(h, "ising_read_window", y0, hgt)) return rcp;
    const int64_t L = h->L;
    x0 = ((x0 % L) + L) % L; y0 = ((y0 % L) + L) % L;
    const int64_t rows_per = std::max<int64_t>(1, std::min<int64_t>(hgt, kStageBytes / w));
    int rc = ensure_stage(h, (size_t)(rows_per * w) + 16);
    if (rc) return rc;
    for (int64_t j = 0; j < hgt; j += rows_per) {
        const int64_t nr = std::min(rows_per, hgt - j);
        cudaError_t e = launch_unpack(h, x0, (y0 + j) % L, w, nr, (int8_t *)h->io_stage);
        if (e != cudaSuccess) return cuda_fail(e, "unpack kernel");
        CUDA_TRY(cudaMemcpyAsync(host_out + j * w, h->io_stage, (size_t)(nr * w), cudaMemcpyDeviceToHost, h->stream));
        CUDA_TRY(cudaStreamSynchronize(h->stream));
    }
    return ISING_OK;
}

extern "C" int ising_read_lattice(ising_t *h, int64_t y0, int64_t ny, int8_t *host_out)
{
    DeviceGuard dev_guard(h);
    if (!h || !host_out) return set_error(ISING_EINVAL, "ising_read_lattice: NULL argument");
    if (y0 < 0 || ny < 1 || y0 + ny > h->L) return set_error(ISING_EINVAL, "ising_read_lattice: rows outside [0, L]");
    return ising_read_window(h, 0, y0, h->L, ny, host_out);
}

extern "C" int ising_write_lattice(ising_t *h, int64_t y0, int64_t ny, const int8_t *host_in)
{
    DeviceGuard dev_guard(h);
    if (!h || !host_in) return set_error(ISING_EINVAL, "ising_write_lattice: NULL argument");
    if (y0 < 0 || ny < 1 || y0 + ny > h->L) return set_error(ISING_EINVAL, "ising_write_lattice: rows outside [0, L]");
    if (int rcp = check_local_rows(h, "ising_write_lattice", y0, ny)) return rcp;
    const int64_t L = h->L;
    const int64_t rows_per = std::max<int64_t>(1, std::min<int64_t>(ny, kStageBytes / L));
    int rc = ensure_stage(h, (size_t)(rows_per * L) + 16);
    if (rc) return rc;
    int *d_bad = (int *)(h->d_acc + 32);
    const bool one_chunk = ny <= rows_per;
    // pass 0 validates every chunk, pass 1 writes: the lattice is untouched on bad input
    for (int pass = 0; pass < 2; ++pass)
        for (int64_t j = 0; j < ny; j += rows_per) {
            const int64_t nr = std::min(rows_per, ny - j);
            if (pass == 0 || !one_chunk)
                CUDA_TRY(cudaMemcpyAsync(h->io_stage, host_in + j * L, (size_t)(nr * L), cudaMemcpyHostToDevice, h->stream));
            cudaError_t e = launch_pack(h, y0 + j, nr, (const int8_t *)h->io_stage, d_bad, pass);
            if (e == cudaErrorInvalidValue)
                return set_error(ISING_EINVAL, "ising_write_lattice: spin value outside the model's set");
            if (e != cudaSuccess) return cuda_fail(e, "pack kernel");
            if (pass == 1) CUDA_TRY(cudaStreamSynchronize(h->stream));   // staging buffer is reused
        }
    return h->tally_on ? tally_resync(h) : ISING_OK;
}

extern "C" int ising_read_packed(ising_t *h, int colour, int64_t word0, int64_t nwords, uint64_t *host_out)
{
    DeviceGuard dev_guard(h);
    if (!h || !host_out) return set_error(ISING_EINVAL, "ising_read_packed: NULL argument");
    if ((colour != 0 && colour != 1) || word0 < 0 || nwords < 0 || word0 + nwords > colour_words(h))
        return set_error(ISING_EINVAL, "ising_read_packed: range outside the colour array");
    if (h->part && (word0 < h->slabs[0].y0 * colour_row_words(h) || word0 + nwords > (h->slabs[0].y0 + h->slabs[0].rows) * colour_row_words(h)))
        return set_error(ISING_EINVAL, "ising_read_packed: words outside this part of the lattice");
    for (const Slab &sl : h->slabs) {                    // the word range, slab by slab
        const int64_t first = sl.y0 * colour_row_words(h), last = first + sl.rows * colour_row_words(h);
        const int64_t a = std::max(word0, first), b = std::min(word0 + nwords, last);
        if (a < b) CUDA_TRY(cudaMemcpyAsync(host_out + (a - word0), sl.lat[colour] + (a - first), (size_t)(b - a) * 8, cudaMemcpyDeviceToHost, h->stream));
    }
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    return ISING_OK;
}

extern "C" int ising_write_packed(ising_t *h, int colour, int64_t word0, int64_t nwords, const uint64_t *host_in)
{
    DeviceGuard dev_guard(h);
    if (!h || !host_in) return set_error(ISING_EINVAL, "ising_write_packed: NULL argument");
    if ((colour != 0 && colour != 1) || word0 < 0 || nwords < 0 || word0 + nwords > colour_words(h))
        return set_error(ISING_EINVAL, "ising_write_packed: range outside the colour array");
    if (h->part && (word0 < h->slabs[0].y0 * colour_row_words(h) || word0 + nwords > (h->slabs[0].y0 + h->slabs[0].rows) * colour_row_words(h)))
        return set_error(ISING_EINVAL, "ising_write_packed: words outside this part of the lattice");
    for (const Slab &sl : h->slabs) {
        const int64_t first = sl.y0 * colour_row_words(h), last = first + sl.rows * colour_row_words(h);
        const int64_t a = std::max(word0, first), b = std::min(word0 + nwords, last);
        if (a < b) CUDA_TRY(cudaMemcpyAsync(sl.lat[colour] + (a - first), host_in + (a - word0), (size_t)(b - a) * 8, cudaMemcpyHostToDevice, h->stream));
    }
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    return h->tally_on ? tally_resync(h) : ISING_OK;
}

// Compact transport format: 1 bit per Ising spin, 2 bits per Blume-Capel spin, rows of one
// colour array in the site order of the packed layout.  For the 1-bit and 2-bit models this IS the packed
// layout (a plain copy); the 4-bit models expand / gather on the device, chunk by chunk through the staging
// buffer, so that an upload moves the information content of the lattice and not its storage size.
static int64_t bits_row_words(const ising_sim *h) { return is_blume_capel(h->model) ? h->L / 64 : h->L / 128; }

static int bits_args(const ising_sim *h, const char *who, int colour, int64_t row0, int64_t nrows, const void *host)
{
    if (!h || !host) return set_error(ISING_EINVAL, std::string(who) + ": NULL argument");
    if ((colour != 0 && colour != 1) || row0 < 0 || nrows < 0 || row0 + nrows > h->L)
        return set_error(ISING_EINVAL, std::string(who) + ": colour or rows out of range");
    if (int rcp = check_local_rows(h, who, row0, nrows)) return rcp;
    if (!is_blume_capel(h->model) && (h->L % 128) != 0)
        return set_error(ISING_EINVAL, std::string(who) + ": one bit per spin needs L to be a multiple of 128 (whole 64-bit words per colour row)");
    return ISING_OK;
}

extern "C" int ising_write_bits(ising_t *h, int colour, int64_t row0, int64_t nrows, const uint64_t *host_in)
{
    DeviceGuard dev_guard(h);
    int rc = bits_args(h, "ising_write_bits", colour, row0, nrows, host_in);
    if (rc) return rc;
    const int64_t rw = bits_row_words(h);
    if (h->model == ISING_MODEL_ISING_LUT)                       // any bit pattern is a lattice: a plain copy
        return ising_write_packed(h, colour, row0 * rw, nrows * rw, host_in);
    const bool bc = is_blume_capel(h->model);
    // Blume-Capel input is validated before anything is written; up to 256 MB it stays in the staging buffer between
    // the two passes (one upload), beyond that every chunk is uploaded twice
    const int64_t stage_cap = bc ? 4 * kStageBytes : kStageBytes;
    const int64_t rows_per = std::max<int64_t>(1, std::min<int64_t>(nrows, stage_cap / (rw * 8)));
    const bool one_chunk = rows_per >= nrows;
    rc = ensure_stage(h, (size_t)(rows_per * rw * 8));
    if (rc) return rc;
    int *d_bad = (int *)(h->d_acc + 32);
    // The copies and the (small) expansion kernels run on a stream of the highest priority, ordered after what is
    // queued on the handle's stream: when another handle's sweeps fill the GPU (bench.py's pipelined end-to-end
    // run) an expansion kernel is then scheduled as soon as blocks retire, not after the running launch.
    if (!h->io_stream) {
        int lo = 0, hi = 0;
        CUDA_TRY(cudaDeviceGetStreamPriorityRange(&lo, &hi));
        CUDA_TRY(cudaStreamCreateWithPriority(&h->io_stream, cudaStreamNonBlocking, hi));
        CUDA_TRY(cudaEventCreateWithFlags(&h->io_event, cudaEventDisableTiming));
    }
    CUDA_TRY(cudaEventRecord(h->io_event, h->stream));
    CUDA_TRY(cudaStreamWaitEvent(h->io_stream, h->io_event, 0));
    cudaStream_t user = h->stream;
    struct Swap {                                               // the launchers use h->stream
        ising_sim *h; cudaStream_t user;
        ~Swap() { h->stream = user; }
    } swap{h, user};
    h->stream = h->io_stream;
    // Blume-Capel: a first pass validates every chunk, so that the lattice is untouched on bad input
    for (int pass = bc ? 0 : 1; pass < 2; ++pass)
        for (int64_t j = 0; j < nrows; j += rows_per) {
            const int64_t nr = std::min(rows_per, nrows - j);
            if (pass == 0 || !bc || !one_chunk)
                CUDA_TRY(cudaMemcpyAsync(h->io_stage, host_in + j * rw, (size_t)(nr * rw * 8), cudaMemcpyHostToDevice, h->stream));
            cudaError_t e = launch_bits(h, colour, row0 + j, nr, (uint32_t *)h->io_stage, pass, d_bad);
            if (e == cudaErrorInvalidValue) return set_error(ISING_EINVAL, "ising_write_bits: a 2-bit code equal to 3");
            if (e != cudaSuccess) return cuda_fail(e, "bit expansion kernel");
        }
    CUDA_TRY(cudaStreamSynchronize(h->io_stream));              // the lattice is written: later work on the user's stream may follow
    h->stream = user;
    return h->tally_on ? tally_resync(h) : ISING_OK;
}

extern "C" int ising_read_bits(ising_t *h, int colour, int64_t row0, int64_t nrows, uint64_t *host_out)
{
    DeviceGuard dev_guard(h);
    int rc = bits_args(h, "ising_read_bits", colour, row0, nrows, host_out);
    if (rc) return rc;
    const int64_t rw = bits_row_words(h);
    if (h->model == ISING_MODEL_ISING_LUT || h->model == ISING_MODEL_BLUME_CAPEL_2BIT)
        return ising_read_packed(h, colour, row0 * rw, nrows * rw, host_out);
    const int64_t rows_per = std::max<int64_t>(1, std::min<int64_t>(nrows, kStageBytes / (rw * 8)));
    rc = ensure_stage(h, (size_t)(rows_per * rw * 8));
    if (rc) return rc;
    for (int64_t j = 0; j < nrows; j += rows_per) {
        const int64_t nr = std::min(rows_per, nrows - j);
        cudaError_t e = launch_bits(h, colour, row0 + j, nr, (uint32_t *)h->io_stage, 2, nullptr);
        if (e != cudaSuccess) return cuda_fail(e, "bit gather kernel");
        CUDA_TRY(cudaMemcpyAsync(host_out + j * rw, h->io_stage, (size_t)(nr * rw * 8), cudaMemcpyDeviceToHost, h->stream));
    }
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    return ISING_OK;
}

// ----------------------------------------------------------- correlation ---
static int ensure_planes(ising_sim *h)
{
    const size_t pw = (size_t)h->L * (size_t)(h->L / 64);
    const size_t bytes = pw * 8 * (is_blume_capel(h->model) ? 4 : 2);
    if (h->planes_bytes >= bytes) return ISING_OK;
    cudaError_t e = cudaMalloc((void **)&h->planes, bytes);
    if (e != cudaSuccess) { cudaGetLastError(); h->planes = nullptr; return set_error(ISING_ENOMEM, "bit planes: cudaMalloc failed"); }
    h->planes_bytes = bytes;
    return ISING_OK;
}

static int ensure_comb(ising_sim *h, int64_t stride)
{
    const size_t bytes = (size_t)h->L * (size_t)comb_words_per_row(h->L, stride) * 8 *
                         (is_blume_capel(h->model) ? 4 : 2);
    if (h->comb_bytes >= bytes) return ISING_OK;
    if (h->comb) { cudaFree(h->comb); h->comb = nullptr; h->comb_bytes = 0; }
    cudaError_t e = cudaMalloc((void **)&h->comb, bytes);
    if (e != cudaSuccess) { cudaGetLastError(); h->comb = nullptr; return set_error(ISING_ENOMEM, "comb planes: cudaMalloc failed"); }
    h->comb_bytes = bytes;
    return ISING_OK;
}

static int ensure_corr(ising_sim *h, int64_t count)
{
    const size_t bytes = (size_t)count * 2 * sizeof(long long);
    if (h->d_corr_bytes < bytes) {
        if (h->d_corr) cudaFree(h->d_corr);
        h->d_corr = nullptr; h->d_corr_bytes = 0;
        cudaError_t e = cudaMalloc((void **)&h->d_corr, bytes);
        if (e != cudaSuccess) { cudaGetLastError(); return set_error(ISING_ENOMEM, "correlation buffer: cudaMalloc failed"); }
        h->d_corr_bytes = bytes;
    }
    const size_t rb = (size_t)count * sizeof(long long);
    if (h->d_rlist_bytes < rb) {
        if (h->d_rlist) cudaFree(h->d_rlist);
        h->d_rlist = nullptr; h->d_rlist_bytes = 0;
        cudaError_t e = cudaMalloc((void **)&h->d_rlist, rb);
        if (e != cudaSuccess) { cudaGetLastError(); return set_error(ISING_ENOMEM, "distance list: cudaMalloc failed"); }
        h->d_rlist_bytes = rb;
    }
    return ISING_OK;
}

// shared tail: planes already built.  stride 0 = full-source r = 1..count.
static int run_corr(ising_sim *h, int64_t stride, int64_t count, const int64_t *r, int64_t *sx, int64_t *sy)
{
    int rc = ensure_corr(h, count);
    if (rc) return rc;
    if (stride >= 2) { rc = ensure_comb(h, stride); if (rc) return rc; }
    long long *d_sx = h->d_corr, *d_sy = h->d_corr + count;
    if (stride > 0)
        CUDA_TRY(cudaMemcpyAsync(h->d_rlist, r, (size_t)count * sizeof(long long), cudaMemcpyHostToDevice, h->stream));
    cudaError_t e = launch_corr(h, stride, count, h->d_rlist, d_sx, d_sy);
    if (e != cudaSuccess) return cuda_fail(e, "correlation kernel");
    CUDA_TRY(cudaMemcpyAsync(sx, d_sx, (size_t)count * sizeof(long long), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(cudaMemcpyAsync(sy, d_sy, (size_t)count * sizeof(long long), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    if (!is_blume_capel(h->model)) {   // popcount of unequal pairs -> pair sum
        const int64_t s = stride > 0 ? stride : 1;
        const int64_t n_src = (h->L / s) * (h->L / s);
        for (int64_t i = 0; i < count; ++i) { sx[i] = n_src - 2 * sx[i]; sy[i] = n_src - 2 * sy[i]; }
    }
    return ISING_OK;
}

static int ensure_gram(ising_sim *h)
{
    const size_t bytes = corr_gram_bytes(h);
    if (h->gram_bytes >= bytes) return ISING_OK;
    if (h->gram) { cudaFree(h->gram); h->gram = nullptr; h->gram_bytes = 0; }
    cudaError_t e = cudaMalloc((void **)&h->gram, bytes);
    if (e != cudaSuccess) { cudaGetLastError(); h->gram = nullptr; return set_error(ISING_ENOMEM, "int8 spin matrix: cudaMalloc failed"); }
    h->gram_bytes = bytes;
    return ISING_OK;
}

// Full-range sums on the tensor cores (corr_gram.cu): planes already built.
static int run_corr_gram(ising_sim *h, int64_t count, int64_t *sx, int64_t *sy)
{
    int rc = ensure_corr(h, count);
    if (rc) return rc;
    rc = ensure_gram(h);
    if (rc) return rc;
    long long *d_sx = h->d_corr, *d_sy = h->d_corr + count;
    cudaError_t e = launch_corr_gram(h, count, d_sx, d_sy);
    if (e != cudaSuccess) return cuda_fail(e, "tensor-core correlation kernels");
    CUDA_TRY(cudaMemcpyAsync(sx, d_sx, (size_t)count * sizeof(long long), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(cudaMemcpyAsync(sy, d_sy, (size_t)count * sizeof(long long), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    return ISING_OK;
}

extern "C" int ising_correlation(ising_t *h, int64_t rmax, int64_t *sx, int64_t *sy)
{
    DeviceGuard dev_guard(h);
    if (!h || !sx || !sy) return set_error(ISING_EINVAL, "ising_correlation: NULL argument");
    if (rmax < 1 || rmax > h->L / 2) return set_error(ISING_EINVAL, "ising_correlation: rmax outside [1, L/2]");
    if (int rcp = no_parts(h, "ising_correlation")) return rcp;
    int rc = ensure_planes(h);
    if (rc) return rc;
    cudaError_t e = launch_planes(h);
    if (e != cudaSuccess) return cuda_fail(e, "bit-plane kernels");
    // tensor cores pay off once the band is wide; narrow bands stay on the bit planes
    const bool tensor = h->corr_path >= 2 || (h->corr_path == 0 && rmax >= 512);
    if (tensor && corr_gram_supported(h, rmax)) return run_corr_gram(h, rmax, sx, sy);
    if (h->corr_path >= 2) return set_error(ISING_EINVAL, "ising_correlation: tensor-core path needs L % 256 == 0 and L >= 512");
    return run_corr(h, 0, rmax, nullptr, sx, sy);
}

extern "C" int ising_set_corr_path(ising_t *h, int path)
{
    DeviceGuard dev_guard(h);
    if (!h) return set_error(ISING_EINVAL, "ising_set_corr_path: NULL handle");
    if (path < 0 || path > 4) return set_error(ISING_EINVAL, "ising_set_corr_path: path must be 0 (auto), 1 (bit planes), 2 (tensor cores), 3 (CTA pairs) or 4 (CTA pairs, fp4)");
    h->corr_path = path;
    return ISING_OK;
}

static bool valid_stride(int64_t s) { return s == 1 || s == 2 || s == 4 || s == 8 || s == 16 || s == 32 || s == 64; }

extern "C" int ising_correlation_list(ising_t *h, int64_t stride, int64_t count, const int64_t *r, int64_t *sx, int64_t *sy)
{
    DeviceGuard dev_guard(h);
    if (!h || !r || !sx || !sy) return set_error(ISING_EINVAL, "ising_correlation_list: NULL argument");
    if (!valid_stride(stride)) return set_error(ISING_EINVAL, "ising_correlation_list: stride must be 1 or a power of two <= 64");
    if (int rcp = no_parts(h, "ising_correlation_list")) return rcp;
    if (count < 1 || count > 65535) return set_error(ISING_EINVAL, "ising_correlation_list: count outside [1, 65535]");
    for (int64_t i = 0; i < count; ++i)
        if (r[i] < 1 || r[i] > h->L / 2) return set_error(ISING_EINVAL, "ising_correlation_list: distance outside [1, L/2]");
    int rc = ensure_planes(h);
    if (rc) return rc;
    cudaError_t e = launch_planes(h);
    if (e != cudaSuccess) return cuda_fail(e, "bit-plane kernels");
    return run_corr(h, stride, count, r, sx, sy);
}

// Sec. 3.3 at t = sweeps_done; the distance lists are host arithmetic (host_logic.cu).
// Results are staged in host vectors and handed out only when every kernel has succeeded.
static int protocol_measure(ising_sim *h, std::vector<int64_t> &r, std::vector<int64_t> &sx, std::vector<int64_t> &sy,
                            std::vector<int64_t> &n_src)
{
    if (int rcp = no_parts(h, "the correlation protocol")) return rcp;
    std::vector<int64_t> all_sources, block_sources;
    host_protocol_lists(h->L, h->t, all_sources, block_sources);
    const int64_t na = (int64_t)all_sources.size(), nb = (int64_t)block_sources.size();
    r = all_sources;
    r.insert(r.end(), block_sources.begin(), block_sources.end());
    sx.assign(na + nb, 0); sy.assign(na + nb, 0); n_src.assign(na + nb, 0);
    int rc = ensure_planes(h);
    if (rc) return rc;
    cudaError_t e = launch_planes(h);
    if (e != cudaSuccess) return cuda_fail(e, "bit-plane kernels");
    rc = run_corr(h, 0, na, nullptr, sx.data(), sy.data());                  // every site a source, r = 1..2R
    if (rc) return rc;
    for (int64_t i = 0; i < na; ++i) n_src[i] = h->L * h->L;
    if (nb > 0) {
        rc = run_corr(h, 16, nb, block_sources.data(), sx.data() + na, sy.data() + na);   // one source per 16 x 16 block
        if (rc) return rc;
        for (int64_t i = 0; i < nb; ++i) n_src[na + i] = (h->L / 16) * (h->L / 16);
    }
    return ISING_OK;
}

extern "C" int ising_correlation_protocol(ising_t *h, int64_t cap, int64_t *r, int64_t *sx, int64_t *sy,
                                          int64_t *n_src, int64_t *count)
{
    DeviceGuard dev_guard(h);
    if (!h || !count) return set_error(ISING_EINVAL, "ising_correlation_protocol: NULL argument");
    std::vector<int64_t> all_sources, block_sources;
    host_protocol_lists(h->L, h->t, all_sources, block_sources);
    const int64_t n = (int64_t)(all_sources.size() + block_sources.size());
    *count = n;
    if (!r && !sx && !sy && !n_src) return ISING_OK;             // size query
    if (!r || !sx || !sy || !n_src || cap < n) return set_error(ISING_EINVAL, "ising_correlation_protocol: cap too small");
    std::vector<int64_t> vr, vx, vy, vn;
    int rc = protocol_measure(h, vr, vx, vy, vn);
    if (rc) return rc;
    std::copy(vr.begin(), vr.end(), r); std::copy(vx.begin(), vx.end(), sx);
    std::copy(vy.begin(), vy.end(), sy); std::copy(vn.begin(), vn.end(), n_src);
    return ISING_OK;
}

// A11 with the correlation measurement: sweep to each time, run the Sec. 3.3 protocol there.
extern "C" int ising_run_protocol_schedule(ising_t *h, int64_t n_times, const uint64_t *times, int64_t cap,
                                           int64_t *r, int64_t *sx, int64_t *sy, int64_t *n_src, int64_t *counts,
                                           ising_obs_t *obs)
{
    DeviceGuard dev_guard(h);
    if (!h || !times || !r || !sx || !sy || !n_src || !counts || n_times < 0)
        return set_error(ISING_EINVAL, "ising_run_protocol_schedule: bad argument");
    uint64_t prev = h->t;
    for (int64_t i = 0; i < n_times; ++i) {
        if (times[i] < prev) return set_error(ISING_EINVAL, "ising_run_protocol_schedule: times must be ascending and >= sweeps_done");
        prev = times[i];
        std::vector<int64_t> a, b;
        host_protocol_lists(h->L, times[i], a, b);
        if ((int64_t)(a.size() + b.size()) > cap)
            return set_error(ISING_EINVAL, "ising_run_protocol_schedule: cap smaller than the distance list of a scheduled time "
                                           "(ising_protocol_distances gives the size)");
    }
    for (int64_t i = 0; i < n_times; ++i) {
        int rc = ising_sweep(h, (int64_t)(times[i] - h->t));
        if (rc) return rc;
        std::vector<int64_t> vr, vx, vy, vn;
        rc = protocol_measure(h, vr, vx, vy, vn);
        if (rc) return rc;
        if (obs) {
            rc = h->tally_on ? ising_tally(h, &obs[i]) : ising_observables(h, &obs[i]);
            if (rc) return rc;
        }
        counts[i] = (int64_t)vr.size();
        std::copy(vr.begin(), vr.end(), r + i * cap); std::copy(vx.begin(), vx.end(), sx + i * cap);
        std::copy(vy.begin(), vy.end(), sy + i * cap); std::copy(vn.begin(), vn.end(), n_src + i * cap);
    }
    return ISING_OK;
}

