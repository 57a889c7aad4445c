// Full-range correlation on the tensor cores (A9 of SURVEY.md Sec. 8(a)).
//
// S_y(r) = sum_y sum_x s(x, y) s(x, (y + r) mod L) = sum_y G[y, (y + r) mod L],  G = A A^T,
// with A the L x L spin matrix as int8 (-1, 0, +1): a banded Gram matrix, the one dense
// contraction on the path.  tcgen05.mma kind::i8 accumulates in int32 (exact: |G| <= L), so
// the sums stay bit-exact integers.  S_x is the same on the transposed matrix.
//
// One persistent CTA per SM, warp-specialised: warp 0 = TMA producer (128-byte-swizzled
// K-major tiles, 4-stage mbarrier ring), warp 1 = MMA issuer (one elected thread, 128 x 256
// int32 accumulator in TMEM, double buffered), warps 2-5 = epilogue (tcgen05.ld, every
// element added to the shared-memory bin of its diagonal j - i, bins flushed to the int64
// result with one atomic per distance per tile).  Tile (I0, J0 = I0 + 256 k) holds the ordered
// pairs (y = I0 + i, y + r = J0 + j): r = J0 - I0 + j - i, kept when 1 <= r <= rmax.
// The default is the fp4 CTA-pair variant further down (gram4_kernel: kind::mxf4, cta_group::2, 256 x 224
// tiles); the int8 kernels stay selectable (ising_set_corr_path(h, 2): this single-CTA kernel, 3: gram2_kernel,
// int8 CTA pairs) and are tested against it.
#include "ising_internal.cuh"

#include <cuda.h>

namespace {

constexpr int TM = 128, TN = 256, TKB = 128;        // tile rows, tile columns, K bytes per stage
constexpr int STAGES = 4;
constexpr int A_BYTES = TM * TKB, B_BYTES = TN * TKB, STAGE_BYTES = A_BYTES + B_BYTES;
constexpr int NBINS = TM + TN - 1;                   // diagonals j - i = -(TM-1) .. TN-1
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 1024 /*alignment slack*/ + 2048 /*bins, barriers*/;

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_load_2d(void *dst, const CUtensorMap *map, uint64_t *bar, int c0, int c1)
{
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1) : "memory");
}
// K-major operand, 128-byte swizzle: 8-row groups of 1024 bytes, descriptor version 1 (sm_100)
__device__ __forceinline__ uint64_t umma_desc(uint32_t smem_addr)
{
    uint64_t d = 0;
    d |= (uint64_t)((smem_addr & 0x3FFFFu) >> 4);          // start address, 16-byte units
    d |= (uint64_t)(1024 >> 4) << 32;                      // stride between 8-row groups
    d |= (uint64_t)1 << 46;                                // descriptor version
    d |= (uint64_t)2 << 61;                                // SWIZZLE_128B
    return d;
}
// kind::i8, signed x signed -> int32, both K-major, M = 128, N = 256
constexpr uint32_t kInstrDesc = (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(TN >> 3) << 17) | ((uint32_t)(TM >> 4) << 24);

__device__ __forceinline__ void umma_i8(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t accumulate)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, {%5, %5, %5, %5}, p;\n\t}"
        ::"r"(tmem_d), "l"(da), "l"(db), "r"(kInstrDesc), "r"(accumulate), "r"(0u) : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t *bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// 32 consecutive accumulator columns of this thread's TMEM lane -> registers (waits for the load)
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
          "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
          "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// Work split: the K dimension (the L columns of the spin matrix) is cut into chunks of kc bytes
// so that the L x kc slab every tile of a launch reads stays resident in L2 (S(r) is linear in
// G, so the chunks simply add up); one launch per chunk.  Inside a launch the tiles are ordered
// column-tile-major and every CTA takes a contiguous run of them: consecutive tiles of a run
// share jk, hence the same diagonal bins, which are flushed only when jk changes.
struct GramParams {
    int L, rmax, n_ib, n_jk;          // row blocks, column tiles per row block
    int k0, n_kb;                     // first K byte of this chunk, 128-byte K blocks per tile
    long long *out;                   // S(r), r = 1..rmax at out[r-1]
};

__device__ __forceinline__ void tile_range(const GramParams &p, int &lo, int &hi)
{
    const long long n = (long long)p.n_ib * p.n_jk;
    lo = (int)(n * blockIdx.x / gridDim.x);
    hi = (int)(n * (blockIdx.x + 1) / gridDim.x);
}

}  // namespace

// ------------------------------------------------------------------ kernel ---
__global__ void __launch_bounds__(192, 1) gram_kernel(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ GramParams p)
{
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    uint8_t *tail = smem + STAGES * STAGE_BYTES;
    int *bins = reinterpret_cast<int *>(tail);                              // NBINS ints (1532 B)
    uint64_t *full = reinterpret_cast<uint64_t *>(tail + 1536);             // [STAGES]
    uint64_t *empty = full + STAGES;                                        // [STAGES]
    uint64_t *tfull = empty + STAGES;                                       // [2]
    uint64_t *tempty = tfull + 2;                                           // [2]
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(tempty + 2);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_kb = p.n_kb;
    int t_lo, t_hi;
    tile_range(p, t_lo, t_hi);

    if (warp == 1 && lane == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
        for (int s = 0; s < 2; ++s) { mbar_init(&tfull[s], 1); mbar_init(&tempty[s], 4); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 2) {   // TMEM: 512 columns = two 128 x 256 int32 accumulators
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_slot)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    for (int i = threadIdx.x; i < NBINS; i += blockDim.x) bins[i] = 0;
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_base = *tmem_slot;

    if (warp == 0) {
        // ===== TMA producer =====
        if (lane == 0) {
            int stage = 0; uint32_t phase = 0;
            for (int t = t_lo; t < t_hi; ++t) {
                const int jk = t / p.n_ib, ib = t - jk * p.n_ib;
                const int I0 = ib * TM;
                int J0 = I0 + jk * TN; if (J0 >= p.L) J0 -= p.L;
                int J1 = J0 + TM; if (J1 >= p.L) J1 -= p.L;                 // second half of the B tile (wraps)
                for (int kb = 0; kb < n_kb; ++kb) {
                    mbar_wait(&empty[stage], phase ^ 1);
                    mbar_expect_tx(&full[stage], STAGE_BYTES);
                    uint8_t *sa = smem + stage * STAGE_BYTES, *sb = sa + A_BYTES;
                    tma_load_2d(sa, &tmap, &full[stage], p.k0 + kb * TKB, I0);
                    tma_load_2d(sb, &tmap, &full[stage], p.k0 + kb * TKB, J0);
                    tma_load_2d(sb + A_BYTES, &tmap, &full[stage], p.k0 + kb * TKB, J1);
                    if (++stage == STAGES) { stage = 0; phase ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer (one thread) =====
        if (lane == 0) {
            int stage = 0; uint32_t phase = 0;
            int as = 0; uint32_t aphase = 0;
            for (int t = t_lo; t < t_hi; ++t) {
                mbar_wait(&tempty[as], aphase ^ 1);
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const uint32_t d_tmem = tmem_base + (uint32_t)(as * TN);
                for (int kb = 0; kb < n_kb; ++kb) {
                    mbar_wait(&full[stage], phase);
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    const uint32_t sa = smem_u32(smem + stage * STAGE_BYTES), sb = sa + A_BYTES;
                    const uint64_t da = umma_desc(sa), db = umma_desc(sb);
#pragma unroll
                    for (int k = 0; k < TKB / 32; ++k)                       // UMMA_K = 32 int8 = 32 bytes = 2 x 16 B
                        umma_i8(d_tmem, da + (uint64_t)(2 * k), db + (uint64_t)(2 * k), (kb | k) ? 1u : 0u);
                    umma_commit(&empty[stage]);                              // frees the smem slot when the MMAs retire
                    if (++stage == STAGES) { stage = 0; phase ^= 1; }
                }
                umma_commit(&tfull[as]);                                     // accumulator complete
                if (++as == 2) { as = 0; aphase ^= 1; }
            }
        }
    } else {
        // ===== epilogue: warps 2..5, TMEM lane quarter = warp % 4 =====
        const int q = warp & 3, row = q * 32 + lane;                        // tile row i of this thread
        const int et = threadIdx.x - 64;                                    // 0..127 among the epilogue threads
        int as = 0; uint32_t aphase = 0;
        for (int t = t_lo; t < t_hi; ++t) {
            const int jk = t / p.n_ib;
            mbar_wait(&tfull[as], aphase);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(as * TN);
#pragma unroll 1
            for (int c = 0; c < TN / 32; ++c) {
                uint32_t v[32];
                tmem_ld32(taddr + (uint32_t)(c * 32), v);
                // element (row, 32 c + k) lies on diagonal j - i: lanes hit consecutive bins, no conflicts
                const uint32_t b0 = smem_u32(bins) + 4u * (uint32_t)((TM - 1) + 32 * c - row);
#pragma unroll
                for (int k = 0; k < 32; ++k)
                    asm volatile("red.shared.add.s32 [%0], %1;" ::"r"(b0 + 4u * k), "r"(v[k]) : "memory");
            }
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            __syncwarp();
            if (lane == 0) mbar_arrive(&tempty[as]);                        // this warp has drained its quarter
            if (++as == 2) { as = 0; aphase ^= 1; }
            // the next tile of the run has the same jk (same bins) unless the run crosses into the
            // next column tile: flush the bins then, r = jk * TN + (bin - (TM - 1))
            if (t + 1 < t_hi && (t + 1) / p.n_ib == jk) continue;
            asm volatile("bar.sync 1, 128;" ::: "memory");
            for (int b = et; b < NBINS; b += 128) {
                const int r = jk * TN + b - (TM - 1);
                const int v = bins[b];
                bins[b] = 0;
                if (r >= 1 && r <= p.rmax && v != 0)
                    atomicAdd(reinterpret_cast<unsigned long long *>(&p.out[r - 1]), (unsigned long long)(long long)v);
            }
            asm volatile("bar.sync 1, 128;" ::: "memory");
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 2) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem_base) : "memory");
}

// ------------------------------------------------ CTA-pair variant (opt-in) ---
// cta_group::2: two CTAs of a cluster (one TPC) share one 256 x 256 tile.  Each CTA loads its own
// 128 rows of A and 128 of the 256 B rows (32 KB per stage instead of 48 KB: a third less L2 -> SM
// traffic, 6 stages), the leader CTA issues tcgen05.mma.cta_group::2 (M = 256), and each CTA's
// TMEM receives the accumulator rows of its own A half, which its epilogue warps bin as before.
namespace {
constexpr int STAGES2 = 6, HALF_BYTES = TM * TKB, STAGE2_BYTES = 2 * HALF_BYTES;
constexpr int SMEM2_BYTES = STAGES2 * STAGE2_BYTES + 1024 + 2048;
constexpr uint32_t kInstrDesc2 = (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(256 >> 3) << 17) | ((uint32_t)(256 >> 4) << 24);

__device__ __forceinline__ uint32_t cluster_rank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_remote(uint64_t *bar, uint32_t cta)
{
    asm volatile("{\n\t.reg .b32 ra;\n\tmapa.shared::cluster.u32 ra, %0, %1;\n\tmbarrier.arrive.shared::cluster.b64 _, [ra];\n\t}"
                 ::"r"(smem_u32(bar)), "r"(cta) : "memory");
}
// 2-SM TMA load: the transaction bytes are counted on the LEADER CTA's barrier (peer bit cleared)
__device__ __forceinline__ void tma_load_2d_2sm(void *dst, const CUtensorMap *map, uint64_t *bar, int c0, int c1)
{
    asm volatile(
        "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar) & 0xFEFFFFFFu), "r"(c0), "r"(c1) : "memory");
}
__device__ __forceinline__ void umma_i8_2sm(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t accumulate)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::i8 [%0], %1, %2, %3, {%5, %5, %5, %5, %5, %5, %5, %5}, p;\n\t}"
        ::"r"(tmem_d), "l"(da), "l"(db), "r"(kInstrDesc2), "r"(accumulate), "r"(0u) : "memory");
}
__device__ __forceinline__ void umma_commit_2sm(uint64_t *bar)      // arrives on the barrier at this offset in BOTH CTAs
{
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
                 ::"r"(smem_u32(bar)), "h"((uint16_t)3) : "memory");
}
}  // namespace

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(192, 1)
gram2_kernel(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ GramParams p)
{
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    uint8_t *tail = smem + STAGES2 * STAGE2_BYTES;
    int *bins = reinterpret_cast<int *>(tail);
    uint64_t *full = reinterpret_cast<uint64_t *>(tail + 1536);             // [STAGES2]  (used on the leader)
    uint64_t *empty = full + STAGES2;                                       // [STAGES2]  (both CTAs)
    uint64_t *tfull = empty + STAGES2;                                      // [2]        (both CTAs)
    uint64_t *tempty = tfull + 2;                                           // [2]        (used on the leader)
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(tempty + 2);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_rank();
    const bool leader = rank == 0;
    const int n_kb = p.n_kb;
    // tiles of 256 rows: p.n_ib row blocks; a contiguous run per CLUSTER, column-tile-major
    const long long n_tiles = (long long)p.n_ib * p.n_jk;
    const int n_cl = gridDim.x >> 1, cl = blockIdx.x >> 1;
    const int t_lo = (int)(n_tiles * cl / n_cl), t_hi = (int)(n_tiles * (cl + 1) / n_cl);

    if (warp == 1 && lane == 0) {
        for (int s = 0; s < STAGES2; ++s) { mbar_init(&full[s], 2); mbar_init(&empty[s], 1); }
        for (int s = 0; s < 2; ++s) { mbar_init(&tfull[s], 1); mbar_init(&tempty[s], 8); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int i = threadIdx.x; i < NBINS; i += blockDim.x) bins[i] = 0;
    cluster_sync_all();                                                      // barriers of both CTAs exist
    if (warp == 2) {
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_slot)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    cluster_sync_all();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_base = *tmem_slot;

    if (warp == 0) {
        // ===== TMA producer (both CTAs): own A half, own half of the B rows =====
        if (lane == 0) {
            int stage = 0; uint32_t phase = 0;
            for (int t = t_lo; t < t_hi; ++t) {
                const int jk = t / p.n_ib, ib = t - jk * p.n_ib;
                const int I0 = ib * 256 + (int)rank * TM;
                int J0 = ib * 256 + jk * TN; if (J0 >= p.L) J0 -= p.L;      // multiple of 256: the tile never wraps
                J0 += (int)rank * TM;
                for (int kb = 0; kb < n_kb; ++kb) {
                    mbar_wait(&empty[stage], phase ^ 1);
                    if (leader) mbar_expect_tx(&full[stage], 2 * STAGE2_BYTES);   // bytes of both CTAs land on this barrier
                    uint8_t *sa = smem + stage * STAGE2_BYTES, *sb = sa + HALF_BYTES;
                    tma_load_2d_2sm(sa, &tmap, &full[stage], p.k0 + kb * TKB, I0);
                    tma_load_2d_2sm(sb, &tmap, &full[stage], p.k0 + kb * TKB, J0);
                    if (!leader) mbar_arrive_remote(&full[stage], 0);
                    if (++stage == STAGES2) { stage = 0; phase ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer: leader CTA only =====
        if (leader && lane == 0) {
            int stage = 0; uint32_t phase = 0;
            int as = 0; uint32_t aphase = 0;
            for (int t = t_lo; t < t_hi; ++t) {
                mbar_wait(&tempty[as], aphase ^ 1);
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const uint32_t d_tmem = tmem_base + (uint32_t)(as * TN);
                for (int kb = 0; kb < n_kb; ++kb) {
                    mbar_wait(&full[stage], phase);
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    const uint32_t sa = smem_u32(smem + stage * STAGE2_BYTES), sb = sa + HALF_BYTES;
                    const uint64_t da = umma_desc(sa), db = umma_desc(sb);
#pragma unroll
                    for (int k = 0; k < TKB / 32; ++k)
                        umma_i8_2sm(d_tmem, da + (uint64_t)(2 * k), db + (uint64_t)(2 * k), (kb | k) ? 1u : 0u);
                    umma_commit_2sm(&empty[stage]);
                    if (++stage == STAGES2) { stage = 0; phase ^= 1; }
                }
                umma_commit_2sm(&tfull[as]);
                if (++as == 2) { as = 0; aphase ^= 1; }
            }
        }
    } else {
        // ===== epilogue (both CTAs): rows I0 + 128 rank + i of the pair tile =====
        const int q = warp & 3, row = q * 32 + lane;
        const int et = threadIdx.x - 64;
        int as = 0; uint32_t aphase = 0;
        for (int t = t_lo; t < t_hi; ++t) {
            const int jk = t / p.n_ib;
            mbar_wait(&tfull[as], aphase);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(as * TN);
#pragma unroll 1
            for (int c = 0; c < TN / 32; ++c) {
                uint32_t v[32];
                tmem_ld32(taddr + (uint32_t)(c * 32), v);
                const uint32_t b0 = smem_u32(bins) + 4u * (uint32_t)((TM - 1) + 32 * c - row);
#pragma unroll
                for (int k = 0; k < 32; ++k)
                    asm volatile("red.shared.add.s32 [%0], %1;" ::"r"(b0 + 4u * k), "r"(v[k]) : "memory");
            }
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            __syncwarp();
            if (lane == 0) { if (leader) mbar_arrive(&tempty[as]); else mbar_arrive_remote(&tempty[as], 0); }
            if (++as == 2) { as = 0; aphase ^= 1; }
            if (t + 1 < t_hi && (t + 1) / p.n_ib == jk) continue;
            asm volatile("bar.sync 1, 128;" ::: "memory");
            for (int b = et; b < NBINS; b += 128) {
                const int r = jk * TN - (int)rank * TM + b - (TM - 1);
                const int v = bins[b];
                bins[b] = 0;
                if (r >= 1 && r <= p.rmax && v != 0)
                    atomicAdd(reinterpret_cast<unsigned long long *>(&p.out[r - 1]), (unsigned long long)(long long)v);
            }
            asm volatile("bar.sync 1, 128;" ::: "memory");
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    cluster_sync_all();                                                      // the peer may still be read by MMAs / arrive remotely
    if (warp == 2) asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, 512;" ::"r"(tmem_base) : "memory");
}

// ---------------------------------------------- fp4 variant (opt-in, path 4) ---
// -1, 0, +1 are exact in e2m1, so the same Gram matrix can run at the fp4 rate: tcgen05.mma
// kind::mxf4 (K = 64 per instruction, 128 smem bytes = 256 elements per stage), fp32 accumulators
// (exact: |sum| <= elements per K chunk < 2^24), every block scale = 1.0.  TMEM must also hold the
// scale columns, so the tile is 256 x 224: two 224-column accumulators (MMA and epilogue overlap) + 32
// scale columns.  224 does not divide L: the matrix carries a replica of its first 256 rows behind
// row L - 1, so a tile that starts below L never wraps.
namespace {
// block-scaled descriptor: a/b format E2M1 (1), scale format UE8M0 (bit 23), N >> 3 at bit 17, M >> 4 at bit 24
constexpr int TN4 = 224;                                         // 2 x 224 accumulator columns + 32 scale columns <= 512
constexpr int STAGE4_BYTES = HALF_BYTES + (TN4 / 2) * TKB, NBINS4 = TM + TN4 - 1;
constexpr int SMEM4_BYTES = STAGES2 * STAGE4_BYTES + 1024 + 2048;
constexpr uint32_t kInstrDescF4 = (1u << 7) | (1u << 10) | ((uint32_t)(TN4 >> 3) << 17) | (1u << 23) | ((uint32_t)(256 >> 4) << 24);
__device__ __forceinline__ void umma_mxf4_2sm(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t accumulate, uint32_t tmem_sf)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::mxf4.block_scale.block32 [%0], %1, %2, %3, [%5], [%5], p;\n\t}"
        ::"r"(tmem_d), "l"(da), "l"(db), "r"(kInstrDescF4), "r"(accumulate), "r"(tmem_sf) : "memory");
}
}  // namespace

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(320, 1)
gram4_kernel(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ CUtensorMap tmap_b,
             const __grid_constant__ GramParams p)
{
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    uint8_t *tail = smem + STAGES2 * STAGE4_BYTES;
    int *bins = reinterpret_cast<int *>(tail);
    uint64_t *full = reinterpret_cast<uint64_t *>(tail + 1536);             // [STAGES2]  (used on the leader)
    uint64_t *empty = full + STAGES2;                                       // [STAGES2]  (both CTAs)
    uint64_t *tfull = empty + STAGES2;                                      // [2]        (both CTAs)
    uint64_t *tempty = tfull + 2;                                           // [2]        (used on the leader)
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(tempty + 2);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_rank();
    const bool leader = rank == 0;
    const int n_kb = p.n_kb;
    // tiles of 256 rows: p.n_ib row blocks; a contiguous run per CLUSTER, column-tile-major
    const long long n_tiles = (long long)p.n_ib * p.n_jk;
    const int n_cl = gridDim.x >> 1, cl = blockIdx.x >> 1;
    const int t_lo = (int)(n_tiles * cl / n_cl), t_hi = (int)(n_tiles * (cl + 1) / n_cl);

    if (warp == 1 && lane == 0) {
        for (int s = 0; s < STAGES2; ++s) { mbar_init(&full[s], 2); mbar_init(&empty[s], 1); }
        for (int s = 0; s < 2; ++s) { mbar_init(&tfull[s], 1); mbar_init(&tempty[s], 16); }   // 8 epilogue warps per CTA
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int i = threadIdx.x; i < NBINS4; i += blockDim.x) bins[i] = 0;
    cluster_sync_all();                                                      // barriers of both CTAs exist
    if (warp == 2) {
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_slot)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    cluster_sync_all();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_base = *tmem_slot;
    // scale factors: every block scale is 1.0 (ue8m0 byte 0x7F).  Columns 448..479 of all 128 lanes are
    // filled with that byte, so whichever bytes the instruction picks as SFA / SFB read as 1.0.
    if (warp >= 2 && warp < 6) {
        const uint32_t sf = tmem_base + ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)(2 * TN4);
        asm volatile(
            "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "
            "{%1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, "
            "%1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1};"
            ::"r"(sf), "r"(0x7F7F7F7Fu) : "memory");
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    cluster_sync_all();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");

    if (warp == 0) {
        // ===== TMA producer (both CTAs): own A half, own half of the B rows =====
        if (lane == 0) {
            int stage = 0; uint32_t phase = 0;
            for (int t = t_lo; t < t_hi; ++t) {
                const int jk = t / p.n_ib, ib = t - jk * p.n_ib;
                const int I0 = ib * 256 + (int)rank * TM;
                int J0 = ib * 256 + jk * TN4; if (J0 >= p.L) J0 -= p.L;     // rows J0 .. J0 + 223 may run past L - 1:
                J0 += (int)rank * (TN4 / 2);                                //   the matrix carries a replica of its first 256 rows
                for (int kb = 0; kb < n_kb; ++kb) {
                    mbar_wait(&empty[stage], phase ^ 1);
                    if (leader) mbar_expect_tx(&full[stage], 2 * STAGE4_BYTES);   // bytes of both CTAs land on this barrier
                    uint8_t *sa = smem + stage * STAGE4_BYTES, *sb = sa + HALF_BYTES;
                    tma_load_2d_2sm(sa, &tmap, &full[stage], p.k0 + kb * TKB, I0);
                    tma_load_2d_2sm(sb, &tmap_b, &full[stage], p.k0 + kb * TKB, J0);
                    if (!leader) mbar_arrive_remote(&full[stage], 0);
                    if (++stage == STAGES2) { stage = 0; phase ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer: leader CTA only =====
        if (leader && lane == 0) {
            int stage = 0; uint32_t phase = 0;
            int as = 0; uint32_t aphase = 0;                             // two 224-column accumulators + the scale columns
            for (int t = t_lo; t < t_hi; ++t) {
                mbar_wait(&tempty[as], aphase ^ 1);
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const uint32_t d_tmem = tmem_base + (uint32_t)(as * TN4);
                for (int kb = 0; kb < n_kb; ++kb) {
                    mbar_wait(&full[stage], phase);
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    const uint32_t sa = smem_u32(smem + stage * STAGE4_BYTES), sb = sa + HALF_BYTES;
                    const uint64_t da = umma_desc(sa), db = umma_desc(sb);
#pragma unroll
                    for (int k = 0; k < TKB / 32; ++k)
                        umma_mxf4_2sm(d_tmem, da + (uint64_t)(2 * k), db + (uint64_t)(2 * k), (kb | k) ? 1u : 0u, tmem_base + (uint32_t)(2 * TN4));
                    umma_commit_2sm(&empty[stage]);
                    if (++stage == STAGES2) { stage = 0; phase ^= 1; }
                }
                umma_commit_2sm(&tfull[as]);
                if (++as == 2) { as = 0; aphase ^= 1; }
            }
        }
    } else {
        // ===== epilogue (both CTAs, 8 warps: two per TMEM lane quarter, each half of the columns) =====
        const int q = warp & 3, row = q * 32 + lane, chalf = (warp - 2) >> 2;
        const int et = threadIdx.x - 64;
        int as = 0; uint32_t aphase = 0;
        for (int t = t_lo; t < t_hi; ++t) {
            const int jk = t / p.n_ib;
            mbar_wait(&tfull[as], aphase);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(as * TN4);
#pragma unroll 1
            for (int c = chalf * 4; c < (chalf ? TN4 / 32 : 4); ++c) {       // 7 chunks of 32 columns: 4 + 3
                uint32_t v[32];
                tmem_ld32(taddr + (uint32_t)(c * 32), v);
                const uint32_t b0 = smem_u32(bins) + 4u * (uint32_t)((TM - 1) + 32 * c - row);
#pragma unroll
                for (int k = 0; k < 32; ++k)
                    asm volatile("red.shared.add.s32 [%0], %1;" ::"r"(b0 + 4u * k), "r"(__float2int_rn(__uint_as_float(v[k]))) : "memory");   // fp32 accumulators hold exact integers
            }
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            __syncwarp();
            if (lane == 0) { if (leader) mbar_arrive(&tempty[as]); else mbar_arrive_remote(&tempty[as], 0); }
            if (++as == 2) { as = 0; aphase ^= 1; }
            if (t + 1 < t_hi && (t + 1) / p.n_ib == jk) continue;
            asm volatile("bar.sync 1, 256;" ::: "memory");
            for (int b = et; b < NBINS4; b += 256) {
                const int r = jk * TN4 - (int)rank * TM + b - (TM - 1);
                const int v = bins[b];
                bins[b] = 0;
                if (r >= 1 && r <= p.rmax && v != 0)
                    atomicAdd(reinterpret_cast<unsigned long long *>(&p.out[r - 1]), (unsigned long long)(long long)v);
            }
            asm volatile("bar.sync 1, 256;" ::: "memory");
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    cluster_sync_all();                                                      // the peer may still be read by MMAs / arrive remotely
    if (warp == 2) asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, 512;" ::"r"(tmem_base) : "memory");
}

// ------------------------------------------------- planes -> int8 matrix ---
// out[y][64 q + i] = nz bit ? (sg bit ? +1 : -1) : 0   (Ising: nz == nullptr, every site non-zero)
__global__ void __launch_bounds__(256) expand_kernel(const uint64_t *__restrict__ sg, const uint64_t *__restrict__ nz,
                                                     int8_t *__restrict__ out, int64_t n_words)
{
    const int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= n_words) return;
    const uint64_t s = sg[w], z = nz ? nz[w] : ~0ull;
    uint4 *o = reinterpret_cast<uint4 *>(out + w * 64);
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        uint32_t v[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            uint32_t word = 0;
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                const int bit = 16 * c + 4 * k + b;
                const uint32_t val = ((z >> bit) & 1ull) ? (((s >> bit) & 1ull) ? 0x01u : 0xFFu) : 0u;
                word |= val << (8 * b);
            }
            v[k] = word;
        }
        o[c] = make_uint4(v[0], v[1], v[2], v[3]);
    }
}

// out[y][32 q + i/2] nibble (i & 1) = e2m1 code of site x = 64 q + i: +1 -> 0x2, -1 -> 0xA, 0 -> 0x0
__global__ void __launch_bounds__(256) expand_fp4_kernel(const uint64_t *__restrict__ sg, const uint64_t *__restrict__ nz,
                                                         uint8_t *__restrict__ out, int64_t n_words, int64_t words_per_row)
{
    const int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= n_words) return;
    const uint64_t s = sg[w], z = nz ? nz[w] : ~0ull;
    uint4 *o = reinterpret_cast<uint4 *>(out + w * 32);
    uint4 *o_rep = (w < 256 * words_per_row) ? reinterpret_cast<uint4 *>(out + (n_words + w) * 32) : nullptr;   // rows 0..255 again behind row L - 1
#pragma unroll
    for (int c = 0; c < 2; ++c) {
        uint32_t v[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            uint32_t word = 0;
#pragma unroll
            for (int b = 0; b < 8; ++b) {
                const int bit = 32 * c + 8 * k + b;
                const uint32_t val = ((z >> bit) & 1ull) ? (((s >> bit) & 1ull) ? 0x2u : 0xAu) : 0u;
                word |= val << (4 * b);
            }
            v[k] = word;
        }
        o[c] = make_uint4(v[0], v[1], v[2], v[3]);
        if (o_rep) o_rep[c] = make_uint4(v[0], v[1], v[2], v[3]);
    }
}

// ------------------------------------------------------------------- host ---
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_tiled()
{
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}

bool corr_gram_supported(const ising_sim *h, int64_t rmax)
{
    return (h->L % 256) == 0 && h->L >= 512 && rmax >= 1;
}

// int8 paths: L x L bytes; fp4 path: (L + 256) rows of L / 2 bytes (replica of the first 256 rows)
size_t corr_gram_bytes(const ising_sim *h)
{
    const bool fp4 = h->corr_path == 0 || h->corr_path == 4;
    return fp4 ? (size_t)(h->L + 256) * (size_t)(h->L / 2) : (size_t)h->L * (size_t)h->L;
}

// S_y (planes sg/nz) and S_x (transposed planes) for r = 1..count via the int8 Gram kernel.
// dev_sx / dev_sy receive the pair sums themselves (no popcount conversion needed).
cudaError_t launch_corr_gram(ising_sim *h, int64_t count, long long *dev_sx, long long *dev_sy)
{
    const int L = (int)h->L, Wq = L / 64;
    const size_t pw = (size_t)L * Wq;
    const bool ising = !is_blume_capel(h->model);
    const int np = ising ? 1 : 2;
    EncodeTiledFn enc = encode_tiled();
    if (!enc) return cudaErrorNotSupported;
    // per call: the attribute is per device, and a process may drive several devices
    cudaError_t ea = cudaFuncSetAttribute(gram_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
    if (ea != cudaSuccess) return ea;
    CUtensorMap tmap;
    const bool fp4_layout = h->corr_path == 0 || h->corr_path == 4;
    const int row_bytes = fp4_layout ? L / 2 : L;               // fp4: two elements per byte
    const cuuint64_t gdim[2] = {(cuuint64_t)row_bytes, (cuuint64_t)(fp4_layout ? L + 256 : L)};
    const cuuint64_t gstride[1] = {(cuuint64_t)row_bytes};
    const cuuint32_t box[2] = {(cuuint32_t)TKB, (cuuint32_t)TM};
    const cuuint32_t estr[2] = {1, 1};
    if (enc(&tmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, h->gram, gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return cudaErrorInvalidValue;
    CUtensorMap tmap_b = tmap;                         // fp4 path: 112-row boxes for the B halves
    if (fp4_layout) {
        const cuuint32_t box_b[2] = {(cuuint32_t)TKB, (cuuint32_t)(TN4 / 2)};
        if (enc(&tmap_b, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, h->gram, gdim, gstride, box_b, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return cudaErrorInvalidValue;
    }
    int dev = 0, n_sm = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    GramParams p;
    p.L = L; p.rmax = (int)count; p.n_ib = L / TM;
    p.n_jk = (int)((count + TM + TN - 1) / TN);          // columns I0 .. I0 + 127 + rmax
    // K chunk: keep the L x kc slab within about half of the 126 MB L2 (measured at L = 2^16: 1024 bytes
    // is the optimum for both kernels; 512 pays more epilogues, 2048 falls out of L2)
    int kc = (int)(((64ll << 20) / L) / TKB * TKB);
    if (kc < 4 * TKB) kc = 4 * TKB;
    if (kc > row_bytes) kc = row_bytes;
    p.n_kb = kc / TKB;
    const bool fp4 = h->corr_path == 0 || h->corr_path == 4;   // default: kind::mxf4 on a packed e2m1 matrix (L/2 bytes per row)
    const bool pair = h->corr_path != 2;              // default: cta_group::2 kernel, 256-row tiles; path 2 = single-CTA kernel
    if (pair) {
        ea = cudaFuncSetAttribute(gram2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM2_BYTES);
        if (ea == cudaSuccess) ea = cudaFuncSetAttribute(gram4_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM4_BYTES);
        if (ea != cudaSuccess) return ea;
        p.n_ib = L / 256;
        p.n_jk = (int)((count + 256 + TN - 1) / TN);      // columns I0 .. I0 + 255 + rmax
        if (fp4) p.n_jk = (int)((count + 256 + TN4 - 1) / TN4);
    }
    const int n_tiles = p.n_ib * p.n_jk;
    int grid = n_tiles < n_sm ? n_tiles : n_sm;
    if (pair) { grid = 2 * (n_tiles < n_sm / 2 ? n_tiles : n_sm / 2); }
    for (int axis = 0; axis < 2; ++axis) {              // 0: S_y from the planes, 1: S_x from the transposed planes
        const uint64_t *sg = h->planes + (axis ? np * pw : 0);
        const uint64_t *nz = ising ? nullptr : sg + pw;
        long long *out = axis ? dev_sx : dev_sy;
        cudaError_t e = cudaMemsetAsync(out, 0, count * sizeof(long long), h->stream);
        if (e != cudaSuccess) return e;
        if (fp4) expand_fp4_kernel<<<(unsigned)((pw + 255) / 256), 256, 0, h->stream>>>(sg, nz, reinterpret_cast<uint8_t *>(h->gram), (int64_t)pw, (int64_t)Wq);
        else expand_kernel<<<(unsigned)((pw + 255) / 256), 256, 0, h->stream>>>(sg, nz, h->gram, (int64_t)pw);
        p.out = out;
        h->launches++;
        for (int k0 = 0; k0 < row_bytes; k0 += kc) {
            p.k0 = k0;
            p.n_kb = (row_bytes - k0 < kc ? row_bytes - k0 : kc) / TKB;
            if (fp4) gram4_kernel<<<grid, 320, SMEM4_BYTES, h->stream>>>(tmap, tmap_b, p);
            else if (pair) gram2_kernel<<<grid, 192, SMEM2_BYTES, h->stream>>>(tmap, p);
            else gram_kernel<<<grid, 192, SMEM_BYTES, h->stream>>>(tmap, p);
            h->launches++;
        }
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}
