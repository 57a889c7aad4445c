// NEXT-2: the paper's own Ising kernel -- one bit per spin and non-uniform
// random bits from a 16-entry look-up table (4 bits per Philox number, 1/2 number per spin).
// Model ISING_MODEL_ISING_LUT; readings L1-L7 of DESIGN.md.  Layout: two colour arrays, each
// L rows x (L/128) uint64 words, bit j of word m of row y = compact site k = 64 m + j
// (x = 2k + ((y + colour) & 1)), 1 = spin +1.
//
// Update kernel: one thread owns one 128-bit column (128 same-colour sites) and walks R rows with
// the opposite-colour rows y-1, y, y+1 in registers (same sliding window as update.cu).  Per
// 32-bit word: eq3 / eq4 from a bit-sliced adder of the four "equal to the spin" words, two random
// words from 4 Philox calls whose 16 numbers each go through a 4-level binary search of the table
// (shared memory, heap order; IADD3 carry + IMAD.X per level), then the paper's flip formula.
#include "ising_internal.cuh"

struct LutParams {
    const uint4 *opp;            // rows of this slab (NEXT-4; the whole lattice when unsharded)
    uint4 *own;
    const char *opp_up, *opp_dn; // the opposite-colour row above / below the slab (neighbouring slabs; see update.cu)
    int y_base;                  // global row of the slab's first row (even)
    int L, cols, R;              // L = rows of this slab; cols = uint4 per colour row = (lattice size) / 256
    uint32_t colour, t;
    const uint32_t *tree;        // 16 carry constants in heap order (device): tree[n] = 2^32 - threshold(node n)
    const uint2 *buckets;        // 4096 entries indexed by the top 12 bits of the number (device), see lut_bits32
    uint32_t bucket_stride;      // 8: bytes per bucket entry, as a run-time value (see lut_bucket_step)
    const uint32_t *t_base;      // sweep number = t + *t_base (see update.cu)
    long long *tally;            // A7: running B, M (device), updated when the kernel is built with TALLY
    RoundKeys rk;
};

// node n of the heap (1..15) splits at table index: level 0 -> 8; level 1 -> 4, 12; ...
// host helper (api.cu) fills tree[n]; here only the search.
__device__ __forceinline__ uint32_t lut_search(uint32_t rnd, uint32_t c_root, const uint32_t *tree)
{
    uint32_t node = 1;
    // level 0: uniform threshold, no load
    asm("{\n\t.reg .u32 t;\n\tadd.cc.u32 t, %1, %2;\n\tmadc.lo.u32 %0, %0, 2, 0;\n\t}" : "+r"(node) : "r"(rnd), "r"(c_root));
#pragma unroll
    for (int level = 1; level < 4; ++level) {
        const uint32_t c = tree[node];
        asm("{\n\t.reg .u32 t;\n\tadd.cc.u32 t, %1, %2;\n\tmadc.lo.u32 %0, %0, 2, 0;\n\t}" : "+r"(node) : "r"(rnd), "r"(c));
    }
    return node;                 // 16 + table index
}

// 32 random bits (8 nibbles) from two Philox calls: nibble u of call 0, then of call 1.
// V = 1: every number goes through the 4-level binary search.
// V = 0 (default): bucket table.  The top 12 bits of the number select an entry {C, meta}: the
// bucket [b 2^20, (b+1) 2^20) holds at most one table threshold t in all but a few buckets, so
// getMaxLE = idx_base + [rnd >= t] = meta + carry(rnd + C), C = 2^32 - t (0 if the bucket has no
// threshold): one shift, one LDS.64, one IADD3 and two IMADs per number.  Buckets with two or more
// thresholds carry meta = 256 (+ anything): the sum of the eight metas then reaches 256 and the
// word is recomputed by the binary search (rare: none at T >= 0.6 Tc, ~0.1 % of numbers at 0.5 Tc).
#define LUT_BUCKET_BITS 12
static const int64_t kLutBucketMinL = 6144;      // automatic variant: bucket table from this size on
#ifndef LUT_MIN_BLOCKS
#define LUT_MIN_BLOCKS 2
#endif
// The entry address is base + 8 (rnd >> 20): the shift is an ALU instruction, the scaling a multiply-add on the FMA
// pipe whose factor 8 comes from a kernel parameter (p.bucket_stride) so that it stays a multiply: written as a
// constant it becomes a second ALU instruction (shift by 17 and mask), and the dispatch slots of the ALU are what
// bounds this kernel.
struct BucketTable { uint32_t base, stride; };     // shared-memory address of entry 0, bytes per entry (= 8)

__device__ __forceinline__ void lut_bucket_step(uint32_t &w, uint32_t &f, uint32_t rnd, const BucketTable bk)
{
    uint32_t ex, ey;
    asm("{\n\t.reg .u32 t, a;\n\t"
        "shr.u32 t, %2, 20;\n\t"
        "mad.lo.u32 a, t, %4, %3;\n\t"
        "ld.shared.v2.u32 {%0, %1}, [a];\n\t}"
        : "=r"(ex), "=r"(ey) : "r"(rnd), "r"(bk.base), "r"(bk.stride));
    asm("{\n\t.reg .u32 t;\n\tadd.cc.u32 t, %1, %2;\n\tmadc.lo.u32 %0, %0, 16, %3;\n\t}" : "+r"(w) : "r"(rnd), "r"(ex), "r"(ey));
    asm("mad.lo.u32 %0, %1, 1, %0;" : "+r"(f) : "r"(ey));
}

// bad: OR of the meta sums of the fast path (>= 256 iff some number fell into a multi-threshold bucket)
template <int V>
__device__ __forceinline__ uint32_t lut_bits32(uint32_t g_lo, const PhiloxRow &pr, const RoundKeys &rk,
                                               uint32_t c_root, const uint32_t *tree, const BucketTable buckets,
                                               uint32_t &bad)
{
    const uint4 a = philox_site4(philox_counter(g_lo), pr, rk), b = philox_site4(philox_counter(g_lo | 1u), pr, rk);
    if (V == 0) {
        uint32_t w = 0, f = 0;   // highest nibble first
        lut_bucket_step(w, f, b.w, buckets); lut_bucket_step(w, f, b.z, buckets);
        lut_bucket_step(w, f, b.y, buckets); lut_bucket_step(w, f, b.x, buckets);
        lut_bucket_step(w, f, a.w, buckets); lut_bucket_step(w, f, a.z, buckets);
        lut_bucket_step(w, f, a.y, buckets); lut_bucket_step(w, f, a.x, buckets);
        bad |= f;
        return w;
    }
    uint32_t w = 0;              // highest nibble first; the "+16" of every node is removed at the end
    w = w * 16u + lut_search(b.w, c_root, tree); w = w * 16u + lut_search(b.z, c_root, tree);
    w = w * 16u + lut_search(b.y, c_root, tree); w = w * 16u + lut_search(b.x, c_root, tree);
    w = w * 16u + lut_search(a.w, c_root, tree); w = w * 16u + lut_search(a.z, c_root, tree);
    w = w * 16u + lut_search(a.y, c_root, tree); w = w * 16u + lut_search(a.x, c_root, tree);
    // sum_j 16 * 16^j = 0x11111110 + ... : every nibble got +16, i.e. +1 carried into the next nibble
    return w - 0x11111110u;      // (the carry out of nibble 7 leaves the word)
}

__device__ __forceinline__ uint32_t lut_flip(uint32_t x, uint32_t up, uint32_t dn, uint32_t sm, uint32_t sd,
                                             uint32_t e4, uint32_t e8)
{
    // Bit-sliced count of the neighbours equal to the spin, pair by pair: c = both of a pair equal, s = exactly
    // one (the spin cancels: (up == x) ^ (dn == x) = up ^ dn).  Equal neighbours = 2 c0 + s0 + 2 c1 + s1, so
    // eq4 = c0 & c1 and ">= 3 equal" = c0 & (c1 | s1) | c1 & s0 (c and s of a pair exclude each other).
    const uint32_t c0 = ~(up ^ x) & ~(dn ^ x), c1 = ~(sm ^ x) & ~(sd ^ x);
    const uint32_t s0 = up ^ dn, s1 = sm ^ sd;
    const uint32_t eq4 = c0 & c1;
    const uint32_t ge3 = (c0 & (c1 | s1)) | (c1 & s0);
    // flip = (eq4 & exp8) | (eq3 & exp4) | (~eq4 & ~eq3), exp8 = e8 & e4, eq3 = ge3 & ~eq4
    //                        = ~ge3 | (e4 & (~eq4 | e8))
    const uint32_t flip = ~ge3 | (e4 & (~eq4 | e8));
    return x ^ flip;
}

template <int P>
__device__ __forceinline__ void lut_side(const uint4 &sm, uint32_t edge, uint32_t sd[4])
{
    if (P == 0) {   // neighbour k-1: shift up by one bit, carry in the top bit of the previous word
        sd[0] = __funnelshift_l(edge, sm.x, 1); sd[1] = __funnelshift_l(sm.x, sm.y, 1);
        sd[2] = __funnelshift_l(sm.y, sm.z, 1); sd[3] = __funnelshift_l(sm.z, sm.w, 1);
    } else {        // neighbour k+1
        sd[0] = __funnelshift_r(sm.x, sm.y, 1); sd[1] = __funnelshift_r(sm.y, sm.z, 1);
        sd[2] = __funnelshift_r(sm.z, sm.w, 1); sd[3] = __funnelshift_r(sm.w, edge, 1);
    }
}

template <int P>
__device__ __noinline__ uint4 lut_row_slow(const uint4 &src, const uint4 &up, const uint4 &sm, const uint4 &dn,
                                           uint32_t edge, uint64_t g0, uint32_t t, const LutParams &p, uint32_t c_root,
                                           const uint32_t *tree);

template <int P, int V>
__device__ __forceinline__ uint4 lut_row(const uint4 &src, const uint4 &up, const uint4 &sm, const uint4 &dn,
                                         uint32_t edge, uint64_t g0, uint32_t t, const LutParams &p, uint32_t c_root,
                                         const uint32_t *tree, const BucketTable bk)
{
    uint32_t sd[4];
    lut_side<P>(sm, edge, sd);
    // g0 = 8 * (first 64-site word of this thread): words 2 col, 2 col + 1 -> g0, g0 + 8
    const PhiloxRow pr = philox_row((uint32_t)(g0 >> 32), t, p.colour, p.rk);
    const uint32_t gl = (uint32_t)g0;         // multiple of 16
    uint32_t bad = 0;
    uint4 o;
    {
        const uint32_t e4 = lut_bits32<V>(gl | 0u, pr, p.rk, c_root, tree, bk, bad), e8 = lut_bits32<V>(gl | 4u, pr, p.rk, c_root, tree, bk, bad);
        o.x = lut_flip(src.x, up.x, dn.x, sm.x, sd[0], e4, e8);
    }
    {
        const uint32_t e4 = lut_bits32<V>(gl | 2u, pr, p.rk, c_root, tree, bk, bad), e8 = lut_bits32<V>(gl | 6u, pr, p.rk, c_root, tree, bk, bad);
        o.y = lut_flip(src.y, up.y, dn.y, sm.y, sd[1], e4, e8);
    }
    {
        const uint32_t e4 = lut_bits32<V>(gl | 8u, pr, p.rk, c_root, tree, bk, bad), e8 = lut_bits32<V>(gl | 12u, pr, p.rk, c_root, tree, bk, bad);
        o.z = lut_flip(src.z, up.z, dn.z, sm.z, sd[2], e4, e8);
    }
    {
        const uint32_t e4 = lut_bits32<V>(gl | 10u, pr, p.rk, c_root, tree, bk, bad), e8 = lut_bits32<V>(gl | 14u, pr, p.rk, c_root, tree, bk, bad);
        o.w = lut_flip(src.w, up.w, dn.w, sm.w, sd[3], e4, e8);
    }
    // one test per row keeps the 16 Philox calls and 128 bucket steps in one basic block; a number in
    // a multi-threshold bucket (rare, see lut_bits32) redoes the row with the binary search
    if (V == 0 && bad >= 256u) return lut_row_slow<P>(src, up, sm, dn, edge, g0, t, p, c_root, tree);
    return o;
}

template <int P>
__device__ __noinline__ uint4 lut_row_slow(const uint4 &src, const uint4 &up, const uint4 &sm, const uint4 &dn,
                                           uint32_t edge, uint64_t g0, uint32_t t, const LutParams &p, uint32_t c_root,
                                           const uint32_t *tree)
{
    return lut_row<P, 1>(src, up, sm, dn, edge, g0, t, p, c_root, tree, BucketTable{0u, 0u});
}

// A7 (optional): change of B and M caused by one updated row, from old / new words and the neighbours.
// A flipped site with d unequal neighbours changes B by 4 d - 8 and M by -2 sigma; d is counted bit-sliced.
template <int P>
__device__ __forceinline__ void lut_tally_row(const uint4 &x4, const uint4 &y4, const uint4 &up, const uint4 &sm, const uint4 &dn,
                                              uint32_t edge, int &dB, int &dM)
{
    uint32_t sd[4];
    lut_side<P>(sm, edge, sd);
    const uint32_t xs[4] = {x4.x, x4.y, x4.z, x4.w}, ys[4] = {y4.x, y4.y, y4.z, y4.w};
    const uint32_t us[4] = {up.x, up.y, up.z, up.w}, ds[4] = {dn.x, dn.y, dn.z, dn.w}, ms[4] = {sm.x, sm.y, sm.z, sm.w};
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const uint32_t x = xs[k], F = x ^ ys[k];
        const uint32_t a = us[k] ^ x, b = ds[k] ^ x, c = ms[k] ^ x, d = sd[k] ^ x;     // 1 where the neighbour differs
        const uint32_t s0 = a ^ b, c0 = a & b, s1 = c ^ d, c1 = c & d;
        const uint32_t b0 = s0 ^ s1, t = s0 & s1, b1 = c0 ^ c1 ^ t, b2 = c0 & c1;       // d = b0 + 2 b1 + 4 b2
        const int cnt = __popc(F), cnt_up = __popc(F & x);
        dB += 4 * (__popc(F & b0) + 2 * __popc(F & b1) + 4 * __popc(F & b2)) - 8 * cnt;
        dM += 2 * cnt - 4 * cnt_up;
    }
}

template <int C, int V, int TALLY>
__global__ void __launch_bounds__(256, LUT_MIN_BLOCKS) lut_update_kernel(const __grid_constant__ LutParams p)
{
    int dB = 0, dM = 0;
    __shared__ uint32_t s_tree[16];
    extern __shared__ __align__(16) unsigned char s_buckets[];          // V = 0: 4096 x 8 bytes
    if (threadIdx.x < 16) s_tree[threadIdx.x] = p.tree[threadIdx.x];
    if (V == 0) {
        const uint4 *src4 = reinterpret_cast<const uint4 *>(p.buckets);
        uint4 *dst4 = reinterpret_cast<uint4 *>(s_buckets);
        for (int i = threadIdx.x; i < (8 << LUT_BUCKET_BITS) / 16; i += blockDim.x) dst4[i] = src4[i];
    }
    __syncthreads();
    pdl_wait();                        // tables (written at create / set_beta) are in; the phase before this one is complete from here on
    pdl_launch_dependents();           // after the wait: at most one later phase sits resident and waiting
    const uint32_t t_eff = p.t + __ldg(p.t_base);
    const uint32_t c_root = s_tree[1];
    const BucketTable bk = {(uint32_t)__cvta_generic_to_shared(s_buckets), p.bucket_stride};
    const int cols = p.cols, L = p.L;
    unsigned tid = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned chunk = tid / (unsigned)cols;
    int col = (int)(tid - chunk * (unsigned)cols);
    int y0 = (int)chunk * p.R;
    if (y0 < L) {                                                      // no early return: every thread reaches block_accumulate
    int yend = min(L, y0 + p.R);

    const size_t rs = (size_t)cols * 16;                               // bytes per colour row
    const char *oppb = reinterpret_cast<const char *>(p.opp);
    char *ownb = reinterpret_cast<char *>(p.own);
    const size_t row0 = (size_t)y0 * rs, cb = (size_t)col * 16;
    // carry half: parity 0 needs the top bit of the previous 32-bit word, parity 1 the low bit of the next
    const int halves = cols * 4;
    const size_t e_p0 = (size_t)((col == 0) ? halves - 1 : 4 * col - 1) * 4;
    const size_t e_p1 = (size_t)((col == cols - 1) ? 0 : 4 * col + 4) * 4;
    const size_t e_even = C == 0 ? e_p0 : e_p1, e_odd = C == 0 ? e_p1 : e_p0;   // y0 even: parity = C on even offsets
    const char *o1 = oppb + row0 + rs + cb;
    const char *ee = oppb + row0 + e_even;
    const char *eo = oppb + row0 + rs + e_odd;
    char *w0 = ownb + row0 + cb;

    uint4 up = *reinterpret_cast<const uint4 *>((y0 == 0) ? p.opp_up + cb : oppb + row0 - rs + cb);
    uint4 sm = *reinterpret_cast<const uint4 *>(oppb + row0 + cb);
    uint4 src = *reinterpret_cast<const uint4 *>(w0);
    uint32_t edge = *reinterpret_cast<const uint32_t *>(ee);
    // g = 8 * (64-site word index): word = y * (2 cols) + 2 col, y the global row
    const uint64_t gs = (uint64_t)cols * 16;
    uint64_t g0 = (uint64_t)(p.y_base + y0) * gs + (uint64_t)col * 16;

    for (int y = y0; y < yend; y += 2) {
        const char *o2 = (y + 2 == L) ? p.opp_dn + cb : o1 + rs;
        uint4 dn = *reinterpret_cast<const uint4 *>(o1);
        uint4 nsrc = *reinterpret_cast<const uint4 *>(w0 + rs);
        uint32_t nedge = *reinterpret_cast<const uint32_t *>(eo);
        uint4 dn2 = *reinterpret_cast<const uint4 *>(o2);
        uint4 o = lut_row<C, V>(src, up, sm, dn, edge, g0, t_eff, p, c_root, s_tree, bk);
        if (TALLY) lut_tally_row<C>(src, o, up, sm, dn, edge, dB, dM);
        *reinterpret_cast<uint4 *>(w0) = o;
        g0 += gs;
        uint4 nsrc2 = src;
        uint32_t nedge2 = 0;
        ee += 2 * rs;
        if (y + 2 < yend) {
            nsrc2 = *reinterpret_cast<const uint4 *>(w0 + 2 * rs);
            nedge2 = *reinterpret_cast<const uint32_t *>(ee);
        }
        o = lut_row<1 - C, V>(nsrc, sm, dn, dn2, nedge, g0, t_eff, p, c_root, s_tree, bk);
        if (TALLY) lut_tally_row<1 - C>(nsrc, o, sm, dn, dn2, nedge, dB, dM);
        *reinterpret_cast<uint4 *>(w0 + rs) = o;
        g0 += gs;
        up = dn; sm = dn2; src = nsrc2; edge = nedge2;
        o1 += 2 * rs; eo += 2 * rs; w0 += 2 * rs;
    }
    }
    if (TALLY) {
        const int v[2] = {dB, dM};
        block_accumulate<2>(v, p.tally);
    }
}

cudaError_t launch_lut_update(ising_sim *h, int slab, int colour, uint32_t t)
{
    LutParams p;
    const Slab &sl = h->slabs[slab];
    const int64_t L = sl.rows;
    p.opp = reinterpret_cast<const uint4 *>(sl.lat[1 - colour]);
    p.own = reinterpret_cast<uint4 *>(sl.lat[colour]);
    p.opp_up = reinterpret_cast<const char *>(halo_up(h, slab, 1 - colour));
    p.opp_dn = reinterpret_cast<const char *>(halo_down(h, slab, 1 - colour));
    p.y_base = (int)sl.y0;
    p.L = (int)L; p.cols = (int)(h->L / 256); p.R = h->rows_per_thread;
    p.colour = (uint32_t)colour; p.t = t;
    p.tree = sl.d_table;
    p.rk = h->rk;
    int64_t chunks = (L + p.R - 1) / p.R;
    int64_t threads = chunks * p.cols;
    int block = h->block_threads;
    unsigned grid = (unsigned)((threads + block - 1) / block);
    p.buckets = reinterpret_cast<const uint2 *>(sl.lut_buckets);
    p.bucket_stride = 8u;
    const size_t smem = 8 << LUT_BUCKET_BITS;
    p.tally = sl.d_acc + 40;
    p.t_base = reinterpret_cast<const uint32_t *>(sl.d_acc + 48) + (h->graph_capture ? 1 : 0);
    cudaError_t le = cudaSuccess;
#define LUT_LAUNCH(C, V, T, SM) le = launch_with_pdl(lut_update_kernel<C, V, T>, grid, block, SM, sl.stream, p, h->pdl_in_graph || !h->graph_capture)
    // variant 0 = automatic: the bucket table pays once its 32 KB fill per block is amortised (L >= 6144, measured with
    // the fill overlapped by programmatic dependent launch: 1777 vs 1676 updates/ns there, 1290 vs 1311 at L = 4096);
    // a small launch starts faster with the table-free binary search.
    // 1 = binary search, 2 = bucket table
    const bool bucket = h->variant == 2 || (h->variant == 0 && h->L >= kLutBucketMinL);
    if (bucket) {
        // per launch: the attribute is per device, and a process may drive several devices
        cudaError_t ea = cudaFuncSetAttribute(lut_update_kernel<0, 0, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (ea == cudaSuccess) ea = cudaFuncSetAttribute(lut_update_kernel<1, 0, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (ea == cudaSuccess) ea = cudaFuncSetAttribute(lut_update_kernel<0, 0, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (ea == cudaSuccess) ea = cudaFuncSetAttribute(lut_update_kernel<1, 0, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (ea != cudaSuccess) return ea;
        if (h->tally_on) { if (colour == 0) LUT_LAUNCH(0, 0, 1, smem); else LUT_LAUNCH(1, 0, 1, smem); }
        else { if (colour == 0) LUT_LAUNCH(0, 0, 0, smem); else LUT_LAUNCH(1, 0, 0, smem); }
    } else {
        if (h->tally_on) { if (colour == 0) LUT_LAUNCH(0, 1, 1, 0); else LUT_LAUNCH(1, 1, 1, 0); }
        else { if (colour == 0) LUT_LAUNCH(0, 1, 0, 0); else LUT_LAUNCH(1, 1, 0, 0); }
    }
#undef LUT_LAUNCH
    h->launches++;
    return le != cudaSuccess ? le : cudaGetLastError();
}

// Resident blocks per SM of the kernel launch_lut_update picks for this handle (0 if the query fails).
int lut_blocks_per_sm(const ising_sim *h, int block)
{
    const bool bucket = h->variant == 2 || (h->variant == 0 && h->L >= kLutBucketMinL);
    const size_t smem = bucket ? (8 << LUT_BUCKET_BITS) : 0;
    const void *fn = bucket ? reinterpret_cast<const void *>(&lut_update_kernel<0, 0, 0>) : reinterpret_cast<const void *>(&lut_update_kernel<0, 1, 0>);
    if (bucket && cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) { cudaGetLastError(); return 0; }
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, block, smem) != cudaSuccess) { cudaGetLastError(); return 0; }
    return per_sm;
}

// L5: word w of colour c = (x | y << 32) of Philox(ctr = (w_lo, w_hi, 0, 2 + c))
__global__ void __launch_bounds__(256) lut_init_kernel(uint64_t *lat0, uint64_t *lat1, int64_t words, int64_t word0, RoundKeys rk)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= words) return;
    const uint64_t w = (uint64_t)(word0 + i);                     // global word index of the slab's word i
    for (int c = 0; c < 2; ++c) {
        const uint4 r = philox4x32_10(make_uint4((uint32_t)w, (uint32_t)(w >> 32), 0u, 2u + c), rk);
        (c ? lat1 : lat0)[i] = (uint64_t)r.x | ((uint64_t)r.y << 32);
    }
}

cudaError_t launch_lut_init(ising_sim *h, int slab)
{
    const Slab &sl = h->slabs[slab];
    const int64_t words = sl.rows * (h->L / 128), word0 = sl.y0 * (h->L / 128);
    lut_init_kernel<<<(unsigned)((words + 255) / 256), 256, 0, sl.stream>>>(sl.lat[0], sl.lat[1], words, word0, h->rk);
    h->launches++;
    return cudaGetLastError();
}

// ----------------------------------------------------------- observables ---
// Same register sliding window as the update kernel: a thread walks R rows of one 128-bit column
// (128 sites) of the CENTRE colour array and reads every word of both arrays once (+2/R halo rows);
// d = unequal neighbours per site from four XORs.  MODE 0 (centre = black only): B = sum (4 - 2 d)
// over black sites (each bond once), M from the black word and the white word of the same position.
// MODE 1 (run for both colours): histogram of s*h = 4 - 2 d, bit-sliced count of the four
// difference words.  One global atomic per block and quantity (block_accumulate).
struct LutObsParams {
    const uint4 *ctr, *nbr;       // rows of this slab
    const char *nbr_up, *nbr_dn;  // the neighbour-colour row above / below the slab
    int centre, L, cols, R;       // L = rows of this slab
    long long *acc;
};

template <int MODE>
__global__ void __launch_bounds__(256) lut_observe_kernel(const __grid_constant__ LutObsParams p)
{
    const int cols = p.cols, L = p.L;
    const unsigned tid = blockIdx.x * blockDim.x + threadIdx.x;
    const unsigned chunk = tid / (unsigned)cols;
    const int col = (int)(tid - chunk * (unsigned)cols);
    const int y0 = (int)chunk * p.R;
    int v[5] = {0, 0, 0, 0, 0};
    if (y0 < L) {
        const int yend = min(L, y0 + p.R);
        const char *nbr = reinterpret_cast<const char *>(p.nbr), *ctr = reinterpret_cast<const char *>(p.ctr);
        const size_t rs = (size_t)cols * 16, cb = (size_t)col * 16;
        const int halves = cols * 4;
        const size_t e0 = (size_t)((col == 0) ? halves - 1 : 4 * col - 1) * 4;   // parity 0: top bit of the previous word
        const size_t e1 = (size_t)((col == cols - 1) ? 0 : 4 * col + 4) * 4;     // parity 1: low bit of the next word
        uint4 up = *reinterpret_cast<const uint4 *>((y0 == 0) ? p.nbr_up + cb : nbr + (size_t)(y0 - 1) * rs + cb);
        uint4 sm = *reinterpret_cast<const uint4 *>(nbr + (size_t)y0 * rs + cb);
        for (int y = y0; y < yend; ++y) {
            const uint4 dn = *reinterpret_cast<const uint4 *>((y + 1 == L) ? p.nbr_dn + cb : nbr + (size_t)(y + 1) * rs + cb);
            const uint4 x4 = *reinterpret_cast<const uint4 *>(ctr + (size_t)y * rs + cb);
            uint32_t sd[4];
            if (((y + p.centre) & 1) == 0) lut_side<0>(sm, *reinterpret_cast<const uint32_t *>(nbr + (size_t)y * rs + e0), sd);
            else lut_side<1>(sm, *reinterpret_cast<const uint32_t *>(nbr + (size_t)y * rs + e1), sd);
            const uint32_t xs[4] = {x4.x, x4.y, x4.z, x4.w}, us[4] = {up.x, up.y, up.z, up.w};
            const uint32_t ds[4] = {dn.x, dn.y, dn.z, dn.w}, ms[4] = {sm.x, sm.y, sm.z, sm.w};
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const uint32_t x = xs[k];
                const uint32_t a = us[k] ^ x, b = ds[k] ^ x, c = ms[k] ^ x, d = sd[k] ^ x;   // 1 where the neighbour differs
                if (MODE == 0) {
                    v[0] += 128 - 2 * (__popc(a) + __popc(b) + __popc(c) + __popc(d));
                    v[1] += 2 * (__popc(x) + __popc(ms[k])) - 64;
                } else {
                    const uint32_t s0 = a ^ b, c0 = a & b, s1 = c ^ d, c1 = c & d;
                    const uint32_t b0 = s0 ^ s1, t = s0 & s1, b1 = c0 ^ c1 ^ t, b2 = c0 & c1;   // d = b0 + 2 b1 + 4 b2
                    v[0] += __popc(~b0 & ~b1 & ~b2); v[1] += __popc(b0 & ~b1); v[2] += __popc(~b0 & b1);
                    v[3] += __popc(b0 & b1); v[4] += __popc(b2);
                }
            }
            up = sm; sm = dn;
        }
    }
    if (MODE == 0) {          // acc[0] = B, acc[1] = M; warp sums fit 32 bits (<= 32 lanes x R rows x 512)
        const int bm[2] = {v[0], v[1]};
        block_accumulate<2>(bm, p.acc);
    } else {                  // d = k  <->  s*h = 4 - 2k  <->  hist index 8 - 2k (acc + 8)
        const int hist[9] = {v[4], 0, v[3], 0, v[2], 0, v[1], 0, v[0]};
        block_accumulate<9>(hist, p.acc + 8);
    }
}

template <int MODE>
static cudaError_t launch_lut_obs(ising_sim *h, int slab, int centre)
{
    LutObsParams p;
    const Slab &sl = h->slabs[slab];
    p.ctr = reinterpret_cast<const uint4 *>(sl.lat[centre]);
    p.nbr = reinterpret_cast<const uint4 *>(sl.lat[1 - centre]);
    p.nbr_up = reinterpret_cast<const char *>(halo_up(h, slab, 1 - centre));
    p.nbr_dn = reinterpret_cast<const char *>(halo_down(h, slab, 1 - centre));
    p.centre = centre;
    p.L = (int)sl.rows; p.cols = (int)(h->L / 256);
    p.R = 64;                 // rows per thread: as long as the grid keeps two full waves of threads
    while (p.R > 4 && (sl.rows / p.R) * p.cols < 148 * 2048 * 2) p.R >>= 1;
    p.acc = sl.d_acc;
    const int64_t threads = ((sl.rows + p.R - 1) / p.R) * p.cols;
    const int block = 128;
    lut_observe_kernel<MODE><<<(unsigned)((threads + block - 1) / block), block, 0, sl.stream>>>(p);
    h->launches++;
    return cudaGetLastError();
}

cudaError_t launch_lut_observables(ising_sim *h, int slab)
{
    cudaError_t e = cudaMemsetAsync(h->slabs[slab].d_acc, 0, 8 * sizeof(long long), h->slabs[slab].stream);
    if (e != cudaSuccess) return e;
    return launch_lut_obs<0>(h, slab, 0);
}

cudaError_t launch_lut_sd_hist(ising_sim *h, int slab)
{
    cudaError_t e = cudaMemsetAsync(h->slabs[slab].d_acc + 8, 0, 9 * sizeof(long long), h->slabs[slab].stream);
    if (e != cudaSuccess) return e;
    e = launch_lut_obs<1>(h, slab, 0);
    if (e != cudaSuccess) return e;
    return launch_lut_obs<1>(h, slab, 1);
}
