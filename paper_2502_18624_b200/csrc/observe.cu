// Integer observables (A8 of SURVEY.md Sec. 8(a)) and the Schwinger-Dyson
// histogram (Eq. 3).  Same register sliding window as the update
// kernel: each thread walks R rows of one 128-bit column (64-bit at 2 bits per spin) of the BLACK array and
// sees every bond exactly once (for even L every bond joins a black and a white
// site).  Warp reduction -> one int64 atomic per block per quantity (block_accumulate).
#include "ising_internal.cuh"
#include "row_format.cuh"

#define ONES 0x11111111u

struct ObsParams {
    const uint4 *ctr, *nbr;   // centre-colour array, neighbour-colour array: the rows of this slab
    const char *nbr_up, *nbr_dn;   // neighbour-colour row above / below the slab (NEXT-4; own last / first row when unsharded)
    int centre;               // colour of the centre sites
    int L, cols, R;           // L = rows of this slab
    long long *acc;
};

__device__ __forceinline__ uint32_t nibble_sum(uint32_t x)  // sum of the 8 nibbles (each <= 15)
{
    uint32_t t = (x & 0x0F0F0F0Fu) + ((x >> 4) & 0x0F0F0F0Fu);
    return (t * 0x01010101u) >> 24;
}

// MODE 0: B, M, Q.  MODE 1: Schwinger-Dyson histogram of s*h over the centre sites.
template <int MODEL, int MODE>
__device__ __forceinline__ void obs_half(uint32_t x, uint32_t up, uint32_t dn, uint32_t sm, uint32_t sd,
                                         int &B, int &M, int &Q, int hist[9])
{
    if (MODEL == ISING_MODEL_ISING) {
        uint32_t d = (up ^ x) + (dn ^ x) + (sm ^ x) + (sd ^ x);   // unequal neighbours per site
        if (MODE == 0) {
            B += 32 - 2 * (int)nibble_sum(d);                      // sum of s*h = sum (4 - 2 d)
            M += 2 * (__popc(x) + __popc(sm)) - 16;                // black half + the white half of this row
            Q += 16;
        } else {
#pragma unroll
            for (int k = 0; k <= 4; ++k) {                         // s*h = 4 - 2k
                uint32_t e = d ^ (ONES * (uint32_t)k);             // nibble == 0 where d == k
                e = (e | (e >> 1) | (e >> 2)) & ONES;
                hist[8 - 2 * k] += 8 - __popc(e);
            }
        }
    } else {
        uint32_t S = up + dn + sm + sd;                            // h + 4 per site
        if (MODE == 0) {
            // Word level, in the codes c = s + 1 ("similar to an energy computation using a short look-up
            // table" -- here no table at all): the nibbles are spread to bytes and summed by 4-way byte dot products
            // (IDP4A).  B accumulates sum_black c S, M sum c and Q sum c^2 over the black word and the white word of
            // the same position; the kernel turns them into B, M, Q at the end (observe_kernel).
            const uint32_t lo = 0x0F0F0F0Fu, one = 0x01010101u;
            const uint32_t Se = S & lo, So = (S >> 4) & lo, ce = x & lo, co = (x >> 4) & lo, we = sm & lo, wo = (sm >> 4) & lo;
            uint32_t b = (uint32_t)B, m = (uint32_t)M, q = (uint32_t)Q;
            b = __dp4a(ce, Se, b); b = __dp4a(co, So, b);
            m = __dp4a(ce + co + we + wo, one, m);                 // bytes <= 8
            q = __dp4a(ce, ce, q); q = __dp4a(co, co, q); q = __dp4a(we, we, q); q = __dp4a(wo, wo, q);
            B = (int)b; M = (int)m; Q = (int)q;
        } else {
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                int code = (x >> (4 * j)) & 15, h = (int)((S >> (4 * j)) & 15u) - 4;
                hist[(code - 1) * h + 4] += 1;
            }
        }
    }
}

template <int MODEL, int MODE>
__global__ void __launch_bounds__(256) observe_kernel(const __grid_constant__ ObsParams p)
{
    // centre sites: colour p.centre (array `ctr`), neighbours in the other array (`nbr`);
    // row parity of the centre colour is (y + centre) & 1
    const int cols = p.cols, L = p.L;
    unsigned tid = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned chunk = tid / (unsigned)cols;
    int col = (int)(tid - chunk * (unsigned)cols);
    int y0 = (int)chunk * p.R;
    int B = 0, M = 0, Q = 0;
    int hist[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
    if (y0 < L) {
        int yend = min(L, y0 + p.R);
        constexpr int VB = RowFmt<MODEL>::kVecBytes;
        const char *nbr = reinterpret_cast<const char *>(p.nbr), *ctr = reinterpret_cast<const char *>(p.ctr);
        const size_t rs = (size_t)cols * VB, cb = (size_t)col * VB;
        const size_t e0 = (size_t)edge_half<MODEL, 0>(col, cols) * 4;   // parity 0: neighbour k-1
        const size_t e1 = (size_t)edge_half<MODEL, 1>(col, cols) * 4;   // parity 1: neighbour k+1
        uint4 up = load_row<MODEL>((y0 == 0) ? p.nbr_up + cb : nbr + (size_t)(y0 - 1) * rs + cb);
        uint4 sm = load_row<MODEL>(nbr + (size_t)y0 * rs + cb);
        for (int y = y0; y < yend; ++y) {
            uint4 dn = load_row<MODEL>((y + 1 == L) ? p.nbr_dn + cb : nbr + (size_t)(y + 1) * rs + cb);
            uint4 x = load_row<MODEL>(ctr + (size_t)y * rs + cb);
            uint32_t sd[4];
            if (((y + p.centre) & 1) == 0) side_words<MODEL, 0>(sm, *reinterpret_cast<const uint32_t *>(nbr + (size_t)y * rs + e0), sd);
            else side_words<MODEL, 1>(sm, *reinterpret_cast<const uint32_t *>(nbr + (size_t)y * rs + e1), sd);
            obs_half<MODEL, MODE>(x.x, up.x, dn.x, sm.x, sd[0], B, M, Q, hist);
            obs_half<MODEL, MODE>(x.y, up.y, dn.y, sm.y, sd[1], B, M, Q, hist);
            obs_half<MODEL, MODE>(x.z, up.z, dn.z, sm.z, sd[2], B, M, Q, hist);
            obs_half<MODEL, MODE>(x.w, up.w, dn.w, sm.w, sd[3], B, M, Q, hist);
            up = sm; sm = dn;
        }
    }
    if (MODE == 0) {          // warp sums fit 32 bits: <= 32 lanes x R rows x 128 sites x 4
        if (MODEL != ISING_MODEL_ISING && y0 < L) {
            // (B, M, Q) hold (sum_black c S, sum c, sum c^2) over this thread's n black and n white sites.  With
            // s = c - 1, h = S - 4:  sum_black s h = sum cS - 4 sum_black c - sum_black S + 4 n, and over the whole
            // lattice sum_black S = 4 sum_white c (every white site is the neighbour of four black ones), so the
            // per-thread shares  B' = sum cS - 4 sum c + 4 n  add up to the bond sum;  M = sum c - 2 n;
            // Q = sum (c - 1)^2 = sum c^2 - 2 sum c + 2 n.
            const int n = (min(L, y0 + p.R) - y0) * 32;
            const int cS = B, c1 = M, c2 = Q;
            B = cS - 4 * c1 + 4 * n; M = c1 - 2 * n; Q = c2 - 2 * c1 + 2 * n;
        }
        const int v[3] = {B, M, Q};
        block_accumulate<3>(v, p.acc);
    } else {
        block_accumulate<9>(hist, p.acc + 8);
    }
}

template <int MODE>
static cudaError_t launch_obs(ising_sim *h, int slab, int centre)
{
    ObsParams p;
    const Slab &sl = h->slabs[slab];
    p.ctr = reinterpret_cast<const uint4 *>(sl.lat[centre]);
    p.nbr = reinterpret_cast<const uint4 *>(sl.lat[1 - centre]);
    p.nbr_up = reinterpret_cast<const char *>(halo_up(h, slab, 1 - centre));
    p.nbr_dn = reinterpret_cast<const char *>(halo_down(h, slab, 1 - centre));
    p.centre = centre;
    p.L = (int)sl.rows; p.cols = (int)(h->L / 64);
    p.R = (h->L >= 65536) ? 64 : (h->L >= 2048) ? 32 : 4;   // rows per thread: halo re-reads 2/R, still >= 1 M threads at R = 64
    p.acc = sl.d_acc;
    int64_t chunks = (sl.rows + p.R - 1) / p.R;
    int64_t threads = chunks * p.cols;
    int block = 128;
    unsigned grid = (unsigned)((threads + block - 1) / block);
    if (h->model == ISING_MODEL_ISING) observe_kernel<ISING_MODEL_ISING, MODE><<<grid, block, 0, sl.stream>>>(p);
    else if (h->model == ISING_MODEL_BLUME_CAPEL) observe_kernel<ISING_MODEL_BLUME_CAPEL, MODE><<<grid, block, 0, sl.stream>>>(p);
    else observe_kernel<ISING_MODEL_BLUME_CAPEL_2BIT, MODE><<<grid, block, 0, sl.stream>>>(p);
    h->launches++;
    return cudaGetLastError();
}

// B, M, Q: centre = black sees every bond once; M and Q also count the white words of
// the centre row (`sm`), so one pass covers both arrays.
cudaError_t launch_observables(ising_sim *h, int slab)
{
    cudaError_t e = cudaMemsetAsync(h->slabs[slab].d_acc, 0, 8 * sizeof(long long), h->slabs[slab].stream);
    if (e != cudaSuccess) return e;
    return launch_obs<0>(h, slab, 0);
}

// Schwinger-Dyson histogram over ALL sites: one pass centred on each colour.
cudaError_t launch_sd_hist(ising_sim *h, int slab)
{
    cudaError_t e = cudaMemsetAsync(h->slabs[slab].d_acc + 8, 0, 9 * sizeof(long long), h->slabs[slab].stream);
    if (e != cudaSuccess) return e;
    e = launch_obs<1>(h, slab, 0);
    if (e != cudaSuccess) return e;
    return launch_obs<1>(h, slab, 1);
}
