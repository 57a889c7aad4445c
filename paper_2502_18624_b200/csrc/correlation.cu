// Correlation pair sums (A9/A10 of SURVEY.md Sec. 8(a)).
//
// Both kernels compute "S_y on a plane set": for bit planes P[y][q] (bit i of word q
// = site x = 64 q + i of row y)
//     S(r) = sum_y sum_x s(x, y) s(x, (y + r) mod L)
// with the pair product evaluated 64 sites at a time:
//     Ising        sum = n_pairs - 2 popc(sg ^ sg')
//     Blume-Capel  sum = popc(nz & nz') - 2 popc(nz & nz' & (sg ^ sg'))
// S_x of the lattice is S_y of the transposed planes (lattice_io.cu).
#include "ising_internal.cuh"

// ------------------------------------------------ full-source, r = 1..rmax ---
// Register tiling: a thread keeps TY source-row words a[0..TY) of one word column q
// and streams the TY + TR - 1 partner rows once; pair (j, i) contributes to distance
// r0 + (i - j).  TR accumulators live in registers across the q loop and the y-tile
// loop, so a partner word loaded once feeds up to TY pair products.
#define TY 8
#define TR 32

template <int MODEL>
__global__ void __launch_bounds__(128) corr_full_kernel(const uint64_t *__restrict__ sg, const uint64_t *__restrict__ nz,
                                                        int L, int Wq, int rmax, long long *__restrict__ accum)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    const int r0 = 1 + TR * blockIdx.x;
    int acc[TR];
#pragma unroll
    for (int k = 0; k < TR; ++k) acc[k] = 0;

    const int ytiles = L / TY;
    for (int yt = blockIdx.y * nwarp + warp; yt < ytiles; yt += gridDim.y * nwarp) {
        const int y0 = yt * TY;
        for (int q = lane; q < Wq; q += 32) {
            uint64_t a[TY], az[TY];
#pragma unroll
            for (int j = 0; j < TY; ++j) {
                a[j] = sg[(size_t)(y0 + j) * Wq + q];
                if (MODEL != ISING_MODEL_ISING) az[j] = nz[(size_t)(y0 + j) * Wq + q];
            }
            int yb = y0 + r0;                 // first partner row
            if (yb >= L) yb -= L;             // r0 <= L/2 and y0 < L: one wrap at most
#pragma unroll
            for (int i = 0; i < TY + TR - 1; ++i) {
                uint64_t b = sg[(size_t)yb * Wq + q], bz = 0;
                if (MODEL != ISING_MODEL_ISING) bz = nz[(size_t)yb * Wq + q];
                if (++yb == L) yb = 0;
#pragma unroll
                for (int j = 0; j < TY; ++j) {
                    const int rr = i - j;
                    if (rr >= 0 && rr < TR) {
                        if (MODEL == ISING_MODEL_ISING) acc[rr] += __popcll(a[j] ^ b);
                        else {
                            uint64_t both = az[j] & bz;
                            acc[rr] += __popcll(both) - 2 * __popcll(both & (a[j] ^ b));
                        }
                    }
                }
            }
        }
    }
#pragma unroll
    for (int k = 0; k < TR; ++k) {
        int v = acc[k];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if (lane == 0 && r0 + k <= rmax) atomicAdd((unsigned long long *)&accum[r0 + k - 1], (unsigned long long)(long long)v);
    }
}

// ----------------------------------------- explicit distance list + stride ---
// One block per distance.  Sources: rows y % stride == 0, bits x % stride == 0.
template <int MODEL>
__global__ void __launch_bounds__(256) corr_list_kernel(const uint64_t *__restrict__ sg, const uint64_t *__restrict__ nz,
                                                        int L, int Wq, int stride, uint64_t mask,
                                                        const long long *__restrict__ rlist, long long *__restrict__ out)
{
    const int r = (int)rlist[blockIdx.x];
    long long acc = 0;
    const int rows = L / stride;
    for (int idx = threadIdx.x; idx < rows * Wq; idx += blockDim.x) {
        int yi = idx / Wq, q = idx - yi * Wq;
        int y = yi * stride;
        int yb = y + r;
        if (yb >= L) yb -= L;
        uint64_t a = sg[(size_t)y * Wq + q], b = sg[(size_t)yb * Wq + q];
        if (MODEL == ISING_MODEL_ISING) acc += __popcll((a ^ b) & mask);
        else {
            uint64_t both = nz[(size_t)y * Wq + q] & nz[(size_t)yb * Wq + q] & mask;
            acc += __popcll(both) - 2 * __popcll(both & (a ^ b));
        }
    }
    __shared__ long long red[8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        long long s = 0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) s += red[w];
        out[blockIdx.x] = s;     // Ising: number of unequal pairs; BC: the signed sum itself
    }
}

static uint64_t stride_mask(int64_t s)
{
    switch (s) {
        case 1: return ~0ull;
        case 2: return 0x5555555555555555ull;
        case 4: return 0x1111111111111111ull;
        case 8: return 0x0101010101010101ull;
        case 16: return 0x0001000100010001ull;
        case 32: return 0x0000000100000001ull;
        default: return 1ull;
    }
}

// stride == 0: full-source tiled kernel for r = 1..count (dev_r ignored), raw popcount
// sums are converted to pair sums on the host (api.cu).  stride >= 1: list kernel.
cudaError_t launch_corr(ising_sim *h, int64_t stride, int64_t count, const long long *dev_r,
                        long long *dev_sx, long long *dev_sy)
{
    const int L = (int)h->L, Wq = L / 64;
    const size_t pw = (size_t)L * Wq;
    const bool ising = h->model == ISING_MODEL_ISING;
    const int np = ising ? 1 : 2;
    const uint64_t *sg = h->planes, *nz = ising ? nullptr : h->planes + pw;
    const uint64_t *sgT = h->planes + np * pw, *nzT = ising ? nullptr : h->planes + (np + 1) * pw;
    if (stride == 0) {
        cudaError_t e = cudaMemsetAsync(dev_sx, 0, count * sizeof(long long), h->stream);
        if (e != cudaSuccess) return e;
        e = cudaMemsetAsync(dev_sy, 0, count * sizeof(long long), h->stream);
        if (e != cudaSuccess) return e;
        int ytiles = L / TY;
        int gy = (ytiles + 4 * 32 - 1) / (4 * 32);       // ~32 y-tiles per warp
        if (gy < 1) gy = 1;
        dim3 grid((unsigned)((count + TR - 1) / TR), (unsigned)gy);
        if (ising) {
            corr_full_kernel<ISING_MODEL_ISING><<<grid, 128, 0, h->stream>>>(sg, nz, L, Wq, (int)count, dev_sy);
            corr_full_kernel<ISING_MODEL_ISING><<<grid, 128, 0, h->stream>>>(sgT, nzT, L, Wq, (int)count, dev_sx);
        } else {
            corr_full_kernel<ISING_MODEL_BLUME_CAPEL><<<grid, 128, 0, h->stream>>>(sg, nz, L, Wq, (int)count, dev_sy);
            corr_full_kernel<ISING_MODEL_BLUME_CAPEL><<<grid, 128, 0, h->stream>>>(sgT, nzT, L, Wq, (int)count, dev_sx);
        }
        h->launches += 2;
        return cudaGetLastError();
    }
    uint64_t mask = stride_mask(stride);
    if (ising) {
        corr_list_kernel<ISING_MODEL_ISING><<<(unsigned)count, 256, 0, h->stream>>>(sg, nz, L, Wq, (int)stride, mask, dev_r, dev_sy);
        corr_list_kernel<ISING_MODEL_ISING><<<(unsigned)count, 256, 0, h->stream>>>(sgT, nzT, L, Wq, (int)stride, mask, dev_r, dev_sx);
    } else {
        corr_list_kernel<ISING_MODEL_BLUME_CAPEL><<<(unsigned)count, 256, 0, h->stream>>>(sg, nz, L, Wq, (int)stride, mask, dev_r, dev_sy);
        corr_list_kernel<ISING_MODEL_BLUME_CAPEL><<<(unsigned)count, 256, 0, h->stream>>>(sgT, nzT, L, Wq, (int)stride, mask, dev_r, dev_sx);
    }
    h->launches += 2;
    return cudaGetLastError();
}
