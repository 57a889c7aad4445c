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
    // warp shuffle -> shared memory across the block's warps -> one int64 atomic per distance per block
    __shared__ int red[4][TR];
#pragma unroll
    for (int k = 0; k < TR; ++k) {
        int v = acc[k];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if (lane == 0) red[warp][k] = v;
    }
    __syncthreads();
    if (threadIdx.x < TR) {
        const int k = threadIdx.x;
        long long v = 0;
        for (int w = 0; w < nwarp; ++w) v += red[w][k];
        if (r0 + k <= rmax && v) atomicAdd((unsigned long long *)&accum[r0 + k - 1], (unsigned long long)v);
    }
}

// ----------------------------------------- explicit distance list + stride ---
// Sources: rows y % stride == 0, bits x % stride == 0; the partner (x, y + r) sits on the same
// comb of bits, so for stride >= 2 the planes are first down-sampled to that comb (all rows,
// L / stride bits per row, zero padded to whole words): 1/stride of the traffic and of the
// XOR + POPC work.  stride = 1 runs on the full planes.

// bits 0, 2, 4, ... of x gathered into the low 32 bits
__device__ __forceinline__ uint64_t gather_even(uint64_t x)
{
    x &= 0x5555555555555555ull;
    x = (x | (x >> 1)) & 0x3333333333333333ull;
    x = (x | (x >> 2)) & 0x0F0F0F0F0F0F0F0Full;
    x = (x | (x >> 4)) & 0x00FF00FF00FF00FFull;
    x = (x | (x >> 8)) & 0x0000FFFF0000FFFFull;
    x = (x | (x >> 16)) & 0x00000000FFFFFFFFull;
    return x;
}

// out[y][cw] packs, for j = 0..stride-1, the 64/stride comb bits of in[y][cw * stride + j]
__global__ void __launch_bounds__(256) comb_kernel(const uint64_t *__restrict__ in, uint64_t *__restrict__ out,
                                                   int L, int Wq, int Wc, int log2s)
{
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (int64_t)L * Wc) return;
    const int y = (int)(idx / Wc), cw = (int)(idx - (int64_t)y * Wc);
    const int s = 1 << log2s, bits = 64 >> log2s;
    uint64_t o = 0;
    for (int j = 0; j < s; ++j) {
        const int q = cw * s + j;
        if (q >= Wq) break;
        uint64_t w = in[(size_t)y * Wq + q];
        if (log2s == 4) {                     // the protocol's stride: bits 0, 16, 32, 48 -> 4 bits
            uint32_t lo = (uint32_t)w & 0x00010001u, hi = (uint32_t)(w >> 32) & 0x00010001u;
            lo = (lo | (lo >> 15)) & 3u; hi = (hi | (hi >> 15)) & 3u;
            w = lo | (hi << 2);
        } else {
            for (int k = 0; k < log2s; ++k) w = gather_even(w);
        }
        o |= w << (j * bits);
    }
    out[idx] = o;
}

// One block per distance.  W = words per row of the planes handed in (full or comb).
template <int MODEL>
__global__ void __launch_bounds__(256) corr_list_kernel(const uint64_t *__restrict__ sg, const uint64_t *__restrict__ nz,
                                                        int L, int W, int stride,
                                                        const long long *__restrict__ rlist, long long *__restrict__ out)
{
    const int r = (int)rlist[blockIdx.x];
    long long acc = 0;
    const int rows = L / stride;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    // a warp per source row, lanes over the words of the row (no per-element division), two rows in flight
    for (int yi = warp; yi < rows; yi += 2 * nwarp) {
        const int yj = yi + nwarp;
        const bool two = yj < rows;
        const int y0 = yi * stride, y1 = two ? yj * stride : y0;
        int yb0 = y0 + r, yb1 = y1 + r;
        if (yb0 >= L) yb0 -= L;
        if (yb1 >= L) yb1 -= L;
        const uint64_t *a0 = sg + (size_t)y0 * W, *b0 = sg + (size_t)yb0 * W;
        const uint64_t *a1 = sg + (size_t)y1 * W, *b1 = sg + (size_t)yb1 * W;
        int cnt = 0;
        for (int q = lane; q < W; q += 32) {
            const uint64_t xa = a0[q] ^ b0[q], xb = a1[q] ^ b1[q];
            if (MODEL == ISING_MODEL_ISING) cnt += __popcll(xa) + (two ? __popcll(xb) : 0);
            else {
                const uint64_t both0 = nz[(size_t)y0 * W + q] & nz[(size_t)yb0 * W + q];
                cnt += __popcll(both0) - 2 * __popcll(both0 & xa);
                if (two) {
                    const uint64_t both1 = nz[(size_t)y1 * W + q] & nz[(size_t)yb1 * W + q];
                    cnt += __popcll(both1) - 2 * __popcll(both1 & xb);
                }
            }
        }
        acc += cnt;
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

// stride == 0: full-source tiled kernel for r = 1..count (dev_r ignored), raw popcount
// sums are converted to pair sums on the host (api.cu).  stride >= 1: list kernel.
cudaError_t launch_corr(ising_sim *h, int64_t stride, int64_t count, const long long *dev_r,
                        long long *dev_sx, long long *dev_sy)
{
    const int L = (int)h->L, Wq = L / 64;
    const size_t pw = (size_t)L * Wq;
    const bool ising = !is_blume_capel(h->model);
    const int np = ising ? 1 : 2;
    const uint64_t *sg = h->planes, *nz = ising ? nullptr : h->planes + pw;
    const uint64_t *sgT = h->planes + np * pw, *nzT = ising ? nullptr : h->planes + (np + 1) * pw;
    // (the four pointers are re-aimed at the comb planes below when stride >= 2)
    if (stride == 0) {
        cudaError_t e = cudaMemsetAsync(dev_sx, 0, count * sizeof(long long), h->stream);
        if (e != cudaSuccess) return e;
        e = cudaMemsetAsync(dev_sy, 0, count * sizeof(long long), h->stream);
        if (e != cudaSuccess) return e;
        // y-tiles are dealt to warps round-robin; enough blocks to fill 148 SMs x 8 even when
        // only a few distance blocks are asked for (the protocol's r <= 32 is one)
        const int ytiles = L / TY, gx = (int)((count + TR - 1) / TR);
        int gy = (ytiles + 4 * 32 - 1) / (4 * 32);       // ~32 y-tiles per warp
        const int want = (148 * 8 + gx - 1) / gx;
        if (gy < want) gy = want;
        if (gy > (ytiles + 3) / 4) gy = (ytiles + 3) / 4;
        if (gy < 1) gy = 1;
        dim3 grid((unsigned)gx, (unsigned)gy);
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
    // list kernel: on the full planes (stride 1) or on their comb (stride >= 2)
    int W = Wq;
    if (stride >= 2) {
        int log2s = 0;
        while ((1 << log2s) < stride) ++log2s;
        W = (int)comb_words_per_row(L, stride);
        const size_t cw = (size_t)L * W;
        const uint64_t *src[4] = {sg, nz, sgT, nzT};
        uint64_t *dst[4] = {h->comb, h->comb + cw, h->comb + (ising ? 1 : 2) * cw, h->comb + 3 * cw};
        for (int k = 0; k < 4; ++k) {
            if (!src[k]) continue;
            comb_kernel<<<(unsigned)((cw + 255) / 256), 256, 0, h->stream>>>(src[k], dst[k], L, Wq, W, log2s);
            h->launches++;
        }
        sg = dst[0]; nz = ising ? nullptr : dst[1]; sgT = dst[2]; nzT = ising ? nullptr : dst[3];
    }
    if (ising) {
        corr_list_kernel<ISING_MODEL_ISING><<<(unsigned)count, 256, 0, h->stream>>>(sg, nz, L, W, (int)stride, dev_r, dev_sy);
        corr_list_kernel<ISING_MODEL_ISING><<<(unsigned)count, 256, 0, h->stream>>>(sgT, nzT, L, W, (int)stride, dev_r, dev_sx);
    } else {
        corr_list_kernel<ISING_MODEL_BLUME_CAPEL><<<(unsigned)count, 256, 0, h->stream>>>(sg, nz, L, W, (int)stride, dev_r, dev_sy);
        corr_list_kernel<ISING_MODEL_BLUME_CAPEL><<<(unsigned)count, 256, 0, h->stream>>>(sgT, nzT, L, W, (int)stride, dev_r, dev_sx);
    }
    h->launches += 2;
    return cudaGetLastError();
}
