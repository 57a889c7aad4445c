// Packed lattice <-> int8 spins (A12 of SURVEY.md Sec. 8(a)), and the 1-bit planes
// the correlation kernels read (A9: "Pair product via 1-bit planes").
#include "ising_internal.cuh"

// ---------------------------------------------------------------- unpack ---
struct UnpackParams {
    const uint64_t *lat[2];
    int64_t L, x0, y0, w, hgt;
    int model;
    int8_t *out;
};

__global__ void __launch_bounds__(256) unpack_kernel(const __grid_constant__ UnpackParams p)
{
    int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= p.w * p.hgt) return;
    int64_t j = idx / p.w, i = idx - j * p.w;
    int64_t x = (p.x0 + i) % p.L, y = (p.y0 + j) % p.L;     // x0, y0 already reduced to [0, L)
    int c = (int)((x + y) & 1);
    int64_t k = x >> 1;
    if (p.model == ISING_MODEL_ISING_LUT) {                  // 1 bit per spin, 64 sites per word
        uint64_t word = p.lat[c][y * (p.L / 128) + (k >> 6)];
        p.out[idx] = (int8_t)(2 * (int)((word >> (k & 63)) & 1u) - 1);
        return;
    }
    if (p.model == ISING_MODEL_BLUME_CAPEL_2BIT) {           // 2 bits per spin, 32 sites per word
        uint64_t word = p.lat[c][y * (p.L / 64) + (k >> 5)];
        p.out[idx] = (int8_t)((int)((word >> (2 * (k & 31))) & 3u) - 1);
        return;
    }
    uint64_t word = p.lat[c][y * (p.L / 32) + (k >> 4)];
    int nib = (int)((word >> (4 * (k & 15))) & 15u);
    p.out[idx] = (int8_t)(p.model == ISING_MODEL_ISING ? 2 * nib - 1 : nib - 1);
}

cudaError_t launch_unpack(ising_sim *h, int64_t x0, int64_t y0, int64_t w, int64_t hgt, int8_t *dev_out)
{
    UnpackParams p;
    p.lat[0] = h->lat[0]; p.lat[1] = h->lat[1];
    p.L = h->L; p.x0 = x0; p.y0 = y0; p.w = w; p.hgt = hgt; p.model = h->model; p.out = dev_out;
    int64_t n = w * hgt;
    unpack_kernel<<<(unsigned)((n + 255) / 256), 256, 0, h->stream>>>(p);
    h->launches++;
    return cudaGetLastError();
}

// ------------------------------------------------------------------ pack ---
struct PackParams {
    uint32_t *lat[2];
    int64_t L, y0, ny;
    int model, dry;
    const int8_t *in;
    int *bad;
};

// one thread per 32-bit half (8 same-colour sites; 16 in the 2-bit layout) of rows [y0, y0 + ny)
__global__ void __launch_bounds__(256) pack_kernel(const __grid_constant__ PackParams p)
{
    const int sites = p.model == ISING_MODEL_BLUME_CAPEL_2BIT ? 16 : 8, bits = 32 / sites;
    const int64_t halves_per_row = p.L / (2 * sites);
    int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= p.ny * halves_per_row * 2) return;
    int c = (int)(idx & 1);
    int64_t rest = idx >> 1;
    int64_t row = rest / halves_per_row, hf = rest - row * halves_per_row;
    int64_t y = p.y0 + row;
    int par = (int)((y + c) & 1);
    uint32_t w = 0;
    bool bad = false;
    for (int j = 0; j < sites; ++j) {
        int64_t x = 2 * (hf * sites + j) + par;
        int v = p.in[row * p.L + x];
        uint32_t nib;
        if (p.model == ISING_MODEL_ISING) { bad |= (v != 1 && v != -1); nib = (v > 0) ? 1u : 0u; }
        else { bad |= (v < -1 || v > 1); nib = (uint32_t)(v + 1) & 3u; }
        w |= nib << (bits * j);
    }
    if (bad) atomicOr(p.bad, 1);
    if (!p.dry) p.lat[c][y * halves_per_row + hf] = w;
}

// 1-bit layout (ISING_MODEL_ISING_LUT): one thread per 32-bit half (32 same-colour sites)
__global__ void __launch_bounds__(256) pack_lut_kernel(const __grid_constant__ PackParams p)
{
    const int64_t halves_per_row = p.L / 64;
    int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= p.ny * halves_per_row * 2) return;
    int c = (int)(idx & 1);
    int64_t rest = idx >> 1;
    int64_t row = rest / halves_per_row, hf = rest - row * halves_per_row;
    int64_t y = p.y0 + row;
    int par = (int)((y + c) & 1);
    uint32_t w = 0;
    bool bad = false;
    for (int j = 0; j < 32; ++j) {
        int v = p.in[row * p.L + 2 * (hf * 32 + j) + par];
        bad |= (v != 1 && v != -1);
        w |= (v > 0 ? 1u : 0u) << j;
    }
    if (bad) atomicOr(p.bad, 1);
    if (!p.dry) p.lat[c][y * halves_per_row + hf] = w;
}

// write = 0: validate only (cudaErrorInvalidValue if a value is outside the model's set;
// synchronises).  write = 1: pack and store, no validation result.
cudaError_t launch_pack(ising_sim *h, int64_t y0, int64_t ny, const int8_t *dev_in, int *dev_bad, int write)
{
    PackParams p;
    p.lat[0] = reinterpret_cast<uint32_t *>(h->lat[0]);
    p.lat[1] = reinterpret_cast<uint32_t *>(h->lat[1]);
    p.L = h->L; p.y0 = y0; p.ny = ny; p.model = h->model; p.dry = !write; p.in = dev_in; p.bad = dev_bad;
    const bool lut = h->model == ISING_MODEL_ISING_LUT;
    int64_t n = ny * (h->L / sites_per_word(h->model)) * 2;      // 32-bit halves of both colours
    cudaError_t e;
    if (!write) {
        e = cudaMemsetAsync(dev_bad, 0, sizeof(int), h->stream);
        if (e != cudaSuccess) return e;
    }
    if (lut) pack_lut_kernel<<<(unsigned)((n + 255) / 256), 256, 0, h->stream>>>(p);
    else pack_kernel<<<(unsigned)((n + 255) / 256), 256, 0, h->stream>>>(p);
    h->launches++;
    e = cudaGetLastError();
    if (e != cudaSuccess || write) return e;
    int bad = 0;
    e = cudaMemcpyAsync(&bad, dev_bad, sizeof(int), cudaMemcpyDeviceToHost, h->stream);
    if (e != cudaSuccess) return e;
    e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return e;
    return bad ? cudaErrorInvalidValue : cudaSuccess;
}

// ---------------------------------------------------------------- planes ---
// plane[y][q] bit i  <->  site x = 64 q + i of row y.
//   sg: 1 iff spin == +1;   nz (Blume-Capel only): 1 iff spin != 0
// and the transposed planes planeT[x][y/64] so that S_x(r) of the lattice is S_y(r) of
// the transpose.  Layout of h->planes: [sg | sgT] (Ising) or [sg | nz | sgT | nzT] (BC),
// each L*L/8 bytes.
__device__ __forceinline__ uint32_t compress_nibble_bit(uint64_t w, int b)   // bit b of 16 nibbles -> 16 bits
{
    uint64_t x = (w >> b) & 0x1111111111111111ull;
    x = (x | (x >> 3)) & 0x0303030303030303ull;
    x = (x | (x >> 6)) & 0x000F000F000F000Full;
    x = (x | (x >> 12)) & 0x000000FF000000FFull;
    x = (x | (x >> 24)) & 0xFFFFull;
    return (uint32_t)x;
}

__device__ __forceinline__ uint32_t compress_pair_bit(uint64_t w, int b)     // bit b of 32 bit pairs -> 32 bits
{
    uint64_t x = (w >> b) & 0x5555555555555555ull;
    x = (x | (x >> 1)) & 0x3333333333333333ull;
    x = (x | (x >> 2)) & 0x0F0F0F0F0F0F0F0Full;
    x = (x | (x >> 4)) & 0x00FF00FF00FF00FFull;
    x = (x | (x >> 8)) & 0x0000FFFF0000FFFFull;
    x = (x | (x >> 16)) & 0xFFFFFFFFull;
    return (uint32_t)x;
}

__device__ __forceinline__ uint64_t spread_even(uint32_t v)   // bit i -> bit 2 i
{
    uint64_t x = v;
    x = (x | (x << 16)) & 0x0000FFFF0000FFFFull;
    x = (x | (x << 8)) & 0x00FF00FF00FF00FFull;
    x = (x | (x << 4)) & 0x0F0F0F0F0F0F0F0Full;
    x = (x | (x << 2)) & 0x3333333333333333ull;
    x = (x | (x << 1)) & 0x5555555555555555ull;
    return x;
}

struct PlaneParams {
    const uint64_t *lat[2];
    int64_t L;
    int model;
    uint64_t *sg, *nz;
};

__global__ void __launch_bounds__(256) planes_kernel(const __grid_constant__ PlaneParams p)
{
    const int64_t Wq = p.L / 64;
    int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= p.L * Wq) return;
    int64_t y = idx / Wq, q = idx - y * Wq;
    uint64_t sg = 0, nz = 0;
    if (p.model == ISING_MODEL_ISING_LUT) {                  // 1-bit layout: 32 sites of each colour per plane word
        for (int c = 0; c < 2; ++c) {
            const uint32_t *row32 = reinterpret_cast<const uint32_t *>(p.lat[c]) + y * Wq;
            sg |= spread_even(row32[q]) << (int)((y + c) & 1);
        }
        p.sg[idx] = sg;
        return;
    }
    if (p.model == ISING_MODEL_BLUME_CAPEL_2BIT) {           // 2-bit layout: one word = 32 sites of a colour
        for (int c = 0; c < 2; ++c) {
            const uint64_t w = p.lat[c][y * Wq + q];
            sg |= spread_even(compress_pair_bit(w, 1)) << (int)((y + c) & 1);       // code 2 = +1
            nz |= spread_even(compress_pair_bit(~w, 0)) << (int)((y + c) & 1);      // code != 1
        }
        p.sg[idx] = sg; p.nz[idx] = nz;
        return;
    }
    for (int c = 0; c < 2; ++c) {
        int par = (int)((y + c) & 1);
        const uint64_t *row = p.lat[c] + y * (p.L / 32);
        uint64_t w0 = row[2 * q], w1 = row[2 * q + 1];
        if (p.model == ISING_MODEL_ISING) {
            uint32_t m = compress_nibble_bit(w0, 0) | (compress_nibble_bit(w1, 0) << 16);
            sg |= spread_even(m) << par;
        } else {
            uint32_t m = compress_nibble_bit(w0, 1) | (compress_nibble_bit(w1, 1) << 16);        // code 2 = +1
            uint32_t z = compress_nibble_bit(~w0, 0) | (compress_nibble_bit(~w1, 0) << 16);      // code != 1
            sg |= spread_even(m) << par;
            nz |= spread_even(z) << par;
        }
    }
    p.sg[idx] = sg;
    if (p.model != ISING_MODEL_ISING) p.nz[idx] = nz;
}

// 64 x 64 bit-block transpose: block (bx, by) reads words in[64 by + j][bx], j = 0..63,
// writes out[64 bx + i][by] with bit j = bit i of in-word j.
__global__ void __launch_bounds__(64) transpose_kernel(const uint64_t *__restrict__ in, uint64_t *__restrict__ out, int64_t Wq)
{
    __shared__ uint64_t tile[64];
    int i = threadIdx.x;
    int64_t bx = blockIdx.x, by = blockIdx.y;
    tile[i] = in[(64 * by + i) * Wq + bx];
    __syncthreads();
    uint64_t o = 0;
#pragma unroll 16
    for (int j = 0; j < 64; ++j) o |= ((tile[j] >> i) & 1ull) << j;
    out[(64 * bx + i) * Wq + by] = o;
}

cudaError_t launch_planes(ising_sim *h)
{
    const int64_t L = h->L, Wq = L / 64, plane_words = L * Wq;
    const int np = is_blume_capel(h->model) ? 2 : 1;
    PlaneParams p;
    p.lat[0] = h->lat[0]; p.lat[1] = h->lat[1];
    p.L = L; p.model = h->model;
    p.sg = h->planes; p.nz = h->planes + plane_words;
    planes_kernel<<<(unsigned)((plane_words + 255) / 256), 256, 0, h->stream>>>(p);
    h->launches++;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    dim3 grid((unsigned)Wq, (unsigned)Wq);
    for (int k = 0; k < np; ++k) {
        transpose_kernel<<<grid, 64, 0, h->stream>>>(h->planes + k * plane_words, h->planes + (np + k) * plane_words, Wq);
        h->launches++;
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}
