// Packed lattice <-> int8 spins (A12 of SURVEY.md Sec. 8(a)), and the 1-bit planes
// the correlation kernels read (A9: "Pair product via 1-bit planes").
#include "ising_internal.cuh"

SlabDir slab_directory(const ising_sim *h)
{
    SlabDir d;
    d.n = (int)h->slabs.size();
    d.y_first = h->slabs[0].y0;
    for (int k = 0; k < ISING_MAX_SLABS; ++k) {
        const bool live = k < d.n;
        d.y_end[k] = live ? h->slabs[k].y0 + h->slabs[k].rows : h->L;
        for (int c = 0; c < 2; ++c) d.lat[c][k] = live ? h->slabs[k].lat[c] : nullptr;
    }
    return d;
}

// ---------------------------------------------------------------- unpack ---
struct UnpackParams {
    SlabDir dir;
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
        uint64_t word = slab_row(p.dir, c, y, p.L / 128)[k >> 6];
        p.out[idx] = (int8_t)(2 * (int)((word >> (k & 63)) & 1u) - 1);
        return;
    }
    if (p.model == ISING_MODEL_BLUME_CAPEL_2BIT) {           // 2 bits per spin, 32 sites per word
        uint64_t word = slab_row(p.dir, c, y, p.L / 64)[k >> 5];
        p.out[idx] = (int8_t)((int)((word >> (2 * (k & 31))) & 3u) - 1);
        return;
    }
    uint64_t word = slab_row(p.dir, c, y, p.L / 32)[k >> 4];
    int nib = (int)((word >> (4 * (k & 15))) & 15u);
    p.out[idx] = (int8_t)(p.model == ISING_MODEL_ISING ? 2 * nib - 1 : nib - 1);
}

cudaError_t launch_unpack(ising_sim *h, int64_t x0, int64_t y0, int64_t w, int64_t hgt, int8_t *dev_out)
{
    UnpackParams p;
    p.dir = slab_directory(h);
    p.L = h->L; p.x0 = x0; p.y0 = y0; p.w = w; p.hgt = hgt; p.model = h->model; p.out = dev_out;
    int64_t n = w * hgt;
    unpack_kernel<<<(unsigned)((n + 255) / 256), 256, 0, h->stream>>>(p);
    h->launches++;
    return cudaGetLastError();
}

// ------------------------------------------------------------------ pack ---
struct PackParams {
    SlabDir dir;
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
    if (!p.dry) reinterpret_cast<uint32_t *>(slab_row(p.dir, c, y, halves_per_row / 2))[hf] = w;
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
    if (!p.dry) reinterpret_cast<uint32_t *>(slab_row(p.dir, c, y, halves_per_row / 2))[hf] = w;
}

// write = 0: validate only (cudaErrorInvalidValue if a value is outside the model's set;
// synchronises).  write = 1: pack and store, no validation result.
cudaError_t launch_pack(ising_sim *h, int64_t y0, int64_t ny, const int8_t *dev_in, int *dev_bad, int write)
{
    PackParams p;
    p.dir = slab_directory(h);
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
__device__ __forceinline__ uint64_t nibble_bit_to_even(uint64_t w, int b)   // bit b of nibble j -> bit 2 j (j = 0..15)
{
    uint64_t x = (w >> b) & 0x1111111111111111ull;
    x = (x | (x >> 2)) & 0x0505050505050505ull;
    x = (x | (x >> 4)) & 0x0055005500550055ull;
    x = (x | (x >> 8)) & 0x0000555500005555ull;
    x = (x | (x >> 16)) & 0x0000000055555555ull;
    return x;
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
    SlabDir dir;
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
            const uint32_t *row32 = reinterpret_cast<const uint32_t *>(slab_row(p.dir, c, y, Wq / 2));
            sg |= spread_even(row32[q]) << (int)((y + c) & 1);
        }
        p.sg[idx] = sg;
        return;
    }
    if (p.model == ISING_MODEL_BLUME_CAPEL_2BIT) {           // 2-bit layout: one word = 32 sites of a colour, pair j at bit 2 j
        for (int c = 0; c < 2; ++c) {
            const uint64_t w = slab_row(p.dir, c, y, Wq)[q];
            sg |= ((w >> 1) & 0x5555555555555555ull) << (int)((y + c) & 1);       // code 2 = +1: high bit of the pair
            nz |= (~w & 0x5555555555555555ull) << (int)((y + c) & 1);             // code != 1: low bit clear
        }
        p.sg[idx] = sg; p.nz[idx] = nz;
        return;
    }
    for (int c = 0; c < 2; ++c) {
        int par = (int)((y + c) & 1);
        const uint64_t *row = slab_row(p.dir, c, y, p.L / 32);
        uint64_t w0 = row[2 * q], w1 = row[2 * q + 1];
        if (p.model == ISING_MODEL_ISING) {
            sg |= (nibble_bit_to_even(w0, 0) | (nibble_bit_to_even(w1, 0) << 32)) << par;
        } else {
            sg |= (nibble_bit_to_even(w0, 1) | (nibble_bit_to_even(w1, 1) << 32)) << par;        // code 2 = +1
            nz |= (nibble_bit_to_even(~w0, 0) | (nibble_bit_to_even(~w1, 0) << 32)) << par;      // code != 1
        }
    }
    p.sg[idx] = sg;
    if (p.model != ISING_MODEL_ISING) p.nz[idx] = nz;
}

// Bit-matrix transpose out[x][y] = in[y][x] of an L x L plane, in 32 x 32 bit tiles (a uint64 word is two
// consecutive 32-bit words, low half first, so the 32-bit view is the same matrix).  A warp holds one tile,
// one row per lane, and transposes it with five rounds of block swaps between lanes (`shfl.xor` by 16, 8, 4,
// 2, 1: about one instruction per word instead of the 3 per word of gathering 32 bits one by one).  A block
// moves a panel of 8 x 32 tiles through shared memory.  W32 = L / 32 words per row; L is a multiple of 64,
// panels may be ragged.
__device__ __forceinline__ uint32_t transpose32(uint32_t a, int lane)
{
    const uint32_t masks[5] = {0x0000FFFFu, 0x00FF00FFu, 0x0F0F0F0Fu, 0x33333333u, 0x55555555u};
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        const int s = 16 >> k;
        const uint32_t m = masks[k];
        const uint32_t x = __shfl_xor_sync(0xffffffffu, a, s);
        a = (lane & s) ? (((x >> s) & m) | (a & ~m)) : ((a & m) | ((x & m) << s));
    }
    return a;
}

__global__ void __launch_bounds__(256) transpose_kernel(const uint32_t *__restrict__ in, uint32_t *__restrict__ out,
                                                        int64_t L, int64_t W32)
{
    // panel: 256 input rows x 32 words (8 x 32 tiles) -> 1024 output rows x 8 words.  blockIdx.x walks the
    // input rows (= the output words), so consecutive blocks write neighbouring 32-byte pieces of the same
    // output rows and the L2 assembles full lines; the reads are 128 contiguous bytes per row.
    __shared__ uint32_t buf[1024 * 9];                      // in: [256][33], out: [1024][9] (odd strides: no bank conflicts)
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    const int64_t row0 = 256 * (int64_t)blockIdx.x, word0 = 32 * (int64_t)blockIdx.y;
#pragma unroll 8
    for (int i = 0; i < 32; ++i) {
        const int row = warp + 8 * i;
        const int64_t y = row0 + row;
        uint32_t v = 0;
        if (y < L && word0 + lane < W32) v = in[y * W32 + word0 + lane];
        buf[row * 33 + lane] = v;
    }
    __syncthreads();
    uint32_t r[32];
#pragma unroll
    for (int tx = 0; tx < 32; ++tx) r[tx] = transpose32(buf[(32 * warp + lane) * 33 + tx], lane);   // tile (ty = warp, tx)
    __syncthreads();
#pragma unroll
    for (int tx = 0; tx < 32; ++tx) buf[(32 * tx + lane) * 9 + warp] = r[tx];                      // output row 32 tx + lane, word ty
    __syncthreads();
    const int64_t x0 = 1024 * (int64_t)blockIdx.y, yw = 8 * (int64_t)blockIdx.x + (lane & 7);
#pragma unroll 8
    for (int i = 0; i < 32; ++i) {
        const int row = 32 * i + 4 * warp + (lane >> 3);
        const int64_t x = x0 + row;
        if (x < L && yw < W32) out[x * W32 + yw] = buf[row * 9 + (lane & 7)];
    }
}

cudaError_t launch_planes(ising_sim *h)
{
    const int64_t L = h->L, Wq = L / 64, plane_words = L * Wq;
    const int np = is_blume_capel(h->model) ? 2 : 1;
    PlaneParams p;
    p.dir = slab_directory(h);
    p.L = L; p.model = h->model;
    p.sg = h->planes; p.nz = h->planes + plane_words;
    planes_kernel<<<(unsigned)((plane_words + 255) / 256), 256, 0, h->stream>>>(p);
    h->launches++;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    const int64_t W32 = 2 * Wq;
    dim3 grid((unsigned)((L + 255) / 256), (unsigned)((W32 + 31) / 32));
    for (int k = 0; k < np; ++k) {
        transpose_kernel<<<grid, 256, 0, h->stream>>>(reinterpret_cast<const uint32_t *>(h->planes + k * plane_words),
                                                     reinterpret_cast<uint32_t *>(h->planes + (np + k) * plane_words), L, W32);
        h->launches++;
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

// ------------------------------------------------------- compact transport ---
// ising_write_bits / ising_read_bits: the lattice at the information content of a spin -- 1 bit per Ising
// spin, 2 bits per Blume-Capel spin -- in the site order of the packed arrays (the layouts of the 1-bit and
// 2-bit models), expanded to / gathered from the 4-bit nibbles on the device.  One thread per 128-bit
// lattice vector (32 sites): 32 input bits (Ising) or 64 (Blume-Capel).
__device__ __forceinline__ uint64_t bits16_to_nibbles(uint32_t v)          // bit j -> nibble j (j = 0..15)
{
    uint64_t x = v & 0xFFFFu;
    x = (x | (x << 24)) & 0x000000FF000000FFull;
    x = (x | (x << 12)) & 0x000F000F000F000Full;
    x = (x | (x << 6)) & 0x0303030303030303ull;
    x = (x | (x << 3)) & 0x1111111111111111ull;
    return x;
}

__device__ __forceinline__ uint32_t nibbles_to_bits16(uint64_t x)          // bit 0 of nibble j -> bit j
{
    x &= 0x1111111111111111ull;
    x = (x | (x >> 3)) & 0x0303030303030303ull;
    x = (x | (x >> 6)) & 0x000F000F000F000Full;
    x = (x | (x >> 12)) & 0x000000FF000000FFull;
    x = (x | (x >> 24)) & 0xFFFFull;
    return (uint32_t)x;
}

__device__ __forceinline__ uint64_t pairs16_to_nibbles(uint32_t v)         // bit pair j -> nibble j (j = 0..15)
{
    uint64_t x = v;
    x = (x | (x << 16)) & 0x0000FFFF0000FFFFull;
    x = (x | (x << 8)) & 0x00FF00FF00FF00FFull;
    x = (x | (x << 4)) & 0x0F0F0F0F0F0F0F0Full;
    x = (x | (x << 2)) & 0x3333333333333333ull;
    return x;
}

__device__ __forceinline__ uint32_t nibbles_to_pairs16(uint64_t x)         // low two bits of nibble j -> bit pair j
{
    x &= 0x3333333333333333ull;
    x = (x | (x >> 2)) & 0x0F0F0F0F0F0F0F0Full;
    x = (x | (x >> 4)) & 0x00FF00FF00FF00FFull;
    x = (x | (x >> 8)) & 0x0000FFFF0000FFFFull;
    x = (x | (x >> 16)) & 0xFFFFFFFFull;
    return (uint32_t)x;
}

struct BitsParams {
    SlabDir dir;
    int64_t L, row0, nrows;      // rows [row0, row0 + nrows) of colour `colour`
    int colour, bc, mode;        // mode 0: validate only, 1: expand into the lattice, 2: gather from the lattice
    int two_bit;                 // the lattice itself is stored at 2 bits per spin: the format is the layout, no expansion
    uint32_t *buf;               // staging: nrows x (L/64) x {1 (Ising) | 2 (Blume-Capel)} uint32, row-major
    int *bad;
};

__global__ void __launch_bounds__(256) bits_kernel(const __grid_constant__ BitsParams p)
{
    const int64_t vecs = p.L / 64;                               // 128-bit vectors per colour row
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= p.nrows * vecs) return;
    const int64_t row = idx / vecs, v = idx - row * vecs;
    if (p.two_bit) {                                             // validate / store one 64-bit word (32 sites) as it is
        const uint32_t a = p.buf[2 * idx], b = p.buf[2 * idx + 1];
        if ((a & (a >> 1) & 0x55555555u) | (b & (b >> 1) & 0x55555555u)) atomicOr(p.bad, 1);
        if (p.mode == 1) slab_row(p.dir, p.colour, p.row0 + row, vecs)[v] = (uint64_t)a | ((uint64_t)b << 32);
        return;
    }
    uint64_t *lat = slab_row(p.dir, p.colour, p.row0 + row, p.L / 32) + 2 * v;
    if (p.mode == 2) {
        const uint64_t w0 = lat[0], w1 = lat[1];
        if (p.bc) {
            p.buf[2 * idx] = nibbles_to_pairs16(w0);
            p.buf[2 * idx + 1] = nibbles_to_pairs16(w1);
        } else {
            p.buf[idx] = nibbles_to_bits16(w0) | (nibbles_to_bits16(w1) << 16);
        }
        return;
    }
    uint64_t w0, w1;
    if (p.bc) {
        const uint32_t a = p.buf[2 * idx], b = p.buf[2 * idx + 1];
        if ((a & (a >> 1) & 0x55555555u) | (b & (b >> 1) & 0x55555555u)) atomicOr(p.bad, 1);      // a pair equal to 3
        w0 = pairs16_to_nibbles(a); w1 = pairs16_to_nibbles(b);
    } else {
        const uint32_t a = p.buf[idx];
        w0 = bits16_to_nibbles(a); w1 = bits16_to_nibbles(a >> 16);
    }
    if (p.mode == 1) { lat[0] = w0; lat[1] = w1; }
}

// mode 0 synchronises and returns cudaErrorInvalidValue on a bad Blume-Capel code; modes 1, 2 are asynchronous
cudaError_t launch_bits(ising_sim *h, int colour, int64_t row0, int64_t nrows, uint32_t *dev_buf, int mode, int *dev_bad)
{
    BitsParams p;
    p.dir = slab_directory(h);
    p.L = h->L; p.row0 = row0; p.nrows = nrows; p.colour = colour; p.bc = is_blume_capel(h->model) ? 1 : 0;
    p.mode = mode; p.buf = dev_buf; p.bad = dev_bad;
    p.two_bit = h->model == ISING_MODEL_BLUME_CAPEL_2BIT ? 1 : 0;
    cudaError_t e;
    if (mode == 0) {
        e = cudaMemsetAsync(dev_bad, 0, sizeof(int), h->stream);
        if (e != cudaSuccess) return e;
    }
    const int64_t n = nrows * (h->L / 64);
    bits_kernel<<<(unsigned)((n + 255) / 256), 256, 0, h->stream>>>(p);
    h->launches++;
    e = cudaGetLastError();
    if (e != cudaSuccess || mode != 0) return e;
    int bad = 0;
    e = cudaMemcpyAsync(&bad, dev_bad, sizeof(int), cudaMemcpyDeviceToHost, h->stream);
    if (e != cudaSuccess) return e;
    e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return e;
    return bad ? cudaErrorInvalidValue : cudaSuccess;
}
