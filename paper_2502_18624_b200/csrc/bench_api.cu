// Measurement and debug entry points (include/ising_bench.h): not part of a simulation.
#include <curand_kernel.h>

#include "ising_internal.cuh"
#include "ising_bench.h"

// ----------------------------------------------------- measurement helpers ---
extern "C" int ising_bench_philox_only(ising_t *h, int n)
{
    DeviceGuard dev_guard(h);
    if (!h || n < 0 || h->model == ISING_MODEL_ISING_LUT || h->slabs.size() != 1) return set_error(ISING_EINVAL, "ising_bench_philox_only: bad argument (4-bit and 2-bit models, unsharded lattice)");
    for (int i = 0; i < n; ++i) {
        cudaError_t e = launch_philox_only(h, (uint32_t)i);
        if (e != cudaSuccess) return cuda_fail(e, "philox-only kernel");
    }
    return ISING_OK;
}

extern "C" int ising_bench_copy(ising_t *h, int n)
{
    DeviceGuard dev_guard(h);
    if (!h || n < 0 || h->model == ISING_MODEL_ISING_LUT || h->slabs.size() != 1) return set_error(ISING_EINVAL, "ising_bench_copy: bad argument (4-bit and 2-bit models, unsharded lattice)");
    for (int i = 0; i < n; ++i) {
        cudaError_t e = launch_copy(h);
        if (e != cudaSuccess) return cuda_fail(e, "copy kernel");
    }
    return ISING_OK;
}

// ------------------------------------------------------------ debug Philox ---
__global__ void debug_philox_kernel(int64_t count, const uint32_t *ctr, const uint32_t *key, uint32_t *out, int with_curand)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    uint4 c = make_uint4(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3]);
    uint4 r;
    if (with_curand) {
        r = curand_Philox4x32_10(c, make_uint2(key[2 * i], key[2 * i + 1]));
    } else {
        RoundKeys rk;
        uint32_t k0 = key[2 * i], k1 = key[2 * i + 1];
        for (int j = 0; j < 10; ++j) { rk.k0[j] = k0; rk.k1[j] = k1; k0 += PHILOX_W0; k1 += PHILOX_W1; }
        if (with_curand == 0 && (i & 1)) {
            // odd entries go through the specialised path the update kernel uses
            PhiloxRow pr = philox_row(c.y, c.z, c.w, rk);
            r = philox_site4(c.x, pr, rk);
        } else {
            r = philox4x32_10(c, rk);
        }
    }
    out[4 * i] = r.x; out[4 * i + 1] = r.y; out[4 * i + 2] = r.z; out[4 * i + 3] = r.w;
}

cudaError_t launch_debug_philox(int64_t count, const uint32_t *d_ctr, const uint32_t *d_key, uint32_t *d_out,
                                int with_curand, cudaStream_t s)
{
    debug_philox_kernel<<<(unsigned)((count + 127) / 128), 128, 0, s>>>(count, d_ctr, d_key, d_out, with_curand);
    return cudaGetLastError();
}

extern "C" int ising_debug_philox(int64_t count, const uint32_t *ctr, const uint32_t *key, uint32_t *out, int with_curand)
{
    if (count < 1 || !ctr || !key || !out) return set_error(ISING_EINVAL, "ising_debug_philox: bad argument");
    uint32_t *d = nullptr;
    CUDA_TRY(cudaMalloc((void **)&d, (size_t)count * 10 * sizeof(uint32_t)));
    uint32_t *d_ctr = d, *d_key = d + 4 * count, *d_out = d + 6 * count;
    cudaError_t e = cudaMemcpy(d_ctr, ctr, (size_t)count * 16, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(d_key, key, (size_t)count * 8, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = launch_debug_philox(count, d_ctr, d_key, d_out, with_curand, 0);
    if (e == cudaSuccess) e = cudaMemcpy(out, d_out, (size_t)count * 16, cudaMemcpyDeviceToHost);
    cudaFree(d);
    if (e != cudaSuccess) return cuda_fail(e, "ising_debug_philox");
    return ISING_OK;
}
