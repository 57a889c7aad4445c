// ising_correlation_noalloc: the full-source pair sums of ising_correlation (A9 of SURVEY.md Sec. 8(a);
// PAPER.md:65) for callers that may not allocate -- code under CUDA graph capture, tight serving loops,
// harnesses that forbid cudaMalloc.  ising_correlation keeps its scratch (bit planes, transposed planes,
// int64 accumulators) in buffers it cudaMallocs on first use; this variant runs the same kernels
// (planes_kernel, transpose_kernel, corr_full_kernel) on a file-scope device array of a fixed size, so it
// calls no cudaMalloc, cudaFree or allocating library routine -- and is limited to L <= ISING_NOALLOC_MAX_L.
//
// The array is shared by every call on a device and keeps the last call's contents: the accumulators are
// cleared at the start of each call, the planes are overwritten completely.  Two calls that overlap on the
// GPU (two handles on two streams, or two host threads) race on it; calls on one stream are ordered.
#include <string.h>

#include "ising_internal.cuh"

// scratch layout: [bit planes: up to 4 x L*L/8 bytes (Blume-Capel: sg, nz, sgT, nzT) | 2 x L/2 int64 accumulators]
static const size_t kNoallocPlaneBytes = 4 * ((size_t)ISING_NOALLOC_MAX_L * ISING_NOALLOC_MAX_L / 8);
static const size_t kNoallocAccBytes = 2 * ((size_t)ISING_NOALLOC_MAX_L / 2) * sizeof(long long);
static const size_t kNoallocBytes = kNoallocPlaneBytes + kNoallocAccBytes;      // 532480 bytes per GPU that loads the library

static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoallocBytes];

// In host code g_noalloc_scratch is a stand-in, not a device address: the address comes from
// cudaGetSymbolAddress, once per device, with that device current.
static const int kMaxDevices = 64;
static void *g_noalloc_addr[kMaxDevices];

static int noalloc_scratch_address(int device, unsigned char **out)
{
    if (device < 0 || device >= kMaxDevices) return set_error(ISING_EINVAL, "ising_correlation_noalloc: device index out of range");
    if (!g_noalloc_addr[device]) {
        void *p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_scratch);            // the caller has made `device` current
        if (e != cudaSuccess || !p) return cuda_fail(e, "cudaGetSymbolAddress(g_noalloc_scratch)");
        g_noalloc_addr[device] = p;
    }
    *out = (unsigned char *)g_noalloc_addr[device];
    return ISING_OK;
}

// Device code names the array directly: the accumulators must start at zero, whatever the last call left.
__global__ void noalloc_clear_kernel(int n_acc)
{
    long long *acc = reinterpret_cast<long long *>(g_noalloc_scratch + kNoallocPlaneBytes);
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_acc; i += gridDim.x * blockDim.x) acc[i] = 0;
}

extern "C" int ising_correlation_noalloc(ising_t *h, int64_t rmax, int64_t *sx, int64_t *sy)
{
    DeviceGuard dev_guard(h);
    if (!h || !sx || !sy) return set_error(ISING_EINVAL, "ising_correlation_noalloc: NULL argument");
    if (h->L > ISING_NOALLOC_MAX_L)
        return set_error(ISING_EINVAL, "ising_correlation_noalloc: L exceeds ISING_NOALLOC_MAX_L (1024), the size the static scratch "
                                       "array holds; use ising_correlation, which allocates its scratch");
    if (rmax < 1 || rmax > h->L / 2) return set_error(ISING_EINVAL, "ising_correlation_noalloc: rmax outside [1, L/2]");
    if (h->part && h->slabs[0].rows != h->L)
        return set_error(ISING_EINVAL, "ising_correlation_noalloc: needs the whole lattice, this handle holds one part of it");
    unsigned char *scratch = nullptr;
    int rc = noalloc_scratch_address(h->device, &scratch);
    if (rc) return rc;
    long long *d_sx = reinterpret_cast<long long *>(scratch + kNoallocPlaneBytes), *d_sy = d_sx + rmax;
    noalloc_clear_kernel<<<4, 256, 0, h->stream>>>((int)(2 * rmax));
    CUDA_TRY(cudaGetLastError());
    h->launches++;
    // the plane and correlation launchers take the plane buffer from the handle: point it at the static
    // scratch for the duration of the call (a handle is not thread-safe, so nobody else looks)
    struct PlanesSwap {
        ising_sim *h; uint64_t *saved;
        ~PlanesSwap() { h->planes = saved; }
    } swap{h, h->planes};
    h->planes = reinterpret_cast<uint64_t *>(scratch);
    cudaError_t e = launch_planes(h);
    if (e != cudaSuccess) return cuda_fail(e, "bit-plane kernels");
    e = launch_corr(h, 0, rmax, nullptr, d_sx, d_sy);                           // bit planes (XOR + POPC), r = 1..rmax
    if (e != cudaSuccess) return cuda_fail(e, "correlation kernel");
    CUDA_TRY(cudaMemcpyAsync(sx, d_sx, (size_t)rmax * sizeof(long long), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(cudaMemcpyAsync(sy, d_sy, (size_t)rmax * sizeof(long long), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    if (!is_blume_capel(h->model)) {            // Ising: the kernels count unequal pairs; pair sum = N - 2 count
        const int64_t n = h->L * h->L;
        for (int64_t i = 0; i < rmax; ++i) { sx[i] = n - 2 * sx[i]; sy[i] = n - 2 * sy[i]; }
    }
    return ISING_OK;
}
