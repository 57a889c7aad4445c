// Integer-pipe probe (measurement helper): dependent chains of one or two
// SASS instruction kinds, 8-way ILP per thread, 16 warps per SM sub-partition, timed with CUDA
// events.  Gives the issue rates (warp-instructions per sub-partition per clock) the ALU
// roofline of the update kernel is derived from.  Not part of a simulation.
#include "ising_internal.cuh"

#define PROBE_ILP 8
#define PROBE_ITERS 256
#define PROBE_REP 4

enum { P_WIDE = 0, P_LOP3, P_IMAD, P_WIDE_LOP3, P_WIDE_2LOP3, P_CARRY_IMADX, P_WIDE_IMAD, P_POPC_IADD, P_COUNT };

template <int OP>
__global__ void __launch_bounds__(256) probe_kernel(uint32_t *out, uint32_t seed, uint32_t M)
{
    uint32_t a[PROBE_ILP], b[PROBE_ILP];
#pragma unroll
    for (int i = 0; i < PROBE_ILP; ++i) {
        a[i] = seed + threadIdx.x * 17 + i;
        b[i] = (seed ^ (i * 0x9E3779B9u)) + threadIdx.x * 0x85EBCA6Bu;
    }
    for (int it = 0; it < PROBE_ITERS; ++it) {
#pragma unroll
        for (int rep = 0; rep < PROBE_REP; ++rep)
#pragma unroll
            for (int i = 0; i < PROBE_ILP; ++i) {
                if (OP == P_WIDE || OP == P_WIDE_LOP3 || OP == P_WIDE_2LOP3 || OP == P_WIDE_IMAD)
                    asm volatile("{.reg .b64 t; .reg .b32 lo; mul.wide.u32 t, %0, %1; mov.b64 {lo, %0}, t;}" : "+r"(a[i]) : "r"(M));
                if (OP == P_LOP3) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[i]) : "r"(b[i]), "r"(seed));
                if (OP == P_WIDE_LOP3 || OP == P_WIDE_2LOP3)
                    asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(b[i]) : "r"(seed), "r"(M));
                if (OP == P_WIDE_2LOP3) asm volatile("lop3.b32 %0, %0, %1, %2, 0x69;" : "+r"(b[i]) : "r"(seed), "r"(M));
                if (OP == P_IMAD) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(M), "r"(seed));
                if (OP == P_WIDE_IMAD) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(b[i]) : "r"(M), "r"(seed));
                if (OP == P_CARRY_IMADX)
                    asm volatile("add.cc.u32 %1, %1, %2; madc.lo.u32 %0, %0, 16, 0;" : "+r"(a[i]), "+r"(b[i]) : "r"(seed));
                if (OP == P_POPC_IADD) {
                    asm volatile("popc.b32 %0, %0;" : "+r"(a[i]));
                    asm volatile("add.u32 %0, %0, %1;" : "+r"(a[i]) : "r"(b[i]));
                }
            }
    }
    uint32_t s = 0;
#pragma unroll
    for (int i = 0; i < PROBE_ILP; ++i) s ^= a[i] ^ b[i];
    if (s == 0x12345u) out[threadIdx.x] = s;     // practically never taken
}

template <int OP>
static cudaError_t time_probe(uint32_t *sink, int instr_per_step, double sm_hz, int n_sm, double *rate)
{
    cudaEvent_t e0, e1;
    cudaError_t e = cudaEventCreate(&e0);
    if (e != cudaSuccess) return e;
    e = cudaEventCreate(&e1);
    if (e != cudaSuccess) { cudaEventDestroy(e0); return e; }
    const int grid = n_sm * 8 * 8;                       // 8 resident blocks of 8 warps = 16 warps per sub-partition, 8 waves
    probe_kernel<OP><<<grid, 256>>>(sink, 1u, 0xD2511F53u);
    cudaEventRecord(e0);
    probe_kernel<OP><<<grid, 256>>>(sink, 3u, 0xD2511F53u);
    cudaEventRecord(e1);
    e = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (e != cudaSuccess) return e;
    const double warp_instr = (double)grid * 8.0 * PROBE_ITERS * PROBE_REP * PROBE_ILP * instr_per_step;
    *rate = warp_instr / (ms * 1e-3) / (n_sm * 4.0) / sm_hz;
    return cudaGetLastError();
}

// rates[i] for the P_* probes above; sm_mhz = the clock the rates are normalised to
extern "C" int ising_bench_pipes(double sm_mhz, double *rates, int cap, int *count)
{
    if (!rates || !count) return set_error(ISING_EINVAL, "ising_bench_pipes: NULL argument");
    *count = P_COUNT;
    if (cap < P_COUNT) return set_error(ISING_EINVAL, "ising_bench_pipes: cap too small");
    int dev = 0, n_sm = 0, khz = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    CUDA_TRY(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    CUDA_TRY(cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev));
    const double hz = (sm_mhz > 0 ? sm_mhz * 1e6 : khz * 1e3);
    uint32_t *sink = nullptr;
    CUDA_TRY(cudaMalloc((void **)&sink, 4096));
    cudaError_t e = time_probe<P_WIDE>(sink, 1, hz, n_sm, &rates[P_WIDE]);
    if (e == cudaSuccess) e = time_probe<P_LOP3>(sink, 1, hz, n_sm, &rates[P_LOP3]);
    if (e == cudaSuccess) e = time_probe<P_IMAD>(sink, 1, hz, n_sm, &rates[P_IMAD]);
    if (e == cudaSuccess) e = time_probe<P_WIDE_LOP3>(sink, 2, hz, n_sm, &rates[P_WIDE_LOP3]);
    if (e == cudaSuccess) e = time_probe<P_WIDE_2LOP3>(sink, 3, hz, n_sm, &rates[P_WIDE_2LOP3]);
    if (e == cudaSuccess) e = time_probe<P_CARRY_IMADX>(sink, 2, hz, n_sm, &rates[P_CARRY_IMADX]);
    if (e == cudaSuccess) e = time_probe<P_WIDE_IMAD>(sink, 2, hz, n_sm, &rates[P_WIDE_IMAD]);
    if (e == cudaSuccess) e = time_probe<P_POPC_IADD>(sink, 2, hz, n_sm, &rates[P_POPC_IADD]);
    cudaFree(sink);
    if (e != cudaSuccess) return cuda_fail(e, "pipe probe");
    return ISING_OK;
}
