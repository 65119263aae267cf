// peaks_kernels.cuh -- microbenchmarks behind the secondary rooflines quoted in DESIGN.md section 5:
// fp64 FMA / ADD issue rate, shared-memory load bandwidth (LDS.64) and 64-bit warp-shuffle rate of
// this device.  MEASURED_PEAKS.json carries only HBM and bf16-GEMM peaks; the sweep kernels are
// bounded by the fp64 pipe and the shared-memory / shuffle pipe as well, so those denominators
// are measured by the library itself (dd4dvar_measure_peaks, `python bench.py --peaks`).
#pragma once
#include <cuda_runtime.h>

__global__ void pk_dfma(double* out, int iters)
{
    double a0 = 1.0 + threadIdx.x * 1e-9, a1 = 1.1, a2 = 1.2, a3 = 1.3, a4 = 1.4, a5 = 1.5, a6 = 1.6, a7 = 1.7;
    const double b = 0.999999, c = 1e-9;
    for (int i = 0; i < iters; ++i) {
        a0 = fma(a0, b, c); a1 = fma(a1, b, c); a2 = fma(a2, b, c); a3 = fma(a3, b, c);
        a4 = fma(a4, b, c); a5 = fma(a5, b, c); a6 = fma(a6, b, c); a7 = fma(a7, b, c);
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
}
__global__ void pk_dadd(double* out, int iters)
{
    double a0 = 1.0 + threadIdx.x * 1e-9, a1 = 1.1, a2 = 1.2, a3 = 1.3, a4 = 1.4, a5 = 1.5, a6 = 1.6, a7 = 1.7;
    const double c = 1e-9;
    for (int i = 0; i < iters; ++i) { a0 += c; a1 += c; a2 += c; a3 += c; a4 += c; a5 += c; a6 += c; a7 += c; }
    out[blockIdx.x * blockDim.x + threadIdx.x] = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
}
__global__ void pk_lds64(double* out, int iters)
{
    __shared__ double sm[4096];
    for (int i = threadIdx.x; i < 4096; i += blockDim.x) sm[i] = i;
    __syncthreads();
    double acc = 0.0;
    int idx = threadIdx.x;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < 8; ++k) acc += sm[(idx + k * 512) & 4095];
        idx = (idx + 1) & 4095;
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc;
}
__global__ void pk_shfl64(double* out, int iters)
{
    double a0 = threadIdx.x, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3;
    for (int i = 0; i < iters; ++i) {
        a0 = __shfl_down_sync(0xffffffffu, a0, 1); a1 = __shfl_up_sync(0xffffffffu, a1, 1);
        a2 = __shfl_down_sync(0xffffffffu, a2, 1); a3 = __shfl_up_sync(0xffffffffu, a3, 1);
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = a0 + a1 + a2 + a3;
}

// out[0] fp64 FMA TFLOP/s, out[1] fp64 ADD Tinstr/s, out[2] LDS.64 bytes/s (all SMs), out[3] 64-bit shuffles/s
// (thread-level), out[4] SM count, out[5] SM clock (MHz, from the device properties' peak clock)
inline int measure_peaks(cudaStream_t st, double out[6])
{
    int dev = 0, nsm = 0, khz = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -4;
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev);
    double* buf = nullptr;
    const int nt = 512, bps = 2, grid = nsm * bps;
    if (cudaMalloc(&buf, sizeof(double) * grid * nt) != cudaSuccess) return -4;
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    float ms = 0.f;
    const int iters = 20000;
    auto timeit = [&](int which) {
        for (int rep = 0; rep < 2; ++rep) {          // first repetition = warm-up
            cudaEventRecord(e0, st);
            if (which == 0) pk_dfma<<<grid, nt, 0, st>>>(buf, iters);
            if (which == 1) pk_dadd<<<grid, nt, 0, st>>>(buf, iters);
            if (which == 2) pk_lds64<<<grid, nt, 0, st>>>(buf, iters / 4);
            if (which == 3) pk_shfl64<<<grid, nt, 0, st>>>(buf, iters);
            cudaEventRecord(e1, st); cudaEventSynchronize(e1);
            cudaEventElapsedTime(&ms, e0, e1);
        }
        return (double)ms * 1e-3;
    };
    const double threads = (double)grid * nt;
    out[0] = 2.0 * 8 * iters * threads / timeit(0) / 1e12;
    out[1] = 8.0 * iters * threads / timeit(1) / 1e12;
    out[2] = 8.0 * 8 * (iters / 4) * threads / timeit(2);
    out[3] = 4.0 * iters * threads / timeit(3);
    out[4] = nsm; out[5] = khz * 1e-3;
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(buf);
    return cudaGetLastError() == cudaSuccess ? 0 : -4;
}
