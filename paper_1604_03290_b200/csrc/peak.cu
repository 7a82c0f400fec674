// Device peak probes for the roofline denominators that MEASURED_PEAKS.json does not hold
// (DESIGN.md "Measurement"): dependency-free FP64 FMA throughput and a streaming FP64 copy.
#include "sph_internal.cuh"

#define PK_CHAINS 8
#define PK_ITERS 4096

__global__ void __launch_bounds__(256) k_dfma_peak(double *out, double a, double b) {
    double acc[PK_CHAINS];
#pragma unroll
    for (int k = 0; k < PK_CHAINS; ++k) acc[k] = (double)(threadIdx.x + k);
    for (int it = 0; it < PK_ITERS; ++it) {
#pragma unroll
        for (int k = 0; k < PK_CHAINS; ++k) acc[k] = fma(acc[k], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < PK_CHAINS; ++k) s += acc[k];
    if (s == 12345.678) out[blockIdx.x * blockDim.x + threadIdx.x] = s;   // never true: keeps the chains alive
}

__global__ void __launch_bounds__(256) k_copy_bw(const double2 *__restrict__ src, double2 *__restrict__ dst, size_t n2) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n2; i += (size_t)gridDim.x * blockDim.x) dst[i] = src[i];
}

extern "C" {

int sph_measure_fp64_peak(void *cuda_stream, double *tflops) {
    if (!tflops) return SPH_ERR_ARG;
    int ndev = 0, sms = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return SPH_ERR_CUDA; }
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int blocks = sms * 16;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    double best = 0.0;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(e0, st);
        k_dfma_peak<<<blocks, 256, 0, st>>>(nullptr, 1.0000001, 1e-9);
        cudaEventRecord(e1, st);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double flop = 2.0 * PK_CHAINS * PK_ITERS * 256.0 * blocks;
        if (rep > 0 && ms > 0.f) best = fmax(best, flop / (ms * 1e-3) * 1e-12);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    *tflops = best;
    return cudaGetLastError() == cudaSuccess ? SPH_OK : SPH_ERR_CUDA;
}

int sph_measure_copy_bw(void *cuda_stream, const double *src, double *dst, size_t bytes, double *gbs) {
    if (!src || !dst || !gbs || bytes < 16 || (((uintptr_t)src | (uintptr_t)dst) & 15)) return SPH_ERR_ARG;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return SPH_ERR_CUDA; }
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    double best = 0.0;
    for (int rep = 0; rep < 6; ++rep) {
        cudaEventRecord(e0, st);
        k_copy_bw<<<sms * 16, 256, 0, st>>>((const double2 *)src, (double2 *)dst, bytes / 16);
        cudaEventRecord(e1, st);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms > 0.f) best = fmax(best, 2.0 * (double)bytes / (ms * 1e-3) * 1e-9);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    *gbs = best;
    return cudaGetLastError() == cudaSuccess ? SPH_OK : SPH_ERR_CUDA;
}

}  // extern "C"
