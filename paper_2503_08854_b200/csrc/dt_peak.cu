// dt_peak.cu -- FP64 FMA issue-rate probe: the "alu" roofline denominator of kernel 1
// (MEASURED_PEAKS.json carries no FP64 figure).  Eight independent register-resident DFMA chains
// per thread, enough CTAs to fill every SM; best of five launches.
#include "dt_common.cuh"

namespace dt {

__global__ void __launch_bounds__(256) k_dfma(double *out, int iters, double b, double c)
{
    double a0 = threadIdx.x * 1e-3, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5,
           a6 = a0 + 6, a7 = a0 + 7;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            a0 = fma(a0, b, c); a1 = fma(a1, b, c); a2 = fma(a2, b, c); a3 = fma(a3, b, c);
            a4 = fma(a4, b, c); a5 = fma(a5, b, c); a6 = fma(a6, b, c); a7 = fma(a7, b, c);
        }
    }
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
}

cudaError_t fp64_peak_device(double *tflops, cudaStream_t stream)
{
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    const int blocks = sms * 8, threads = 256, iters = 2048;
    double *out = nullptr;
    e = cudaMalloc((void **)&out, (size_t)blocks * threads * sizeof(double));
    if (e != cudaSuccess) return e;
    cudaEvent_t a, b;
    cudaEventCreate(&a);
    cudaEventCreate(&b);
    double best = 0.0;
    for (int rep = 0; rep < 6; ++rep) {
        cudaEventRecord(a, stream);
        k_dfma<<<blocks, threads, 0, stream>>>(out, iters, 0.999999, 1e-9);
        cudaEventRecord(b, stream);
        e = cudaEventSynchronize(b);
        if (e != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, a, b);
        const double flops = 2.0 * 64.0 * (double)iters * (double)blocks * (double)threads;
        if (rep > 0 && ms > 0.f) best = fmax(best, flops / (ms * 1e-3) * 1e-12);
    }
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    cudaFree(out);
    *tflops = best;
    return e;
}

}  // namespace dt
