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

// ---- random-gather probe: what the part gives a gather-bound kernel (profiles/r2_probes.md) ---------------
// Every thread issues independent 4-B loads at hashed addresses of a large buffer, eight in flight.  With
// hint64 the loads carry .L2::64B: ncu shows 64 B of DRAM traffic per gather instead of 127 B, at the same
// rate (37 G gathers/s over 8 GiB on B200): the rate is bound by DRAM row activations, not by bytes.
template <bool HINT64>
__global__ void __launch_bounds__(1024) k_random_gather(const float *buf, unsigned long long mask, int per, float *out)
{
    const unsigned long long tid = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long h = (tid + 1) * 0x9E3779B97F4A7C15ull;
    float acc = 0.f;
    for (int it = 0; it < per; it += 8) {
        float v[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            h = h * 6364136223846793005ull + 1442695040888963407ull;
            const float *a = buf + ((h >> 20) & mask);
            if (HINT64)
                asm volatile("ld.global.nc.L2::64B.f32 %0, [%1];" : "=f"(v[q]) : "l"(a));
            else
                asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(v[q]) : "l"(a));
        }
#pragma unroll
        for (int q = 0; q < 8; ++q) acc += v[q];
    }
    if (acc == 123.456f) out[tid] = acc;
}

cudaError_t random_gather_probe(int64_t buffer_bytes, int hint64, double *gathers_per_s, cudaStream_t stream)
{
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    unsigned long long words = 1;
    while (words * 2 * 4 <= (unsigned long long)buffer_bytes) words *= 2;      // power of two: index by mask
    float *buf = nullptr, *out = nullptr;
    e = cudaMalloc((void **)&buf, words * 4);
    if (e != cudaSuccess) return e;
    // a buffer that fits the L2 (<= 64 MiB) is gathered from four times as long: the L2-resident rate is the
    // denominator of the dense gather schedule (bench.py `l2_gather_bound`)
    const int blocks = sms * 2, threads = 1024, per = buffer_bytes <= (64ll << 20) ? 1024 : 256;
    e = cudaMalloc((void **)&out, (size_t)blocks * threads * 4);
    if (e != cudaSuccess) { cudaFree(buf); return e; }
    cudaMemsetAsync(buf, 0, words * 4, stream);
    cudaEvent_t a, b;
    cudaEventCreate(&a);
    cudaEventCreate(&b);
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(a, stream);
        if (hint64)
            k_random_gather<true><<<blocks, threads, 0, stream>>>(buf, words - 1, per, out);
        else
            k_random_gather<false><<<blocks, threads, 0, stream>>>(buf, words - 1, per, out);
        cudaEventRecord(b, stream);
        e = cudaEventSynchronize(b);
        if (e != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, a, b);
        if (rep > 0 && ms > 0.f) best = fmax(best, (double)blocks * threads * per / (ms * 1e-3));
    }
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    cudaFree(buf);
    cudaFree(out);
    *gathers_per_s = best;
    return e;
}

}  // namespace dt
