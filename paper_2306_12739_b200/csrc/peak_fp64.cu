// dns_debug_fp64_peak (include/dns_debug.h): sustained fp64 throughput of the current device, measured the way
// MEASURED_PEAKS.json measures bf16: a register-resident kernel with no memory traffic, timed with CUDA
// events, repeated back to back for a stated duration.  kind 0: independent DFMA chains; kind 1: independent chains of
// mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4, the only fp64 tensor shape sm_100a executes natively; tcgen05 has no f64 kind).
// The result is the denominator of every fp64 roofline fraction bench.py prints.
#include <cstdint>

#include "dns_internal.h"

namespace {

constexpr int CHAINS = 8, ITERS = 4096;

__global__ void __launch_bounds__(256) k_peak_dfma(double* out, double a, double b) {
    double x[CHAINS];
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) x[c] = (double)(threadIdx.x + c);
#pragma unroll 1
    for (int it = 0; it < ITERS; ++it) {
#pragma unroll
        for (int c = 0; c < CHAINS; ++c) x[c] = fma(x[c], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) s += x[c];
    if (s == 12345.678) out[0] = s;                       // never true: keeps the chains alive
}

__global__ void __launch_bounds__(256) k_peak_dmma(double* out, double a, double b) {
    double acc[CHAINS][2];
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) acc[c][0] = acc[c][1] = (double)(threadIdx.x + c);
#pragma unroll 1
    for (int it = 0; it < ITERS; ++it) {
#pragma unroll
        for (int c = 0; c < CHAINS; ++c)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(acc[c][0]), "+d"(acc[c][1])
                         : "d"(a), "d"(b));
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) s += acc[c][0] + acc[c][1];
    if (s == 12345.678) out[0] = s;
}

// kind 2: every thread interleaves CHAINS independent DFMA chains with MIXM independent DMMA chains.  If the two instruction
// kinds had pipes of their own the sum of their rates would exceed either peak; on B200 it does not.
constexpr int MIXM = 2;
__global__ void __launch_bounds__(256) k_peak_mix(double* out, double a, double b) {
    double x[CHAINS];
    double acc[MIXM][2];
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) x[c] = (double)(threadIdx.x + c);
#pragma unroll
    for (int c = 0; c < MIXM; ++c) acc[c][0] = acc[c][1] = (double)(threadIdx.x + c);
#pragma unroll 1
    for (int it = 0; it < ITERS; ++it) {
#pragma unroll
        for (int c = 0; c < CHAINS; ++c) {
            x[c] = fma(x[c], a, b);
            if (c < MIXM)
                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                             : "+d"(acc[c][0]), "+d"(acc[c][1])
                             : "d"(a), "d"(b));
        }
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) s += x[c];
#pragma unroll
    for (int c = 0; c < MIXM; ++c) s += acc[c][0] + acc[c][1];
    if (s == 12345.678) out[0] = s;
}

}  // namespace

extern "C" int dns_debug_fp64_peak(int kind, double seconds, double* tflops) {
    if (!tflops || kind < 0 || kind > 2 || !(seconds > 0.0) || seconds > 30.0) return DNS_EINVAL;
    int dev = 0, nsm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        cudaGetLastError();
        return DNS_ECUDA;
    }
    double* out = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (cudaMalloc((void**)&out, 64) != cudaSuccess || cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) {
        cudaGetLastError();
        if (out) cudaFree(out);
        return DNS_ECUDA;
    }
    const int grid = nsm * 8, block = 256;
    // fused multiply-adds per launch: DFMA = 1 per thread and instruction; DMMA m8n8k4 = 8*8*4 = 256 per warp and instruction
    const double fma_dfma = (double)grid * block * CHAINS * ITERS, fma_dmma = (double)grid * (block / 32) * ITERS * 256.0;
    const double fma_per_launch = kind == 0 ? fma_dfma : (kind == 1 ? fma_dmma * CHAINS : fma_dfma + fma_dmma * MIXM);
    auto launch = [&]() {
        if (kind == 0) k_peak_dfma<<<grid, block>>>(out, 0.999999, 1e-9);
        else if (kind == 1) k_peak_dmma<<<grid, block>>>(out, 0.999999, 1e-9);
        else k_peak_mix<<<grid, block>>>(out, 0.999999, 1e-9);
    };
    for (int w = 0; w < 3; ++w) launch();
    cudaDeviceSynchronize();
    double total_ms = 0.0, total_fma = 0.0;
    while (total_ms < seconds * 1e3) {
        cudaEventRecord(e0);
        for (int r = 0; r < 10; ++r) launch();
        cudaEventRecord(e1);
        if (cudaEventSynchronize(e1) != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        total_ms += ms;
        total_fma += 10.0 * fma_per_launch;
        if (ms <= 0.f) break;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    if (cudaGetLastError() != cudaSuccess || total_ms <= 0.0) return DNS_ECUDA;
    *tflops = 2.0 * total_fma / (total_ms * 1e-3) * 1e-12;
    return DNS_OK;
}
