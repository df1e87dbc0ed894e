// peak.cu -- FP64 roofline denominator probe (not on the projection path).
// MEASURED_PEAKS.json has no FP64 figure, so bench.py measures it with these two
// kernels: independent DFMA chains, and independent DMMA (mma.sync m8n8k4 f64) chains.
#include "kernels.h"

namespace hpsd {

__global__ void __launch_bounds__(256) dfma_probe_kernel(int iters, double *sink) {
    double a[8];
    const double x = 1.0 + 1e-9 * threadIdx.x, y = 1e-9 * blockIdx.x;
#pragma unroll
    for (int k = 0; k < 8; ++k) a[k] = k;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int k = 0; k < 8; ++k) a[k] = fma(a[k], x, y);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += a[k];
    if (s == 123.456) sink[0] = s;
}

__device__ __forceinline__ void dmma884(double &d0, double &d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

__global__ void __launch_bounds__(256) dmma_probe_kernel(int iters, double *sink) {
    double c[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) c[k] = 0.0;
    const double a = 1.0 + 1e-9 * threadIdx.x, b = 1e-9 * (blockIdx.x + 1);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
#pragma unroll
            for (int k = 0; k < 8; ++k) dmma884(c[2 * k], c[2 * k + 1], a, b);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 16; ++k) s += c[k];
    if (s == 123.456) sink[0] = s;
}

int launch_fp64_probe(int kind, int iters, double *flops_host, cudaStream_t st) {
    static double *sink = nullptr;
    if (!sink && cudaMalloc(&sink, 64) != cudaSuccess) return HPSD_ECUDA_;
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int ctas = sms * 8, threads = 256;
    if (kind == 0) {
        dfma_probe_kernel<<<ctas, threads, 0, st>>>(iters, sink);
        if (flops_host) *flops_host = (double)ctas * threads * (double)iters * 64.0 * 2.0;
    } else {
        dmma_probe_kernel<<<ctas, threads, 0, st>>>(iters, sink);
        if (flops_host) *flops_host = (double)ctas * (threads / 32) * (double)iters * 32.0 * 512.0;
    }
    HPSD_LAUNCH_CHECK();
    return 0;
}

}  // namespace hpsd
