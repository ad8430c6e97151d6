// probe.cu -- roofline denominators measured on the box: a register-resident DFMA loop and a DMMA.8x8x4 loop over the whole chip.
#include "common.cuh"

namespace sww {

__global__ void __launch_bounds__(256) k_probe_dfma(double* out, int iters, double seed) {
    double a[16];
#pragma unroll
    for (int i = 0; i < 16; i++) a[i] = seed + i * 1e-3 + threadIdx.x * 1e-6;
    const double m = 1.0000001, c = 1e-9;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int r = 0; r < 4; r++)
#pragma unroll
            for (int i = 0; i < 16; i++) a[i] = fma(a[i], m, c);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 16; i++) s += a[i];
    if (s == 123.456) out[0] = s;
}

__global__ void __launch_bounds__(256) k_probe_dmma(double* out, int iters, double seed) {
    double c[16][2];
#pragma unroll
    for (int i = 0; i < 16; i++) c[i][0] = c[i][1] = seed * i;
    double a = 1.0 + 1e-9 * threadIdx.x, b = 1e-9 * (threadIdx.x & 7);
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int r = 0; r < 4; r++)
#pragma unroll
            for (int i = 0; i < 16; i++)
                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                             : "+d"(c[i][0]), "+d"(c[i][1])
                             : "d"(a), "d"(b));
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 16; i++) s += c[i][0] + c[i][1];
    if (s == 123.456) out[0] = s;
}

}  // namespace sww

extern "C" int sww_probe_fp64_peak(int which, double* flops_per_s) {
    using namespace sww;
    if (!flops_per_s || which < 0 || which > 1) return SWW_EINVAL;
    int dev = 0, sms = 0;
    SWW_CUDA(cudaGetDevice(&dev));
    SWW_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    double* out = nullptr;
    SWW_CUDA(cudaMalloc(&out, 8));
    cudaEvent_t e0, e1;
    SWW_CUDA(cudaEventCreate(&e0));
    SWW_CUDA(cudaEventCreate(&e1));
    const int iters = 4096, blocks = sms * 8, threads = 256;
    double best = 0.0;
    for (int rep = 0; rep < 5; rep++) {
        SWW_CUDA(cudaEventRecord(e0));
        if (which == 0)
            k_probe_dfma<<<blocks, threads>>>(out, iters, 0.5);
        else
            k_probe_dmma<<<blocks, threads>>>(out, iters, 0.5);
        SWW_LAUNCHED();
        SWW_CUDA(cudaEventRecord(e1));
        SWW_CUDA(cudaEventSynchronize(e1));
        float ms = 0;
        SWW_CUDA(cudaEventElapsedTime(&ms, e0, e1));
        double flops;
        if (which == 0)
            flops = 2.0 * 64.0 * iters * (double)blocks * threads;  // 64 DFMA per thread per iteration
        else
            flops = 2.0 * 256.0 * 64.0 * iters * (double)blocks * (threads / 32);  // 64 DMMA (8x8x4 = 256 FMA) per warp per iteration
        double f = flops / (ms * 1e-3);
        if (rep > 0 && f > best) best = f;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    *flops_per_s = best;
    return SWW_OK;
}
