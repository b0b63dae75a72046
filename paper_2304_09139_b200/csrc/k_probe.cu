// k_probe.cu -- FP64-pipe issue-rate probe: the measured denominator of the "alu" roofline
// (no FP64 entry exists in MEASURED_PEAKS.json, so the library measures one).
// Every thread runs 8 independent dependent-DFMA (or DADD) chains, or every warp 8 independent
// chains of the FP64 matrix instruction (mma.sync m8n8k4, SASS DMMA.8x8x4 = 256 FMAs per warp =
// 8 per thread); the result is thread-level FP64 instructions (FMAs) per second over the whole GPU.
#include "../../include/shd.h"
#include <cuda_runtime.h>

namespace {

template <int KIND>
__global__ void __launch_bounds__(256) k_fp64_chain(double* out, int iters, double seed)
{
    double a0 = seed + threadIdx.x, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5,
           a6 = a0 + 6, a7 = a0 + 7;
    const double m = 0.99999, c = 1e-9;
    for (int i = 0; i < iters; i++) {
#pragma unroll
        for (int u = 0; u < 8; u++) {
            if (KIND == 0) {
                a0 = __fma_rn(a0, m, c); a1 = __fma_rn(a1, m, c); a2 = __fma_rn(a2, m, c); a3 = __fma_rn(a3, m, c);
                a4 = __fma_rn(a4, m, c); a5 = __fma_rn(a5, m, c); a6 = __fma_rn(a6, m, c); a7 = __fma_rn(a7, m, c);
            } else {
                a0 = __dadd_rn(a0, c); a1 = __dadd_rn(a1, c); a2 = __dadd_rn(a2, c); a3 = __dadd_rn(a3, c);
                a4 = __dadd_rn(a4, c); a5 = __dadd_rn(a5, c); a6 = __dadd_rn(a6, c); a7 = __dadd_rn(a7, c);
            }
        }
    }
    double s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    if (s == 123.456) out[0] = s;   // never true; keeps the chains alive
}

__global__ void __launch_bounds__(256) k_fp64_dmma(double* out, int iters, double seed)
{
    double c[8][2];
#pragma unroll
    for (int i = 0; i < 8; i++) { c[i][0] = seed + i; c[i][1] = seed - i; }
    const double a = 1e-3 * (threadIdx.x & 31), b = 1e-3;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 8; i++)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; i++) s += c[i][0] + c[i][1];
    if (s == 123.456) out[0] = s;
}

}  // namespace

extern "C" int shd_fp64_peak(int kind, double seconds, double* instr_per_s)
{
    if (!instr_per_s || (kind < 0 || kind > 2) || !(seconds > 0.0) || seconds > 10.0) return SHD_EINVAL;
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return SHD_ECUDA;
    double* d_out = nullptr;
    if (cudaMalloc((void**)&d_out, 8) != cudaSuccess) return SHD_ENOMEM;
    const int blocks = prop.multiProcessorCount * 8, threads = 256;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    int iters = 2000;
    double best = 0.0, spent = 0.0, work = 0.0;
    for (int rep = 0; rep < 64 && spent < seconds; rep++) {
        cudaEventRecord(e0, 0);
        if (kind == 0) k_fp64_chain<0><<<blocks, threads>>>(d_out, iters, 1.0);
        else if (kind == 1) k_fp64_chain<1><<<blocks, threads>>>(d_out, iters, 1.0);
        else k_fp64_dmma<<<blocks, threads>>>(d_out, iters, 1.0);   // 8 DMMAs = 64 FMAs per thread and iteration
        cudaEventRecord(e1, 0);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(d_out); return SHD_ECUDA; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        double rate = (double)blocks * threads * (double)iters * 64.0 / (ms * 1e-3);
        if (rep > 0 && rate > best) best = rate;
        if (rep > 0) { spent += ms * 1e-3; work += (double)blocks * threads * (double)iters * 64.0; }
        if (ms < 20.f) iters *= 2;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d_out);
    instr_per_s[0] = best;
    instr_per_s[1] = spent > 0.0 ? work / spent : 0.0;
    return SHD_OK;
}
