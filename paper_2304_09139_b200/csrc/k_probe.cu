// k_probe.cu -- FP64-pipe issue-rate probe: the measured denominator of the "alu" roofline
// (no FP64 entry exists in MEASURED_PEAKS.json, so the library measures one).
// Every thread runs 8 independent dependent-DFMA (or DADD) chains, or every warp 8 independent
// chains of the FP64 matrix instruction (mma.sync m8n8k4, SASS DMMA.8x8x4 = 256 FMAs per warp =
// 8 per thread); the result is thread-level FP64 instructions (FMAs) per second over the whole GPU.
#include "../../include/shd_bench.h"
#include <cuda_runtime.h>
#include <cstdint>
#include <vector>

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

// ---------------------------------------------------------------------------------------------------
// INT8 tensor-core probe (exact digit-sliced contraction on tcgen05.mma.kind::i8).
// (1) exactness: D(128 x 64, s32) = A(128 x 128, s8) B(64 x 128, s8)^T through UTCIMMA with the operands
//     in shared memory (no swizzle, K-major core matrices), accumulator in TMEM, read back with
//     tcgen05.ld and compared with the integer product on the host;
// (2) rate: one CTA per SM issues M=128, N=256, K=32 instructions back to back from one thread.
namespace {

__device__ __forceinline__ uint32_t p_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
// shared-memory matrix descriptor: K-major, SWIZZLE_NONE; core matrix = 8 rows x 16 bytes (128 B contiguous),
// K-adjacent core matrices 128 B apart (LBO), 8-row groups 256 B apart (SBO); version 1 (sm_100)
__device__ __forceinline__ uint64_t p_desc(uint32_t addr) {
    return (uint64_t)((addr >> 4) & 0x3FFF) | ((uint64_t)(128 >> 4) << 16) | ((uint64_t)(256 >> 4) << 32) | ((uint64_t)1 << 46);
}
// instruction descriptor of kind::i8: D = s32, A = B = s8, both K-major, N >> 3 at bit 17, M >> 4 at bit 24
__device__ __forceinline__ uint32_t p_idesc(int m, int n) {
    return (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(m >> 4) << 24);
}
__device__ __forceinline__ void p_mma_i8(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
    uint32_t z = 0;
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, {%5, %5, %5, %5}, p;\n\t}"
                 ::"r"(tmem_d), "l"(da), "l"(db), "r"(idesc), "r"(accumulate), "r"(z) : "memory");
}
__device__ __forceinline__ void p_wait(uint32_t bar) {
    uint32_t ok = 0;
    while (!ok)
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(bar) : "memory");
}

// MODE 0: exactness (KB = 4 K-blocks, N = 64, result to D); MODE 1: rate (iters x 4 instructions, N = 256)
template <int MODE>
__global__ void __launch_bounds__(128) k_i8_probe(const signed char* A, const signed char* B, int* D, int iters)
{
    constexpr int NN = MODE == 0 ? 64 : 256, KB = MODE == 0 ? 4 : 2, COLS = MODE == 0 ? 64 : 512;
    __shared__ __align__(1024) signed char sA[KB][128 * 32];
    __shared__ __align__(1024) signed char sB[KB][NN * 32];
    __shared__ __align__(8) unsigned long long bar;
    __shared__ uint32_t tmem_base;
    const int tid = threadIdx.x, warp = tid >> 5;
    if (MODE == 0) {
        const int K = 32 * KB;
        for (int i = tid; i < 128 * K; i += 128) {
            int r = i / K, kk = i % K;
            sA[kk / 32][(r / 8) * 256 + ((kk % 32) / 16) * 128 + (r % 8) * 16 + kk % 16] = A[i];
        }
        for (int i = tid; i < NN * K; i += 128) {
            int r = i / K, kk = i % K;
            sB[kk / 32][(r / 8) * 256 + ((kk % 32) / 16) * 128 + (r % 8) * 16 + kk % 16] = B[i];
        }
    } else {
        for (int i = tid; i < KB * 128 * 32; i += 128) (&sA[0][0])[i] = (signed char)(i % 7 - 3);
        for (int i = tid; i < KB * NN * 32; i += 128) (&sB[0][0])[i] = (signed char)(i % 5 - 2);
    }
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(p_smem_u32(&bar)));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(p_smem_u32(&tmem_base)), "n"(COLS));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // generic-proxy smem writes -> UMMA reads
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    const uint32_t tb = tmem_base;
    if (tid == 0) {
        const uint32_t idesc = p_idesc(128, NN);
        for (int it = 0; it < (MODE == 0 ? 1 : iters); it++)
#pragma unroll
            for (int kb = 0; kb < (MODE == 0 ? KB : 4); kb++)
                p_mma_i8(tb + (MODE == 1 && (it & 1) ? (uint32_t)NN : 0u), p_desc(p_smem_u32(&sA[kb % KB][0])),
                         p_desc(p_smem_u32(&sB[kb % KB][0])), idesc, (it | kb) ? 1u : 0u);
        asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(p_smem_u32(&bar)) : "memory");
    }
    p_wait(p_smem_u32(&bar));
    asm volatile("tcgen05.fence::after_thread_sync;");
    for (int c0 = 0; c0 < (MODE == 0 ? NN : 8); c0 += 8) {
        uint32_t v[8];
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                     : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
                     : "r"(tb + ((uint32_t)(warp * 32) << 16) + c0));
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
        if (MODE == 0)
            for (int i = 0; i < 8; i++) D[tid * NN + c0 + i] = (int)v[i];
        else if (v[0] == 0x12345678u) D[0] = (int)v[1];
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tb), "n"(COLS));
}

}  // namespace

// ---------------------------------------------------------------------------------------------------
// FP64 under a tcgen05.mma.kind::i8 stream (the measurement behind k_grad8's integer epilogue): one CTA
// per SM; warp 16 issues M=128 N=256 K=32 instructions back to back, warps 0..15 run dependent chains (4 per thread)
// of DADD (KIND 0) or IMAD (KIND 1).  The chains are sized to outlast the MMA stream, so the progress they make WHILE
// it runs follows from the two durations.  Also the SM clock under that load (clock64 against globaltimer).
namespace {
template <int KIND>
__global__ void __launch_bounds__(544) k_mix_probe(int mma_iters, int alu_iters, long long* out, double* sink)
{
    __shared__ __align__(1024) signed char sA[2][128 * 32];
    __shared__ __align__(1024) signed char sB[2][256 * 32];
    __shared__ __align__(8) unsigned long long bar;
    __shared__ uint32_t tmem_base;
    const int tid = threadIdx.x, warp = tid >> 5;
    for (int i = tid; i < 2 * 128 * 32; i += blockDim.x) (&sA[0][0])[i] = (signed char)(i % 7 - 3);
    for (int i = tid; i < 2 * 256 * 32; i += blockDim.x) (&sB[0][0])[i] = (signed char)(i % 5 - 2);
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(p_smem_u32(&bar)));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(p_smem_u32(&tmem_base)));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    const uint32_t tb = tmem_base;
    if (warp == 16) {
        if (tid == 512) {
            unsigned long long g0, g1;
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g0));
            const long long t0 = clock64();
            const uint32_t idesc = p_idesc(128, 256);
            for (int it = 0; it < mma_iters; it++)
#pragma unroll
                for (int kb = 0; kb < 4; kb++)
                    p_mma_i8(tb + ((it & 1) ? 256u : 0u), p_desc(p_smem_u32(&sA[kb & 1][0])), p_desc(p_smem_u32(&sB[kb & 1][0])),
                             idesc, (it | kb) ? 1u : 0u);
            asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(p_smem_u32(&bar)) : "memory");
            p_wait(p_smem_u32(&bar));
            const long long t1 = clock64();
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
            if (blockIdx.x == 0) { out[1] = t1 - t0; out[2] = (long long)(g1 - g0); }
        }
    } else {
        const long long t0 = clock64();
        if (KIND == 0) {
            double a0 = tid, a1 = tid + 1, a2 = tid + 2, a3 = tid + 3;
            for (int it = 0; it < alu_iters; it++)
#pragma unroll
                for (int u = 0; u < 16; u++) {
                    a0 = __dadd_rn(a0, 1e-9); a1 = __dadd_rn(a1, 1e-9); a2 = __dadd_rn(a2, 1e-9); a3 = __dadd_rn(a3, 1e-9);
                }
            if (a0 + a1 + a2 + a3 == 1.2345) sink[0] = a0;
        } else {
            int a0 = tid, a1 = tid + 1, a2 = tid + 2, a3 = tid + 3;
            for (int it = 0; it < alu_iters; it++)
#pragma unroll
                for (int u = 0; u < 16; u++) { a0 = a0 * 3 + tid; a1 = a1 * 3 + tid; a2 = a2 * 3 + tid; a3 = a3 * 3 + tid; }
            if (a0 + a1 + a2 + a3 == 12345) sink[0] = a0;
        }
        if (tid == 0 && blockIdx.x == 0) out[0] = clock64() - t0;
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tb));
}
}  // namespace

// out[0]: cycles per DADD per warp, chains alone (16 warps per SM);  out[1]: the same averaged over the time a back-to-back
// tcgen05.mma.kind::i8 stream runs on the SM (progress the chains make during the stream / their progress alone = out[0] / out[1]);
// out[2], out[3]: the same for IMAD chains;  out[4]: cycles per N = 256 instruction alone, out[5]: beside the DADD chains,
// out[6]: beside the IMAD chains;  out[7]: SM clock in MHz during the MMA stream (clock64 against globaltimer).
extern "C" int shd_mix_probe(double out[8])
{
    if (!out) return SHD_EINVAL;
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return SHD_ECUDA;
    long long* d = nullptr;
    double* sink = nullptr;
    if (cudaMalloc((void**)&d, 3 * sizeof(long long)) != cudaSuccess || cudaMalloc((void**)&sink, 8) != cudaSuccess) { cudaFree(d); return SHD_ENOMEM; }
    const int sms = prop.multiProcessorCount, mma_iters = 4000, alu_iters = 8000;
    const double per = 16.0 * 4.0;                  // chain instructions per thread and iteration
    long long h[3];
    auto run = [&](int kind, int mi, int ai) -> cudaError_t {
        cudaMemset(d, 0, 3 * sizeof(long long));
        for (int r = 0; r < 2; r++) {
            if (kind == 0) k_mix_probe<0><<<sms, 544>>>(mi, ai, d, sink); else k_mix_probe<1><<<sms, 544>>>(mi, ai, d, sink);
        }
        cudaError_t e = cudaMemcpy(h, d, sizeof(h), cudaMemcpyDeviceToHost);
        return e == cudaSuccess ? cudaGetLastError() : e;
    };
    cudaError_t e = cudaSuccess;
    for (int kind = 0; kind < 2 && e == cudaSuccess; kind++) {
        if ((e = run(kind, 0, alu_iters)) != cudaSuccess) break;
        const double alone = (double)h[0] / (alu_iters * per);
        if ((e = run(kind, mma_iters, alu_iters)) != cudaSuccess) break;
        // the chains ran h[0] cycles in all, h[1] of them beside the MMA stream and the rest alone at `alone` cycles per instruction
        const double done_alone = ((double)h[0] - (double)h[1]) / alone, done_beside = alu_iters * per - done_alone;
        out[2 * kind] = alone;
        out[2 * kind + 1] = done_beside > 0.0 ? (double)h[1] / done_beside : 1e30;
        out[5 + kind] = (double)h[1] / (mma_iters * 4.0);
        if (kind == 0) out[7] = (double)h[1] / (double)h[2] * 1e3;
    }
    if (e == cudaSuccess && (e = run(0, mma_iters, 1)) == cudaSuccess) out[4] = (double)h[1] / (mma_iters * 4.0);
    cudaFree(d); cudaFree(sink);
    return e == cudaSuccess ? SHD_OK : SHD_ECUDA;
}

extern "C" int shd_i8_probe(double* tops, long* mismatches)
{
    if (!tops || !mismatches) return SHD_EINVAL;
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return SHD_ECUDA;
    constexpr int M = 128, N = 64, K = 128;
    std::vector<signed char> hA(M * K), hB(N * K);
    unsigned s = 12345u;
    for (auto& x : hA) { s = s * 1664525u + 1013904223u; x = (signed char)((s >> 24) & 0xff); }
    for (auto& x : hB) { s = s * 1664525u + 1013904223u; x = (signed char)((s >> 24) & 0xff); }
    signed char *dA = nullptr, *dB = nullptr;
    int* dD = nullptr;
    if (cudaMalloc((void**)&dA, M * K) != cudaSuccess || cudaMalloc((void**)&dB, N * K) != cudaSuccess ||
        cudaMalloc((void**)&dD, M * N * sizeof(int)) != cudaSuccess) { cudaFree(dA); cudaFree(dB); cudaFree(dD); return SHD_ENOMEM; }
    cudaMemcpy(dA, hA.data(), M * K, cudaMemcpyHostToDevice);
    cudaMemcpy(dB, hB.data(), N * K, cudaMemcpyHostToDevice);
    cudaMemset(dD, 0xff, M * N * sizeof(int));
    k_i8_probe<0><<<1, 128>>>(dA, dB, dD, 1);
    std::vector<int> hD(M * N);
    cudaError_t e = cudaMemcpy(hD.data(), dD, M * N * sizeof(int), cudaMemcpyDeviceToHost);
    long bad = 0;
    for (int i = 0; i < M; i++)
        for (int j = 0; j < N; j++) {
            int ref = 0;
            for (int k = 0; k < K; k++) ref += (int)hA[i * K + k] * (int)hB[j * K + k];
            bad += ref != hD[i * N + j];
        }
    *mismatches = bad;
    const int iters = 20000;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    k_i8_probe<1><<<prop.multiProcessorCount, 128>>>(dA, dB, dD, iters);
    cudaEventRecord(e0, 0);
    k_i8_probe<1><<<prop.multiProcessorCount, 128>>>(dA, dB, dD, iters);
    cudaEventRecord(e1, 0);
    if (e == cudaSuccess) e = cudaEventSynchronize(e1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    *tops = 2.0 * (double)prop.multiProcessorCount * iters * 4.0 * 128.0 * 256.0 * 32.0 / (ms * 1e-3) / 1e12;
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(dA); cudaFree(dB); cudaFree(dD);
    return e == cudaSuccess ? SHD_OK : SHD_ECUDA;
}
