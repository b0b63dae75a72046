// pipe.cuh -- device helpers shared by the rho and gradient kernels: mbarrier + TMA 1-D bulk copies
// (cp.async.bulk, SASS UBLKCP), the FP64 matrix instruction (mma.sync m8n8k4, SASS DMMA.8x8x4) and
// the limb-level product-accumulate built from it (shd_internal.h).
#pragma once
#include "dd.cuh"
#include <cstdint>

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    } while (!ok);
}
__device__ __forceinline__ void tma_load_1d(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

// C(8x8) += A(8x4) B(4x8) in FP64.  Fragments (lane = 4 g + t): a = A[g][t], b = B[t][g],
// c0 = C[g][2t], c1 = C[g][2t+1].
struct Frag2 { double c0, c1; };
__device__ __forceinline__ void dmma(Frag2& c, double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c.c0), "+d"(c.c1) : "d"(a), "d"(b));
}

// one limb of one complex operand fragment, loaded / used in program order (volatile): the rho and
// gradient kernels write their LDS -> DMMA software pipeline as straight-line code
struct F2 { double r, i; };
__device__ __forceinline__ F2 lds2(uint32_t addr) {
    F2 f;
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(f.r), "=d"(f.i) : "r"(addr));
    return f;
}
__device__ __forceinline__ F2 add2(F2 a, F2 b) { return F2{__dadd_rn(a.r, b.r), __dadd_rn(a.i, b.i)}; }
__device__ __forceinline__ void dmma_v(Frag2& c, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c.c0), "+d"(c.c1) : "d"(a), "d"(b));
}

// one complex operand fragment: limbs 0..2 of (re, im) plus x12 = x1 + x2
struct LimbFrag { double r0, i0, r1, i1, r2, i2, r12, i12; };
// three LDS.128 at plane stride `ps` bytes (shared-memory byte address)
__device__ __forceinline__ LimbFrag lds_frag(uint32_t addr, uint32_t ps) {
    LimbFrag f;
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(f.r0), "=d"(f.i0) : "r"(addr));
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(f.r1), "=d"(f.i1) : "r"(addr + ps));
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(f.r2), "=d"(f.i2) : "r"(addr + 2 * ps));
    f.r12 = __dadd_rn(f.r1, f.r2);
    f.i12 = __dadd_rn(f.i1, f.i2);
    return f;
}

// limb accumulators of one 8x8 block of one real bilinear sum
struct Acc3 { Frag2 l0, l1, l2; };
__device__ __forceinline__ void acc3_zero(Acc3& a) {
    a.l0 = Frag2{0.0, 0.0}; a.l1 = Frag2{0.0, 0.0}; a.l2 = Frag2{0.0, 0.0};
}
// fold an exact burst into a (hi, lo) running sum
__device__ __forceinline__ void fold_burst(double l0, double l1, double l2, double2& m) {
    dd s = two_sum(l0, l1);
    double e = __dadd_rn(s.l, l2);
    dd t = two_sum(m.x, s.h);
    m.x = t.h;
    m.y = __dadd_rn(m.y, __dadd_rn(t.l, e));
}
