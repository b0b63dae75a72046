// k_grad.cu -- step a4: dPhi/dr_{j,a} = (4 pi / L) sum_k v_k n_a Im[ exp(-i k.r_j) rho(k) ]
// (Eq. 6, sign D:R2) as two contractions over q followed by one over p:
//   T_j[p]   = sum_{q,sigma} W(p,q,sigma) conj(B_j[q]^sigma)          = sum_q ( C1 br + C2 bi )
//   T''_j[p] = -i sum_{q,sigma} sigma q W conj(B^sigma)               = sum_q ( C2 (q br) - C1 (q bi) )
//   grad_a   = (4 pi/L) sum_p ( w_a(p) Im[conj(A_j[p]) T_j[p]] + [a = last axis] Re[conj(A_j[p]) T''_j[p]] )
// with C1 = W+ + W-, C2 = -i (W+ - W-), W = v rho (built by k_ctable), so both signs of the last
// axis share the same products: 24 DFMA per particle-wavevector pair.
// One CTA owns 32 particles and walks all p-blocks; per p-block it streams the q-chunks of the
// rho.v operand C (k_ctable output, shared by every CTA, L2 resident) and of the particles' own
// B-table into shared memory with TMA bulk copies (cp.async.bulk + mbarrier, 2-stage ring); each
// thread owns 2 particles x 2 p.  Exact limb bursts (64 q) are folded into double-double sums kept in
// shared memory; the p-contraction and the reduction over the 16 threads that share a particle
// run in double-double in a fixed order (deterministic, no atomics).
#include "dd.cuh"
#include "shd_internal.h"
#include <cstdint>

namespace {

constexpr int TJ = 16, TP = 16;
constexpr int GSLAB = SHD_QCH * 4096;          // 8 q x (8 planes x 32 x 16 B)
constexpr int GSTAGE = 2 * GSLAB;              // B slab + C slab
constexpr int MAIN_BYTES = 16 * 256 * 16;      // 16 dd accumulators per thread
constexpr int GSMEM = SHD_GRAD_STAGES * GSTAGE + MAIN_BYTES;

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE;\n"
        "bra WAIT_LOOP;\n"
        "DONE:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_1d(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

struct Half { double r0, i0, r1, i1, r2, i2, r12, i12; };   // one complex value, 4 limb pairs
__device__ __forceinline__ Half lds_half(uint32_t addr) {   // planes 512 B apart
    Half e;
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(e.r0), "=d"(e.i0) : "r"(addr));
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(e.r1), "=d"(e.i1) : "r"(addr + 512));
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(e.r2), "=d"(e.i2) : "r"(addr + 1024));
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(e.r12), "=d"(e.i12) : "r"(addr + 1536));
    return e;
}
struct Acc { double l0, l1, l2; };

__device__ __forceinline__ dd limbs_to_dd(double x0, double x1, double x2) {
    return fast_two_sum(__dadd_rn(x0, x1), x2);    // x0 + x1 is exact (46 bits)
}

__global__ void __launch_bounds__(TJ * TP, 1) k_grad(
    int d, long N, double L, long Npad, int npb, int Qpad, int Ppad, int qscale_log2,
    const int* __restrict__ qchunks, const int* __restrict__ wT,
    const double* __restrict__ A, const double* __restrict__ Bg, const double* __restrict__ C,
    const shd_scalars* __restrict__ scal, double* __restrict__ grad_hi, double* __restrict__ grad_lo,
    const int* __restrict__ skip)
{
    if (skip && *skip) return;
    extern __shared__ __align__(1024) unsigned char smem[];
    __shared__ __align__(8) unsigned long long bars[SHD_GRAD_STAGES];
    const int tid = threadIdx.x;
    const int tj = tid % TJ, tp = tid / TJ;
    const long jb = blockIdx.x;
    const uint32_t s0 = smem_u32(smem);
    double2* mainacc = reinterpret_cast<double2*>(smem + SHD_GRAD_STAGES * GSTAGE);   // [16][256]

    int total = 0;
    for (int pb = 0; pb < npb; pb++) total += qchunks[pb];

    if (tid == 0) {
        for (int s = 0; s < SHD_GRAD_STAGES; s++) mbar_init(smem_u32(&bars[s]), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int a = 0; a < 16; a++) mainacc[a * 256 + tid] = make_double2(0.0, 0.0);
    __syncthreads();

    // producer cursor (thread 0 only)
    int lpb = 0, lqc = 0, issued = 0;
    auto issue = [&](int stage) {
        uint32_t bar = smem_u32(&bars[stage]);
        mbar_expect_tx(bar, GSTAGE);
        const double* srcB = Bg + (((size_t)jb * Qpad + (size_t)lqc * SHD_QCH) * 8) * 64;
        const double* srcC = C + (((size_t)lpb * Qpad + (size_t)lqc * SHD_QCH) * 8) * 64;
        tma_load_1d(s0 + stage * GSTAGE, srcB, GSLAB, bar);
        tma_load_1d(s0 + stage * GSTAGE + GSLAB, srcC, GSLAB, bar);
        issued++;
        if (++lqc == qchunks[lpb]) { lqc = 0; lpb++; }
    };
    if (tid == 0)
        for (int s = 0; s < SHD_GRAD_STAGES && issued < total; s++) issue(s);

    Acc acc[2][2][4];
#pragma unroll
    for (int uj = 0; uj < 2; uj++)
#pragma unroll
        for (int up = 0; up < 2; up++)
#pragma unroll
            for (int x = 0; x < 4; x++) acc[uj][up][x] = Acc{0.0, 0.0, 0.0};
    dd g[2][3];
#pragma unroll
    for (int uj = 0; uj < 2; uj++)
#pragma unroll
        for (int a = 0; a < 3; a++) g[uj][a] = dd{0.0, 0.0};

    const uint32_t offB = (uint32_t)tj * 16;            // j_local = uj*16 + tj
    const uint32_t offC = GSLAB + (uint32_t)tp * 16;    // p_local = up*16 + tp
    const double qs = ldexp(1.0, qscale_log2);

    int c = 0;
    for (int pb = 0; pb < npb; pb++) {
        const int nqc = qchunks[pb];
        for (int qc = 0; qc < nqc; qc++, c++) {
            const int s = c % SHD_GRAD_STAGES;
            mbar_wait(smem_u32(&bars[s]), (uint32_t)((c / SHD_GRAD_STAGES) & 1));
            const uint32_t sb = s0 + s * GSTAGE;
#pragma unroll 1
            for (int qi = 0; qi < SHD_QCH; qi++) {
                Half c1[2], c2[2];
#pragma unroll
                for (int up = 0; up < 2; up++) {
                    c1[up] = lds_half(sb + offC + qi * 4096 + up * (TP * 16));
                    c2[up] = lds_half(sb + offC + qi * 4096 + 2048 + up * (TP * 16));
                }
#pragma unroll
                for (int uj = 0; uj < 2; uj++) {
                    // runs of 4 DFMAs sharing the B-side limb BL; SG = +1 / -1
#define RUN_B(BL, SG, lv, CC, LIMB, XR, XI)                                                          \
    _Pragma("unroll") for (int up = 0; up < 2; up++) {                                                \
        acc[uj][up][XR].lv = __fma_rn(SG BL, CC[up].r##LIMB, acc[uj][up][XR].lv);                     \
        acc[uj][up][XI].lv = __fma_rn(SG BL, CC[up].i##LIMB, acc[uj][up][XI].lv);                     \
    }
#define SIX_RUNS(BV, SG, CC, XR, XI)            \
    RUN_B(BV##0, SG, l0, CC, 0, XR, XI)         \
    RUN_B(BV##0, SG, l2, CC, 2, XR, XI)         \
    RUN_B(BV##0, SG, l1, CC, 1, XR, XI)         \
    RUN_B(BV##2, SG, l2, CC, 0, XR, XI)         \
    RUN_B(BV##1, SG, l1, CC, 0, XR, XI)         \
    RUN_B(BV##12, SG, l2, CC, 12, XR, XI)
                    {
                        Half b = lds_half(sb + offB + qi * 4096 + uj * (TJ * 16));       // (br, bi) limbs
                        SIX_RUNS(b.r, +, c1, 0, 1)     // T  += C1 * br
                        SIX_RUNS(b.i, +, c2, 0, 1)     // T  += C2 * bi
                    }
                    {
                        Half w = lds_half(sb + offB + qi * 4096 + 2048 + uj * (TJ * 16)); // (q br, q bi) limbs
                        SIX_RUNS(w.r, +, c2, 2, 3)     // T'' += C2 * (q br)
                        SIX_RUNS(w.i, -, c1, 2, 3)     // T'' -= C1 * (q bi)
                    }
#undef SIX_RUNS
#undef RUN_B
                }
            }
            const bool last = (qc == nqc - 1);
            if (((qc + 1) * SHD_QCH) % (SHD_BURST / 2) == 0 || last) {
                // fold the exact burst into the dd sums (shared memory, thread-private slots)
#pragma unroll
                for (int uj = 0; uj < 2; uj++)
#pragma unroll
                    for (int up = 0; up < 2; up++)
#pragma unroll
                        for (int x = 0; x < 4; x++) {
                            Acc& a = acc[uj][up][x];
                            double2* slot = &mainacc[((uj * 2 + up) * 4 + x) * 256 + tid];
                            double2 m = *slot;
                            dd sm = two_sum(a.l0, a.l1);
                            double e = __dadd_rn(sm.l, a.l2);
                            dd t = two_sum(m.x, sm.h);
                            m.x = t.h;
                            m.y = __dadd_rn(m.y, __dadd_rn(t.l, e));
                            *slot = m;
                            a.l0 = 0.0; a.l1 = 0.0; a.l2 = 0.0;
                        }
            }
            if (last) {
                // p-contraction for this p-block
#pragma unroll
                for (int uj = 0; uj < 2; uj++) {
                    const long j = jb * 32 + uj * TJ + tj;
#pragma unroll
                    for (int up = 0; up < 2; up++) {
                        const int pl = up * TP + tp;
                        const int p = pb * 32 + pl;
                        dd T[4];
#pragma unroll
                        for (int x = 0; x < 4; x++) {
                            double2* slot = &mainacc[((uj * 2 + up) * 4 + x) * 256 + tid];
                            double2 m = *slot;
                            T[x] = fast_two_sum(m.x, m.y);
                            *slot = make_double2(0.0, 0.0);
                        }
                        if (j < N) {
                            const double2* ap = reinterpret_cast<const double2*>(A) +
                                                (((size_t)pb * Npad + j) * 4) * 32 + pl;
                            double2 a0 = ap[0], a1 = ap[32], a2 = ap[64];
                            dd ar = limbs_to_dd(a0.x, a1.x, a2.x), ai = limbs_to_dd(a0.y, a1.y, a2.y);
                            dd I = dd_dot2(ar, T[1], ai, T[0], -1.0);     // Im[conj(A) T]
                            dd R = dd_dot2(ar, T[2], ai, T[3], 1.0);      // Re[conj(A) T'']
#pragma unroll
                            for (int a = 0; a < 3; a++) {
                                if (a < d) {
                                    int w = wT[a * Ppad + p];
                                    if (w != 0) g[uj][a] = dd_add(g[uj][a], dd_mul_d(I, (double)w));
                                    if (a == d - 1) g[uj][a] = dd_add(g[uj][a], dd_scale2(R, qs));
                                }
                            }
                        }
                    }
                }
            }
            __syncthreads();
            if (tid == 0 && issued < total) issue(s);
        }
    }

    // reduce over the 16 threads (tp) that share a particle: gred[a][j_local][tp]
    double2* gred = reinterpret_cast<double2*>(smem);
#pragma unroll
    for (int uj = 0; uj < 2; uj++)
#pragma unroll
        for (int a = 0; a < 3; a++)
            gred[(a * 32 + uj * TJ + tj) * TP + tp] = make_double2(g[uj][a].h, g[uj][a].l);
    __syncthreads();
    if (tid < 32 * d) {
        const int a = tid / 32, jl = tid % 32;
        const long j = jb * 32 + jl;
        if (j < N) {
            dd sum{0.0, 0.0};
            for (int t = 0; t < TP; t++) {
                double2 v = gred[(a * 32 + jl) * TP + t];
                sum = dd_add(sum, dd{v.x, v.y});
            }
            // (4 pi / L) / cscale
            dd pref = dd_div_d(dd_mul_d(dd{0x1.921fb54442d18p+2, 0x1.1a62633145c07p-52}, 2.0), L);
            sum = dd_mul(sum, pref);
            sum = dd_scale2(sum, 1.0 / scal->cscale);
            grad_hi[(size_t)a * N + j] = sum.h;
            grad_lo[(size_t)a * N + j] = sum.l;
        }
    }
}

}  // namespace

cudaError_t shd_grad_configure()
{
    return cudaFuncSetAttribute(k_grad, cudaFuncAttributeMaxDynamicSharedMemorySize, GSMEM);
}

cudaError_t shd_launch_grad(shd_ctx* h, double* grad_hi, double* grad_lo)
{
    k_grad<<<(unsigned)h->njb, TJ * TP, GSMEM, h->stream>>>(
        h->d, h->N, h->L, h->Npad, h->npb, h->Qpad, h->npb * 32, h->qscale_log2, h->d_qchunks, h->d_wT,
        h->d_A, h->d_Bg, h->d_C, h->d_scal, grad_hi, grad_lo, h->d_skip);
    h->last_launches += 1;
    return cudaGetLastError();
}
