// k_grad8.cu -- step a4 on the INT8 tensor cores (see k_grad.cu for the mathematics and k_rho8.cu for the
// digit-sliced exact integer contraction).  The q-contraction
//   T_j[p] = sum_q (C1 br + C2 bi),   T''_j[p] = sum_q (D1 br + D2 bi)
// is the matrix product  T[j, (p, out)] = sum_{(q, c)} b_j[(q, c)] W[(p, out), (q, c)]  with out in
// {T re, T im, T'' re, T'' im}, c in {re, im} and W built from C1, C2, D1, D2 by k_wtable8 (k_finish.cu).
// One CTA owns 128 particles (the M = 128 rows) and a segment of the step list; a step is 16 q (K = 32) of
// a block of 8 p (N side: 13 digit blocks of 8 p x 4 out = 32 columns, digits ascending, so one
// tcgen05.mma.kind::i8 per particle-side digit lands all its digit pairs in the tensor-memory columns of
// their digit sums; 18 instructions per step).  The s32 sums are exact (<= 2 Qn products per pair, Qn <= 5000).
// At the end of a block (or of the segment) the sixteen epilogue warps read tensor memory, four threads per
// particle (one per quarter of the block's 8 p): the 13 digit sums of each output are combined exactly into three
// 64-bit integers on the integer pipe, tensor memory is released, and only then the (128-bit) integer becomes a
// double-double that is contracted with the particle's own A_j[p] exactly as in k_grad.cu; the per-axis sums
// stay in registers across blocks.  Warp 16: TMA producer, warp 17: MMA issuer.
#include "pipe.cuh"
#include "shd_internal.h"

namespace {

constexpr int G8_ND = SHD_I8_DIGITS;
constexpr int G8_ASLAB = 128 * 32;                   // one digit of the particle operand of a step
constexpr int G8_WSLAB = 32 * 32;                    // one digit of the shared operand W
constexpr int G8_A = G8_ND * G8_ASLAB;               // 53248
constexpr int G8_W = G8_ND * G8_WSLAB;               // 13312
constexpr int G8_STAGE = G8_A + G8_W;
constexpr int G8_NST = 3;
constexpr int G8_SMEM = G8_NST * G8_STAGE;
constexpr int G8_EPI_WARPS = 16;                    // epilogue warps: four threads per particle, 2 p of the block's 8 each
constexpr int G8_THREADS = (G8_EPI_WARPS + 2) * 32;

__device__ __forceinline__ uint64_t g8_desc(uint32_t addr) {
    return (uint64_t)((addr >> 4) & 0x3FFF) | ((uint64_t)(128 >> 4) << 16) | ((uint64_t)(256 >> 4) << 32) | ((uint64_t)1 << 46);
}
__device__ __forceinline__ uint32_t g8_idesc(int n) {
    return (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
}
__device__ __forceinline__ void g8_mma(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
    uint32_t z = 0;
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, {%5, %5, %5, %5}, p;\n\t}"
                 ::"r"(tmem_d), "l"(da), "l"(db), "r"(idesc), "r"(accumulate), "r"(z) : "memory");
}
__device__ __forceinline__ void g8_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ dd limbs_to_dd8(double x0, double x1, double x2) {
    return fast_two_sum(__dadd_rn(x0, x1), x2);
}
// T 2^e as a double-double (relative error <= 2^-105; |T| < 2^127).  Sign and magnitude first, so that the four
// 32-bit words of the magnitude are non-overlapping terms of one sign (no cancellation); every word becomes a
// double through the 2^52 trick with its scale in the exponent field ((2^52 + u) 2^k - 2^52 2^k = u 2^k, one
// exact addition), and two exact pair sums are merged.  15 additions instead of three conversions and two
// double-double sums: the epilogue warps are bound by the FP64 pipe.
__device__ __forceinline__ dd s128_scaled_to_dd(__int128 T, int e) {
    const bool neg = T < 0;
    const unsigned __int128 M = neg ? (unsigned __int128)(-T) : (unsigned __int128)T;
    const unsigned long long mh = (unsigned long long)(M >> 64), ml = (unsigned long long)M;
    const int e0 = 0x43300000 + (e << 20);
    const double x0 = __dadd_rn(__hiloint2double(e0, (int)(unsigned)ml), -__hiloint2double(e0, 0));
    const double x1 = __dadd_rn(__hiloint2double(e0 + (32 << 20), (int)(unsigned)(ml >> 32)), -__hiloint2double(e0 + (32 << 20), 0));
    const double x2 = __dadd_rn(__hiloint2double(e0 + (64 << 20), (int)(unsigned)mh), -__hiloint2double(e0 + (64 << 20), 0));
    const double x3 = __dadd_rn(__hiloint2double(e0 + (96 << 20), (int)(unsigned)(mh >> 32)), -__hiloint2double(e0 + (96 << 20), 0));
    const dd hi = fast_two_sum(x3, x2), lo = fast_two_sum(x1, x0);   // exact: |x3| >= |x2| or x3 = 0, same below
    dd r = fast_two_sum(hi.h, __dadd_rn(hi.l, lo.h));
    r.l = __dadd_rn(r.l, lo.l);
    return neg ? dd{-r.h, -r.l} : r;
}

// ND = 13: full precision; 7 / 4: the most significant digits only (shd_set_precision 2 / 1; see k_rho8.cu)
template <int ND>
__global__ void __launch_bounds__(G8_THREADS, 1) k_grad8(
    int d, long N, long Npad, long njb128, int Ppad, int qscale_log2, int nkq,
    const int2* __restrict__ steps, int nsteps, int nseg, const int* __restrict__ wT,
    const double* __restrict__ A, const signed char* __restrict__ Bg8, const signed char* __restrict__ W8,
    double* __restrict__ gpart, const int* __restrict__ skip)
{
    if (skip && *skip) return;
    extern __shared__ __align__(1024) unsigned char smem[];
    // a stage holds the ND digit slabs in use of both operands; the fewer digits, the deeper the ring
    constexpr int STG = ND * (G8_ASLAB + G8_WSLAB), NST = G8_SMEM / STG < 8 ? G8_SMEM / STG : 8;
    __shared__ __align__(8) unsigned long long full_bar[8], empty_bar[8], tfull_bar, tempty_bar;
    __shared__ uint32_t tmem_base;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    // segment fastest: the CTAs of one particle block run side by side and share its digit slabs in L2
    const int seg = (int)(blockIdx.x % nseg);
    const long jb = blockIdx.x / nseg;
    const int c_begin = (int)((long)nsteps * seg / nseg), c_end = (int)((long)nsteps * (seg + 1) / nseg);
    const int total = c_end - c_begin;
    const uint32_t s0 = smem_u32(smem);
    if (tid == 0) {
        for (int s = 0; s < NST; s++) { mbar_init(smem_u32(&full_bar[s]), 1); mbar_init(smem_u32(&empty_bar[s]), 1); }
        mbar_init(smem_u32(&tfull_bar), 1);
        mbar_init(smem_u32(&tempty_bar), G8_EPI_WARPS * 32);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(&tmem_base)));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    const uint32_t tb = tmem_base;
    constexpr int OFF = G8_ND - ND;                  // first (least significant) digit used

    if (warp == G8_EPI_WARPS) {
        if (lane == 0) {
            const signed char* gA = Bg8 + (size_t)jb * nkq * G8_A;
            for (int i = 0; i < total; i++) {
                const int s = i % NST;
                if (i >= NST) mbar_wait(smem_u32(&empty_bar[s]), (uint32_t)((i / NST - 1) & 1));
                const uint32_t bar = smem_u32(&full_bar[s]);
                const int2 st = steps[c_begin + i];           // x: pb8 * nkq + kstep,  y: kstep | end << 16
                mbar_expect_tx(bar, ND * (G8_ASLAB + G8_WSLAB));
                tma_load_1d(s0 + s * STG, gA + (size_t)(st.y & 0xffff) * G8_A + OFF * G8_ASLAB, ND * G8_ASLAB, bar);
                tma_load_1d(s0 + s * STG + ND * G8_ASLAB, W8 + (size_t)st.x * G8_W + OFF * G8_WSLAB, ND * G8_WSLAB, bar);
            }
        }
    } else if (warp == G8_EPI_WARPS + 1) {
        if (lane == 0) {
            int nblock = 0;
            bool fresh = true;                                 // next step starts a new accumulation
            for (int i = 0; i < total; i++) {
                const int s = i % NST;
                const int2 st = steps[c_begin + i];
                if (fresh && nblock > 0) {                     // tensor memory must have been drained by the epilogue
                    mbar_wait(smem_u32(&tempty_bar), (uint32_t)((nblock - 1) & 1));
                    asm volatile("tcgen05.fence::after_thread_sync;");
                }
                mbar_wait(smem_u32(&full_bar[s]), (uint32_t)((i / NST) & 1));
                asm volatile("tcgen05.fence::after_thread_sync;");
                const uint32_t sA = s0 + s * STG, sW = sA + ND * G8_ASLAB;
                // descriptors differ only in the 14-bit address field: one base per operand, compile-time offsets
                const uint64_t dA0 = g8_desc(sA), dW0 = g8_desc(sW);
                auto issue = [&](int ii, uint32_t acc) {            // relative digit i' (absolute OFF + i')
                    const int n = (ii + 1) * 32, l0 = ND - 1 - ii;          // its partners: relative digits l0 .. ND - 1
                    const uint64_t da = dA0 + (uint64_t)((ii * G8_ASLAB) >> 4);
                    if (n <= 256) {
                        g8_mma(tb, da, dW0 + (uint64_t)((l0 * G8_WSLAB) >> 4), g8_idesc(n), acc);
                    } else {
                        g8_mma(tb, da, dW0 + (uint64_t)((l0 * G8_WSLAB) >> 4), g8_idesc(256), acc);
                        g8_mma(tb + 256, da, dW0 + (uint64_t)(((l0 + 8) * G8_WSLAB) >> 4), g8_idesc(n - 256), acc);
                    }
                };
                // A block's first step runs from the most significant digit down (its first instruction covers all
                // columns and initialises them); the other steps run upwards, short instructions first and long ones
                // last, so that the tensor core's queue holds long instructions while this thread crosses the step
                // boundary (k_rho8.cu).
                if (fresh || ND < G8_ND) {
#pragma unroll
                    for (int ii = ND - 1; ii >= 0; ii--) issue(ii, (!fresh || ii < ND - 1) ? 1u : 0u);
                } else {
#pragma unroll
                    for (int ii = 0; ii < ND; ii++) issue(ii, 1u);
                }
                g8_commit(smem_u32(&empty_bar[s]));
                fresh = false;
                if ((st.y >> 16) || i == total - 1) {          // block (or segment) end: hand the sums to the epilogue
                    g8_commit(smem_u32(&tfull_bar));
                    nblock++;
                    fresh = true;
                }
            }
        }
    } else {
        // ---- 16 epilogue warps: thread = (particle = TMEM lane, quarter of the block's 8 p); columns 32 c + 4 p_local + out
        const int quarter = warp >> 2, row = tid & 127;
        const long j = jb * 128 + row;
        const double qs = ldexp(1.0, qscale_log2);
        const double2* Aj = reinterpret_cast<const double2*>(A) + (size_t)(j >> 2) * 3 * 32 * 4 + (j & 3);
        dd g0{0.0, 0.0}, g1{0.0, 0.0}, g2{0.0, 0.0}, g3{0.0, 0.0};
        int nblock = 0;
        // next block (or segment) end at or after step i: 32 steps per look, one load latency per block
        auto next_end = [&](int& i, int2& st) {
            for (;;) {
                const int ii = i + lane < total - 1 ? i + lane : total - 1;
                const int2 sl = steps[c_begin + ii];
                const unsigned m = __ballot_sync(0xffffffffu, (sl.y >> 16) || ii == total - 1);
                if (m) {
                    const int f = __ffs(m) - 1;
                    st.x = __shfl_sync(0xffffffffu, sl.x, f);
                    st.y = __shfl_sync(0xffffffffu, sl.y, f);
                    i += f;
                    return;
                }
                i += 32;
            }
        };
        int i = 0;
        int2 st;
        if (total > 0) next_end(i, st);
        while (i < total) {
            const int pb8 = st.x / nkq;
            // this block's A_j[p] (three limbs each) and axis weights.  With fewer digits the epilogue's own latencies
            // bound the kernel and registers are free: the loads go out before the wait for the tensor core
            double2 araw[2][3];
            int wg[2][3];
            auto load_A = [&]() {
#pragma unroll
                for (int pp = 0; pp < 2; pp++) {
                    const int p = pb8 * 8 + quarter * 2 + pp;
                    araw[pp][0] = araw[pp][1] = araw[pp][2] = make_double2(0.0, 0.0);
                    wg[pp][0] = wg[pp][1] = wg[pp][2] = 0;
                    if (j < N && p < Ppad) {
                        const double2* ap = Aj + ((size_t)(p >> 5) * (Npad / 4) * 3 * 32 + (p & 31)) * 4;
                        asm volatile("ld.global.nc.v2.f64 {%0,%1}, [%2];" : "=d"(araw[pp][0].x), "=d"(araw[pp][0].y) : "l"(ap));
                        asm volatile("ld.global.nc.v2.f64 {%0,%1}, [%2];" : "=d"(araw[pp][1].x), "=d"(araw[pp][1].y) : "l"(ap + 128));
                        asm volatile("ld.global.nc.v2.f64 {%0,%1}, [%2];" : "=d"(araw[pp][2].x), "=d"(araw[pp][2].y) : "l"(ap + 256));
#pragma unroll
                        for (int ax = 0; ax < 3; ax++)
                            if (ax < d) wg[pp][ax] = wT[ax * Ppad + p];
                    }
                }
            };
            if constexpr (ND < G8_ND) load_A();
            mbar_wait(smem_u32(&tfull_bar), (uint32_t)(nblock & 1));
            asm volatile("tcgen05.fence::after_thread_sync;");
            // Drain: the thread's 16 columns (4 p x 4 outputs) of each of the ND digit sums, combined EXACTLY on the
            // integer pipe into NG 64-bit group values G_g = sum_c 2^(8 (c - 4 g)) S_c (four sums per group, the top
            // group takes a fifth).  Column block c holds the absolute digit sum s = ND - 1 + 2 OFF + c, a sum
            // of ND - c digit pairs of <= 2 Qn <= 10^4 products each: |S_c| <= (ND - c) 10^4 2^14, which bounds
            // the groups by 2^54.6, 2^53.9 and (top five, 5 + 4 2^8 + 3 2^16 + 2 2^24 + 2^32 pairs-weights) 2^59.3.
            // Nothing else happens before the release, so the tensor core idles only for these loads.
            constexpr int NG = (ND + 2) / 4;
            long long G[NG][8];
            const uint32_t taddr = tb + ((uint32_t)((warp & 3) * 32) << 16) + 8 * quarter;
#pragma unroll
            for (int c = 0; c < ND; c++) {
                uint32_t v[8];
                asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                             : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
                             : "r"(taddr + c * 32));
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                const int g = (c / 4 < NG - 1) ? c / 4 : NG - 1, sh = 8 * (c - 4 * g);
#pragma unroll
                for (int e = 0; e < 8; e++) {
                    const long long x = (long long)(int)v[e];
                    G[g][e] = sh == 0 ? x : G[g][e] + x * (1ll << sh);
                }
            }
            // tensor memory is drained: the next block's instructions start while the rest of the epilogue runs
            asm volatile("tcgen05.fence::before_thread_sync;");
            mbar_arrive(smem_u32(&tempty_bar));
            int inext = i + 1;                                 // the block after this one
            int2 stn = st;
            if (inext < total) next_end(inext, stn);
            if constexpr (ND == G8_ND) load_A();               // (13 digits: after the release, the registers are needed above)
            if constexpr (ND < G8_ND) {
                // Fewer digits (operands of 54 or 30 bits): the sums are worth no more than a double, so the
                // contraction with A_j[p] runs in plain FP64 (products rounded once, ~2^-53 relative, below the
                // operand truncation); only the running per-axis sums stay double-double.  A tenth of the FP64
                // instructions of the full path: at these digit counts the epilogue, not the tensor core, is
                // what bounds the kernel.
                const double w0 = __longlong_as_double((long long)(1023 + 8 * (ND - 1 + 2 * OFF) - 204) << 52);
#pragma unroll
                for (int pp = 0; pp < 2; pp++) {
                    double T[4];
#pragma unroll
                    for (int o4 = 0; o4 < 4; o4++) {
                        double t = (double)G[0][4 * pp + o4];
                        if (NG > 1) t = __fma_rn((double)G[NG - 1][4 * pp + o4], 4294967296.0, t);
                        T[o4] = __dmul_rn(t, w0);
                    }
                    const double ar = __dadd_rn(__dadd_rn(araw[pp][0].x, araw[pp][1].x), araw[pp][2].x);
                    const double ai = __dadd_rn(__dadd_rn(araw[pp][0].y, araw[pp][1].y), araw[pp][2].y);
                    const int p = pb8 * 8 + quarter * 2 + pp;
                    if (j < N && p < Ppad) {
                        const double I = __fma_rn(ar, T[1], -__dmul_rn(ai, T[0]));      // Im[conj(A) T]
                        const double R = __fma_rn(ar, T[2], __dmul_rn(ai, T[3]));       // Re[conj(A) T'']
#define GACC8F(AX)                                                                            \
    if (AX < d) {                                                                             \
        const int wgt = AX < 3 ? wg[pp][AX < 3 ? AX : 0] : 0;                                 \
        if (wgt != 0) g##AX = dd_add_d(g##AX, __dmul_rn(I, (double)wgt));                     \
        if (AX == d - 1) g##AX = dd_add_d(g##AX, __dmul_rn(R, qs));                           \
    }
                        GACC8F(0) GACC8F(1) GACC8F(2) GACC8F(3)
#undef GACC8F
                    }
                }
            } else {
                dd Tall[2][4];
#pragma unroll
                for (int e = 0; e < 8; e++) {
                    __int128 T = (__int128)G[0][e];                     // sum_c 2^(8 c) S_c, exact
#pragma unroll
                    for (int g = 1; g < NG; g++) T += (__int128)G[g][e] << (32 * g);
                    Tall[e >> 2][e & 3] = s128_scaled_to_dd(T, 8 * (ND - 1 + 2 * OFF) - 204);
                }
#pragma unroll
                for (int pp = 0; pp < 2; pp++) {
                    const dd* T = Tall[pp];
                    const dd ar = limbs_to_dd8(araw[pp][0].x, araw[pp][1].x, araw[pp][2].x);
                    const dd ai = limbs_to_dd8(araw[pp][0].y, araw[pp][1].y, araw[pp][2].y);
                    const int p = pb8 * 8 + quarter * 2 + pp;
                    if (j < N && p < Ppad) {
                        const dd I = dd_dot2(ar, T[1], ai, T[0], -1.0);         // Im[conj(A) T]
                        const dd R = dd_dot2(ar, T[2], ai, T[3], 1.0);          // Re[conj(A) T'']
#define GACC8(AX)                                                                             \
    if (AX < d) {                                                                             \
        const int wgt = AX < 3 ? wg[pp][AX < 3 ? AX : 0] : 0;                                 \
        if (wgt != 0) g##AX = dd_add(g##AX, dd_mul_d(I, (double)wgt));                        \
        if (AX == d - 1) g##AX = dd_add(g##AX, dd_scale2(R, qs));                             \
    }
                        GACC8(0) GACC8(1) GACC8(2) GACC8(3)
#undef GACC8
                    }
                }
            }
            nblock++;
            i = inext;
            st = stn;
        }
        if (j < N) {
            double2* o = reinterpret_cast<double2*>(gpart);
            const size_t slot = (size_t)(seg * 4 + quarter) * d;       // four partials per segment (the p quarters)
            if (d > 0) o[(slot + 0) * N + j] = make_double2(g0.h, g0.l);
            if (d > 1) o[(slot + 1) * N + j] = make_double2(g1.h, g1.l);
            if (d > 2) o[(slot + 2) * N + j] = make_double2(g2.h, g2.l);
            if (d > 3) o[(slot + 3) * N + j] = make_double2(g3.h, g3.l);
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tb));
}

}  // namespace

cudaError_t shd_grad8_configure()
{
    cudaError_t e = cudaFuncSetAttribute(k_grad8<13>, cudaFuncAttributeMaxDynamicSharedMemorySize, G8_SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_grad8<7>, cudaFuncAttributeMaxDynamicSharedMemorySize, G8_SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_grad8<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, G8_SMEM);
    return e;
}

// k_gradsum (k_grad.cu) adds the segments' partial gradients and applies 4 pi / L / cscale
cudaError_t shd_launch_grad8_main(shd_ctx* h)
{
#define LAUNCH_GRAD8(NDV)                                                                            \
    k_grad8<NDV><<<(unsigned)(h->njb128 * h->nseg8), G8_THREADS, G8_SMEM, h->stream>>>(                      \
        h->d, h->N, h->Npad, h->njb128, h->npb * 32, h->qscale_log2, h->nkq8,                          \
        reinterpret_cast<const int2*>(h->d_steps8), h->nsteps8, h->nseg8, h->d_wT,                     \
        h->d_A, h->d_Bg8, h->d_W8, h->d_gpart, h->d_skip)
    if (h->nlimb >= 3) LAUNCH_GRAD8(13);
    else if (h->nlimb == 2) LAUNCH_GRAD8(7);
    else LAUNCH_GRAD8(4);
#undef LAUNCH_GRAD8
    h->last_launches += 1;
    return cudaGetLastError();
}
