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
// 64-bit integers on the integer pipe, tensor memory is released, and the exact (128-bit) integer T is contracted
// with the particle's own A_j[p] -- the integer trunc(a 2^102) k_tables stores in sign-magnitude form -- in
// INTEGER arithmetic: (|T| |A|) >> 96 by 64-bit multiplies, signed 192-bit per-axis accumulators in registers across
// blocks, one conversion to double-double per CTA.  Measured on B200 (profiles/r2a_summary.md): FP64 instructions all
// but stall while tcgen05.mma.kind::i8 streams on the same SM (DADD chains of 16 warps make no progress during a
// back-to-back N = 256 stream, IMAD chains are unaffected), so the double-double epilogue of round 1 (332 FP64
// instructions per thread and block) took 11.7 us per block against 9.9 us of tensor work and slowed the issue.
// Warp 16: TMA producer (one lane); warp 17: MMA issuer, all 32 lanes in the loop (descriptors stay in uniform
// registers, no per-instruction election loop), one elected lane issues.
#include "pipe.cuh"
#include "shd_internal.h"
#include <algorithm>
#include <cstdio>
#include <cstdlib>

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
// issued by the elected lane of a converged warp (elected = 1 in one lane)
__device__ __forceinline__ void g8_mma(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate, uint32_t elected) {
    uint32_t z = 0;
    asm volatile("{\n\t.reg .pred p, q;\n\tsetp.ne.b32 p, %4, 0;\n\tsetp.ne.b32 q, %6, 0;\n\t"
                 "@q tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, {%5, %5, %5, %5}, p;\n\t}"
                 ::"r"(tmem_d), "l"(da), "l"(db), "r"(idesc), "r"(accumulate), "r"(z), "r"(elected) : "memory");
}
__device__ __forceinline__ void g8_commit(uint32_t bar, uint32_t elected) {
    asm volatile("{\n\t.reg .pred q;\n\tsetp.ne.b32 q, %1, 0;\n\t"
                 "@q tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n\t}" ::"r"(bar), "r"(elected) : "memory");
}
typedef unsigned long long ull;
// signed 192-bit integer (two's complement), the per-axis gradient accumulator of a thread
struct acc192 { ull w0, w1, w2; };
// a += neg ? -r : r   (r = 192-bit magnitude)
__device__ __forceinline__ void acc_addsub(acc192& a, ull r0, ull r1, ull r2, bool neg) {
    const ull m = neg ? ~0ull : 0ull;
    unsigned __int128 s = (unsigned __int128)a.w0 + (r0 ^ m) + (neg ? 1u : 0u);
    a.w0 = (ull)s;
    s = (unsigned __int128)a.w1 + (r1 ^ m) + (ull)(s >> 64);
    a.w1 = (ull)s;
    a.w2 = a.w2 + (r2 ^ m) + (ull)(s >> 64);
}
// g += v w  (mod 2^192; v two's complement, 0 <= w < 2^32)
__device__ __forceinline__ void acc_mac(acc192& g, const acc192& v, uint32_t w) {
    unsigned __int128 c = (unsigned __int128)v.w0 * w + g.w0;
    g.w0 = (ull)c;
    c = (unsigned __int128)v.w1 * w + g.w1 + (ull)(c >> 64);
    g.w1 = (ull)c;
    g.w2 = v.w2 * w + g.w2 + (ull)(c >> 64);
}
// (|T| |A|) >> 96 with |T| = (t1 : t0) < 2^127 and |A| = (a1 : a0) <= 2^102 (+ a few units): the product is below 2^230,
// the result below 2^134.  HI = false: t1 = 0 (the 4-digit precision, |T| < 2^56).
template <bool HI>
__device__ __forceinline__ void mul_shr96(ull t0, ull t1, ull a0, ull a1, ull& r0, ull& r1, ull& r2) {
    const unsigned __int128 p00 = (unsigned __int128)t0 * a0, p01 = (unsigned __int128)t0 * a1;
    unsigned __int128 mid = (p00 >> 64) + (ull)p01, up = p01 >> 64;
    if (HI) {
        const unsigned __int128 p10 = (unsigned __int128)t1 * a0, p11 = (unsigned __int128)t1 * a1;
        mid += (ull)p10;
        up += (p10 >> 64) + p11;
    }
    up += mid >> 64;
    const ull l1 = (ull)mid, l2 = (ull)up, l3 = (ull)(up >> 64);
    r0 = (l1 >> 32) | (l2 << 32);
    r1 = (l2 >> 32) | (l3 << 32);
    r2 = l3 >> 32;
}
// g 2^e as a double-double (relative error <= 2^-104): sign and magnitude, the six 32-bit words of the magnitude
// become doubles through the 2^52 trick with their scale in the exponent field ((2^52 + u) 2^k - 2^52 2^k = u 2^k,
// exact) and are summed from the top.  Once per CTA and axis.
__device__ __forceinline__ dd acc192_to_dd(acc192 g, int e) {
    const bool neg = (long long)g.w2 < 0;
    if (neg) { acc192 z{0, 0, 0}; acc_addsub(z, g.w0, g.w1, g.w2, true); g = z; }
    const uint32_t w[6] = {(uint32_t)g.w0, (uint32_t)(g.w0 >> 32), (uint32_t)g.w1, (uint32_t)(g.w1 >> 32),
                           (uint32_t)g.w2, (uint32_t)(g.w2 >> 32)};
    dd r{0.0, 0.0};
#pragma unroll
    for (int k = 5; k >= 0; k--) {
        const int e0 = 0x43300000 + ((e + 32 * k) << 20);
        const double x = __dadd_rn(__hiloint2double(e0, (int)w[k]), -__hiloint2double(e0, 0));
        r = dd_add_d(r, x);
    }
    return neg ? dd{-r.h, -r.l} : r;
}

// ND = 13: full precision; 7 / 4: the most significant digits only (shd_set_precision 2 / 1; see k_rho8.cu)
// D = the dimension d: the epilogue is bound by instruction issue (about 1500 instructions per thread and block), so the
// per-axis accumulations exist only for the axes there are: axis a < NI takes I w_a[p] (NI = d - 1 prefix axes; d = 1: the one
// axis, split as n = S p + q), axis d - 1 takes R 2^qscale
template <int ND, int D>
__global__ void __launch_bounds__(G8_THREADS, 1) k_grad8(
    int d, long N, long Npad, long njb128, int Ppad, int qscale_log2, int nkq,
    const int2* __restrict__ steps, int nsteps, int nseg, const int* __restrict__ wT,
    const ulonglong2* __restrict__ Afix, const signed char* __restrict__ Bg8, const signed char* __restrict__ W8,
    double* __restrict__ gpart, long nunits, long long* __restrict__ clk, const int* __restrict__ skip)
{
    if (skip && *skip) return;
    extern __shared__ __align__(1024) unsigned char smem[];
    // a stage holds the ND digit slabs in use of both operands; the fewer digits, the deeper the ring
    constexpr int STG = ND * (G8_ASLAB + G8_WSLAB), NST = G8_SMEM / STG < 8 ? G8_SMEM / STG : 8;
    // tempty_bar[g]: column blocks 4 g .. 4 g + 3 of the accumulator set have been read AND zeroed by the epilogue
    constexpr int NTG = (ND + 3) / 4;
    __shared__ __align__(8) unsigned long long full_bar[8], empty_bar[8], tfull_bar, tempty_bar[4];
    __shared__ uint32_t tmem_base;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    // PERSISTENT: one CTA per SM walks the work units u = blockIdx.x, blockIdx.x + gridDim.x, ... (unit = particle block x
    // segment of the step list, all of the same length; segment fastest, so that the CTAs of one particle block run side
    // by side and share its digit slabs in L2).  The TMA ring and the tensor-memory hand-shake run on across units: the
    // producer is already loading the next unit while the epilogue of the last block of a unit -- and its conversion and
    // write-out -- runs beside the next unit's first instructions, and nothing is set up twice.
    // HAND-OVER: one accumulator set (32 ND of the 512 columns) is all tensor memory holds, so at a block end the tensor
    // core waits for the epilogue to read it -- 0.9 us, bound by the tensor-memory read bandwidth.  To hide most of that the
    // epilogue ZEROES each group of four column blocks right after reading it (tcgen05.st is four times faster than the
    // read) and releases the group on its own barrier; every instruction accumulates (no initialising instruction), and
    // the first K-step of the next block runs in ASCENDING digit order -- digit i' touches column blocks 0 .. i' only --
    // waiting for a group just before the first instruction that needs it.
    const uint32_t s0 = smem_u32(smem);
    if (tid == 0) {
        for (int s = 0; s < NST; s++) { mbar_init(smem_u32(&full_bar[s]), 1); mbar_init(smem_u32(&empty_bar[s]), 1); }
        mbar_init(smem_u32(&tfull_bar), 1);
        for (int g = 0; g < NTG; g++) mbar_init(smem_u32(&tempty_bar[g]), G8_EPI_WARPS * 32);
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
          int s = 0;                                            // ring position and the parity of its "empty" phase,
          uint32_t epar = 0u;                                   //   kept incrementally (no division in the loop)
          bool first_round = true;
          for (long u = blockIdx.x; u < nunits; u += gridDim.x) {
            const int seg = (int)(u % nseg);
            const long jb = u / nseg;
            const int c_begin = (int)((long)nsteps * seg / nseg), total = (int)((long)nsteps * (seg + 1) / nseg) - c_begin;
            const signed char* gA = Bg8 + (size_t)jb * nkq * G8_A;
            for (int i = 0; i < total; i++) {
                if (!first_round) mbar_wait(smem_u32(&empty_bar[s]), epar);
                const uint32_t bar = smem_u32(&full_bar[s]);
                const int2 st = steps[c_begin + i];           // x: pb8 * nkq + kstep,  y: kstep | end << 16
                mbar_expect_tx(bar, ND * (G8_ASLAB + G8_WSLAB));
                tma_load_1d(s0 + s * STG, gA + (size_t)(st.y & 0xffff) * G8_A + OFF * G8_ASLAB, ND * G8_ASLAB, bar);
                tma_load_1d(s0 + s * STG + ND * G8_ASLAB, W8 + (size_t)st.x * G8_W + OFF * G8_WSLAB, ND * G8_WSLAB, bar);
                if (++s == NST) { s = 0; if (first_round) first_round = false; else epar ^= 1u; }
            }
          }
        }
    } else if (warp == G8_EPI_WARPS + 1) {
        {
            uint32_t elected;
            asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(elected));
            unsigned long long g0 = 0;
            long long c0 = 0;
            if (blockIdx.x == 0 && clk) { asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g0)); c0 = clock64(); }
            uint32_t tpar = 0u;                                // parity of the tensor-memory hand-shake (blocks handed over so far)
            int s = 0;                                         // ring position and the parity of its "full" phase
            uint32_t fpar = 0u;
            bool fresh = true;                                 // next step starts a new accumulation
          for (long u = blockIdx.x; u < nunits; u += gridDim.x) {
            const int seg = (int)(u % nseg);
            const int c_begin = (int)((long)nsteps * seg / nseg), total = (int)((long)nsteps * (seg + 1) / nseg) - c_begin;
            for (int i = 0; i < total; i++) {
                const int2 st = steps[c_begin + i];
                mbar_wait(smem_u32(&full_bar[s]), fpar);
                asm volatile("tcgen05.fence::after_thread_sync;");
                const uint32_t sA = s0 + s * STG, sW = sA + ND * G8_ASLAB;
                // descriptors differ only in the 14-bit address field: one base per operand, compile-time offsets
                const uint64_t dA0 = g8_desc(sA), dW0 = g8_desc(sW);
                auto issue = [&](int ii, uint32_t acc) {            // relative digit i' (absolute OFF + i')
                    const int n = (ii + 1) * 32, l0 = ND - 1 - ii;          // its partners: relative digits l0 .. ND - 1
                    const uint64_t da = dA0 + (uint64_t)((ii * G8_ASLAB) >> 4);
                    if (n <= 256) {
                        g8_mma(tb, da, dW0 + (uint64_t)((l0 * G8_WSLAB) >> 4), g8_idesc(n), acc, elected);
                    } else {
                        // two instructions of n / 2 columns each, not 256 + the rest: an instruction reads its 4 KB A
                        // slab and 32 n bytes of the other operand from shared memory, about 32 + n / 4 cycles, against
                        // n / 2 cycles of arithmetic, so below n = 128 the operand fetch is what it costs (measured:
                        // the 256 + rest split is 2.5 % slower in k_grad8, 1 % in k_rho8; profiles/r2b_summary.md)
                        const int n1 = n / 2;                                  // 144 .. 208: a multiple of 16
                        g8_mma(tb, da, dW0 + (uint64_t)((l0 * G8_WSLAB) >> 4), g8_idesc(n1), acc, elected);
                        g8_mma(tb + n1, da, dW0 + (uint64_t)((l0 * G8_WSLAB + n1 * 32) >> 4), g8_idesc(n - n1), acc, elected);
                    }
                };
                // Every step runs upwards, short instructions first and long ones last, so that the tensor core's queue
                // holds long instructions while this thread crosses the step boundary (k_rho8.cu); all accumulate (the
                // accumulator set is zero at a block's start: zeroed by the epilogue, or at kernel start).  A block's
                // first step waits for column group g (read and zeroed) before its first instruction that touches it.
#pragma unroll
                for (int ii = 0; ii < ND; ii++) {
                    if (fresh && (ii & 3) == 0) {
                        mbar_wait(smem_u32(&tempty_bar[ii >> 2]), tpar);
                        asm volatile("tcgen05.fence::after_thread_sync;");
                    }
                    issue(ii, 1u);
                }
                g8_commit(smem_u32(&empty_bar[s]), elected);
                fresh = false;
                if ((st.y >> 16) || i == total - 1) {          // block (or segment) end: hand the sums to the epilogue
                    g8_commit(smem_u32(&tfull_bar), elected);
                    tpar ^= 1u;
                    fresh = true;
                }
                if (++s == NST) { s = 0; fpar ^= 1u; }
            }
          }
          if (blockIdx.x == 0 && clk && elected) {
              unsigned long long g1;
              asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
              clk[0] = clock64() - c0;
              clk[1] = (long long)(g1 - g0);
          }
        }
    } else {
        // ---- 16 epilogue warps: thread = (particle = TMEM lane, quarter of the block's 8 p); columns 32 c + 4 p_local + out
        const int quarter = warp >> 2, row = tid & 127;
        const long NpadA = njb128 * 128;
        uint32_t nblock = 0;                                   // blocks drained by this CTA so far (tensor-memory hand-shake)
        {
            // the accumulator set starts at zero: every thread clears its own 8 columns of every column block, then
            // releases all groups (phase 0 of the tempty barriers = "zero at kernel start")
            const uint32_t taddr0 = tb + ((uint32_t)((warp & 3) * 32) << 16) + 8 * quarter;
            const uint32_t z = 0;
#pragma unroll
            for (int c = 0; c < ND; c++)
                asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%1,%1,%1,%1,%1,%1,%1};" ::"r"(taddr0 + c * 32), "r"(z) : "memory");
            asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
            asm volatile("tcgen05.fence::before_thread_sync;");
#pragma unroll
            for (int g = 0; g < NTG; g++) mbar_arrive(smem_u32(&tempty_bar[g]));
        }
      for (long u = blockIdx.x; u < nunits; u += gridDim.x) {
        const int seg = (int)(u % nseg);
        const long jb = u / nseg;
        const int c_begin = (int)((long)nsteps * seg / nseg), total = (int)((long)nsteps * (seg + 1) / nseg) - c_begin;
        const long j = jb * 128 + row;
        const ulonglong2* Aj = Afix + (size_t)j * 2;
        constexpr int NI = D == 1 ? 1 : D - 1;
        acc192 g[D];
#pragma unroll
        for (int ax = 0; ax < D; ax++) g[ax] = acc192{0, 0, 0};
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
            // this block's A_j[p] (sign-magnitude integers trunc(a 2^102), k_tables) and axis weights, requested before
            // the wait for the tensor core
            ulonglong2 ar[2], ai[2];
            int wg[2][NI];
#pragma unroll
            for (int pp = 0; pp < 2; pp++) {
                const int p = pb8 * 8 + quarter * 2 + pp;             // < Ppad8 (the table is allocated and zeroed up to there)
                const ulonglong2* ap = Aj + (size_t)p * NpadA * 2;
                asm volatile("ld.global.nc.v2.u64 {%0,%1}, [%2];" : "=l"(ar[pp].x), "=l"(ar[pp].y) : "l"(ap));
                asm volatile("ld.global.nc.v2.u64 {%0,%1}, [%2];" : "=l"(ai[pp].x), "=l"(ai[pp].y) : "l"(ap + 1));
#pragma unroll
                for (int ax = 0; ax < NI; ax++) wg[pp][ax] = p < Ppad ? wT[ax * Ppad + p] : 0;
            }
            mbar_wait(smem_u32(&tfull_bar), (uint32_t)(nblock & 1));
            asm volatile("tcgen05.fence::after_thread_sync;");
            // Drain: the thread's 8 columns (2 p x 4 outputs) of each of the ND digit sums, combined EXACTLY on the
            // integer pipe into NG 64-bit group values G_g = sum_c 2^(8 (c - 4 g)) S_c (four sums per group, the top
            // group takes a fifth).  Column block c holds the absolute digit sum s = ND - 1 + 2 OFF + c, a sum
            // of ND - c digit pairs of <= 2 Qn <= 10^4 products each: |S_c| <= (ND - c) 10^4 2^14, which bounds
            // the groups by 2^54.6, 2^53.9 and (top five, 5 + 4 2^8 + 3 2^16 + 2 2^24 + 2^32 pairs-weights) 2^59.3.
            // The loads go out four at a time (one wait per four); nothing else happens before the release.
            constexpr int NG = (ND + 2) / 4;
            long long G[NG][8];
            const uint32_t taddr = tb + ((uint32_t)((warp & 3) * 32) << 16) + 8 * quarter;
#pragma unroll
            for (int c0 = 0; c0 < ND; c0 += 4) {
                uint32_t v[4][8];
#pragma unroll
                for (int cc = 0; cc < 4; cc++)
                    if (c0 + cc < ND)
                        asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                                     : "=r"(v[cc][0]), "=r"(v[cc][1]), "=r"(v[cc][2]), "=r"(v[cc][3]), "=r"(v[cc][4]), "=r"(v[cc][5]),
                                       "=r"(v[cc][6]), "=r"(v[cc][7])
                                     : "r"(taddr + (c0 + cc) * 32));
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                {
                    // this group of column blocks is in registers: zero it and hand it back to the tensor core
                    const uint32_t z = 0;
#pragma unroll
                    for (int cc = 0; cc < 4; cc++)
                        if (c0 + cc < ND)
                            asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%1,%1,%1,%1,%1,%1,%1};"
                                         ::"r"(taddr + (c0 + cc) * 32), "r"(z) : "memory");
                    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
                    asm volatile("tcgen05.fence::before_thread_sync;");
                    mbar_arrive(smem_u32(&tempty_bar[c0 >> 2]));
                }
#pragma unroll
                for (int cc = 0; cc < 4; cc++) {
                    const int c = c0 + cc;
                    if (c < ND) {
                        const int gq = (c / 4 < NG - 1) ? c / 4 : NG - 1, sh = 8 * (c - 4 * gq);
#pragma unroll
                        for (int e = 0; e < 8; e++) {
                            const long long x = (long long)(int)v[cc][e];
                            G[gq][e] = sh == 0 ? x : G[gq][e] + x * (1ll << sh);
                        }
                    }
                }
            }
            // tensor memory is drained and zeroed: the next block's instructions run while the rest of the epilogue does
            int inext = i + 1;                                 // the block after this one
            int2 stn = st;
            if (inext < total) next_end(inext, stn);
            // T = sum_g G_g 2^(32 g) (exact, |T| < 2^127), as sign and magnitude
            ull t0[8], t1[8];
            bool tn[8];
#pragma unroll
            for (int e = 0; e < 8; e++) {
                __int128 T = (__int128)G[0][e];
#pragma unroll
                for (int gq = 1; gq < NG; gq++) T += (__int128)G[gq][e] << (32 * gq);
                tn[e] = T < 0;
                const unsigned __int128 M = tn[e] ? (unsigned __int128)(-T) : (unsigned __int128)T;
                t0[e] = (ull)M;
                t1[e] = (ull)(M >> 64);
            }
#pragma unroll
            for (int pp = 0; pp < 2; pp++) {
                const ull ar0 = ar[pp].x, ar1 = ar[pp].y & 0x7fffffffffffffffULL, ai0 = ai[pp].x, ai1 = ai[pp].y & 0x7fffffffffffffffULL;
                const bool arn = (long long)ar[pp].y < 0, ain = (long long)ai[pp].y < 0;
                const ull* T0 = t0 + 4 * pp;
                const ull* T1 = t1 + 4 * pp;
                const bool* TN = tn + 4 * pp;
                constexpr bool HI = ND > 4;
                ull r0, r1, r2;
                // I = Im[conj(A) T] = ar T_im - ai T_re,   R = Re[conj(A) T''] = ar T''_re + ai T''_im   (units 2^(e0) below)
                acc192 I{0, 0, 0}, R{0, 0, 0};
                mul_shr96<HI>(T0[1], T1[1], ar0, ar1, r0, r1, r2); acc_addsub(I, r0, r1, r2, arn != TN[1]);
                mul_shr96<HI>(T0[0], T1[0], ai0, ai1, r0, r1, r2); acc_addsub(I, r0, r1, r2, ain == TN[0]);
                mul_shr96<HI>(T0[2], T1[2], ar0, ar1, r0, r1, r2); acc_addsub(R, r0, r1, r2, arn != TN[2]);
                mul_shr96<HI>(T0[3], T1[3], ai0, ai1, r0, r1, r2); acc_addsub(R, r0, r1, r2, ain != TN[3]);
#pragma unroll
                for (int ax = 0; ax < NI; ax++) {
                    const int wgt = wg[pp][ax];
                    if (wgt != 0) {
                        acc192 v = I;
                        if (wgt < 0) { v = acc192{0, 0, 0}; acc_addsub(v, I.w0, I.w1, I.w2, true); }
                        acc_mac(g[ax], v, (uint32_t)(wgt < 0 ? -wgt : wgt));
                    }
                }
                acc_mac(g[D - 1], R, 1u << qscale_log2);
            }
            nblock++;
            i = inext;
            st = stn;
        }
        if (j < N) {
            constexpr int E0 = 8 * (ND - 1 + 2 * OFF) - 210;      // units of the accumulators: 2^(8 s0 - 204 - 102 + 96)
            double2* o = reinterpret_cast<double2*>(gpart);
            const size_t slot = (size_t)(seg * 4 + quarter) * D;       // four partials per segment (the p quarters)
#pragma unroll
            for (int ax = 0; ax < D; ax++) {
                const dd r = acc192_to_dd(g[ax], E0);
                o[(slot + ax) * N + j] = make_double2(r.h, r.l);
            }
        }
      }
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tb));
}

}  // namespace

cudaError_t shd_grad8_configure()
{
    if (getenv("SHD_DEBUG")) {
        cudaFuncAttributes a;
        cudaFuncGetAttributes(&a, k_grad8<13, 2>);
        fprintf(stderr, "k_grad8<13, 2>: regs %d maxThreadsPerBlock %d static smem %zu local %zu\n", a.numRegs, a.maxThreadsPerBlock, a.sharedSizeBytes, a.localSizeBytes);
    }
    cudaError_t e = cudaSuccess;
#define CONF_GRAD8(NDV)                                                                                                       \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_grad8<NDV, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, G8_SMEM);    \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_grad8<NDV, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, G8_SMEM);    \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_grad8<NDV, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, G8_SMEM);    \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_grad8<NDV, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, G8_SMEM);
    CONF_GRAD8(13)
    CONF_GRAD8(7)
    CONF_GRAD8(4)
#undef CONF_GRAD8
    return e;
}

// k_gradsum (k_grad.cu) adds the segments' partial gradients and applies 4 pi / L / cscale; nc = particles of the chunk
cudaError_t shd_launch_grad8_main(shd_ctx* h, long nc)
{
    const long njb = (nc + 127) / 128, nunits = njb * h->nseg8;
    const unsigned grid = (unsigned)std::min<long>(nunits, h->sms);        // persistent: one CTA per SM
#define LAUNCH_GRAD8_(NDV, DV)                                                                       \
    k_grad8<NDV, DV><<<grid, G8_THREADS, G8_SMEM, h->stream>>>(                                              \
        h->d, nc, h->Npad, h->njb128, h->npb * 32, h->qscale_log2, h->nkq8,                            \
        reinterpret_cast<const int2*>(h->d_steps8), h->nsteps8, h->nseg8, h->d_wT,                     \
        reinterpret_cast<const ulonglong2*>(h->d_Afix), h->d_Bg8, h->d_W8, h->d_gpart, nunits, h->d_scal->clk + 2, h->d_skip)
#define LAUNCH_GRAD8(NDV)                                                                            \
    do {                                                                                             \
        if (h->d == 1) LAUNCH_GRAD8_(NDV, 1);                                                        \
        else if (h->d == 2) LAUNCH_GRAD8_(NDV, 2);                                                   \
        else if (h->d == 3) LAUNCH_GRAD8_(NDV, 3);                                                   \
        else LAUNCH_GRAD8_(NDV, 4);                                                                  \
    } while (0)
    if (h->nlimb >= 3) LAUNCH_GRAD8(13);
    else if (h->nlimb == 2) LAUNCH_GRAD8(7);
    else LAUNCH_GRAD8(4);
#undef LAUNCH_GRAD8
#undef LAUNCH_GRAD8_
    h->last_launches += 1;
    return cudaGetLastError();
}
