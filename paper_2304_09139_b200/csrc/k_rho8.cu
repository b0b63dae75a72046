// k_rho8.cu -- step a2 on the INT8 tensor cores: rho(+/-)[p,q] = sum_j A_j[p] B_j[q]^(+/-) (Eq. 4) as an
// EXACT integer contraction.
//
// Every real operand x (|x| <= 1) is the 13-digit balanced base-256 integer X = trunc(x 2^102) = sum_i d_i 256^i,
// d_i in [-128, 127] (k_tables writes the digits as s8, K-major over particles, in the shared-memory layout of
// the tensor core).  sum_j x_j y_j = 2^-204 sum_s 256^s S_s,  S_s = sum_{i+l=s} sum_j d_i(j) e_l(j);  the sums
// with s >= 12 are kept (91 digit pairs; the rest is below 2^-98 per product, the accuracy of the third FP64
// limb).  Each S_s is an s32 accumulator in TENSOR MEMORY: |S_s| <= 13 * 8192 * 2^14 < 2^31 for at most 8192
// particles per CTA, so the integer arithmetic is exact.
//
// One CTA owns 64 p x 16 q cells and a range of particles.  Rows of the M = 128 side are (p, re/im); the N
// side holds (digit l, q, re/im) with the digits ascending, so ONE tcgen05.mma.kind::i8 per A digit i
// multiplies it with all its partners l = 12-i .. 12 and lands every pair in the TMEM columns of its digit sum:
// column 32 (i + l - 12) + (q, re/im).  18 instructions (N = 32 .. 256) per 32 particles cover the 91 pairs
// and all four real products of the complex multiply.  13 x 32 = 416 of the 512 TMEM columns are used.
// Warp 4: TMA producer (cp.async.bulk, 65 KB per stage, 3 stages; 5 / 8 stages with 7 / 4 digits).  Warp 5: MMA issuer (one thread);
// tcgen05.commit releases a stage when the tensor core has read it.  Warps 0-3: epilogue: tcgen05.ld, the 13
// integer sums of every cell scaled by exact powers of two and added in double-double, partials written in
// the layout k_finish1 sums over the particle splits.
#include "pipe.cuh"
#include "shd_internal.h"

namespace {

constexpr int R8_ND = SHD_I8_DIGITS;                 // 13
constexpr int R8_ASLAB = 128 * 32;                   // one A digit of one stage: 128 rows x 32 particles
constexpr int R8_BSLAB = 32 * 32;                    // one B digit: 32 rows (16 q x re/im) x 32 particles
constexpr int R8_A = R8_ND * R8_ASLAB;               // 53248
constexpr int R8_B = R8_ND * R8_BSLAB;               // 13312
constexpr int R8_STAGE = R8_A + R8_B;                // 66560
constexpr int R8_NST = 3;
constexpr int R8_SMEM = R8_NST * R8_STAGE;

__device__ __forceinline__ uint64_t umma_desc(uint32_t addr) {      // K-major, no swizzle: LBO 128 B, SBO 256 B
    return (uint64_t)((addr >> 4) & 0x3FFF) | ((uint64_t)(128 >> 4) << 16) | ((uint64_t)(256 >> 4) << 32) | ((uint64_t)1 << 46);
}
__device__ __forceinline__ uint32_t umma_idesc_i8(int n) {          // D = s32, A = B = s8, M = 128
    return (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
}
// issued by the elected lane of a converged warp (elected = 1 in one lane): the whole warp runs the issue loop, so
// the descriptors stay in uniform registers and there is no per-instruction election loop (k_grad8.cu)
__device__ __forceinline__ void umma_i8(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate, uint32_t elected) {
    uint32_t z = 0;
    asm volatile("{\n\t.reg .pred p, q;\n\tsetp.ne.b32 p, %4, 0;\n\tsetp.ne.b32 q, %6, 0;\n\t"
                 "@q tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, {%5, %5, %5, %5}, p;\n\t}"
                 ::"r"(tmem_d), "l"(da), "l"(db), "r"(idesc), "r"(accumulate), "r"(z), "r"(elected) : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar, uint32_t elected) {
    asm volatile("{\n\t.reg .pred q;\n\tsetp.ne.b32 q, %1, 0;\n\t"
                 "@q tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n\t}" ::"r"(bar), "r"(elected) : "memory");
}

// ND = 13: full precision.  ND = 7 / 4: the "fast" precisions of shd_set_precision(h, 2 / 1) on this engine: only the
// ND most significant digits of both operands (54 / 30 bits) and the digit pairs with i' + l' >= ND - 1
// (28 / 10 instead of 91), in 32 ND tensor-memory columns.
template <int ND>
__global__ void __launch_bounds__(192, 1) k_rho8(
    const signed char* __restrict__ A8, const signed char* __restrict__ B8,
    const int* __restrict__ tile_pb, const int* __restrict__ tile_qb, int ntiles,
    long nk_total, int ksteps_per_split, double* __restrict__ part, long long* __restrict__ clk, const int* __restrict__ skip)
{
    if (skip && *skip) return;
    extern __shared__ __align__(1024) unsigned char smem[];
    // a stage holds the ND digit slabs in use of both operands; the fewer digits, the deeper the ring
    constexpr int STG = ND * (R8_ASLAB + R8_BSLAB), NST = R8_SMEM / STG < 8 ? R8_SMEM / STG : 8;
    __shared__ __align__(8) unsigned long long full_bar[8], empty_bar[8], done_bar;
    __shared__ uint32_t tmem_base;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int tile = blockIdx.x % ntiles;
    const long split = blockIdx.x / ntiles;
    const int pb = tile_pb[tile], qb = tile_qb[tile];
    const long k0 = split * ksteps_per_split;
    const int nk = ksteps_per_split;
    const uint32_t s0 = smem_u32(smem);
    if (tid == 0) {
        for (int s = 0; s < NST; s++) { mbar_init(smem_u32(&full_bar[s]), 1); mbar_init(smem_u32(&empty_bar[s]), 1); }
        mbar_init(smem_u32(&done_bar), 1);
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
    constexpr int OFF = R8_ND - ND;                  // first (least significant) digit used

    if (warp == 4) {
        if (lane == 0) {
            const signed char* gA = A8 + ((size_t)pb * nk_total + k0) * R8_A;
            const signed char* gB = B8 + ((size_t)qb * nk_total + k0) * R8_B;
            gA += OFF * R8_ASLAB;
            gB += OFF * R8_BSLAB;
            for (int i0 = 0; i0 < nk; i0 += NST) {                 // unrolled over the ring positions (as below)
                const uint32_t par = (uint32_t)((i0 / NST - 1) & 1);
#pragma unroll
              for (int s = 0; s < NST; s++) {
                if (i0 + s >= nk) break;
                if (i0 > 0) mbar_wait(smem_u32(&empty_bar[s]), par);
                const uint32_t bar = smem_u32(&full_bar[s]);
                mbar_expect_tx(bar, ND * (R8_ASLAB + R8_BSLAB));
                tma_load_1d(s0 + s * STG, gA, ND * R8_ASLAB, bar);
                tma_load_1d(s0 + s * STG + ND * R8_ASLAB, gB, ND * R8_BSLAB, bar);
                gA += R8_A;
                gB += R8_B;
              }
            }
        }
    } else if (warp == 5) {
        {
            uint32_t elected;
            asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(elected));
            // the ring position is a compile-time constant inside the unrolled inner loop: shared-memory addresses
            // and descriptors of a step are constants off one base, the step boundary costs a few instructions
            unsigned long long g0 = 0;
            long long c0 = 0;
            if (blockIdx.x == 0 && clk) { asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g0)); c0 = clock64(); }
            const uint64_t dbase = umma_desc(s0);
            for (int i0 = 0; i0 < nk; i0 += NST) {
                const uint32_t par = (uint32_t)((i0 / NST) & 1);
#pragma unroll
              for (int s = 0; s < NST; s++) {
                const int i = i0 + s;
                if (i >= nk) break;
                mbar_wait(smem_u32(&full_bar[s]), par);
                asm volatile("tcgen05.fence::after_thread_sync;");
                // the most significant A digit first: its partners are all ND B digits = all 32 ND columns, so on the
                // first K-step it initialises every accumulator (accumulate = 0), everything else accumulates.
                // Descriptors differ only in the 14-bit address field: one base per operand, compile-time offsets.
                const uint64_t dA0 = dbase + (uint64_t)((s * STG) >> 4), dB0 = dA0 + (uint64_t)((ND * R8_ASLAB) >> 4);
                // Order inside a K-step: ascending digits, i.e. the short instructions (N = 32, 64, ...) first and the
                // long ones last, so that the tensor core's queue holds long instructions while this thread crosses
                // the step boundary (commit, barrier wait, descriptors): 4 % at 13 digits.  The very first step runs
                // descending: its first instruction covers all columns and initialises them.
                auto issue = [&](int ii, uint32_t acc) {            // relative digit i' (absolute OFF + i')
                    const int n = (ii + 1) * 32, l0 = ND - 1 - ii;          // its partners: relative digits l0 .. ND - 1
                    const uint64_t da = dA0 + (uint64_t)((ii * R8_ASLAB) >> 4);
                    if (n <= 256) {
                        umma_i8(tb, da, dB0 + (uint64_t)((l0 * R8_BSLAB) >> 4), umma_idesc_i8(n), acc, elected);
                    } else {
                        // two instructions of n / 2 columns each, not 256 + the rest: an instruction reads its 4 KB A
                        // slab and 32 n bytes of the other operand from shared memory, about 32 + n / 4 cycles, against
                        // n / 2 cycles of arithmetic, so below n = 128 the operand fetch is what it costs (measured:
                        // the 256 + rest split is 2.5 % slower in k_grad8, 1 % in k_rho8; profiles/r2b_summary.md)
                        const int n1 = n / 2;                                  // 144 .. 208: a multiple of 16
                        umma_i8(tb, da, dB0 + (uint64_t)((l0 * R8_BSLAB) >> 4), umma_idesc_i8(n1), acc, elected);
                        umma_i8(tb + n1, da, dB0 + (uint64_t)((l0 * R8_BSLAB + n1 * 32) >> 4), umma_idesc_i8(n - n1), acc, elected);
                    }
                };
                if (i == 0 || ND < R8_ND) {                         // (with fewer digits the order makes no difference)
#pragma unroll
                    for (int ii = ND - 1; ii >= 0; ii--) issue(ii, (i > 0 || ii < ND - 1) ? 1u : 0u);
                } else {
#pragma unroll
                    for (int ii = 0; ii < ND; ii++) issue(ii, 1u);
                }
                umma_commit(smem_u32(&empty_bar[s]), elected); // arrives when the tensor core is done with stage s
              }
            }
            umma_commit(smem_u32(&done_bar), elected);
            if (blockIdx.x == 0 && clk && elected) {
                unsigned long long g1;
                asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
                clk[0] = clock64() - c0;
                clk[1] = (long long)(g1 - g0);
            }
        }
    } else {
        // ---- epilogue warps 0..3: warp w reads TMEM lanes 32 w .. 32 w + 31 (rows r = 2 p_local + c)
        mbar_wait(smem_u32(&done_bar), 0u);
        asm volatile("tcgen05.fence::after_thread_sync;");
        const int r = tid, pl = r >> 1, c = r & 1;
        double2* out = reinterpret_cast<double2*>(part) + ((size_t)(split * ntiles + tile) * 4) * 1024;
        for (int c0 = 0; c0 < 32; c0 += 8) {
            dd sum[8];
#pragma unroll
            for (int e = 0; e < 8; e++) sum[e] = dd{0.0, 0.0};
#pragma unroll
            for (int sidx = 0; sidx < ND; sidx++) {             // absolute digit sum s = ND - 1 + 2 OFF + sidx, weight 2^(8 s - 204)
                uint32_t v[8];
                asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                             : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
                             : "r"(tb + ((uint32_t)(warp * 32) << 16) + sidx * 32 + c0));
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                const double w = __longlong_as_double((long long)(1023 + 8 * (ND - 1 + 2 * OFF + sidx) - 204) << 52);
#pragma unroll
                for (int e = 0; e < 8; e++) sum[e] = dd_add_d(sum[e], __dmul_rn((double)(int)v[e], w));
            }
#pragma unroll
            for (int e = 0; e < 8; e++) {
                const int col = c0 + e, ql = col >> 1, cp = col & 1;
                const int x = c == 0 ? (cp == 0 ? 0 : 2) : (cp == 0 ? 3 : 1);   // X1 ar br, X2 ai bi, X3 ar bi, X4 ai br
                out[(size_t)x * 1024 + pl * 16 + ql] = make_double2(sum[e].h, sum[e].l);
            }
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tb));
}

}  // namespace

cudaError_t shd_rho8_configure()
{
    cudaError_t e = cudaFuncSetAttribute(k_rho8<13>, cudaFuncAttributeMaxDynamicSharedMemorySize, R8_SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_rho8<7>, cudaFuncAttributeMaxDynamicSharedMemorySize, R8_SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_rho8<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, R8_SMEM);
    return e;
}

cudaError_t shd_launch_rho8(shd_ctx* h, int nsplits)
{
    const unsigned grid = (unsigned)(h->ntiles8 * nsplits);      // the splits of one chunk
#define LAUNCH_RHO8(NDV)                                                                              \
    k_rho8<NDV><<<grid, 192, R8_SMEM, h->stream>>>(h->d_A8, h->d_B8, h->d_tile8_pb, h->d_tile8_qb, h->ntiles8, \
                                                   h->nk8, h->ksteps8, h->d_part, h->d_scal->clk, h->d_skip)
    if (h->nlimb >= 3) LAUNCH_RHO8(13);
    else if (h->nlimb == 2) LAUNCH_RHO8(7);
    else LAUNCH_RHO8(4);
#undef LAUNCH_RHO8
    h->last_launches += 1;
    return cudaGetLastError();
}
