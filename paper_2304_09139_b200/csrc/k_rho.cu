// k_rho.cu -- step a2: rho(+/-)[p,q] = sum_j A_j[p] B_j[q]^(+/-)   (Eq. 4, conjugated D:R1).
//
// One CTA owns a 32 x 32 tile of (p,q) cells and a contiguous range of particles.  Each of its 8
// warps owns 8 p x 16 q cells (two 8x8 blocks) and accumulates, per block, the four real bilinear sums
//   X1 = sum ar br, X2 = sum ai bi, X3 = sum ar bi, X4 = sum ai br
// from which rho+ = (X1 - X2) + i (X3 + X4) and rho- = (X1 + X2) + i (X4 - X3): both signs of
// the last axis come out of the same four sums (12 FP64 FMAs per particle-wavevector pair).
// The FMAs are FP64 matrix instructions (DMMA.8x8x4, k = 4 particles) on the limb planes of the
// operands (shd_internal.h): 6 per real sum, 48 per warp and k-step.
// Operand slabs (8 particles x 32 entries x 48 B for A and for B) are streamed from the
// fragment-major tables by TMA bulk copies (cp.async.bulk + full/empty mbarriers), issued by a ninth
// (producer) warp, through a 6-stage ring; no block-wide barrier in the main loop.
// Every 128 particles the exact limb accumulators are folded into double-double sums (TwoSum) kept
// in thread-private shared-memory slots.
// No atomics: each (tile, split) writes its own partial, summed in fixed order by k_finish.
#include "pipe.cuh"
#include "shd_internal.h"

namespace {

constexpr int NW = 8;                                        // warps per CTA
constexpr int GROUP_BYTES = SHD_GROUP_DOUBLES * 8;           // 6144
constexpr int PLANE_BYTES = 32 * 4 * 16;                     // 2048: one limb plane of a group
constexpr int SLAB_BYTES = (SHD_NPS / 4) * GROUP_BYTES;      // one table, one stage
constexpr int STAGE_BYTES = 2 * SLAB_BYTES;                  // A slab + B slab
constexpr int RING_BYTES = SHD_RHO_STAGES * STAGE_BYTES;
constexpr int MAIN_BYTES = 16 * 256 * 16;                    // 16 dd sums per thread
constexpr int RHO_SMEM = RING_BYTES + MAIN_BYTES;
constexpr int KSTEPS_PER_BURST = SHD_BURST / 4;

// NL = 3: three limbs (double-double accuracy).  NL = 2: the "fast" precision of shd_set_precision(h, 2):
// limbs x0, x1 only (L0 and L1, both exact), i.e. operands rounded to 44 bits, half the FMAs; error ~2^-45
// per term instead of ~2^-98.  NL = 1: limb x0 only (22-bit operands, one sixth of the FMAs, error ~2^-23
// per term) for the first decades of a quench ("tunable precision").
template <int NL>
__global__ void __launch_bounds__(NW * 32 + 128, 1) k_rho(
    const double* __restrict__ A, const double* __restrict__ B,
    const int* __restrict__ tile_pb, const int* __restrict__ tile_qb, const int* __restrict__ tile_wmap, int ntiles,
    long Npad, long chunks_per_split, double* __restrict__ part, const int* __restrict__ skip)
{
    if (skip && *skip) return;
    extern __shared__ __align__(1024) unsigned char smem[];
    __shared__ __align__(8) unsigned long long full_bar[SHD_RHO_STAGES], empty_bar[SHD_RHO_STAGES];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int tile = blockIdx.x % ntiles;
    const long split = blockIdx.x / ntiles;
    const int pb = tile_pb[tile], qb = tile_qb[tile];
    // unit (8 p x 16 q) of this consumer warp: 2 (p strip) + (q half), or -1 when the tile has fewer valid
    // units than warps (tiles on the circle boundary; with <= 4 valid units they sit on warps 0..3, one
    // per scheduler, and the CTA runs its FMAs in about half the time); byte 8 = number of active warps
    const int unit = warp < NW ? tile_wmap[tile * 9 + warp] : -1;
    const int nactive = tile_wmap[tile * 9 + 8];
    const long g0 = split * chunks_per_split * (SHD_NPS / 4);          // first group of 4 particles
    const double* gA = A + ((size_t)pb * (Npad / 4) + g0) * SHD_GROUP_DOUBLES;
    const double* gB = B + ((size_t)qb * (Npad / 4) + g0) * SHD_GROUP_DOUBLES;
    const uint32_t s0 = smem_u32(smem);
    const int nchunks = (int)chunks_per_split;
    double2* mainacc = reinterpret_cast<double2*>(smem + RING_BYTES);   // [16][256]

    if (tid == 0) {
        for (int s = 0; s < SHD_RHO_STAGES; s++) {
            mbar_init(smem_u32(&full_bar[s]), 1);
            mbar_init(smem_u32(&empty_bar[s]), nactive);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp < NW) {
#pragma unroll
        for (int a = 0; a < 16; a++) mainacc[a * 256 + tid] = make_double2(0.0, 0.0);
    }
    __syncthreads();
    if (warp >= NW) {
        // producer warpgroup: hands its registers to the consumers (setmaxnreg), then one lane streams.
        asm volatile("setmaxnreg.dec.sync.aligned.u32 24;");
        // producer warp (one lane): it does nothing else, so a stage is refilled the moment the last
        // consumer warp releases it
        if (warp == NW && lane == 0)
            for (int chunk = 0; chunk < nchunks; chunk++) {
                const int s = chunk % SHD_RHO_STAGES;
                if (chunk >= SHD_RHO_STAGES)
                    mbar_wait(smem_u32(&empty_bar[s]), (uint32_t)((chunk / SHD_RHO_STAGES - 1) & 1));
                const uint32_t bar = smem_u32(&full_bar[s]);
                const size_t off = (size_t)chunk * (SHD_NPS / 4) * SHD_GROUP_DOUBLES;
                mbar_expect_tx(bar, STAGE_BYTES);
                tma_load_1d(s0 + s * STAGE_BYTES, gA + off, SLAB_BYTES, bar);
                tma_load_1d(s0 + s * STAGE_BYTES + SLAB_BYTES, gB + off, SLAB_BYTES, bar);
            }
        return;
    }
    asm volatile("setmaxnreg.inc.sync.aligned.u32 232;");
    if (unit < 0) return;            // no valid cell in this warp's unit (no block-wide barrier follows)

    // warp tile: p_local = 8 (unit / 2) + g, q_local = 16 (unit % 2) + 8 t + {2 tq, 2 tq + 1}
    const uint32_t fragoff = (uint32_t)(lane >> 2) * 64 + (uint32_t)(lane & 3) * 16;
    const uint32_t offA = (uint32_t)(unit >> 1) * 8 * 64 + fragoff;
    const uint32_t offB = SLAB_BYTES + (uint32_t)(unit & 1) * 16 * 64 + fragoff;

    Acc3 acc[2][4];
#pragma unroll
    for (int t = 0; t < 2; t++)
#pragma unroll
        for (int x = 0; x < 4; x++) acc3_zero(acc[t][x]);

    // k-steps (groups of 4 particles) run through a software pipeline: every LDS is issued at least one
    // round of 8 DMMAs ahead of its first use and the limb-0 fragments of the next k-step are loaded
    // under the last round (the DMMAs and the LDS are volatile: the order below is the schedule).
#define ROUND(LV, Ax, Bx)                                                   \
    _Pragma("unroll") for (int t = 0; t < 2; t++) {                         \
        dmma_v(acc[t][0].LV, Ax.r, Bx[t].r);                                \
        dmma_v(acc[t][1].LV, Ax.i, Bx[t].i);                                \
        dmma_v(acc[t][2].LV, Ax.r, Bx[t].i);                                \
        dmma_v(acc[t][3].LV, Ax.i, Bx[t].r);                                \
    }
    constexpr int GPS = SHD_NPS / 4;                 // groups (k-steps) per stage
    const int nk = nchunks * GPS;
    F2 a0, b0[2];
    if (nk > 0) {
        mbar_wait(smem_u32(&full_bar[0]), 0u);
        a0 = lds2(s0 + offA);
#pragma unroll
        for (int t = 0; t < 2; t++) b0[t] = lds2(s0 + offB + t * 8 * 64);
    }
    constexpr bool FULL = NL >= 3, TWO = NL >= 2;
    for (int k = 0; k < nk; k++) {
        const int c = k / GPS, g = k % GPS, s = c % SHD_RHO_STAGES;
        const uint32_t pA = s0 + s * STAGE_BYTES + g * GROUP_BYTES + offA;
        const uint32_t pB = s0 + s * STAGE_BYTES + g * GROUP_BYTES + offB;
        F2 a1{0.0, 0.0}, a2{0.0, 0.0}, a12{0.0, 0.0};
        if (TWO) a1 = lds2(pA + PLANE_BYTES);
        if (FULL) a2 = lds2(pA + 2 * PLANE_BYTES);
        ROUND(l0, a0, b0)
        F2 b1[2] = {{0.0, 0.0}, {0.0, 0.0}}, b2[2] = {{0.0, 0.0}, {0.0, 0.0}};
        if (TWO) {
#pragma unroll
            for (int t = 0; t < 2; t++) b1[t] = lds2(pB + t * 8 * 64 + PLANE_BYTES);
            ROUND(l1, a1, b0)
        }
        if (FULL) {
#pragma unroll
            for (int t = 0; t < 2; t++) b2[t] = lds2(pB + t * 8 * 64 + 2 * PLANE_BYTES);
            ROUND(l2, a2, b0)
            a12 = add2(a1, a2);
        }
        if (TWO) { ROUND(l1, a0, b1) }
        if (FULL) { ROUND(l2, a0, b2) }
        if (g == GPS - 1) {
            // every LDS of stage s has been consumed by an issued DMMA: release the stage
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(&empty_bar[s]));
        }
        F2 bs[2] = {{0.0, 0.0}, {0.0, 0.0}};
        if (FULL) {
#pragma unroll
            for (int t = 0; t < 2; t++) bs[t] = add2(b1[t], b2[t]);
        }
        if (k + 1 < nk) {
            const int cn = (k + 1) / GPS, gn = (k + 1) % GPS, sn = cn % SHD_RHO_STAGES;
            if (gn == 0) mbar_wait(smem_u32(&full_bar[sn]), (uint32_t)((cn / SHD_RHO_STAGES) & 1));
            const uint32_t nb = s0 + sn * STAGE_BYTES + gn * GROUP_BYTES;
            a0 = lds2(nb + offA);
#pragma unroll
            for (int t = 0; t < 2; t++) b0[t] = lds2(nb + offB + t * 8 * 64);
        }
        if (FULL) { ROUND(l2, a12, bs) }
        if ((k + 1) % KSTEPS_PER_BURST == 0 || k == nk - 1) {
#pragma unroll
            for (int t = 0; t < 2; t++)
#pragma unroll
                for (int x = 0; x < 4; x++) {
                    Acc3& r = acc[t][x];
                    double2* s0p = &mainacc[((t * 4 + x) * 2 + 0) * 256 + tid];
                    double2* s1p = &mainacc[((t * 4 + x) * 2 + 1) * 256 + tid];
                    double2 m0 = *s0p, m1 = *s1p;
                    fold_burst(r.l0.c0, r.l1.c0, r.l2.c0, m0);
                    fold_burst(r.l0.c1, r.l1.c1, r.l2.c1, m1);
                    *s0p = m0; *s1p = m1;
                    acc3_zero(r);
                }
        }
    }
#undef ROUND

    // partial sums: part[((split*ntiles + tile)*4 + x)*1024 + cell] as (hi, lo)
    double2* out = reinterpret_cast<double2*>(part) + ((size_t)(split * ntiles + tile) * 4) * 1024;
    const int pl = (unit >> 1) * 8 + (lane >> 2);
#pragma unroll
    for (int t = 0; t < 2; t++)
#pragma unroll
        for (int x = 0; x < 4; x++)
#pragma unroll
            for (int e = 0; e < 2; e++) {
                const int ql = (unit & 1) * 16 + t * 8 + (lane & 3) * 2 + e;
                double2 m = mainacc[((t * 4 + x) * 2 + e) * 256 + tid];
                dd r = fast_two_sum(m.x, m.y);
                out[(size_t)x * 1024 + pl * 32 + ql] = make_double2(r.h, r.l);
            }
}

}  // namespace

cudaError_t shd_rho_configure()
{
    cudaError_t e = cudaFuncSetAttribute(k_rho<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, RHO_SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_rho<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, RHO_SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_rho<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, RHO_SMEM);
    return e;
}

cudaError_t shd_launch_rho(shd_ctx* h, int nsplits)
{
    if (h->rho_engine >= 1) return shd_launch_rho8(h, nsplits);      // INT8 tensor-core engine (k_rho8.cu)
    unsigned grid = (unsigned)(h->ntiles * nsplits);        // the splits of one chunk
#define LAUNCH_RHO(NLV)                                                                                   \
    k_rho<NLV><<<grid, NW * 32 + 128, RHO_SMEM, h->stream>>>(h->d_A, h->d_B, h->d_tile_pb, h->d_tile_qb,    \
        h->d_tile_wmap, h->ntiles, h->Npad, h->chunks_per_split, h->d_part, h->d_skip)
    if (h->nlimb >= 3) LAUNCH_RHO(3);
    else if (h->nlimb == 2) LAUNCH_RHO(2);
    else LAUNCH_RHO(1);
#undef LAUNCH_RHO
    h->last_launches += 1;
    return cudaGetLastError();
}
