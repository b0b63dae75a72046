// k_rho.cu -- step a2: rho(+/-)[p,q] = sum_j A_j[p] B_j[q]^(+/-)   (Eq. 4, conjugated D:R1).
//
// One CTA owns a 32 x 32 tile of (p,q) cells and a contiguous range of particles; each of its
// 256 threads owns a 2 x 2 micro-tile of cells, i.e. 16 real bilinear accumulators
//   X1 = sum ar br, X2 = sum ai bi, X3 = sum ar bi, X4 = sum ai br
// from which rho+ = (X1 - X2) + i (X3 + X4) and rho- = (X1 + X2) + i (X4 - X3): both signs of
// the last axis come out of the same four sums (12 DFMA per particle-wavevector pair).
// Operand slabs (16 particles x 32 entries x 64 B for A and for B) are streamed from the
// tile-major tables by TMA bulk copies (cp.async.bulk + mbarrier) through a 3-stage ring.
// Every 128 particles the exact limb accumulators are folded into double-double sums (TwoSum).
// No atomics: each (tile, split) writes its own partial, summed in fixed order by k_finish.
#include "dd.cuh"
#include "shd_internal.h"
#include <cstdint>

namespace {

constexpr int TX = 16, TY = 16, U = 2, T = 2;
constexpr int STAGE_BYTES = 2 * SHD_NPS * 2048;            // A slab + B slab
constexpr int SLAB_BYTES = SHD_NPS * 2048;

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

struct Ent { double r0, i0, r1, i1, r2, i2, r12, i12; };
__device__ __forceinline__ Ent lds_ent(uint32_t addr) {   // 4 limb-pair planes, 512 B apart
    Ent e;
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(e.r0), "=d"(e.i0) : "r"(addr));
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(e.r1), "=d"(e.i1) : "r"(addr + 512));
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(e.r2), "=d"(e.i2) : "r"(addr + 1024));
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(e.r12), "=d"(e.i12) : "r"(addr + 1536));
    return e;
}
struct Acc { double l0, l1, l2; };

// fold an exact burst into a (hi, lo) running sum
__device__ __forceinline__ void flush_acc(Acc& a, dd& m) {
    dd s = two_sum(a.l0, a.l1);
    double e = __dadd_rn(s.l, a.l2);
    dd t = two_sum(m.h, s.h);
    m.h = t.h;
    m.l = __dadd_rn(m.l, __dadd_rn(t.l, e));
    a.l0 = 0.0; a.l1 = 0.0; a.l2 = 0.0;
}

__global__ void __launch_bounds__(TX * TY, 1) k_rho(
    const double* __restrict__ A, const double* __restrict__ B,
    const int* __restrict__ tile_pb, const int* __restrict__ tile_qb, int ntiles,
    long Npad, long chunks_per_split, double* __restrict__ part, const int* __restrict__ skip)
{
    if (skip && *skip) return;
    extern __shared__ __align__(1024) unsigned char smem[];
    __shared__ __align__(8) unsigned long long bars[SHD_RHO_STAGES];
    const int tid = threadIdx.x;
    const int tx = tid % TX, ty = tid / TX;
    const int tile = blockIdx.x % ntiles;
    const long split = blockIdx.x / ntiles;
    const int pb = tile_pb[tile], qb = tile_qb[tile];
    const long j0 = split * chunks_per_split * SHD_NPS;
    const double* gA = A + ((size_t)pb * Npad + j0) * SHD_TILE_ENTRY_DOUBLES;
    const double* gB = B + ((size_t)qb * Npad + j0) * SHD_TILE_ENTRY_DOUBLES;
    const uint32_t s0 = smem_u32(smem);
    const int nchunks = (int)chunks_per_split;

    if (tid == 0) {
        for (int s = 0; s < SHD_RHO_STAGES; s++) mbar_init(smem_u32(&bars[s]), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0) {
        for (int s = 0; s < SHD_RHO_STAGES && s < nchunks; s++) {
            uint32_t bar = smem_u32(&bars[s]);
            mbar_expect_tx(bar, STAGE_BYTES);
            tma_load_1d(s0 + s * STAGE_BYTES, gA + (size_t)s * SHD_NPS * SHD_TILE_ENTRY_DOUBLES, SLAB_BYTES, bar);
            tma_load_1d(s0 + s * STAGE_BYTES + SLAB_BYTES, gB + (size_t)s * SHD_NPS * SHD_TILE_ENTRY_DOUBLES, SLAB_BYTES, bar);
        }
    }

    Acc acc[U][T][4];
    dd main_[U][T][4];
#pragma unroll
    for (int u = 0; u < U; u++)
#pragma unroll
        for (int t = 0; t < T; t++)
#pragma unroll
            for (int x = 0; x < 4; x++) {
                acc[u][t][x] = Acc{0.0, 0.0, 0.0};
                main_[u][t][x] = dd{0.0, 0.0};
            }

    const uint32_t offA = (uint32_t)ty * 16;             // p_local = u*TY + ty
    const uint32_t offB = SLAB_BYTES + (uint32_t)tx * 16; // q_local = t*TX + tx

    for (int c = 0; c < nchunks; c++) {
        const int s = c % SHD_RHO_STAGES;
        mbar_wait(smem_u32(&bars[s]), (uint32_t)((c / SHD_RHO_STAGES) & 1));
        const uint32_t sb = s0 + s * STAGE_BYTES;
#pragma unroll 1
        for (int i = 0; i < SHD_NPS; i++) {
            Ent a[U], b[T];
#pragma unroll
            for (int u = 0; u < U; u++) a[u] = lds_ent(sb + offA + i * 2048 + u * (TY * 16));
#pragma unroll
            for (int t = 0; t < T; t++) b[t] = lds_ent(sb + offB + i * 2048 + t * (TX * 16));
#pragma unroll
            for (int u = 0; u < U; u++) {
                // runs of DFMAs that share the A-side operand (register reuse cache), with the
                // three updates of each L2 / two of each L1 spaced two runs apart
#define RUN_A(AL, lvr, BRL, lvi, BIL, XR, XI)                                                   \
    _Pragma("unroll") for (int t = 0; t < T; t++) {                                             \
        acc[u][t][XR].lvr = __fma_rn(AL, b[t].BRL, acc[u][t][XR].lvr);                          \
        acc[u][t][XI].lvi = __fma_rn(AL, b[t].BIL, acc[u][t][XI].lvi);                          \
    }
                RUN_A(a[u].r0, l0, r0, l0, i0, 0, 2)
                RUN_A(a[u].r0, l2, r2, l2, i2, 0, 2)
                RUN_A(a[u].r0, l1, r1, l1, i1, 0, 2)
                RUN_A(a[u].r2, l2, r0, l2, i0, 0, 2)
                RUN_A(a[u].r1, l1, r0, l1, i0, 0, 2)
                RUN_A(a[u].r12, l2, r12, l2, i12, 0, 2)
                RUN_A(a[u].i0, l0, r0, l0, i0, 3, 1)
                RUN_A(a[u].i0, l2, r2, l2, i2, 3, 1)
                RUN_A(a[u].i0, l1, r1, l1, i1, 3, 1)
                RUN_A(a[u].i2, l2, r0, l2, i0, 3, 1)
                RUN_A(a[u].i1, l1, r0, l1, i0, 3, 1)
                RUN_A(a[u].i12, l2, r12, l2, i12, 3, 1)
#undef RUN_A
            }
        }
        if (((c + 1) * SHD_NPS) % SHD_BURST == 0 || c == nchunks - 1) {
#pragma unroll
            for (int u = 0; u < U; u++)
#pragma unroll
                for (int t = 0; t < T; t++)
#pragma unroll
                    for (int x = 0; x < 4; x++) flush_acc(acc[u][t][x], main_[u][t][x]);
        }
        __syncthreads();   // everyone is done reading stage s
        if (tid == 0 && c + SHD_RHO_STAGES < nchunks) {
            uint32_t bar = smem_u32(&bars[s]);
            size_t off = (size_t)(c + SHD_RHO_STAGES) * SHD_NPS * SHD_TILE_ENTRY_DOUBLES;
            mbar_expect_tx(bar, STAGE_BYTES);
            tma_load_1d(sb, gA + off, SLAB_BYTES, bar);
            tma_load_1d(sb + SLAB_BYTES, gB + off, SLAB_BYTES, bar);
        }
    }

    // partial sums: part[((split*ntiles + tile)*4 + x)*1024 + cell] as (hi, lo)
    double2* out = reinterpret_cast<double2*>(part) + ((size_t)(split * ntiles + tile) * 4) * 1024;
#pragma unroll
    for (int u = 0; u < U; u++)
#pragma unroll
        for (int t = 0; t < T; t++) {
            int cell = (u * TY + ty) * 32 + (t * TX + tx);
#pragma unroll
            for (int x = 0; x < 4; x++) {
                dd m = fast_two_sum(main_[u][t][x].h, main_[u][t][x].l);
                out[(size_t)x * 1024 + cell] = make_double2(m.h, m.l);
            }
        }
}

}  // namespace

cudaError_t shd_rho_configure()
{
    return cudaFuncSetAttribute(k_rho, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                SHD_RHO_STAGES * STAGE_BYTES);
}

cudaError_t shd_launch_rho(shd_ctx* h)
{
    unsigned grid = (unsigned)(h->ntiles * h->nsplit);
    k_rho<<<grid, TX * TY, SHD_RHO_STAGES * STAGE_BYTES, h->stream>>>(
        h->d_A, h->d_B, h->d_tile_pb, h->d_tile_qb, h->ntiles, h->Npad, h->chunks_per_split, h->d_part, h->d_skip);
    h->last_launches += 1;
    return cudaGetLastError();
}
