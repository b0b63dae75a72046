// k_grad.cu -- step a4: dPhi/dr_{j,a} = (4 pi / L) sum_k v_k n_a Im[ exp(-i k.r_j) rho(k) ]
// (Eq. 6, sign D:R2) as two contractions over q followed by one over p:
//   T_j[p]   = sum_{q,sigma} W(p,q,sigma) conj(B_j[q]^sigma)          = sum_q ( C1 br + C2 bi )
//   T''_j[p] = -i sum_{q,sigma} sigma q W conj(B^sigma)               = sum_q ( C2 (q br) - C1 (q bi) )
//   grad_a   = (4 pi/L) sum_p ( w_a(p) Im[conj(A_j[p]) T_j[p]] + [a = last axis] Re[conj(A_j[p]) T''_j[p]] )
// with C1 = W+ + W-, C2 = -i (W+ - W-), W = v rho (built by k_ctable), so both signs of the last
// axis share the same products: 24 FP64 FMAs per particle-wavevector pair.
// One CTA owns 32 particles and walks all p-blocks; per p-block it streams the q-groups (4 q) of the
// rho.v operand C (k_ctable output, shared by every CTA, L2 resident) and of the particles' own
// B-table into shared memory with TMA bulk copies (cp.async.bulk + full/empty mbarriers, 6-stage ring,
// no block-wide barrier in the main loop).  Each warp owns 8 particles x 16 p (two 8x8 blocks) and
// issues the FMAs as FP64 matrix instructions (DMMA.8x8x4, k = 4 q) on the limb planes: 96 per warp and
// k-step.  Exact limb bursts (64 q) are folded into double-double sums kept in thread-private
// shared-memory slots; the p-contraction and the reduction over the 8 threads that share a particle
// run in double-double in a fixed order (deterministic, no atomics).
#include "pipe.cuh"
#include "shd_internal.h"

namespace {

constexpr int NW = 8;
constexpr int PLANE_BYTES = 32 * 4 * 16;                     // 2048
constexpr int GSLAB = (SHD_QCH / 4) * SHD_GGROUP_DOUBLES * 8;  // 12288: 6 planes of one q-group
constexpr int GSTAGE = 2 * GSLAB;                            // Bg slab + C slab
constexpr int RING_BYTES = SHD_GRAD_STAGES * GSTAGE;
constexpr int MAIN_BYTES = 16 * 256 * 16;                    // 16 dd accumulators per thread
constexpr int GSMEM = RING_BYTES + MAIN_BYTES;
constexpr int KSTEPS_PER_BURST = SHD_BURST / 8;              // two products per q and accumulator

__device__ __forceinline__ dd limbs_to_dd(double x0, double x1, double x2) {
    return fast_two_sum(__dadd_rn(x0, x1), x2);    // x0 + x1 is exact (46 bits)
}

__global__ void __launch_bounds__(NW * 32, 1) k_grad(
    int d, long N, double L, long Npad, int npb, int Qpad, int Ppad, int qscale_log2,
    const int* __restrict__ qchunks, const int* __restrict__ wT,
    const double* __restrict__ A, const double* __restrict__ Bg, const double* __restrict__ C,
    const shd_scalars* __restrict__ scal, double* __restrict__ grad_hi, double* __restrict__ grad_lo,
    const int* __restrict__ skip)
{
    if (skip && *skip) return;
    extern __shared__ __align__(1024) unsigned char smem[];
    __shared__ __align__(8) unsigned long long full_bar[SHD_GRAD_STAGES], empty_bar[SHD_GRAD_STAGES];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const long jb = blockIdx.x;
    const uint32_t s0 = smem_u32(smem);
    double2* mainacc = reinterpret_cast<double2*>(smem + RING_BYTES);   // [16][256]

    int total = 0;
    for (int pb = 0; pb < npb; pb++) total += qchunks[pb];

    if (tid == 0) {
        for (int s = 0; s < SHD_GRAD_STAGES; s++) {
            mbar_init(smem_u32(&full_bar[s]), 1);
            mbar_init(smem_u32(&empty_bar[s]), NW);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
#pragma unroll
    for (int a = 0; a < 16; a++) mainacc[a * 256 + tid] = make_double2(0.0, 0.0);
    __syncthreads();

    // producer cursor (thread 0 only)
    int lpb = 0, lqc = 0, issued = 0;
    auto issue = [&]() {
        const int stage = issued % SHD_GRAD_STAGES;
        const uint32_t bar = smem_u32(&full_bar[stage]);
        mbar_expect_tx(bar, GSTAGE);
        const double* srcB = Bg + ((size_t)jb * (Qpad / 4) + (size_t)lqc * (SHD_QCH / 4)) * SHD_GGROUP_DOUBLES;
        const double* srcC = C + ((size_t)lpb * (Qpad / 4) + (size_t)lqc * (SHD_QCH / 4)) * SHD_GGROUP_DOUBLES;
        tma_load_1d(s0 + stage * GSTAGE, srcB, GSLAB, bar);
        tma_load_1d(s0 + stage * GSTAGE + GSLAB, srcC, GSLAB, bar);
        issued++;
        if (++lqc == qchunks[lpb]) { lqc = 0; lpb++; }
    };
    if (tid == 0)
        while (issued < SHD_GRAD_STAGES && issued < total) issue();

    // warp tile: j_local = 8 (warp % 4) + g,  p_local = 16 (warp / 4) + 8 t + {2 tq, 2 tq + 1}
    const int jb8 = warp & 3, ph = warp >> 2;
    const uint32_t fragoff = (uint32_t)(lane >> 2) * 64 + (uint32_t)(lane & 3) * 16;
    const uint32_t offB = (uint32_t)jb8 * 8 * 64 + fragoff;
    const uint32_t offC = GSLAB + (uint32_t)ph * 16 * 64 + fragoff;
    const double qs = ldexp(1.0, qscale_log2);
    const int jl = jb8 * 8 + (lane >> 2);
    const long j = jb * 32 + jl;

    Acc3 acc[2][4];
#pragma unroll
    for (int t = 0; t < 2; t++)
#pragma unroll
        for (int x = 0; x < 4; x++) acc3_zero(acc[t][x]);
    dd g0{0.0, 0.0}, g1{0.0, 0.0}, g2{0.0, 0.0};

    int c = 0;
    for (int pb = 0; pb < npb; pb++) {
        const int nqc = qchunks[pb];
        for (int qc = 0; qc < nqc; qc++, c++) {
            const int s = c % SHD_GRAD_STAGES;
            mbar_wait(smem_u32(&full_bar[s]), (uint32_t)((c / SHD_GRAD_STAGES) & 1));
            const uint32_t sb = s0 + s * GSTAGE;
#pragma unroll
            for (int gq = 0; gq < SHD_QCH / 4; gq++) {
                const uint32_t gb = sb + gq * (SHD_GGROUP_DOUBLES * 8);
                const LimbFrag b = lds_frag(gb + offB, PLANE_BYTES);                    // (br, bi)
                LimbFrag w = lds_frag(gb + offB + 3 * PLANE_BYTES, PLANE_BYTES);        // (q br, q bi)
                w.i0 = -w.i0; w.i1 = -w.i1; w.i2 = -w.i2; w.i12 = -w.i12;               // T'' -= C1 (q bi)
                LimbFrag c1[2], c2[2];
#pragma unroll
                for (int t = 0; t < 2; t++) {
                    c1[t] = lds_frag(gb + offC + t * 8 * 64, PLANE_BYTES);
                    c2[t] = lds_frag(gb + offC + t * 8 * 64 + 3 * PLANE_BYTES, PLANE_BYTES);
                }
                // six rounds of 16 DMMAs; the two products of one accumulator are 8 DMMAs apart
#define GROUND(LV, AL, BL)                                                  \
    _Pragma("unroll") for (int t = 0; t < 2; t++) {                         \
        dmma(acc[t][0].LV, b.r##AL, c1[t].r##BL);                           \
        dmma(acc[t][1].LV, b.r##AL, c1[t].i##BL);                           \
        dmma(acc[t][2].LV, w.r##AL, c2[t].r##BL);                           \
        dmma(acc[t][3].LV, w.r##AL, c2[t].i##BL);                           \
    }                                                                       \
    _Pragma("unroll") for (int t = 0; t < 2; t++) {                         \
        dmma(acc[t][0].LV, b.i##AL, c2[t].r##BL);                           \
        dmma(acc[t][1].LV, b.i##AL, c2[t].i##BL);                           \
        dmma(acc[t][2].LV, w.i##AL, c1[t].r##BL);                           \
        dmma(acc[t][3].LV, w.i##AL, c1[t].i##BL);                           \
    }
                GROUND(l0, 0, 0)
                GROUND(l2, 0, 2)
                GROUND(l1, 0, 1)
                GROUND(l2, 2, 0)
                GROUND(l1, 1, 0)
                GROUND(l2, 12, 12)
#undef GROUND
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(&empty_bar[s]));
            const bool last = (qc == nqc - 1);
            if (((qc + 1) * (SHD_QCH / 4)) % KSTEPS_PER_BURST == 0 || last) {
                // fold the exact burst into the dd sums (shared memory, thread-private slots)
#pragma unroll
                for (int t = 0; t < 2; t++)
#pragma unroll
                    for (int x = 0; x < 4; x++) {
                        Acc3& r = acc[t][x];
                        double2* p0 = &mainacc[((t * 4 + x) * 2 + 0) * 256 + tid];
                        double2* p1 = &mainacc[((t * 4 + x) * 2 + 1) * 256 + tid];
                        double2 m0 = *p0, m1 = *p1;
                        fold_burst(r.l0.c0, r.l1.c0, r.l2.c0, m0);
                        fold_burst(r.l0.c1, r.l1.c1, r.l2.c1, m1);
                        *p0 = m0; *p1 = m1;
                        acc3_zero(r);
                    }
            }
            if (last) {
                // p-contraction for this p-block
#pragma unroll
                for (int t = 0; t < 2; t++)
#pragma unroll
                    for (int e = 0; e < 2; e++) {
                        const int pl = ph * 16 + t * 8 + (lane & 3) * 2 + e;
                        const int p = pb * 32 + pl;
                        dd T[4];
#pragma unroll
                        for (int x = 0; x < 4; x++) {
                            double2* slot = &mainacc[((t * 4 + x) * 2 + e) * 256 + tid];
                            double2 m = *slot;
                            T[x] = fast_two_sum(m.x, m.y);
                            *slot = make_double2(0.0, 0.0);
                        }
                        if (j < N) {
                            const double2* ap = reinterpret_cast<const double2*>(A) +
                                                ((((size_t)pb * (Npad / 4) + (j >> 2)) * 3) * 32 + pl) * 4 + (j & 3);
                            double2 a0 = ap[0], a1 = ap[128], a2 = ap[256];
                            dd ar = limbs_to_dd(a0.x, a1.x, a2.x), ai = limbs_to_dd(a0.y, a1.y, a2.y);
                            dd I = dd_dot2(ar, T[1], ai, T[0], -1.0);     // Im[conj(A) T]
                            dd R = dd_dot2(ar, T[2], ai, T[3], 1.0);      // Re[conj(A) T'']
#define GACC(AX)                                                                              \
    if (AX < d) {                                                                             \
        const int wgt = wT[AX * Ppad + p];                                                    \
        if (wgt != 0) g##AX = dd_add(g##AX, dd_mul_d(I, (double)wgt));                        \
        if (AX == d - 1) g##AX = dd_add(g##AX, dd_scale2(R, qs));                             \
    }
                            GACC(0) GACC(1) GACC(2)
#undef GACC
                        }
                    }
            }
            // refill, one stage behind: the stage of chunk c-1 has been released by (nearly) every warp
            if (tid == 0 && c >= 1 && issued < total) {
                const int sp = (c - 1) % SHD_GRAD_STAGES;
                mbar_wait(smem_u32(&empty_bar[sp]), (uint32_t)(((c - 1) / SHD_GRAD_STAGES) & 1));
                issue();
            }
        }
    }

    // reduce over the 8 threads that share a particle: gred[a][j_local][4 ph + tq]
    __syncthreads();
    double2* gred = reinterpret_cast<double2*>(smem);
    gred[(0 * 32 + jl) * 8 + ph * 4 + (lane & 3)] = make_double2(g0.h, g0.l);
    gred[(1 * 32 + jl) * 8 + ph * 4 + (lane & 3)] = make_double2(g1.h, g1.l);
    gred[(2 * 32 + jl) * 8 + ph * 4 + (lane & 3)] = make_double2(g2.h, g2.l);
    __syncthreads();
    if (tid < 32 * d) {
        const int a = tid / 32, jr = tid % 32;
        const long jo = jb * 32 + jr;
        if (jo < N) {
            dd sum{0.0, 0.0};
            for (int t = 0; t < 8; t++) {
                double2 v = gred[(a * 32 + jr) * 8 + t];
                sum = dd_add(sum, dd{v.x, v.y});
            }
            // (4 pi / L) / cscale
            dd pref = dd_div_d(dd_mul_d(dd{0x1.921fb54442d18p+2, 0x1.1a62633145c07p-52}, 2.0), L);
            sum = dd_mul(sum, pref);
            sum = dd_scale2(sum, 1.0 / scal->cscale);
            grad_hi[(size_t)a * N + jo] = sum.h;
            grad_lo[(size_t)a * N + jo] = sum.l;
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
    k_grad<<<(unsigned)h->njb, NW * 32, GSMEM, h->stream>>>(
        h->d, h->N, h->L, h->Npad, h->npb, h->Qpad, h->npb * 32, h->qscale_log2, h->d_qchunks, h->d_wT,
        h->d_A, h->d_Bg, h->d_C, h->d_scal, grad_hi, grad_lo, h->d_skip);
    h->last_launches += 1;
    return cudaGetLastError();
}
