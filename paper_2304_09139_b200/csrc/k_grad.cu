// k_grad.cu -- step a4: dPhi/dr_{j,a} = (4 pi / L) sum_k v_k n_a Im[ exp(-i k.r_j) rho(k) ]
// (Eq. 6, sign D:R2) as two contractions over q followed by one over p:
//   T_j[p]   = sum_{q,sigma} W(p,q,sigma) conj(B_j[q]^sigma)          = sum_q ( C1 br + C2 bi )
//   T''_j[p] = -i sum_{q,sigma} sigma q W conj(B^sigma)               = sum_q ( D1 br + D2 bi ),  D1 = q C2, D2 = -q C1
//   grad_a   = (4 pi/L) sum_p ( w_a(p) Im[conj(A_j[p]) T_j[p]] + [a = last axis] Re[conj(A_j[p]) T''_j[p]] )
// with C1 = W+ + W-, C2 = -i (W+ - W-), W = v rho (built by k_ctable), so both signs of the last
// axis share the same products: 24 FP64 FMAs per particle-wavevector pair.  The weight q of the last
// axis sits on the SHARED operand (C, D: 16 KB per slab, L2 resident), not on the particles' table, which
// therefore holds only the phasor limbs (half the bytes to write in k_tables and to stream here).
//
// Work unit (one CTA) = 64 particles x one segment of the step list.  A step is one group of 4 q of
// one block of 16 p (host-built list, shd_api.cu); a block's q-range ends at the circle boundary of
// its smallest p, so 16-wide blocks waste 4 % of the cells where 32-wide ones wasted 9 %.  Segments
// have equal length and may cut a block anywhere: the p-contraction is linear in T, so a partial T
// gives a partial gradient; partial gradients are summed in fixed order by k_gradsum.
// Each warp owns 8 particles x 16 p (two 8x8 blocks) and issues the FMAs as FP64 matrix
// instructions (DMMA.8x8x4, k = 4 q) on the limb planes: 96 per warp and step.  Operand slabs (the
// particles' own Bg table, 2 x 6 KB, and the 16-p slab of C and D, 16 KB, L2 resident) arrive by TMA bulk
// copies, issued by a ninth (producer) warp, through a 4-stage full/empty mbarrier ring.  The operand fragment loads are software
// pipelined: every LDS is issued one round of 16 DMMAs (or more) ahead of its first use and the
// first fragments of the next step are loaded under the last round, so the two warps of a
// scheduler never stall on shared memory at the same time (they wait on the same stage).
// A block ends after <= 64 steps (one exact limb burst, 256 q): the limbs are folded into double-double
// T, T'' and parked in thread-private shared-memory slots; their p-contraction with A (double-double,
// deterministic, no atomics) is deferred and spread over the next four steps, A loaded a step ahead,
// so that no warp waits on global memory or on a long dependent chain while the FP64 pipe idles.
#include "pipe.cuh"
#include "shd_internal.h"

namespace {

constexpr int NW = 8;
constexpr int NST = SHD_GRAD_STAGES;
constexpr int PLANE_B = 32 * 4 * 16;                         // 2048: one limb plane of a 32-particle Bg slab
constexpr int PLANE_C = 16 * 4 * 16;                         // 1024: one limb plane of a 16-p C slab
constexpr int BSLAB = 3 * PLANE_B;                           // 6144: limbs of b
constexpr int CSLAB = 16 * PLANE_C;                          // 16384: C1, C2, D1, D2, each x0, x1, x2, x1 + x2
constexpr int GSTAGE = 2 * BSLAB + CSLAB;                    // 28672
constexpr int RING_BYTES = NST * GSTAGE;
constexpr int MAIN_BYTES = 16 * 256 * 16;                    // 16 dd accumulators per thread
constexpr int GSMEM = RING_BYTES + MAIN_BYTES;

__device__ __forceinline__ dd limbs_to_dd(double x0, double x1, double x2) {
    return fast_two_sum(__dadd_rn(x0, x1), x2);    // x0 + x1 is exact (44 bits)
}

// one round: 16 DMMAs on limb level LV; particle-side limb b, shared-side limbs of C1, C2, D1, D2
#define GROUND(LV, Bx, X)                                                   \
    _Pragma("unroll") for (int t = 0; t < 2; t++) {                         \
        dmma_v(acc[t][0].LV, Bx.r, X[0][t].r);                              \
        dmma_v(acc[t][1].LV, Bx.r, X[0][t].i);                              \
        dmma_v(acc[t][2].LV, Bx.r, X[2][t].r);                              \
        dmma_v(acc[t][3].LV, Bx.r, X[2][t].i);                              \
    }                                                                       \
    _Pragma("unroll") for (int t = 0; t < 2; t++) {                         \
        dmma_v(acc[t][0].LV, Bx.i, X[1][t].r);                              \
        dmma_v(acc[t][1].LV, Bx.i, X[1][t].i);                              \
        dmma_v(acc[t][2].LV, Bx.i, X[3][t].r);                              \
        dmma_v(acc[t][3].LV, Bx.i, X[3][t].i);                              \
    }
// fragments of limb plane L of the four shared operands (o = 0..3: C1, C2, D1, D2), both 8-p blocks
#define LOADX(X, base, L)                                                   \
    _Pragma("unroll") for (int o = 0; o < 4; o++)                           \
        _Pragma("unroll") for (int t = 0; t < 2; t++) X[o][t] = lds2((base) + t * 512 + (o * 4 + (L)) * PLANE_C);

// NL = 2 / 1: the two-limb / one-limb "fast" precisions of shd_set_precision (see k_rho.cu)
template <int NL>
__global__ void __launch_bounds__(NW * 32 + 128, 1) k_grad(
    int d, long N, long Npad, long njb64, int Qpad, int Ppad, int qscale_log2,
    const int2* __restrict__ steps, int nsteps, int nseg, const int* __restrict__ wT,
    const double* __restrict__ A, const double* __restrict__ Bg, const double* __restrict__ C,
    double* __restrict__ gpart, const int* __restrict__ skip)
{
    if (skip && *skip) return;
    extern __shared__ __align__(1024) unsigned char smem[];
    __shared__ __align__(8) unsigned long long full_bar[NST], empty_bar[NST];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const long jb = blockIdx.x % njb64;
    const int seg = (int)(blockIdx.x / njb64);
    const int c_begin = (int)((long)nsteps * seg / nseg), c_end = (int)((long)nsteps * (seg + 1) / nseg);
    const int total = c_end - c_begin;
    const uint32_t s0 = smem_u32(smem);
    double2* mainacc = reinterpret_cast<double2*>(smem + RING_BYTES);   // [16][256]

    if (tid == 0) {
        for (int s = 0; s < NST; s++) {
            mbar_init(smem_u32(&full_bar[s]), 1);
            mbar_init(smem_u32(&empty_bar[s]), NW);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();        // (the T slots behind the ring need no initialisation: written before read)

    if (warp >= NW) {
        // producer warpgroup: hands its registers to the consumers (setmaxnreg), then one lane streams.
        asm volatile("setmaxnreg.dec.sync.aligned.u32 24;");
        // producer warp (one lane): stage of step i <- Bg slabs of the two 32-particle halves + C slab;
        // it does nothing else, so a refill is issued the moment the last consumer warp releases a stage
        if (warp == NW && lane == 0) {
            const double* gB = Bg + (size_t)(2 * jb) * (Qpad / 4) * SHD_GROUP_DOUBLES;
            const size_t halfB = (size_t)(Qpad / 4) * SHD_GROUP_DOUBLES;
            for (int i = 0; i < total; i++) {
                const int stage = i % NST;
                if (i >= NST) mbar_wait(smem_u32(&empty_bar[stage]), (uint32_t)((i / NST - 1) & 1));
                const uint32_t bar = smem_u32(&full_bar[stage]);
                const int2 st = steps[c_begin + i];
                const int qg = st.y & 0xffff;
                mbar_expect_tx(bar, GSTAGE);
                tma_load_1d(s0 + stage * GSTAGE, gB + (size_t)qg * SHD_GROUP_DOUBLES, BSLAB, bar);
                tma_load_1d(s0 + stage * GSTAGE + BSLAB, gB + halfB + (size_t)qg * SHD_GROUP_DOUBLES, BSLAB, bar);
                tma_load_1d(s0 + stage * GSTAGE + 2 * BSLAB, C + (size_t)st.x * (CSLAB / 8), CSLAB, bar);
            }
        }
        __syncthreads();        // the two block-wide barriers of the consumers' epilogue
        __syncthreads();
        return;
    }
    asm volatile("setmaxnreg.inc.sync.aligned.u32 232;");

    // warp tile: j_local = 8 warp + g,  p_local = 8 t + {2 tq, 2 tq + 1}
    const uint32_t fragoff = (uint32_t)(lane >> 2) * 64 + (uint32_t)(lane & 3) * 16;
    const uint32_t offB = (uint32_t)(warp >> 2) * BSLAB + (uint32_t)(warp & 3) * 8 * 64 + fragoff;
    const uint32_t offC = 2 * BSLAB + fragoff;
    const double qs = ldexp(1.0, qscale_log2);
    const long j = jb * 64 + warp * 8 + (lane >> 2);

    Acc3 acc[2][4];
#pragma unroll
    for (int t = 0; t < 2; t++)
#pragma unroll
        for (int x = 0; x < 4; x++) acc3_zero(acc[t][x]);
    dd g0{0.0, 0.0}, g1{0.0, 0.0}, g2{0.0, 0.0}, g3{0.0, 0.0};

    // deferred p-contraction state (warp-uniform): quarter pk = (t, e) of block ppb is pending
    bool pend = false;
    int pk = 0, ppb = 0;
    double2 pa0 = make_double2(0.0, 0.0), pa1 = pa0, pa2 = pa0;
    const double2* Aj = reinterpret_cast<const double2*>(A) + (size_t)(j >> 2) * 3 * 32 * 4 + (j & 3);
    auto load_quarter = [&](int k, int pb16, double2& a0, double2& a1, double2& a2) {
        const int p = pb16 * 16 + (k >> 1) * 8 + (lane & 3) * 2 + (k & 1);
        if (j < N) {
            const double2* ap = Aj + ((size_t)(p >> 5) * (Npad / 4) * 3 * 32 + (p & 31)) * 4;
            asm volatile("ld.global.nc.v2.f64 {%0,%1}, [%2];" : "=d"(a0.x), "=d"(a0.y) : "l"(ap));
            asm volatile("ld.global.nc.v2.f64 {%0,%1}, [%2];" : "=d"(a1.x), "=d"(a1.y) : "l"(ap + 128));
            asm volatile("ld.global.nc.v2.f64 {%0,%1}, [%2];" : "=d"(a2.x), "=d"(a2.y) : "l"(ap + 256));
        }
    };
    auto contract_quarter = [&](int k, int pb16, double2 a0, double2 a1, double2 a2) {
        const int t = k >> 1, e = k & 1;
        const int p = pb16 * 16 + t * 8 + (lane & 3) * 2 + e;
        dd T[4];
#pragma unroll
        for (int x = 0; x < 4; x++) {
            double2 m = mainacc[((t * 4 + x) * 2 + e) * 256 + tid];
            T[x] = dd{m.x, m.y};
        }
        if (j < N) {
            dd ar = limbs_to_dd(a0.x, a1.x, a2.x), ai = limbs_to_dd(a0.y, a1.y, a2.y);
            dd I = dd_dot2(ar, T[1], ai, T[0], -1.0);     // Im[conj(A) T]
            dd R = dd_dot2(ar, T[2], ai, T[3], 1.0);      // Re[conj(A) T'']
#define GACC(AX)                                                                              \
    if (AX < d) {                                                                             \
        const int wgt = AX < 3 ? wT[(AX < 3 ? AX : 0) * Ppad + p] : 0;                        \
        if (wgt != 0) g##AX = dd_add(g##AX, dd_mul_d(I, (double)wgt));                        \
        if (AX == d - 1) g##AX = dd_add(g##AX, dd_scale2(R, qs));                             \
    }
            GACC(0) GACC(1) GACC(2) GACC(3)
#undef GACC
        }
    };

    F2 b0, X0[4][2];
    if (total > 0) {
        mbar_wait(smem_u32(&full_bar[0]), 0u);
        b0 = lds2(s0 + offB);
        LOADX(X0, s0 + offC, 0)
    }
    constexpr bool FULL = NL >= 3, TWO = NL >= 2;
    for (int c = 0; c < total; c++) {
        const int s = c % NST;
        const uint32_t pB = s0 + s * GSTAGE + offB, pC = s0 + s * GSTAGE + offC;
        const int2 st = steps[c_begin + c];
        if (pend) load_quarter(pk, ppb, pa0, pa1, pa2);
        F2 b1{0.0, 0.0}, b2{0.0, 0.0}, b12{0.0, 0.0};
        if (TWO) b1 = lds2(pB + 1 * PLANE_B);
        if (FULL) b2 = lds2(pB + 2 * PLANE_B);
        F2 X1[4][2];
        if (TWO) {
            GROUND(l0, b0, X0)
            LOADX(X1, pC, 1)
            GROUND(l1, b1, X0)
        }
        if (FULL) {
            F2 X2[4][2];
            LOADX(X2, pC, 2)
            GROUND(l2, b2, X0)
            b12 = add2(b1, b2);
            GROUND(l1, b0, X1)
            F2 XS[4][2];                         // x1 + x2 of the shared operands comes from the table (k_ctable)
            LOADX(XS, pC, 3)
            GROUND(l2, b0, X2)
            if (c + 1 < total) {
                const int sn = (c + 1) % NST;
                mbar_wait(smem_u32(&full_bar[sn]), (uint32_t)(((c + 1) / NST) & 1));
                b0 = lds2(s0 + sn * GSTAGE + offB);
                LOADX(X0, s0 + sn * GSTAGE + offC, 0)
            }
            GROUND(l2, b12, XS)
        } else {
            F2 b0n = b0, X0n[4][2];
            if (c + 1 < total) {
                const int sn = (c + 1) % NST;
                mbar_wait(smem_u32(&full_bar[sn]), (uint32_t)(((c + 1) / NST) & 1));
                b0n = lds2(s0 + sn * GSTAGE + offB);
                LOADX(X0n, s0 + sn * GSTAGE + offC, 0)
            }
            if (TWO) { GROUND(l1, b0, X1) } else { GROUND(l0, b0, X0) }
            b0 = b0n;
            if (c + 1 < total) {
#pragma unroll
                for (int o = 0; o < 4; o++)
#pragma unroll
                    for (int t = 0; t < 2; t++) X0[o][t] = X0n[o][t];
            }
        }
        // Release the stage only now: every LDS from it has been CONSUMED by an issued DMMA.  An LDS that
        // is merely issued before the arrive may still be in flight when the refill lands (measured: one
        // warp in ~10^5 got a stale limb when the arrive sat between the x1+x2 loads and their round).
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&empty_bar[s]));
        // deferred p-contraction: one quarter of the previous block per step, its A limbs loaded at the
        // top of this step (global-memory latency hidden under the 96 DMMAs above)
        if (pend) {
            contract_quarter(pk, ppb, pa0, pa1, pa2);
            if (++pk == 4) pend = false;
        }
        const int flags = st.y >> 16;
        if ((flags & 1) || c == total - 1) {
            // end of a block of <= 64 steps (one exact burst) or of the segment: limbs -> dd T, T'' parked
            // in the thread-private shared-memory slots until the next steps contract them with A
            while (pend) {                         // blocks shorter than 4 steps: finish the previous one now
                load_quarter(pk, ppb, pa0, pa1, pa2);
                contract_quarter(pk, ppb, pa0, pa1, pa2);
                if (++pk == 4) pend = false;
            }
#pragma unroll
            for (int t = 0; t < 2; t++)
#pragma unroll
                for (int x = 0; x < 4; x++) {
                    Acc3& r = acc[t][x];
                    double2 m0 = make_double2(0.0, 0.0), m1 = make_double2(0.0, 0.0);
                    fold_burst(r.l0.c0, r.l1.c0, r.l2.c0, m0);
                    fold_burst(r.l0.c1, r.l1.c1, r.l2.c1, m1);
                    mainacc[((t * 4 + x) * 2 + 0) * 256 + tid] = m0;
                    mainacc[((t * 4 + x) * 2 + 1) * 256 + tid] = m1;
                    acc3_zero(r);
                }
            pend = true; pk = 0; ppb = st.x / (Qpad / 4);
        }
    }
    if (pend) {
        // the last block of the segment: all remaining quarters' A limbs in flight at once
        double2 qa[4][3];
#pragma unroll
        for (int k = 0; k < 4; k++)
            if (k >= pk) load_quarter(k, ppb, qa[k][0], qa[k][1], qa[k][2]);
#pragma unroll
        for (int k = 0; k < 4; k++)
            if (k >= pk) contract_quarter(k, ppb, qa[k][0], qa[k][1], qa[k][2]);
        pend = false;
    }

    // reduce over the 4 threads that share a particle: gred[a][j_local 64][tq 4]
    __syncthreads();
    double2* gred = reinterpret_cast<double2*>(smem);
    const int jl = warp * 8 + (lane >> 2);
    gred[(0 * 64 + jl) * 4 + (lane & 3)] = make_double2(g0.h, g0.l);
    gred[(1 * 64 + jl) * 4 + (lane & 3)] = make_double2(g1.h, g1.l);
    gred[(2 * 64 + jl) * 4 + (lane & 3)] = make_double2(g2.h, g2.l);
    gred[(3 * 64 + jl) * 4 + (lane & 3)] = make_double2(g3.h, g3.l);
    __syncthreads();
    if (tid < 64 * d) {
        const int a = tid / 64, jr = tid % 64;
        const long jo = jb * 64 + jr;
        if (jo < N) {
            dd sum{0.0, 0.0};
            for (int t = 0; t < 4; t++) {
                double2 v = gred[(a * 64 + jr) * 4 + t];
                sum = dd_add(sum, dd{v.x, v.y});
            }
            reinterpret_cast<double2*>(gpart)[((size_t)seg * d + a) * N + jo] = make_double2(sum.h, sum.l);
        }
    }
}

// grad = (4 pi / L) / cscale * sum_seg gpart[seg], fixed order.  gpart holds the nc particles of one chunk
// ([seg][d][nc]); they are particles j_first .. j_first + nc - 1 of the caller's arrays (axis stride N).
__global__ void __launch_bounds__(256) k_gradsum(
    long nc, int d, long j_first, long N, int nseg, double L, const double* __restrict__ gpart,
    const shd_scalars* __restrict__ scal, double* __restrict__ grad_hi, double* __restrict__ grad_lo,
    const int* __restrict__ skip)
{
    if (skip && *skip) return;
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    const long n = nc * d;
    if (i >= n) return;
    dd sum{0.0, 0.0};
    for (int s = 0; s < nseg; s++) {
        double2 v = reinterpret_cast<const double2*>(gpart)[(size_t)s * n + i];
        sum = dd_add(sum, dd{v.x, v.y});
    }
    dd pref = dd_div_d(dd_mul_d(dd{0x1.921fb54442d18p+2, 0x1.1a62633145c07p-52}, 2.0), L);   // 4 pi / L
    sum = dd_mul(sum, pref);
    sum = dd_scale2(sum, 1.0 / scal->cscale);
    const long o = (i / nc) * N + j_first + i % nc;
    grad_hi[o] = sum.h;
    grad_lo[o] = sum.l;
}

}  // namespace

cudaError_t shd_grad_configure()
{
    cudaError_t e = cudaFuncSetAttribute(k_grad<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, GSMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_grad<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, GSMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_grad<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, GSMEM);
    return e;
}

// gradient of the chunk's particles j_first .. j_first + nc - 1 (their tables are in place) into the caller's arrays
cudaError_t shd_launch_grad(shd_ctx* h, long j_first, long nc, double* grad_hi, double* grad_lo)
{
    const long n = (long)h->d * nc;
    if (h->rho_engine == 2) {          // INT8 tensor-core gradient pass (k_grad8.cu)
        cudaError_t e = shd_launch_grad8_main(h, nc);
        if (e != cudaSuccess) return e;
        k_gradsum<<<(unsigned)((n + 255) / 256), 256, 0, h->stream>>>(
            nc, h->d, j_first, h->N, 4 * h->nseg8, h->L, h->d_gpart, h->d_scal, grad_hi, grad_lo, h->d_skip);
        h->last_launches += 1;
        return cudaGetLastError();
    }
    const long njb = (nc + SHD_JT - 1) / SHD_JT;
#define LAUNCH_GRAD(NLV)                                                                                 \
    k_grad<NLV><<<(unsigned)(njb * h->nseg), NW * 32 + 128, GSMEM, h->stream>>>(                           \
        h->d, nc, h->Npad, njb, h->Qpad, h->npb * 32, h->qscale_log2,                                      \
        reinterpret_cast<const int2*>(h->d_steps), h->nsteps, h->nseg, h->d_wT,                            \
        h->d_A, h->d_Bg, h->d_C, h->d_gpart, h->d_skip)
    if (h->nlimb >= 3) LAUNCH_GRAD(3);
    else if (h->nlimb == 2) LAUNCH_GRAD(2);
    else LAUNCH_GRAD(1);
#undef LAUNCH_GRAD
    k_gradsum<<<(unsigned)((n + 255) / 256), 256, 0, h->stream>>>(
        nc, h->d, j_first, h->N, h->nseg, h->L, h->d_gpart, h->d_scal, grad_hi, grad_lo, h->d_skip);
    h->last_launches += 2;
    return cudaGetLastError();
}
