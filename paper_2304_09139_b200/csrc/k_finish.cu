// k_finish.cu -- step a3: sum the per-split partials in fixed order, form rho(k), |rho|^2,
// Phi = sum_k v_k |rho(k)|^2 (Eq. 2), S_max = max_k |rho(k)|^2 / N (Eq. 1) and its
// argmax, all in double-double and bit-reproducible (fixed reduction trees, no atomics);
// then build the limb-split gradient operand C[p,q] from W = v rho (Eq. 6).
#include "dd.cuh"
#include "shd_internal.h"

#include <cstdio>

namespace {

struct red { dd phi; dd smax; long long arg; double maxvs; };

__device__ __forceinline__ red red_combine(red a, red b) {
    red r;
    r.phi = dd_add(a.phi, b.phi);
    // larger |rho|^2 wins; ties go to the lower canonical index; arg < 0 marks "empty"
    bool takeb = b.arg >= 0 && (a.arg < 0 || dd_less(a.smax, b.smax) ||
                                (!dd_less(b.smax, a.smax) && b.arg < a.arg));
    r.smax = takeb ? b.smax : a.smax;
    r.arg = takeb ? b.arg : a.arg;
    r.maxvs = fmax(a.maxvs, b.maxvs);
    return r;
}
__device__ __forceinline__ red red_shfl(red a, int off) {
    red b;
    b.phi.h = __shfl_down_sync(0xffffffffu, a.phi.h, off);
    b.phi.l = __shfl_down_sync(0xffffffffu, a.phi.l, off);
    b.smax.h = __shfl_down_sync(0xffffffffu, a.smax.h, off);
    b.smax.l = __shfl_down_sync(0xffffffffu, a.smax.l, off);
    b.arg = __shfl_down_sync(0xffffffffu, a.arg, off);
    b.maxvs = __shfl_down_sync(0xffffffffu, a.maxvs, off);
    return b;
}
__device__ red block_reduce(red v) {
    __shared__ red sh[32];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v = red_combine(v, red_shfl(v, off));
    int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) sh[w] = v;
    __syncthreads();
    int nw = (blockDim.x + 31) >> 5;
    if (w == 0) {
        red z; z.phi = dd{0, 0}; z.smax = dd{-1, 0}; z.arg = -1; z.maxvs = 0;
        v = l < nw ? sh[l] : z;
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) v = red_combine(v, red_shfl(v, off));
    }
    return v;   // valid in thread 0
}

__device__ __forceinline__ void account(red& r, dd re, dd im, double v, long long k) {
    dd s = dd_add(dd_mul(re, re), dd_mul(im, im));
    r.phi = dd_add(r.phi, dd_mul_d(s, v));
    if (r.arg < 0 || dd_less(r.smax, s) || (!dd_less(s, r.smax) && k < r.arg)) { r.smax = s; r.arg = k; }
    r.maxvs = fmax(r.maxvs, v * v * s.h);
}

// one thread per (tile, cell).  The four real sums X of a cell are the left fold, in fixed order, of the partials of
// all particle splits: X = (((xin + part_0) + part_1) + ...).  An evaluation whose tables are built chunk by chunk
// (bounded workspace) calls this once per chunk with the running sums xin / xout (fin = 0), a sharded one once more
// with the ranks' running sums as the partials; the result does not depend on where the chunk boundaries fall.
// fin != 0: rho(k), |rho|^2, Phi, S_max partials; else only xout is written.
__global__ void __launch_bounds__(256) k_finish1(
    const double* __restrict__ part, int nsplit, const double* __restrict__ xin, double* __restrict__ xout, int fin,
    int ntiles, int tp, int tq, const int* __restrict__ tile_pb,
    const int* __restrict__ tile_qb, const int* __restrict__ cell_kp, const int* __restrict__ cell_km,
    int Ppad, int Qpad, long M, const double* __restrict__ v, double* __restrict__ rho, double* __restrict__ blockred,
    const int* __restrict__ skip)
{
    if (skip && *skip) return;
    long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    red r; r.phi = dd{0, 0}; r.smax = dd{-1, 0}; r.arg = -1; r.maxvs = 0;
    if (idx < (long)ntiles * 1024) {
        int tile = (int)(idx >> 10), cell = (int)(idx & 1023);
        // tiles are tp x tq = 1024 cells: 32 x 32 (k_rho) or 64 x 16 (k_rho8)
        int p = tile_pb[tile] * tp + cell / tq, q = tile_qb[tile] * tq + cell % tq;
        const bool inside = p < Ppad && q < Qpad;
        int kp = inside ? cell_kp[(size_t)p * Qpad + q] : -1, km = inside ? cell_km[(size_t)p * Qpad + q] : -1;
        if (kp >= 0 || km >= 0) {
            const double2* src = reinterpret_cast<const double2*>(part);
            dd X[4];
#pragma unroll
            for (int x = 0; x < 4; x++) {
                dd acc = dd{0, 0};
                if (xin) {
                    double2 t = reinterpret_cast<const double2*>(xin)[((size_t)tile * 4 + x) * 1024 + cell];
                    acc = dd{t.x, t.y};
                }
                for (int s = 0; s < nsplit; s++) {
                    double2 t = src[((size_t)(s * (long)ntiles + tile) * 4 + x) * 1024 + cell];
                    acc = dd_add(acc, dd{t.x, t.y});
                }
                X[x] = acc;
                if (xout) reinterpret_cast<double2*>(xout)[((size_t)tile * 4 + x) * 1024 + cell] = make_double2(acc.h, acc.l);
            }
            if (fin && kp >= 0) {
                dd re = dd_sub(X[0], X[1]), im = dd_add(X[2], X[3]);
                rho[kp] = re.h; rho[M + kp] = re.l; rho[2 * M + kp] = im.h; rho[3 * M + kp] = im.l;
                account(r, re, im, v ? v[kp] : 1.0, kp);
            }
            if (fin && km >= 0) {
                dd re = dd_add(X[0], X[1]), im = dd_sub(X[3], X[2]);
                rho[km] = re.h; rho[M + km] = re.l; rho[2 * M + km] = im.h; rho[3 * M + km] = im.l;
                account(r, re, im, v ? v[km] : 1.0, km);
            }
        }
    }
    if (!fin) return;
    r = block_reduce(r);
    if (threadIdx.x == 0) {
        double* o = blockred + (size_t)blockIdx.x * 8;
        o[0] = r.phi.h; o[1] = r.phi.l; o[2] = r.smax.h; o[3] = r.smax.l;
        o[4] = (double)r.arg; o[5] = r.maxvs;
    }
}

__global__ void __launch_bounds__(1024) k_finish2(const double* __restrict__ blockred, int nblocks, long N,
                                                  shd_scalars* __restrict__ scal, const int* __restrict__ skip)
{
    if (skip && *skip) return;
    red r; r.phi = dd{0, 0}; r.smax = dd{-1, 0}; r.arg = -1; r.maxvs = 0;
    for (int b = threadIdx.x; b < nblocks; b += blockDim.x) {
        const double* o = blockred + (size_t)b * 8;
        red t; t.phi = dd{o[0], o[1]}; t.smax = dd{o[2], o[3]}; t.arg = (long long)o[4]; t.maxvs = o[5];
        r = red_combine(r, t);
    }
    r = block_reduce(r);
    if (threadIdx.x == 0) {
        dd sm = dd_div_d(r.smax, (double)N);
        scal->phi[0] = r.phi.h; scal->phi[1] = r.phi.l;
        scal->smax[0] = sm.h; scal->smax[1] = sm.l;
        scal->argmax = r.arg;
        scal->maxvs = r.maxvs;
        double mw = sqrt(r.maxvs);
        // |C components| <= 2 max|v rho| < 2^(ilogb(mw)+2)
        scal->cscale = (mw > 0.0 && isfinite(mw)) ? ldexp(1.0, -(ilogb(mw) + 2)) : 1.0;
        scal->nonfinite = (isfinite(r.phi.h) && isfinite(r.smax.h)) ? 0 : 1;
    }
}

struct limbs { double x0, x1, x2; };
__device__ __forceinline__ limbs split_limbs(dd x) {
    const double C0 = 1.5 * 4503599627370496.0 / (double)(1 << SHD_W0);
    const double C1 = 1.5 * 4503599627370496.0 / ((double)(1 << SHD_W0) * (double)(1 << SHD_W1));
    limbs r;
    r.x0 = __dadd_rn(__dadd_rn(x.h, C0), -C0);
    double rem = __dadd_rn(x.h, -r.x0);
    r.x1 = __dadd_rn(__dadd_rn(rem, C1), -C1);
    r.x2 = __dadd_rn(__dadd_rn(rem, -r.x1), x.l);
    return r;
}

// Shared operand of the gradient pass: C1 = W+ + W-,  C2 = -i (W+ - W-),  W = v rho scaled by cscale (a
// power of two), and the q-weighted pair D1 = q C2, D2 = -q C1 scaled by 2^-qscale_log2 (exact).
// layout [pb16][q/4][plane 16][16 p][q%4][re,im]; plane 4 o + l: operand o (C1, C2, D1, D2), limb l of
// (re, im) for l = 0..2 and x1 + x2 for l = 3 (stored so that the gradient pass need not form it).
__global__ void __launch_bounds__(256) k_ctable(
    int npb16, int Qpad, int qscale_log2, const int* __restrict__ cell_kp, const int* __restrict__ cell_km, long M,
    const double* __restrict__ v, const double* __restrict__ rho, const shd_scalars* __restrict__ scal,
    double* __restrict__ C, const int* __restrict__ skip)
{
    if (skip && *skip) return;
    long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    long ncell = (long)npb16 * 16 * Qpad;
    if (idx >= ncell) return;
    // idx enumerates (pb16, q/4, p%16, q%4) with q%4 fastest so that stores are coalesced
    const int q4 = (int)(idx & 3), pi = (int)((idx >> 2) & 15);
    long t = idx >> 6;
    const int qg = (int)(t % (Qpad / 4));
    const int pb = (int)(t / (Qpad / 4));
    const int p = pb * 16 + pi, q = qg * 4 + q4;
    int kp = cell_kp[(size_t)p * Qpad + q], km = cell_km[(size_t)p * Qpad + q];
    double sc = scal->cscale;
    dd wpr{0, 0}, wpi{0, 0}, wmr{0, 0}, wmi{0, 0};
    if (kp >= 0) {
        double vv = v ? v[kp] : 1.0;
        wpr = dd_scale2(dd_mul_d(dd{rho[kp], rho[M + kp]}, vv), sc);
        wpi = dd_scale2(dd_mul_d(dd{rho[2 * M + kp], rho[3 * M + kp]}, vv), sc);
    }
    if (km >= 0) {
        double vv = v ? v[km] : 1.0;
        wmr = dd_scale2(dd_mul_d(dd{rho[km], rho[M + km]}, vv), sc);
        wmi = dd_scale2(dd_mul_d(dd{rho[2 * M + km], rho[3 * M + km]}, vv), sc);
    }
    dd op[4][2];
    op[0][0] = dd_add(wpr, wmr); op[0][1] = dd_add(wpi, wmi);                 // C1
    dd dr = dd_sub(wpr, wmr), di = dd_sub(wpi, wmi);
    op[1][0] = di; op[1][1] = dd_neg(dr);                                     // C2 = -i (dr + i di) = di - i dr
    const double qw = ldexp((double)q, -qscale_log2);                         // q 2^-qs <= 1
    op[2][0] = dd_mul_d(op[1][0], qw); op[2][1] = dd_mul_d(op[1][1], qw);     // D1 =  q C2
    op[3][0] = dd_mul_d(op[0][0], -qw); op[3][1] = dd_mul_d(op[0][1], -qw);   // D2 = -q C1
    double2* dst = reinterpret_cast<double2*>(C) + ((((size_t)pb * (Qpad / 4) + qg) * 16) * 16 + pi) * 4 + q4;
#pragma unroll
    for (int o = 0; o < 4; o++) {
        limbs a = split_limbs(op[o][0]), b = split_limbs(op[o][1]);
        dst[(o * 4 + 0) * 64] = make_double2(a.x0, b.x0);
        dst[(o * 4 + 1) * 64] = make_double2(a.x1, b.x1);
        dst[(o * 4 + 2) * 64] = make_double2(a.x2, b.x2);
        dst[(o * 4 + 3) * 64] = make_double2(__dadd_rn(a.x1, a.x2), __dadd_rn(b.x1, b.x2));
    }
}

// Shared operand of the INT8 gradient pass (k_grad8.cu): W[(p, out), (q, c)] with out = T re, T im, T'' re,
// T'' im and c = re, im of b:  (C1r, C2r), (C1i, C2i), (D1r, D2r), (D1i, D2i), as 13 s8 digits of
// trunc(x 2^102), layout [pb8][q/16][digit][32 rows (4 p%8 + out) x 32 K (2 (q%16) + c)] in the tensor
// core's K-major core-matrix layout.  One thread per (p, q).
__device__ __forceinline__ __int128 f_fix102(double x) {
    const long long b = __double_as_longlong(x);
    const int e = (int)((b >> 52) & 0x7ff);
    if (e == 0) return 0;
    const unsigned long long m = ((unsigned long long)b & 0xfffffffffffffULL) | (1ULL << 52);
    const int sh = e - 1075 + 102;
    __int128 v = sh >= 0 ? ((__int128)m << sh) : (sh > -64 ? (__int128)(m >> (-sh)) : (__int128)0);
    return b < 0 ? -v : v;
}
__global__ void __launch_bounds__(256) k_wtable8(
    int npb8, int Ppad, int Qpad, int qscale_log2, const int* __restrict__ cell_kp, const int* __restrict__ cell_km,
    long M, const double* __restrict__ v, const double* __restrict__ rho, const shd_scalars* __restrict__ scal,
    signed char* __restrict__ W8, const int* __restrict__ skip)
{
    if (skip && *skip) return;
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    const int nkq = Qpad / 16;
    if (idx >= (long)npb8 * 8 * Qpad) return;
    // idx enumerates (pb8, q/16, p%8, q%16), q%16 fastest
    const int ql = (int)(idx & 15), pl = (int)((idx >> 4) & 7);
    const long t = idx >> 7;
    const int kq = (int)(t % nkq), pb = (int)(t / nkq);
    const int p = pb * 8 + pl, q = kq * 16 + ql;
    int kp = -1, km = -1;
    if (p < Ppad) { kp = cell_kp[(size_t)p * Qpad + q]; km = cell_km[(size_t)p * Qpad + q]; }
    const double sc = scal->cscale;
    dd wpr{0, 0}, wpi{0, 0}, wmr{0, 0}, wmi{0, 0};
    if (kp >= 0) {
        double vv = v ? v[kp] : 1.0;
        wpr = dd_scale2(dd_mul_d(dd{rho[kp], rho[M + kp]}, vv), sc);
        wpi = dd_scale2(dd_mul_d(dd{rho[2 * M + kp], rho[3 * M + kp]}, vv), sc);
    }
    if (km >= 0) {
        double vv = v ? v[km] : 1.0;
        wmr = dd_scale2(dd_mul_d(dd{rho[km], rho[M + km]}, vv), sc);
        wmi = dd_scale2(dd_mul_d(dd{rho[2 * M + km], rho[3 * M + km]}, vv), sc);
    }
    dd op[4][2];
    op[0][0] = dd_add(wpr, wmr); op[0][1] = dd_add(wpi, wmi);                 // C1
    const dd dr = dd_sub(wpr, wmr), di = dd_sub(wpi, wmi);
    op[1][0] = di; op[1][1] = dd_neg(dr);                                     // C2
    const double qw = ldexp((double)q, -qscale_log2);
    op[2][0] = dd_mul_d(op[1][0], qw); op[2][1] = dd_mul_d(op[1][1], qw);     // D1 =  q C2
    op[3][0] = dd_mul_d(op[0][0], -qw); op[3][1] = dd_mul_d(op[0][1], -qw);   // D2 = -q C1
    // rows: out 0 = T re: (C1r, C2r); 1 = T im: (C1i, C2i); 2 = T'' re: (D1r, D2r); 3 = T'' im: (D1i, D2i)
    signed char* base = W8 + ((size_t)pb * nkq + kq) * (SHD_I8_DIGITS * 1024);
    const __int128 off = ((__int128)0x0000008080808080ULL << 64) | (__int128)0x8080808080808080ULL;
#pragma unroll
    for (int out = 0; out < 4; out++)
#pragma unroll
        for (int c = 0; c < 2; c++) {
            const dd x = op[2 * (out >> 1) + c][out & 1];
            const unsigned __int128 y = (unsigned __int128)(f_fix102(x.h) + f_fix102(x.l) + off);
            const int row = 4 * pl + out, k = 2 * ql + c;
            const int o = (row >> 3) * 256 + (k >> 4) * 128 + (row & 7) * 16 + (k & 15);
#pragma unroll
            for (int i = 0; i < SHD_I8_DIGITS; i++) base[i * 1024 + o] = (signed char)((int)((y >> (8 * i)) & 0xff) - 128);
        }
}

// NEXT-3 (Eq. 7, Eq. 3): S(k) = |rho(k)|^2 / N for every k of the handle's Q, and the
// sum over Q of (S(k) - 1)^2 that the order metric tau integrates, in double-double, fixed tree.
__global__ void __launch_bounds__(256) k_sfactor1(long M, long N, const double* __restrict__ rho,
                                                  double* __restrict__ S_out, double* __restrict__ blockred)
{
    const long k = (long)blockIdx.x * blockDim.x + threadIdx.x;
    red r; r.phi = dd{0, 0}; r.smax = dd{-1, 0}; r.arg = -1; r.maxvs = 0;
    if (k < M) {
        dd re{rho[k], rho[M + k]}, im{rho[2 * M + k], rho[3 * M + k]};
        dd s = dd_div_d(dd_add(dd_mul(re, re), dd_mul(im, im)), (double)N);
        if (S_out) S_out[k] = s.h;
        dd e = dd_add_d(s, -1.0);
        r.phi = dd_mul(e, e);
    }
    r = block_reduce(r);
    if (threadIdx.x == 0) { blockred[2 * blockIdx.x] = r.phi.h; blockred[2 * blockIdx.x + 1] = r.phi.l; }
}
__global__ void __launch_bounds__(1024) k_sfactor2(const double* __restrict__ blockred, int nblocks,
                                                   double* __restrict__ out)
{
    red r; r.phi = dd{0, 0}; r.smax = dd{-1, 0}; r.arg = -1; r.maxvs = 0;
    for (int b = threadIdx.x; b < nblocks; b += blockDim.x)
        r.phi = dd_add(r.phi, dd{blockred[2 * b], blockred[2 * b + 1]});
    r = block_reduce(r);
    if (threadIdx.x == 0) { out[0] = r.phi.h; out[1] = r.phi.l; }
}

// Radially averaged S(k) (Fig. 2a, Fig. S1a): bin b holds the wavevectors order[start[b] .. start[b+1]) (the
// host sorted them by their integer n.n; ascending k inside a bin).  One warp per bin: lane l adds members l, l+32, ...
// in double-double, then the butterfly: a fixed tree, bit-reproducible.  mean = sum / count.
__global__ void __launch_bounds__(128) k_sfactor_shells(long nbins, const long* __restrict__ start, const int* __restrict__ order,
                                                        long M, long N, const double* __restrict__ rho,
                                                        double* __restrict__ mean_hi, double* __restrict__ mean_lo)
{
    const long b = (long)blockIdx.x * 4 + (threadIdx.x >> 5);
    if (b >= nbins) return;
    const int lane = threadIdx.x & 31;
    const long s0 = start[b], s1 = start[b + 1];
    dd sum{0.0, 0.0};
    for (long i = s0 + lane; i < s1; i += 32) {
        const long k = order[i];
        dd re{rho[k], rho[M + k]}, im{rho[2 * M + k], rho[3 * M + k]};
        sum = dd_add(sum, dd_div_d(dd_add(dd_mul(re, re), dd_mul(im, im)), (double)N));
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        dd o{__shfl_xor_sync(0xffffffffu, sum.h, off), __shfl_xor_sync(0xffffffffu, sum.l, off)};
        sum = dd_add(sum, o);
    }
    if (lane == 0) {
        const dd m = s1 > s0 ? dd_div_d(sum, (double)(s1 - s0)) : dd{0.0, 0.0};
        mean_hi[b] = m.h;
        mean_lo[b] = m.l;
    }
}

}  // namespace

// S_out (device, M doubles) may be NULL; tau2 (device, 2 doubles) receives sum_k (S(k)-1)^2 as (hi, lo)
cudaError_t shd_launch_sfactor(shd_ctx* h, double* S_out, double* scratch, double* tau2)
{
    const int nb = (int)((h->M + 255) / 256);
    k_sfactor1<<<nb, 256, 0, h->stream>>>(h->M, h->Nsys, h->d_rho, S_out, scratch);
    k_sfactor2<<<1, 1024, 0, h->stream>>>(scratch, nb, tau2);
    h->last_launches += 2;
    return cudaGetLastError();
}

// Fold `nparts` partial arrays (part: [nparts][ntiles][4][1024] (hi, lo)) into the running sums: xin (or zero) -> xout
// (either may be NULL); fin: also rho, Phi, S_max, argmax (k_finish2).
cudaError_t shd_launch_fold(shd_ctx* h, const double* part, int nparts, const double* xin, double* xout, bool fin)
{
    const bool i8 = h->rho_engine >= 1;
    const int ntiles = i8 ? h->ntiles8 : h->ntiles;
    const int nb = (int)(((long)ntiles * 1024 + 255) / 256);
    k_finish1<<<nb, 256, 0, h->stream>>>(part, nparts, xin, xout, fin ? 1 : 0, ntiles, i8 ? SHD_I8_PT : 32,
                                         i8 ? SHD_I8_QT : 32, i8 ? h->d_tile8_pb : h->d_tile_pb,
                                         i8 ? h->d_tile8_qb : h->d_tile_qb, h->d_cell_kp, h->d_cell_km,
                                         h->npb * 32, h->Qpad, h->M, h->d_v, h->d_rho, h->d_blockred, h->d_skip);
    h->last_launches += 1;
    if (fin) {
        k_finish2<<<1, 1024, 0, h->stream>>>(h->d_blockred, nb, h->Nsys, h->d_scal, h->d_skip);
        h->last_launches += 1;
    }
    return cudaGetLastError();
}

cudaError_t shd_launch_sfactor_shells(shd_ctx* h, long nbins, const long* d_start, const int* d_order, double* d_mean_hi, double* d_mean_lo)
{
    k_sfactor_shells<<<(unsigned)((nbins + 3) / 4), 128, 0, h->stream>>>(nbins, d_start, d_order, h->M, h->Nsys, h->d_rho, d_mean_hi, d_mean_lo);
    h->last_launches += 1;
    return cudaGetLastError();
}

cudaError_t shd_launch_wtable8(shd_ctx* h);
cudaError_t shd_launch_wtable8(shd_ctx* h)
{
    const long n = (long)h->npb8 * 8 * h->Qpad;
    k_wtable8<<<(unsigned)((n + 255) / 256), 256, 0, h->stream>>>(
        h->npb8, h->npb * 32, h->Qpad, h->qscale_log2, h->d_cell_kp, h->d_cell_km, h->M, h->d_v, h->d_rho, h->d_scal,
        h->d_W8, h->d_skip);
    h->last_launches += 1;
    return cudaGetLastError();
}

cudaError_t shd_launch_ctable(shd_ctx* h)
{
    if (h->rho_engine == 2) return shd_launch_wtable8(h);   // the INT8 gradient pass reads W8 instead
    long ncell = (long)h->npb16 * 16 * h->Qpad;
    k_ctable<<<(unsigned)((ncell + 255) / 256), 256, 0, h->stream>>>(
        h->npb16, h->Qpad, h->qscale_log2, h->d_cell_kp, h->d_cell_km, h->M, h->d_v, h->d_rho, h->d_scal, h->d_C, h->d_skip);
    h->last_launches += 1;
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------------------------
// shd_structure_factor_noalloc (include/shd.h): k_sfactor1 / k_sfactor2 as above, with the per-block partial sums in a
// file-scope device array instead of a cudaMalloc'ed buffer, for callers that must not allocate.  2 doubles per block of
// 256 wavevectors: SHD_NOALLOC_MAX_Q / 256 blocks = 256 KiB, held by every GPU that loads this library until exit.
// Every call on a device shares the array: calls whose kernels overlap on the GPU race on it (shd.h says so).  Nothing
// in it has to start at zero: k_sfactor2 reads the 2 nb doubles that the nb blocks of k_sfactor1 of the same call wrote.
static __device__ __align__(256) double g_sf_scratch[2 * (SHD_NOALLOC_MAX_Q / 256)];

namespace {

// In HOST code the name g_sf_scratch is a stand-in the runtime uses to find the array, not a device address: a kernel
// handed `g_sf_scratch` from here would fault (or, where the GPU reaches host memory, write somewhere else).  The device
// address is per device: resolved once for each, with that device current, and kept.
constexpr int SF_MAX_DEVICES = 64;
double* g_sf_scratch_addr[SF_MAX_DEVICES];

cudaError_t sf_scratch_address(int dev, double** out)
{
    double* p = __atomic_load_n(&g_sf_scratch_addr[dev], __ATOMIC_ACQUIRE);
    if (!p) {
        void* sym = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&sym, g_sf_scratch);     // `dev` is the current device (caller checked)
        if (e != cudaSuccess) return e;
        if (!sym) return cudaErrorInvalidSymbol;
        p = (double*)sym;
        __atomic_store_n(&g_sf_scratch_addr[dev], p, __ATOMIC_RELEASE);   // two racing first calls store the same value
    }
    *out = p;
    return cudaSuccess;
}

int sf_fail(shd_ctx* h, int code, const char* msg) { h->err = msg; return code; }

}  // namespace

extern "C" int shd_structure_factor_noalloc(shd_ctx* h, double* S_out, double* dev2, int wait)
{
    if (!h) return SHD_EINVAL;
    if (!dev2) return sf_fail(h, SHD_EINVAL, "shd_structure_factor_noalloc: dev2 is NULL");
    if (h->M > SHD_NOALLOC_MAX_Q) {
        char msg[192];
        snprintf(msg, sizeof msg, "shd_structure_factor_noalloc: |Q| = %ld exceeds SHD_NOALLOC_MAX_Q = %ld (the static scratch "
                 "array); use shd_structure_factor", h->M, (long)SHD_NOALLOC_MAX_Q);
        return sf_fail(h, SHD_EINVAL, msg);
    }
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    cudaPointerAttributes attr;
    if (e == cudaSuccess) e = cudaPointerGetAttributes(&attr, h->d_rho);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return sf_fail(h, SHD_ECUDA, cudaGetErrorString(e)); }
    if (dev < 0 || dev >= SF_MAX_DEVICES || attr.type != cudaMemoryTypeDevice || attr.device != dev)
        return sf_fail(h, SHD_EINVAL, "shd_structure_factor_noalloc: the handle's device is not the current device");
    double* scratch = nullptr;
    e = sf_scratch_address(dev, &scratch);
    if (e == cudaSuccess) e = shd_launch_sfactor(h, S_out, scratch, dev2);
    if (e == cudaSuccess && wait) e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return sf_fail(h, SHD_ECUDA, cudaGetErrorString(e)); }
    return SHD_OK;
}
