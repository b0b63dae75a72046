// k_tables.cu -- step a1 of the hot path: per-particle phasor tables in limb form.
//
// For every particle j and axis a:  u = r_{j,a} / L to ~160 bits (three-word quotient with exact
// FMA remainders), z_a = exp(2 pi i frac(u)) by a double-double sincos (256-entry table of roots
// of unity + Taylor series), then the per-axis integer-power recurrences
//   A_j[p], B_j[q]  (see shd_internal.h)
// in complex double-double (TwoProd/TwoSum on FP64 FMA; BASELINE.json north_star item 2), each
// entry split into limbs and written in the tile-major layouts the rho / gradient kernels stream
// with TMA bulk copies.
#include "dd.cuh"
#include <cstdint>
#include "shd_internal.h"
#include "sincos_table.inc"
#include <algorithm>

namespace {

// t = frac(m * (hi + lo) / L) as a dd in [-1/2, 1/2], m a power of two
__device__ dd frac_turns(double hi, double lo, double L, double m) {
    double q1 = __ddiv_rn(hi, L);
    double r1 = __fma_rn(-q1, L, hi);            // exact remainder
    dd se = two_sum(r1, lo);
    double q2 = __ddiv_rn(se.h, L);
    double r2 = __fma_rn(-q2, L, se.h);          // exact remainder
    double q3 = __ddiv_rn(__dadd_rn(r2, se.l), L);
    double a1 = __dmul_rn(q1, m), a2 = __dmul_rn(q2, m), a3 = __dmul_rn(q3, m);
    double k = rint(a1);
    double f1 = __dadd_rn(a1, -k);               // exact
    dd t = two_sum(f1, a2);
    t.l = __dadd_rn(t.l, a3);
    return fast_two_sum(t.h, t.l);
}

// exp(2 pi i t) for a dd t with |t| <= 1/2 (+ rounding)
__device__ cdd expi_turns(dd t) {
    double k = rint(__dmul_rn(t.h, 256.0));
    dd f = dd_add_d(t, -k * (1.0 / 256.0));      // |f| <= 1/512
    int idx = ((int)k) & 255;
    dd th = dd_mul(f, dd{SHD_TWOPI_HI, SHD_TWOPI_LO});
    dd x = dd_mul(th, th);
    // cos = sum_{m=0..7} (-1)^m x^m / (2m)!,  sin = th * sum_{m=0..7} (-1)^m x^m / (2m+1)!
    dd c = dd{SHD_INVFACT[14][0], SHD_INVFACT[14][1]};
    dd s = dd{SHD_INVFACT[15][0], SHD_INVFACT[15][1]};
#pragma unroll
    for (int m = 6; m >= 0; m--) {
        c = dd_sub(dd{SHD_INVFACT[2 * m][0], SHD_INVFACT[2 * m][1]}, dd_mul(c, x));
        s = dd_sub(dd{SHD_INVFACT[2 * m + 1][0], SHD_INVFACT[2 * m + 1][1]}, dd_mul(s, x));
    }
    s = dd_mul(s, th);
    cdd w{c, s};
    cdd root{dd{SHD_ROOTS256[idx][0], SHD_ROOTS256[idx][1]}, dd{SHD_ROOTS256[idx][2], SHD_ROOTS256[idx][3]}};
    return cdd_mul(root, w);
}

// z^e by binary powering (start of a chunk of a power table: ~2 log2(e) complex dd products; the phase error of the
// result is e times the base's, as for the recurrence)
__device__ cdd cdd_pow(cdd z, int e) {
    cdd r{dd{1.0, 0.0}, dd{0.0, 0.0}};
    while (e > 0) {
        if (e & 1) r = cdd_mul(r, z);
        e >>= 1;
        if (e) z = cdd_mul(z, z);
    }
    return r;
}

struct limbs { double x0, x1, x2; };

// The 13 balanced base-256 digits d_i in [-128, 127] of X = trunc(x 2^102), x = hi + lo, |x| <= 1 (a few ulps more
// are fine): the bytes of X + sum_i 128 256^i, minus 128 (no carries); sum_i d_i 256^i = X.  X is assembled in two
// 64-bit words split at 2^56: hi 2^46 = H + r (H integer, 0 <= r < 1, both exact), so
// X = H 2^56 + trunc(r 2^56) + trunc(lo 2^102); the last two terms are below 2^57 in magnitude.
// Returned packed: byte i of lo = digit i (i = 0..6), byte i of hi = digit 7 + i (i = 0..5), as s8 bit patterns
// (offset byte - 128 = offset byte ^ 0x80, applied to all bytes of a word at once).
struct digits13_t { unsigned long long lo, hi; };
struct fix102_t { long long lo, hi; };                               // X = hi 2^56 + lo, |lo| < 2^57
__device__ __forceinline__ fix102_t fix102(dd x) {
    const double t = __dmul_rn(x.h, 0x1p46);                       // exact
    const double H = floor(t);
    const double r = __dadd_rn(t, -H);                             // exact, in [0, 1)
    fix102_t f;
    f.lo = __double2ll_rz(__dmul_rn(r, 0x1p56)) + __double2ll_rz(__dmul_rn(x.l, 0x1p102));
    f.hi = __double2ll_rz(H);
    return f;
}
__device__ __forceinline__ digits13_t digits13(fix102_t f) {
    long long xlo = f.lo, xhi = f.hi;
    xlo += 0x80808080808080LL;                                     // digits 0..6 of the offset
    xhi += 0x808080808080LL + (xlo >> 56);                         // digits 7..12, carry (arithmetic shift: may be -1)
    digits13_t d;
    d.lo = ((unsigned long long)xlo & 0xffffffffffffffULL) ^ 0x80808080808080ULL;
    d.hi = ((unsigned long long)xhi & 0xffffffffffffULL) ^ 0x808080808080ULL;
    return d;
}
__device__ __forceinline__ digits13_t digits13(dd x) { return digits13(fix102(x)); }
// The same integer X as sign and magnitude in 128 bits (the INT8 gradient pass contracts its exact integer sums
// with A_j[p] in integer arithmetic, k_grad8.cu): x = |X| low 64 bits, y = |X| high bits | sign << 63.
__device__ __forceinline__ ulonglong2 signmag102(fix102_t f) {
    const __int128 X = ((__int128)f.hi << 56) + (__int128)f.lo;
    const bool neg = X < 0;
    const unsigned __int128 M = neg ? (unsigned __int128)(-X) : (unsigned __int128)X;
    return make_ulonglong2((unsigned long long)M, (unsigned long long)(M >> 64) | (neg ? 0x8000000000000000ULL : 0ULL));
}
__device__ __forceinline__ uint32_t digit_byte(const digits13_t& d, int i) {       // i compile-time after unrolling
    return i < 7 ? (uint32_t)(d.lo >> (8 * i)) & 0xffu : (uint32_t)(d.hi >> (8 * (i - 7))) & 0xffu;
}

// |x| <= 1 (normalised dd) -> limbs (shd_internal.h)
__device__ __forceinline__ limbs split_limbs(dd x) {
    const double C0 = 1.5 * 4503599627370496.0 / (double)(1 << SHD_W0);                 // 1.5 * 2^(52-W0)
    const double C1 = 1.5 * 4503599627370496.0 / ((double)(1 << SHD_W0) * (double)(1 << SHD_W1));
    limbs r;
    r.x0 = __dadd_rn(__dadd_rn(x.h, C0), -C0);
    double rem = __dadd_rn(x.h, -r.x0);          // exact
    r.x1 = __dadd_rn(__dadd_rn(rem, C1), -C1);
    r.x2 = __dadd_rn(__dadd_rn(rem, -r.x1), x.l);
    return r;
}

constexpr int R3MAX = 128;   // d >= 3: max |n_1| supported by the local power table
constexpr int R4MAX = 32;    // d == 4: max |n_2|
constexpr int TB = 64;       // particles (threads) per block
constexpr int TG = 8;        // table entries staged per flush: 8 x 16 B = one 128-byte row per limb plane
constexpr int TABLES_LIMB_SMEM = TB * 3 * TG * 16;
// digit transpose tile: rows of 4 packed digit words x TB particles, padded by 16 bytes so that the 16-byte reads of
// flush8 (eight rows per shared-memory wavefront) fall into eight different bank groups
constexpr int DROW = 4 * TB * 4 + 16;
constexpr int TABLES_SMEM = TABLES_LIMB_SMEM + TG * 2 * DROW;

// Staging tile: a thread owns one particle, so its 16-byte stores would land far apart in global
// memory.  They go to shared memory instead (tile[particle][plane][TG entries], 16-byte chunks
// XOR-swizzled by the bit-reversed particle index: conflict-free for the writes and for both read
// patterns below) and the block then writes runs of 512 contiguous bytes:
//   rho layout       T[block][j/4][limb 3][32 entries][j%4][re,im]            (A and B)
//   gradient layout  Bg[j/32][q/4][limb 3][j%32][q%4][re,im]
// DLO = first digit in use (0, 6 or 9 for 13, 7 or 4 digits, shd_set_precision): lower digit slabs are not written
// LIMBS = false: no FP64 limb table is written (both passes on the INT8 engine): the limb staging is compiled out
template <int DLO, bool LIMBS>
struct Stager {
    double2* tile;        // [TB][planes][TG]
    int planes;           // 3 limbs
    double* table;        // A or B
    double* Bg;           // gradient layout (or nullptr)
    long Npad, j0, N;
    int Qpad;
    // ---- s8 digit tables of the INT8 passes (k_rho8.cu, k_grad8.cu); all in the tensor core's K-major
    // core-matrix layout: 8 rows x 16 bytes per core matrix (128 B contiguous), K-adjacent core matrices
    // 128 B apart, 8-row groups 256 B apart.
    long NpadG;           // particle slots of the gradient-pass tables (multiple of 128)
    signed char* gdig;    // gradient pass, particle operand (B thread only, or nullptr): row = particle % 128 of
    int nkq;              //   block particle / 128, K index = 2 (q % 16) + re/im of K-step q / 16 (nkq per block)
    uint32_t gacc[SHD_I8_DIGITS][4];   // this particle's 16 bytes per digit for the 8 entries of a flush group
    __device__ __forceinline__ void putg8(int slot, const digits13_t& dr, const digits13_t& di) {
        if (gdig == nullptr) return;
        const int w = slot >> 1, sh = (slot & 1) * 16;             // bytes 2 slot (re) and 2 slot + 1 (im)
#pragma unroll
        for (int i = DLO; i < SHD_I8_DIGITS; i++) {
            const uint32_t v = (digit_byte(dr, i) | (digit_byte(di, i) << 8)) << sh;
#pragma unroll
            for (int ww = 0; ww < 4; ww++)
                if (ww == w) gacc[i][ww] = (sh == 0 ? 0u : gacc[i][ww]) | v;
        }
    }
    // q0 = first entry of the group (multiple of 8): one 16-byte store per digit, 8 particles = one 128-byte line
    __device__ __forceinline__ void flushg8(int q0, int count, bool live) {
        if (gdig == nullptr) return;
        const long j = j0 + threadIdx.x;
        if (!live) {
#pragma unroll
            for (int i = DLO; i < SHD_I8_DIGITS; i++) gacc[i][0] = gacc[i][1] = gacc[i][2] = gacc[i][3] = 0u;
        }
        if (j < NpadG) {
            const int row = (int)(j & 127);
            signed char* base = gdig + (((size_t)(j >> 7) * nkq + (size_t)(q0 >> 4)) * SHD_I8_DIGITS) * 4096 +
                                (row >> 3) * 256 + ((q0 >> 3) & 1) * 128 + (row & 7) * 16;
#pragma unroll
            for (int i = DLO; i < SHD_I8_DIGITS; i++) {
                uint4 v = make_uint4(gacc[i][0], gacc[i][1], gacc[i][2], gacc[i][3]);
                if (count < 8) {                                    // ragged tail: entries >= count are zero digits
                    uint32_t* pv = &v.x;
#pragma unroll
                    for (int ww = 0; ww < 4; ww++) {
                        if (2 * ww >= count) pv[ww] = 0u;
                        else if (2 * ww + 1 >= count) pv[ww] &= 0xffffu;
                    }
                }
                *reinterpret_cast<uint4*>(base + (size_t)i * 4096) = v;
            }
        }
    }
    ulonglong2* afix;     // A table of the INT8 gradient pass (or nullptr): [p][NpadA][re, im] sign-magnitude 128-bit integers
    long NpadA;
    __device__ __forceinline__ void put_fix(int p, const fix102_t& fr, const fix102_t& fi, bool live) {
        if (afix == nullptr || j0 + threadIdx.x >= NpadA) return;
        ulonglong2* dst = afix + ((size_t)p * NpadA + j0 + threadIdx.x) * 2;     // a warp writes 1 KB contiguous
        dst[0] = live ? signmag102(fr) : make_ulonglong2(0ULL, 0ULL);
        dst[1] = live ? signmag102(fi) : make_ulonglong2(0ULL, 0ULL);
    }
    signed char* dig;     // rho pass (or nullptr): row = 2 (entry % rows8) + re/im of block entry / rows8,
    long nk8;             //   K index = particle % 32 of K-step particle / 32 (nk8 K-steps per block)
    int rows8;            // entries per block: 64 (A) or 16 (B)
    signed char* dtile;   // shared-memory transpose tile [TG entries][2] rows of DROW bytes: [4 digit words][TB particles] + pad
    // digits of one table entry for both INT8 tables (computed once)
    __device__ __forceinline__ void put_digits(int slot, cdd z, bool live, int entry = -1) {
        if (dig == nullptr && gdig == nullptr && afix == nullptr) return;
        const fix102_t fr = fix102(z.re), fi = fix102(z.im);
        if (entry >= 0) put_fix(entry, fr, fi, live);
        if (dig == nullptr && gdig == nullptr) return;
        digits13_t dr = digits13(fr), di = digits13(fi);
        if (!live) dr.lo = dr.hi = di.lo = di.hi = 0ULL;                            // particles beyond N: zero digits
        put8(slot, dr, di);
        putg8(slot, dr, di);
    }
    // first 32-bit word of the packed digits in use (words: digits 0-3, 4-6, 7-10, 11-12)
    static constexpr int W0 = DLO < 4 ? 0 : DLO < 7 ? 1 : DLO < 11 ? 2 : 3;
    // the packed digit words go to the tile as they are (conflict-free 32-bit stores); flush8 separates the bytes
    __device__ __forceinline__ void put8(int slot, const digits13_t& dr, const digits13_t& di) {
        if (dig == nullptr) return;
        uint32_t* t = reinterpret_cast<uint32_t*>(dtile + (size_t)(slot * 2) * DROW) + threadIdx.x;
        const uint32_t wr[4] = {(uint32_t)dr.lo, (uint32_t)(dr.lo >> 32), (uint32_t)dr.hi, (uint32_t)(dr.hi >> 32)};
        const uint32_t wi[4] = {(uint32_t)di.lo, (uint32_t)(di.lo >> 32), (uint32_t)di.hi, (uint32_t)(di.hi >> 32)};
#pragma unroll
        for (int w = W0; w < 4; w++) {
            t[w * TB] = wr[w];
            t[DROW / 4 + w * TB] = wi[w];
        }
    }
    // after the block-wide barrier of flush(): thread = (row of the group, 16 particles of the block).  Per digit word it
    // reads the 16 particles' words (four 16-byte loads), transposes 4 x 4 bytes by byte permutes (eight per four words) and
    // writes one 16-byte chunk per digit (16 particles of one row of one digit); consecutive threads write consecutive
    // chunks of a 128-byte line (8 rows)
    __device__ __forceinline__ void flush8(int e0, int count) {
        if (dig == nullptr) return;
        const size_t slab = (size_t)rows8 * 2 * 32;
        const int nrow = 2 * count;                                                 // rows of this group
        signed char* base = dig + ((size_t)(e0 / rows8) * nk8 + (size_t)(j0 >> 5)) * SHD_I8_DIGITS * slab;
        const int r_first = 2 * (e0 % rows8);
        static_assert(TB == 2 * TG * (TB / 16), "one pass of the block covers one digit");
        const int rl = threadIdx.x % (2 * TG), kh = threadIdx.x / (2 * TG);
        if (rl < nrow && (j0 >> 5) + (kh >> 1) < nk8) {            // (the last block may reach past the table's K-steps)
            const int r = r_first + rl;
            const uint32_t* src = reinterpret_cast<const uint32_t*>(dtile + (size_t)rl * DROW) + kh * 16;
            signed char* dst = base + (size_t)(kh >> 1) * SHD_I8_DIGITS * slab + (r >> 3) * 256 + (kh & 1) * 128 + (r & 7) * 16;
#pragma unroll
            for (int w = W0; w < 4; w++) {
                constexpr int first[4] = {0, 4, 7, 11};
                uint32_t o[4][4];                                   // o[byte of the word = digit][group of four particles]
#pragma unroll
                for (int g = 0; g < 4; g++) {
                    const uint4 a = *reinterpret_cast<const uint4*>(src + w * TB + 4 * g);
                    const uint32_t t0 = __byte_perm(a.x, a.y, 0x5140), t1 = __byte_perm(a.z, a.w, 0x5140);
                    const uint32_t t2 = __byte_perm(a.x, a.y, 0x7362), t3 = __byte_perm(a.z, a.w, 0x7362);
                    o[0][g] = __byte_perm(t0, t1, 0x5410); o[1][g] = __byte_perm(t0, t1, 0x7632);
                    o[2][g] = __byte_perm(t2, t3, 0x5410); o[3][g] = __byte_perm(t2, t3, 0x7632);
                }
#pragma unroll
                for (int bb = 0; bb < 4; bb++) {
                    const int dg = first[w] + bb;
                    if (dg >= DLO && dg < (w < 3 ? first[w + 1 < 4 ? w + 1 : 3] : SHD_I8_DIGITS))
                        *reinterpret_cast<uint4*>(dst + (size_t)dg * slab) = make_uint4(o[bb][0], o[bb][1], o[bb][2], o[bb][3]);
                }
            }
        }
    }
    __device__ __forceinline__ static int swz(int r) { return ((r & 1) << 2) | (r & 2) | ((r >> 2) & 1); }
    __device__ __forceinline__ void put(int plane0, int slot, cdd z, bool live) {
        if (!LIMBS || (table == nullptr && Bg == nullptr)) return;
        limbs a = split_limbs(z.re), b = split_limbs(z.im);
        if (!live) a.x0 = a.x1 = a.x2 = b.x0 = b.x1 = b.x2 = 0.0;    // particles beyond N: zero limbs (a chunk's table is reused)
        const int t = threadIdx.x, c = slot ^ swz(t);
        double2* row = tile + (t * planes + plane0) * TG;
        row[0 * TG + c] = make_double2(a.x0, b.x0);
        row[1 * TG + c] = make_double2(a.x1, b.x1);
        row[2 * TG + c] = make_double2(a.x2, b.x2);
    }
    // entries e0 .. e0+count-1 (e0 a multiple of TG) of every particle of the block
    __device__ __forceinline__ void flush(int e0, int count, bool live) {
        __syncthreads();
        flush8(e0, count);
        flushg8(e0, count, live);
        const int blk = e0 >> 5, off = e0 & 31;
        // rho layout: (j/4, limb, entry, j%4), j%4 fastest.  Thread = (half of the block's 8-particle rows, entry c,
        // j%4); it walks the 8 row groups and 3 limbs with compile-time strides on both sides (a warp writes 512
        // contiguous bytes per store), so an iteration is one shared load, one global store and a predicate.
        if (LIMBS && table != nullptr) {
            const int t = threadIdx.x, half = t >> 5, jj = t & 3, c = (t >> 2) & 7, r0 = 4 * half + jj;
            const double2* src = tile + r0 * planes * TG + (c ^ swz(r0));
            double2* dst = reinterpret_cast<double2*>(table) +
                           ((((size_t)blk * (Npad / 4) + (j0 >> 2) + half) * 3) * 32 + off + c) * 4 + jj;
            const bool cok = c < count;
#pragma unroll
            for (int a = 0; a < TB / 8; a++) {
                const bool ok = cok && j0 + 8 * a + r0 < Npad;
#pragma unroll
                for (int l = 0; l < 3; l++)
                    if (ok) dst[(size_t)(6 * a + l) * 128] = src[(a * 8 * 3 + l) * TG];
            }
        }
        if (LIMBS && Bg != nullptr) {
            // gradient layout: (j/32, q-group, plane, j%32, q%4), q%4 fastest.  Thread = (j%16, q%4); the walk over
            // (j/32, q-group, plane, upper half of j%32) has compile-time strides on the shared-memory side and
            // loop-invariant ones on the global side
            const int t = threadIdx.x, q4 = t & 3, jl0 = t >> 2;
            const size_t qstride = (size_t)(Qpad / 4) * 3 * 128;          // double2 per 32-particle block
            double2* dstB = reinterpret_cast<double2*>(Bg) + (size_t)(j0 >> 5) * qstride + (size_t)(e0 >> 2) * 3 * 128 +
                            (size_t)jl0 * 4 + q4;
#pragma unroll
            for (int jbl = 0; jbl < TB / 32; jbl++)
#pragma unroll
                for (int u = 0; u < 2; u++) {
                    const int row = jbl * 32 + 16 * u + jl0;
                    const double2* srcB = tile + row * 3 * TG;
                    const int sw = swz(row);
                    const bool jok = j0 + row < N;
#pragma unroll
                    for (int qg = 0; qg < 2; qg++) {
                        const int c = qg * 4 + q4;
                        if (jok && c < count) {
#pragma unroll
                            for (int pl = 0; pl < 3; pl++)
                                dstB[(size_t)jbl * qstride + (size_t)((qg * 3 + pl) * 128 + 64 * u)] = srcB[pl * TG + (c ^ sw)];
                        }
                    }
                }
        }
        __syncthreads();
    }
};

// which = 0: A table.  which = 1: B table (+ the same limbs in the gradient layout Bg).
// HID = true: d >= 3 (A entries are products of per-axis powers kept in local tables); false: d <= 2 (one recurrence)
template <int DLO, bool LIMBS, bool HID>
__global__ void __launch_bounds__(TB, 8) k_tables(
    int d, long N, long j_first, double L, long Npad, int P, int Qn, int S1d, int qscale_log2,
    const int* __restrict__ pn0, const int* __restrict__ pn1, const int* __restrict__ pn2, int Qpad,
    const double* __restrict__ pos_hi, const double* __restrict__ pos_lo,
    double* __restrict__ A, double* __restrict__ B, double* __restrict__ Bg, int with_grad,
    signed char* __restrict__ A8, signed char* __restrict__ B8, long nk8, signed char* __restrict__ Bg8, int nkq8,
    ulonglong2* __restrict__ Afix, long NpadA, int ech, const int* __restrict__ skip)
{
    if (skip && *skip) return;
    // blockIdx.z: chunk of `ech` table entries (a multiple of 8).  With few particles one thread per particle walking the
    // whole table is a long serial recurrence on a mostly idle GPU, so the entries are dealt out over blockIdx.z and every
    // chunk starts from the base's power (cdd_pow); with many particles ech covers the whole table (one chunk).
    const int e_begin = blockIdx.z * ech;
    extern __shared__ __align__(16) unsigned char tables_smem[];
    double2* tile = reinterpret_cast<double2*>(tables_smem);
    const int which = blockIdx.y;
    const long j0 = (long)blockIdx.x * TB;
    const long j = j0 + threadIdx.x;             // slot in the (chunk's) tables; particle j_first + j of the handle
    const bool live = j_first + j < N;
    const long jc = live ? j_first + j : N - 1;  // dead threads shadow the last particle (keeps barriers uniform)
    const cdd one{dd{1.0, 0.0}, dd{0.0, 0.0}};
    const bool gradB = which == 1 && with_grad != 0;
    Stager<DLO, LIMBS> st;
    st.tile = tile; st.planes = 3;
    st.table = which == 0 ? A : B;                      // may be nullptr: the INT8 rho pass does not read B limbs
    st.Bg = gradB ? Bg : nullptr;                       // nullptr too when the gradient pass runs on INT8
    st.Npad = Npad; st.j0 = j0; st.N = N - j_first; st.Qpad = Qpad; st.NpadG = NpadA;
    st.gdig = gradB ? Bg8 : nullptr; st.nkq = nkq8;
    st.dig = which == 0 ? A8 : B8; st.nk8 = nk8; st.rows8 = which == 0 ? SHD_I8_PT : SHD_I8_QT;
    // (the limb staging tile comes first when a limb table is written; the digit transpose tile follows it)
    const bool limb_tile = LIMBS && (A != nullptr || B != nullptr || Bg != nullptr);
    st.dtile = reinterpret_cast<signed char*>(tables_smem) + (limb_tile ? TABLES_LIMB_SMEM : 0);
    st.afix = (which == 0 && with_grad != 0) ? Afix : nullptr; st.NpadA = NpadA;
    if (which == 0) {
        // ---- A table
        cdd base;
        if (d == 1) base = expi_turns(frac_turns(pos_hi[jc], pos_lo[jc], L, (double)S1d));
        else base = expi_turns(frac_turns(pos_hi[jc], pos_lo[jc], L, 1.0));
        const int e_end = min(P, e_begin + ech);
        if (e_begin >= P) return;
        if (!HID) {
            cdd cur = e_begin == 0 ? one : cdd_pow(base, e_begin);
            for (int p0 = e_begin; p0 < e_end; p0 += TG) {
                const int cnt = min(TG, e_end - p0);
                if (cnt == TG) {
                    // full group: slots known at compile time (no selects in the byte staging), and the integer
                    // work of one entry overlaps the serial double-double recurrence of the next
#pragma unroll
                    for (int s = 0; s < TG; s++) {
                        st.put(0, s, cur, live);
                        st.put_digits(s, cur, live, p0 + s);
                        cur = cdd_mul(cur, base);
                    }
                } else {
                    for (int s = 0; s < cnt; s++) {
                        st.put(0, s, cur, live);
                        st.put_digits(s, cur, live, p0 + s);
                        cur = cdd_mul(cur, base);
                    }
                }
                st.flush(p0, cnt, live);
            }
        } else {
            cdd z1 = expi_turns(frac_turns(pos_hi[N + jc], pos_lo[N + jc], L, 1.0));
            cdd pw1[R3MAX + 1];
            int r1max = 0;
            for (int p = e_begin; p < e_end; p++) { int a = abs(pn1[p]); r1max = a > r1max ? a : r1max; }
            pw1[0] = one;
            for (int m = 1; m <= r1max; m++) pw1[m] = cdd_mul(pw1[m - 1], z1);
            cdd pw2[R4MAX + 1];                      // d == 4: powers of the third axis' base phasor
            if (d == 4) {
                cdd z2 = expi_turns(frac_turns(pos_hi[2 * N + jc], pos_lo[2 * N + jc], L, 1.0));
                int r2max = 0;
                for (int p = e_begin; p < e_end; p++) { int a = abs(pn2[p]); r2max = a > r2max ? a : r2max; }
                pw2[0] = one;
                for (int m = 1; m <= r2max; m++) pw2[m] = cdd_mul(pw2[m - 1], z2);
            }
            int n0cur = pn0[e_begin];
            cdd cur0 = n0cur == 0 ? one : cdd_pow(base, n0cur);
            for (int p0 = e_begin; p0 < e_end; p0 += TG) {
                const int cnt = min(TG, e_end - p0);
                for (int s = 0; s < cnt; s++) {
                    const int n0 = pn0[p0 + s], n1 = pn1[p0 + s];
                    while (n0cur < n0) { cur0 = cdd_mul(cur0, base); n0cur++; }
                    cdd f = n1 >= 0 ? pw1[n1] : cdd_conj(pw1[-n1]);
                    if (d == 4) {
                        const int n2 = pn2[p0 + s];
                        f = cdd_mul(f, n2 >= 0 ? pw2[n2] : cdd_conj(pw2[-n2]));
                    }
                    const cdd az = cdd_mul(cur0, f);
                    st.put(0, s, az, live);
                    st.put_digits(s, az, live, p0 + s);
                }
                st.flush(p0, cnt, live);
            }
        }
    } else {
        // ---- B table: powers of the last axis' base phasor
        const int a = d - 1;
        cdd base = expi_turns(frac_turns(pos_hi[(size_t)a * N + jc], pos_lo[(size_t)a * N + jc], L, 1.0));
        const int e_end = min(Qn, e_begin + ech);
        if (e_begin >= Qn) return;
        cdd cur = e_begin == 0 ? one : cdd_pow(base, e_begin);
        for (int q0 = e_begin; q0 < e_end; q0 += TG) {
            const int cnt = min(TG, e_end - q0);
            if (cnt == TG) {
#pragma unroll
                for (int s = 0; s < TG; s++) {
                    st.put(0, s, cur, live);
                    st.put_digits(s, cur, live);
                    cur = cdd_mul(cur, base);
                }
            } else {
                for (int s = 0; s < cnt; s++) {
                    st.put(0, s, cur, live);
                    st.put_digits(s, cur, live);
                    cur = cdd_mul(cur, base);
                }
            }
            st.flush(q0, cnt, live);
        }
    }
}

}  // namespace

cudaError_t shd_tables_configure()
{
    cudaError_t e = cudaSuccess;
#define CONF_TABLES(DLOV)                                                                                                   \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_tables<DLOV, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, TABLES_SMEM);  \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_tables<DLOV, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, TABLES_SMEM);   \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_tables<DLOV, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, TABLES_SMEM); \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_tables<DLOV, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, TABLES_SMEM);
    CONF_TABLES(0)
    CONF_TABLES(6)
    CONF_TABLES(9)
#undef CONF_TABLES
    return e;
}

// what: 1 = the tables of the rho pass, 2 = the tables of the gradient pass (bit mask); j_first = first particle of the chunk
cudaError_t shd_launch_tables(shd_ctx* h, const double* pos_hi, const double* pos_lo, long j_first, int what)
{
    const int e = h->rho_engine;
    const bool rho = (what & 1) != 0, grad = (what & 2) != 0;
    // every slot of the chunk's tables is written (zeros beyond the handle's last particle)
    const long slots = std::max(std::max(h->Npad, h->nk8 * 32), std::max(h->njb128 * 128, h->njb64 * 64));
    // entries per chunk (blockIdx.z): the whole table when the particles alone fill the GPU, else 32- or 16-entry
    // chunks.  Decided from the handle's particle count, not from the size of the tables in use: a chunk start is a
    // binary power, rounded differently from the recurrence, and results must not depend on the workspace cap.
    const int emax = std::max(h->P, h->Qn);
    int ech = ((emax + 7) / 8) * 8;
    // (d >= 3: a chunk start also rebuilds the local power tables, so chunks are twice as long; measured at cfg3: 0.189 ms
    // with 16-entry chunks, 0.178 with 32, 0.176 with 48, 0.203 with 64)
    if (h->N < 96 * 1024 && emax > 32) ech = (h->N < 24 * 1024 && h->d <= 2) ? 16 : 32;
    dim3 grid((unsigned)((slots + TB - 1) / TB), 2, (unsigned)((emax + ech - 1) / ech));
    double* A = (e == 2 || !(rho || grad)) ? nullptr : ((e == 1 && !grad) ? nullptr : h->d_A);   // FP64 rho pass and FP64 gradient pass
    double* B = (e == 0 && rho) ? h->d_B : nullptr;
    double* Bg = (e != 2 && grad) ? h->d_Bg : nullptr;
    signed char* A8 = (e >= 1 && rho) ? h->d_A8 : nullptr;
    signed char* B8 = (e >= 1 && rho) ? h->d_B8 : nullptr;
    signed char* Bg8 = (e == 2 && grad) ? h->d_Bg8 : nullptr;
    ulonglong2* Afix = (e == 2 && grad) ? reinterpret_cast<ulonglong2*>(h->d_Afix) : nullptr;
    // the staging tiles are used by the limb tables and the rho pass's digit tables only: the INT8 gradient pass's
    // tables (Afix, Bg8) go out from registers
    // (8 CTAs of 64 threads per SM by registers; without the 24 KB limb tile the shared memory allows them too)
    const size_t smem = ((A || B || Bg) ? TABLES_LIMB_SMEM : 0) + ((A8 || B8) ? TABLES_SMEM - TABLES_LIMB_SMEM : 0);
    const bool limbs = A || B || Bg, hid = h->d > 2;
#define LAUNCH_TABLES_(DLOV, LV, HV)                                                                               \
    k_tables<DLOV, LV, HV><<<grid, TB, smem, h->stream>>>(h->d, h->N, j_first, h->L, h->Npad, h->P, h->Qn, h->S1d, h->qscale_log2, \
                                         h->d_pn0, h->d_pn1, h->d_pn2, h->Qpad, pos_hi, pos_lo, A, B, Bg, grad ? 1 : 0, \
                                         A8, B8, h->nk8, Bg8, h->nkq8, Afix, h->njb128 * 128, ech, h->d_skip)
#define LAUNCH_TABLES(DLOV)                                                                                       \
    do {                                                                                                          \
        if (limbs) { if (hid) LAUNCH_TABLES_(DLOV, true, true); else LAUNCH_TABLES_(DLOV, true, false); }         \
        else       { if (hid) LAUNCH_TABLES_(DLOV, false, true); else LAUNCH_TABLES_(DLOV, false, false); }       \
    } while (0)
    // the INT8 engines read only the 13, 7 or 4 most significant digits (shd_set_precision): the rest is not written
    if (e == 0 || h->nlimb >= 3) LAUNCH_TABLES(0);
    else if (h->nlimb == 2) LAUNCH_TABLES(6);
    else LAUNCH_TABLES(9);
#undef LAUNCH_TABLES
#undef LAUNCH_TABLES_
    h->last_launches += 1;
    return cudaGetLastError();
}
