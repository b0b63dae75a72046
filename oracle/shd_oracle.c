/*
 * shd_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, binary128 (__float128 / libquadmath) CPU oracle for the hot path of
 * arXiv:2304.09139 (Morse, Kim, Steinhardt, Torquato).  It evaluates the *definitions*
 * of the paper; it shares no code, header, table or constant with the CUDA library in
 * paper_2304_09139_b200/csrc, and nothing in the product path may call it.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs use it.
 *
 * Citations: "P:n" = /root/reference/PAPER.md line n;  "S8c" = SURVEY.md section 8(c);
 * "D:Rn" = reading n in DESIGN.md.
 *
 * Conventions (S8c, D:R1..R3):
 *   box [0,L)^d periodic, integer vector n <-> wavevector k = 2 pi n / L
 *   rho(n)  = sum_j exp(+i k.r_j)         (= conj of the paper's n~(k), Eq. 4)
 *   Phi     = sum_{n in Q} v_n |rho(n)|^2 (Eq. 2 P:39 with the constant dropped)
 *   S(n)    = |rho(n)|^2 / N              (Eq. 3),  S_max = max_{n in Q} S(n)  (Eq. 1)
 *   grad    = dPhi/dr_{j,a} = (4 pi / L) sum_n v_n n_a Im[ exp(-i k.r_j) rho(n) ]
 *             (= -F_j of Eq. 6 P:72 restricted to the half space Q)
 *   Q       = { n in Z^d : 0 < n.n <= m_star, first non-zero component positive },
 *             canonical order = lexicographic ascending, component 0 slowest
 *
 * Positions come as double-double pairs (hi, lo), SoA axis-major: x[a*N + j].
 * Pins: tests/test_oracle_*.py (closed forms, brute force, finite differences, mpmath).
 * Every function below is pinned unless its comment says "parity unpinned".
 */
#include <quadmath.h>
#include <stdlib.h>
#include <string.h>
#include <stdio.h>
#include <math.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef __float128 q128;

/* ------------------------------------------------------------------ helpers */

int shdo_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void shdo_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* pairwise (cascade) summation of x[0..n) in binary128 */
static q128 pairwise_sum(const q128 *x, long n)
{
    if (n <= 8) {
        q128 s = 0;
        for (long i = 0; i < n; i++) s += x[i];
        return s;
    }
    long h = n / 2;
    return pairwise_sum(x, h) + pairwise_sum(x + h, n - h);
}

/* exact promotion of a double-double to binary128 (S8c step 1) */
static inline q128 promote(double hi, double lo) { return (q128)hi + (q128)lo; }

/* conversions used by the Python harness ---------------------------------- */
void shdo_from_dd(long n, const double *hi, const double *lo, q128 *out)
{
    for (long i = 0; i < n; i++) out[i] = promote(hi[i], lo[i]);
}

void shdo_to_dd(long n, const q128 *in, double *hi, double *lo)
{
    for (long i = 0; i < n; i++) {
        double h = (double)in[i];
        hi[i] = h;
        lo[i] = (double)(in[i] - (q128)h);
    }
}

/* out[i] = | (hi[i]+lo[i]) - ref[i] |  rounded to double (for tolerance checks) */
void shdo_absdiff_dd(long n, const q128 *ref, const double *hi, const double *lo, double *out)
{
    for (long i = 0; i < n; i++) out[i] = (double)fabsq(promote(hi[i], lo[i]) - ref[i]);
}

/* out[i] = | (are+i aim) - (bre + i bim) | for complex dd vs complex binary128 */
void shdo_cabsdiff_dd(long n, const q128 *ref_re, const q128 *ref_im,
                      const double *re_hi, const double *re_lo,
                      const double *im_hi, const double *im_lo, double *out)
{
    for (long i = 0; i < n; i++) {
        q128 dr = promote(re_hi[i], re_lo[i]) - ref_re[i];
        q128 di = promote(im_hi[i], im_lo[i]) - ref_im[i];
        out[i] = (double)sqrtq(dr * dr + di * di);
    }
}

/* decimal string of one binary128 value, `digits` significant digits */
void shdo_format(const q128 *x, int digits, char *buf, int buflen)
{
    quadmath_snprintf(buf, (size_t)buflen, "%.*Qe", digits - 1, *x);
}

/* parse a decimal string to binary128 */
void shdo_parse(const char *s, q128 *out) { *out = strtoflt128(s, NULL); }

/* ------------------------------------------------------------- a0: the set Q */

/* is n in the half space: first non-zero component positive (D:R7) */
static int in_half_space(int d, const int *n)
{
    for (int a = 0; a < d; a++) {
        if (n[a] > 0) return 1;
        if (n[a] < 0) return 0;
    }
    return 0; /* n = 0 */
}

/*
 * Enumerate Q for (d, m_star) in canonical order (D:R6-R8).
 * n_out may be NULL (count only); otherwise it receives M*d ints, row-major (k, a).
 * Returns M.
 */
long shdo_enumerate(int d, long m_star, int *n_out)
{
    if (d < 1 || d > 4 || m_star < 1) return -1;
    int R = (int)floor(sqrt((double)m_star));
    while ((long)(R + 1) * (R + 1) <= m_star) R++;
    while ((long)R * R > m_star) R--;
    long M = 0;
    int n[4] = {0, 0, 0, 0};
    int lo1 = (d >= 2) ? -R : 0, hi1 = (d >= 2) ? R : 0;
    int lo2 = (d >= 3) ? -R : 0, hi2 = (d >= 3) ? R : 0;
    int lo3 = (d >= 4) ? -R : 0, hi3 = (d >= 4) ? R : 0;
    for (int n0 = -R; n0 <= R; n0++)
        for (int n1 = lo1; n1 <= hi1; n1++)
            for (int n2 = lo2; n2 <= hi2; n2++)
                for (int n3 = lo3; n3 <= hi3; n3++) {
                    n[0] = n0; n[1] = n1; n[2] = n2; n[3] = n3;
                    long nn = (long)n0 * n0 + (long)n1 * n1 + (long)n2 * n2 + (long)n3 * n3;
                    if (nn == 0 || nn > m_star) continue;
                    if (!in_half_space(d, n)) continue;
                    if (n_out) for (int a = 0; a < d; a++) n_out[M * d + a] = n[a];
                    M++;
                }
    return M;
}

/* ------------------------------------------------ phase of one (particle, n) */

/*
 * theta = 2 pi frac( sum_a n_a r_{j,a} / L ), reduced EXACTLY before the final
 * division (S8c direct mode step 2): n_a*hi and n_a*lo are exact in binary128
 * (<= 32+53 bits), fmodq is exact, the <= 2d reduced pieces are each < L in size.
 */
static inline q128 phase_direct(int d, long N, q128 Lq, const double *pos_hi,
                                const double *pos_lo, long j, const int *n)
{
    q128 acc = 0;
    for (int a = 0; a < d; a++) {
        q128 na = (q128)n[a];
        acc += fmodq(na * (q128)pos_hi[a * N + j], Lq);
        acc += fmodq(na * (q128)pos_lo[a * N + j], Lq);
    }
    q128 t = acc / Lq;
    t -= rintq(t);
    return 2 * M_PIq * t;
}

/* --------------------------------------------------- a2: rho(n), direct mode */

/*
 * rho(n) = sum_j exp(+i k.r_j) for the M vectors n[] (Eq. 4, conjugated: D:R1).
 * One sincosq per (j, n); pairwise summation over j.  rho_re, rho_im: M binary128 each.
 */
void shdo_rho_direct(int d, long N, double L, const double *pos_hi, const double *pos_lo,
                     long M, const int *n, q128 *rho_re, q128 *rho_im)
{
    q128 Lq = (q128)L;
#pragma omp parallel
    {
        q128 *c = (q128 *)malloc(sizeof(q128) * (size_t)N);
        q128 *s = (q128 *)malloc(sizeof(q128) * (size_t)N);
#pragma omp for schedule(dynamic, 4)
        for (long k = 0; k < M; k++) {
            for (long j = 0; j < N; j++) {
                q128 th = phase_direct(d, N, Lq, pos_hi, pos_lo, j, n + k * d);
                sincosq(th, &s[j], &c[j]);
            }
            rho_re[k] = pairwise_sum(c, N);
            rho_im[k] = pairwise_sum(s, N);
        }
        free(c);
        free(s);
    }
}

/* ------------------------------------------------------- a3: Phi and S_max */

/*
 * Phi = sum_n v_n |rho(n)|^2 (Eq. 2; D:R3), S_max = max_n |rho(n)|^2 / N
 * (Eq. 1, Eq. 3; inclusive cutoff D:R4).  v may be NULL (v == 1).
 * s_out (may be NULL) receives |rho(n)|^2 per n.
 */
void shdo_energy(long N, long M, const q128 *rho_re, const q128 *rho_im, const double *v,
                 q128 *phi, q128 *smax, long *argmax, q128 *s_out)
{
    q128 *t = (q128 *)calloc((size_t)(M > 0 ? M : 1), sizeof(q128));
    q128 best = -1;
    long arg = -1;
    for (long k = 0; k < M; k++) {
        q128 s2 = rho_re[k] * rho_re[k] + rho_im[k] * rho_im[k];
        if (s_out) s_out[k] = s2;
        t[k] = (v ? (q128)v[k] : (q128)1) * s2;
        if (s2 > best) { best = s2; arg = k; }
    }
    *phi = pairwise_sum(t, M);
    *smax = (M > 0) ? best / (q128)N : 0;
    if (argmax) *argmax = arg;
    free(t);
}

/* -------------------------------------------------- a4: gradient, direct mode */

/*
 * dPhi/dr_{j,a} = (4 pi / L) sum_n v_n n_a ( cos(th) Im rho(n) - sin(th) Re rho(n) ),
 * th = k.r_j  (Eq. 6 P:72 with F = -grad, half-space sum; D:R2).
 * Evaluated for the nj particles jlist[] (or all N when jlist == NULL, nj == N);
 * grad is axis-major over the evaluated subset: grad[a*nj + i].
 */
void shdo_grad_direct(int d, long N, double L, const double *pos_hi, const double *pos_lo,
                      long M, const int *n, const double *v, const q128 *rho_re,
                      const q128 *rho_im, long nj, const long *jlist, q128 *grad)
{
    q128 Lq = (q128)L;
    q128 pref = 4 * M_PIq / Lq;
#pragma omp parallel
    {
        q128 *t = (q128 *)malloc(sizeof(q128) * (size_t)M * (size_t)d);
#pragma omp for schedule(dynamic, 4)
        for (long i = 0; i < nj; i++) {
            long j = jlist ? jlist[i] : i;
            for (long k = 0; k < M; k++) {
                q128 th = phase_direct(d, N, Lq, pos_hi, pos_lo, j, n + k * d);
                q128 s, c;
                sincosq(th, &s, &c);
                q128 w = (v ? (q128)v[k] : (q128)1) * (c * rho_im[k] - s * rho_re[k]);
                for (int a = 0; a < d; a++) t[a * M + k] = (q128)n[k * d + a] * w;
            }
            for (int a = 0; a < d; a++) grad[a * nj + i] = pref * pairwise_sum(t + a * M, M);
        }
        free(t);
    }
}

/* ------------------------------------------------------------ factored mode */

/*
 * Factored mode (S8c): the same definition, but exp(i k.r_j) = prod_a E_a[n_a] with every
 * table entry E_a[m] = exp(2 pi i frac(m r_{j,a} / L)) evaluated DIRECTLY by a reduced
 * sincosq (no recurrence).  d = 1 uses n = 256 c + b with two directly evaluated tables.
 * Only there to make N ~ 1e5 affordable; validated against direct mode in tests.
 */
static inline void axis_phasor(q128 Lq, double hi, double lo, long m, q128 *c, q128 *s)
{
    q128 mq = (q128)m;
    q128 acc = fmodq(mq * (q128)hi, Lq) + fmodq(mq * (q128)lo, Lq);
    q128 t = acc / Lq;
    t -= rintq(t);
    sincosq(2 * M_PIq * t, s, c);
}

typedef struct {
    int d;
    long R;       /* max |n_a| */
    long stride;  /* entries per axis table */
    int split1d;  /* d == 1: two-level tables */
} fact_shape;

static fact_shape fact_shape_of(int d, long M, const int *n)
{
    fact_shape f;
    long R = 0;
    for (long i = 0; i < M * d; i++) { long v = labs((long)n[i]); if (v > R) R = v; }
    f.d = d; f.R = R; f.split1d = (d == 1);
    f.stride = (d == 1) ? 0 : (2 * R + 1);
    return f;
}

/* fill per-particle tables; tc/ts sized d*(2R+1) for d>=2, (256 + R/256+1) for d==1 */
static void fill_tables(const fact_shape *f, long N, q128 Lq, const double *pos_hi,
                        const double *pos_lo, long j, q128 *tc, q128 *ts)
{
    if (f->split1d) {
        long nc = f->R / 256 + 1;
        for (long b = 0; b < 256; b++) axis_phasor(Lq, pos_hi[j], pos_lo[j], b, &tc[b], &ts[b]);
        for (long c = 0; c < nc; c++)
            axis_phasor(Lq, pos_hi[j], pos_lo[j], 256 * c, &tc[256 + c], &ts[256 + c]);
    } else {
        for (int a = 0; a < f->d; a++)
            for (long m = -f->R; m <= f->R; m++)
                axis_phasor(Lq, pos_hi[a * N + j], pos_lo[a * N + j], m,
                            &tc[a * f->stride + m + f->R], &ts[a * f->stride + m + f->R]);
    }
}

static inline void table_phasor(const fact_shape *f, const q128 *tc, const q128 *ts,
                                const int *n, q128 *c, q128 *s)
{
    if (f->split1d) {
        long m = n[0];
        long hi = m / 256, lo = m % 256; /* m > 0 in the d=1 half space */
        q128 c1 = tc[256 + hi], s1 = ts[256 + hi], c2 = tc[lo], s2 = ts[lo];
        *c = c1 * c2 - s1 * s2;
        *s = c1 * s2 + s1 * c2;
    } else {
        q128 cr = tc[n[0] + f->R], sr = ts[n[0] + f->R];
        for (int a = 1; a < f->d; a++) {
            q128 c2 = tc[a * f->stride + n[a] + f->R], s2 = ts[a * f->stride + n[a] + f->R];
            q128 nr = cr * c2 - sr * s2;
            sr = cr * s2 + sr * c2;
            cr = nr;
        }
        *c = cr; *s = sr;
    }
}

static long table_len(const fact_shape *f)
{
    return f->split1d ? (256 + f->R / 256 + 1) : (long)f->d * f->stride;
}

/*
 * rho(n) for all n, factored mode.  Loops j outermost (tables per particle), accumulating
 * per-thread partial sums in blocks of particles that are then pairwise-combined.
 */
void shdo_rho_factored(int d, long N, double L, const double *pos_hi, const double *pos_lo,
                       long M, const int *n, q128 *rho_re, q128 *rho_im)
{
    q128 Lq = (q128)L;
    fact_shape f = fact_shape_of(d, M, n);
    long tl = table_len(&f);
    const long BLK = 64; /* particles per partial sum */
    long nblk = (N + BLK - 1) / BLK;
    q128 *pre = (q128 *)calloc((size_t)nblk * (size_t)M, sizeof(q128));
    q128 *pim = (q128 *)calloc((size_t)nblk * (size_t)M, sizeof(q128));
#pragma omp parallel
    {
        q128 *tc = (q128 *)malloc(sizeof(q128) * (size_t)tl);
        q128 *ts = (q128 *)malloc(sizeof(q128) * (size_t)tl);
#pragma omp for schedule(dynamic, 1)
        for (long b = 0; b < nblk; b++) {
            long j1 = (b + 1) * BLK < N ? (b + 1) * BLK : N;
            for (long j = b * BLK; j < j1; j++) {
                fill_tables(&f, N, Lq, pos_hi, pos_lo, j, tc, ts);
                for (long k = 0; k < M; k++) {
                    q128 c, s;
                    table_phasor(&f, tc, ts, n + k * d, &c, &s);
                    pre[b * M + k] += c;
                    pim[b * M + k] += s;
                }
            }
        }
        free(tc);
        free(ts);
    }
#pragma omp parallel
    {
        q128 *t = (q128 *)malloc(sizeof(q128) * (size_t)nblk);
#pragma omp for
        for (long k = 0; k < M; k++) {
            for (long b = 0; b < nblk; b++) t[b] = pre[b * M + k];
            rho_re[k] = pairwise_sum(t, nblk);
            for (long b = 0; b < nblk; b++) t[b] = pim[b * M + k];
            rho_im[k] = pairwise_sum(t, nblk);
        }
        free(t);
    }
    free(pre);
    free(pim);
}

/* gradient for all particles (or a subset), factored mode */
void shdo_grad_factored(int d, long N, double L, const double *pos_hi, const double *pos_lo,
                        long M, const int *n, const double *v, const q128 *rho_re,
                        const q128 *rho_im, long nj, const long *jlist, q128 *grad)
{
    q128 Lq = (q128)L;
    q128 pref = 4 * M_PIq / Lq;
    fact_shape f = fact_shape_of(d, M, n);
    long tl = table_len(&f);
#pragma omp parallel
    {
        q128 *tc = (q128 *)malloc(sizeof(q128) * (size_t)tl);
        q128 *ts = (q128 *)malloc(sizeof(q128) * (size_t)tl);
        q128 *t = (q128 *)malloc(sizeof(q128) * (size_t)M * (size_t)d);
#pragma omp for schedule(dynamic, 4)
        for (long i = 0; i < nj; i++) {
            long j = jlist ? jlist[i] : i;
            fill_tables(&f, N, Lq, pos_hi, pos_lo, j, tc, ts);
            for (long k = 0; k < M; k++) {
                q128 c, s;
                table_phasor(&f, tc, ts, n + k * d, &c, &s);
                q128 w = (v ? (q128)v[k] : (q128)1) * (c * rho_im[k] - s * rho_re[k]);
                for (int a = 0; a < d; a++) t[a * M + k] = (q128)n[k * d + a] * w;
            }
            for (int a = 0; a < d; a++) grad[a * nj + i] = pref * pairwise_sum(t + a * M, M);
        }
        free(tc);
        free(ts);
        free(t);
    }
}

/* --------------------------------------------- whole evaluation, convenience */

/*
 * One energy+gradient evaluation on binary128 positions x[a*N+j] (used by the minimizer
 * and the finite-difference pins).  mode 0 = direct, 1 = factored.
 * Positions are split into (hi, lo) doubles first, which is exact when x came from a dd
 * and otherwise rounds at 2^-106 relative -- the same input class the CUDA path sees.
 */
void shdo_eval_q(int d, long N, double L, const q128 *x, long M, const int *n, const double *v,
                 int mode, q128 *phi, q128 *smax, long *argmax, q128 *grad /* may be NULL */)
{
    double *hi = (double *)malloc(sizeof(double) * (size_t)N * d);
    double *lo = (double *)malloc(sizeof(double) * (size_t)N * d);
    shdo_to_dd(N * d, x, hi, lo);
    q128 *re = (q128 *)malloc(sizeof(q128) * (size_t)M);
    q128 *im = (q128 *)malloc(sizeof(q128) * (size_t)M);
    if (mode == 0) shdo_rho_direct(d, N, L, hi, lo, M, n, re, im);
    else shdo_rho_factored(d, N, L, hi, lo, M, n, re, im);
    shdo_energy(N, M, re, im, v, phi, smax, argmax, NULL);
    if (grad) {
        if (mode == 0) shdo_grad_direct(d, N, L, hi, lo, M, n, v, re, im, N, NULL, grad);
        else shdo_grad_factored(d, N, L, hi, lo, M, n, v, re, im, N, NULL, grad);
    }
    free(hi); free(lo); free(re); free(im);
}

/* ------------------------------------------------------- a5: L-BFGS oracle */

static q128 qdot(long n, const q128 *a, const q128 *b)
{
    q128 s = 0;
    for (long i = 0; i < n; i++) s += a[i] * b[i];
    return s;
}

/*
 * Textbook L-BFGS in binary128 (S8c "Minimization oracle"; D:R12, R13): two-loop recursion,
 * history m, H0 = gamma I with gamma = s.y / y.y, backtracking Armijo (c1 = 1e-4, start at
 * step 1, halve), pair skipped when s.y <= 0, first step length 1/|g|; stops when
 * S_max < smax_tol, after max_evals evaluations, or when 40 halvings find no decrease.
 * x (in/out): binary128 positions x[a*N+j].  Outcome is compared, never the trajectory
 * (the ground-state manifold is degenerate) -- "several correct results".
 * Returns 0 converged, 1 max_evals, 2 line-search stall.  report = {iters, evals}.
 */
int shdo_minimize_lbfgs(int d, long N, double L, q128 *x, long M, const int *n, const double *v,
                        int mode, int m, double smax_tol, long max_evals, long *report,
                        q128 *phi_out, q128 *smax_out)
{
    long nd = N * d;
    q128 *g = (q128 *)malloc(sizeof(q128) * nd), *gn = (q128 *)malloc(sizeof(q128) * nd);
    q128 *xn = (q128 *)malloc(sizeof(q128) * nd), *p = (q128 *)malloc(sizeof(q128) * nd);
    q128 *S = (q128 *)malloc(sizeof(q128) * nd * m), *Y = (q128 *)malloc(sizeof(q128) * nd * m);
    q128 *rho_h = (q128 *)malloc(sizeof(q128) * m), *alpha = (q128 *)malloc(sizeof(q128) * m);
    q128 phi, smax, phin, smaxn;
    long arg, evals = 0, iters = 0;
    int hist = 0, head = 0, status = 1;
    shdo_eval_q(d, N, L, x, M, n, v, mode, &phi, &smax, &arg, g); evals++;
    while (1) {
        if ((double)smax < smax_tol) { status = 0; break; }
        if (evals >= max_evals) { status = 1; break; }
        /* two-loop recursion: p = -H g */
        for (long i = 0; i < nd; i++) p[i] = g[i];
        for (int t = 0; t < hist; t++) {
            int idx = (head - 1 - t + 2 * m) % m;
            alpha[idx] = rho_h[idx] * qdot(nd, S + (long)idx * nd, p);
            for (long i = 0; i < nd; i++) p[i] -= alpha[idx] * Y[(long)idx * nd + i];
        }
        q128 gamma;
        if (hist > 0) {
            int idx = (head - 1 + m) % m;
            gamma = qdot(nd, S + (long)idx * nd, Y + (long)idx * nd) /
                    qdot(nd, Y + (long)idx * nd, Y + (long)idx * nd);
        } else {
            gamma = 1 / sqrtq(qdot(nd, g, g));
        }
        for (long i = 0; i < nd; i++) p[i] *= gamma;
        for (int t = hist - 1; t >= 0; t--) {
            int idx = (head - 1 - t + 2 * m) % m;
            q128 beta = rho_h[idx] * qdot(nd, Y + (long)idx * nd, p);
            for (long i = 0; i < nd; i++) p[i] += (alpha[idx] - beta) * S[(long)idx * nd + i];
        }
        for (long i = 0; i < nd; i++) p[i] = -p[i];
        q128 gp = qdot(nd, g, p);
        if (gp >= 0) { /* not a descent direction: restart with steepest descent */
            hist = 0; head = 0;
            q128 gg = qdot(nd, g, g);
            for (long i = 0; i < nd; i++) p[i] = -g[i] / sqrtq(gg);
            gp = qdot(nd, g, p);
        }
        /* backtracking Armijo */
        q128 step = 1;
        int ok = 0;
        for (int ls = 0; ls < 40 && evals < max_evals; ls++) {
            for (long i = 0; i < nd; i++) xn[i] = x[i] + step * p[i];
            shdo_eval_q(d, N, L, xn, M, n, v, mode, &phin, &smaxn, &arg, gn); evals++;
            if (phin <= phi + (q128)1e-4 * step * gp) { ok = 1; break; }
            step /= 2;
        }
        if (!ok) { status = (evals >= max_evals) ? 1 : 2; break; }
        /* history update */
        q128 *s = S + (long)head * nd, *y = Y + (long)head * nd;
        for (long i = 0; i < nd; i++) { s[i] = xn[i] - x[i]; y[i] = gn[i] - g[i]; }
        q128 sy = qdot(nd, s, y);
        if (sy > 0) { rho_h[head] = 1 / sy; head = (head + 1) % m; if (hist < m) hist++; }
        memcpy(x, xn, sizeof(q128) * nd);
        memcpy(g, gn, sizeof(q128) * nd);
        phi = phin; smax = smaxn; iters++;
    }
    report[0] = iters; report[1] = evals;
    *phi_out = phi; *smax_out = smax;
    free(g); free(gn); free(xn); free(p); free(S); free(Y); free(rho_h); free(alpha);
    return status;
}

/* ---------------------------------------------------------- a5: FIRE oracle */

/*
 * FIRE ("fast inertial relaxation engine", the minimizer the paper uses: P:75, ref.[37] P:152)
 * in binary128.  The paper restates none of its parameters (D:R12), so this is the published
 * algorithm with its published defaults, written out step by step; unit masses, force
 * F = -grad Phi, semi-implicit Euler as the MD integrator:
 *     evaluate F(x)
 *     P = F.v
 *     if P > 0:  v <- (1-alpha) v + alpha |v| F/|F|;
 *                if more than N_min = 5 steps since the last P <= 0:
 *                    dt <- min(dt f_inc, dt_max), alpha <- alpha f_alpha      (f_inc 1.1, f_alpha 0.99)
 *     else:      v <- 0, dt <- dt f_dec, alpha <- alpha_start                 (f_dec 0.5, alpha_start 0.1)
 *     v <- v + dt F;  x <- x + dt v
 * dt starts at dt0, dt_max = 10 dt0.  Stops when S_max < smax_tol (checked on every
 * evaluation, before the move) or after max_evals evaluations.  Like the L-BFGS oracle it is
 * compared by OUTCOME only.  Returns 0 converged, 1 max_evals, 3 non-finite Phi.
 * report = {steps, evals}.
 */
int shdo_minimize_fire(int d, long N, double L, q128 *x, long M, const int *n, const double *v,
                       int mode, double dt0, double smax_tol, long max_evals, long *report,
                       q128 *phi_out, q128 *smax_out)
{
    const long nd = N * d;
    /* the parameters are the DOUBLES nearest to 1.1, 0.5, 0.1, 0.99 (what a caller can pass) */
    const q128 f_inc = (q128)1.1, f_dec = (q128)0.5, alpha_start = (q128)0.1, f_alpha = (q128)0.99;
    const int n_min = 5;
    q128 *g = (q128 *)malloc(sizeof(q128) * nd), *vel = (q128 *)calloc(nd, sizeof(q128));
    q128 phi = 0, smax = 0, dt = dt0, dt_max = (q128)(10.0 * dt0), alpha = alpha_start;
    long arg, evals = 0, steps = 0, since = 0;
    int status = 1;
    while (1) {
        shdo_eval_q(d, N, L, x, M, n, v, mode, &phi, &smax, &arg, g); evals++;
        if (!finiteq(phi)) { status = 3; break; }
        if ((double)smax < smax_tol) { status = 0; break; }
        if (evals >= max_evals) { status = 1; break; }
        q128 P = 0, vv = 0, ff = 0;
        for (long i = 0; i < nd; i++) { P -= g[i] * vel[i]; vv += vel[i] * vel[i]; ff += g[i] * g[i]; }
        if (P > 0) {
            q128 c = (ff > 0) ? alpha * sqrtq(vv / ff) : 0;
            for (long i = 0; i < nd; i++) vel[i] = (1 - alpha) * vel[i] - c * g[i];
            if (since > n_min) {
                dt = dt * f_inc; if (dt > dt_max) dt = dt_max;
                alpha *= f_alpha;
            }
            since++;
        } else {
            for (long i = 0; i < nd; i++) vel[i] = 0;
            dt *= f_dec; alpha = alpha_start; since = 0;
        }
        for (long i = 0; i < nd; i++) { vel[i] -= dt * g[i]; x[i] += dt * vel[i]; }
        steps++;
    }
    report[0] = steps; report[1] = evals;
    *phi_out = phi; *smax_out = smax;
    free(g); free(vel);
    return status;
}

/* ------------------------------------------------ NEXT-3: S(k) and the tau lattice sum */

/*
 * Structure factor S(k) = |rho(k)|^2 / N (Eq. 3) for the M given wavevectors and
 * dev2 = sum_k (S(k) - 1)^2, the lattice sum behind the order metric of Eq. 7:
 * with int dk -> (2 pi)^d / V sum over all non-zero k (= twice the half-space sum) and
 * rho = N / V, D = 1/K:  tau = K^d V / N^2 * 2 * dev2.
 */
void shdo_structure_factor(long N, long M, const q128 *rho_re, const q128 *rho_im, q128 *S, q128 *dev2)
{
    q128 *t = (q128 *)malloc(sizeof(q128) * (size_t)M);
    for (long k = 0; k < M; k++) {
        S[k] = (rho_re[k] * rho_re[k] + rho_im[k] * rho_im[k]) / (q128)N;
        t[k] = (S[k] - 1) * (S[k] - 1);
    }
    *dev2 = pairwise_sum(t, M);
    free(t);
}

/*
 * Radially averaged structure factor (Fig. 2a, Fig. S1a: S(k) against |k|, beyond K too when the wavevector
 * set reaches there).  |k|^2 = (2 pi / L)^2 n.n, so a radial bin is a range of the INTEGER n.n: bin b collects the
 * wavevectors with edges[b] <= n.n < edges[b+1] (edges ascending, nbins + 1 of them); count[b] = how many,
 * S_mean[b] = (sum of S(k) over them) / count[b] (0 for an empty bin).  Only half-space vectors are listed, and
 * S(-k) = S(k), so the mean over the half shell is the mean over the whole shell.  Plain loops, binary128.
 */
void shdo_structure_factor_shells(int d, long N, long M, const int *n, const q128 *rho_re, const q128 *rho_im,
                                  long nbins, const long *edges, long *count, q128 *S_mean)
{
    for (long b = 0; b < nbins; b++) { count[b] = 0; S_mean[b] = 0; }
    for (long k = 0; k < M; k++) {
        long nn = 0;
        for (int a = 0; a < d; a++) nn += (long)n[k * d + a] * (long)n[k * d + a];
        const q128 S = (rho_re[k] * rho_re[k] + rho_im[k] * rho_im[k]) / (q128)N;
        for (long b = 0; b < nbins; b++)
            if (edges[b] <= nn && nn < edges[b + 1]) { count[b]++; S_mean[b] += S; break; }
    }
    for (long b = 0; b < nbins; b++)
        if (count[b] > 0) S_mean[b] /= (q128)count[b];
}
