/*
 * shd.h -- C-ABI boundary of the B200-native stealthy-hyperuniform hot path
 *          (arXiv:2304.09139, Morse, Kim, Steinhardt, Torquato).
 *
 * "P:n" = /root/reference/PAPER.md line n.  "D:Rn" = reading n in DESIGN.md.
 *
 * What the library computes (one periodic box [0,L)^d, N point particles):
 *   Q      = { n in Z^d : 0 < n.n <= m_star, first non-zero component of n positive }   (D:R6-R8)
 *            wavevector k = 2 pi n / L; canonical order = lexicographic ascending, n_0 slowest (D:R7)
 *   rho(k) = sum_j exp(+i k.r_j)               (= complex conjugate of n~(k), Eq. 4; D:R1)
 *   Phi    = sum_{k in Q} v(k) |rho(k)|^2      (Eq. 2 P:39 with the structure-independent constant dropped; D:R3)
 *   S_max  = max_{k in Q} |rho(k)|^2 / N       (Eq. 1 P:27 with Eq. 3; inclusive cutoff D:R4)
 *   grad   = dPhi/dr_{j,a} = (4 pi / L) sum_{k in Q} v(k) n_a Im[ exp(-i k.r_j) rho(k) ]
 *            (= -F_j of Eq. 6; the true derivative, D:R2)
 * all in double-double (~106-bit) accuracy ("tunable precision using double-doubles").
 *
 * Conventions
 *   - Every function returns int: SHD_OK (0) or a negative SHD_E* code; nothing throws.
 *   - pos_*, grad_*, and the four shd_get_rho outputs are DEVICE pointers (cudaMalloc'ed memory,
 *     e.g. torch tensors' data_ptr()), owned by the caller, never retained after the call returns.
 *     Everything else (phi, smax, n_out, v, reports) is HOST memory.
 *   - dd values are (hi, lo) pairs of doubles, value = hi + lo.  Layout of particle vectors is
 *     SoA axis-major: x[a*N + j] = component a of particle j  (two arrays: *_hi and *_lo).
 *     Any finite position is valid (Phi is L-periodic, D:R10); |lo| <= ulp(hi)/2 is expected.
 *   - Work is enqueued on the handle's stream; calls that return a scalar synchronise that stream.
 *   - A handle is not thread-safe; different handles are independent.  No global state.
 *   - There is no CPU fallback: without a CUDA device every compute call returns SHD_ECUDA.
 */
#ifndef SHD_H
#define SHD_H

#ifdef __cplusplus
extern "C" {
#endif

#define SHD_OK        0
#define SHD_EINVAL   -1   /* bad d / N / L / K / m_star / NULL pointer / option            */
#define SHD_ENOMEM   -2   /* host or device allocation failed                              */
#define SHD_ECUDA    -3   /* CUDA runtime error; text in shd_last_error()                  */
#define SHD_ENAN     -4   /* non-finite position or non-finite Phi                         */
#define SHD_ESTALL   -5   /* shd_minimize: line search found no decrease (report written)  */
#define SHD_EMAXEVAL -6   /* shd_minimize: max_evals reached before smax_tol (report written) */

typedef struct shd_ctx shd_ctx;

/*
 * Create a handle for dimension d in {1,2,3,4} (d = 4: m_star <= 1024), N >= 1 particles, box edge
 * L > 0, cutoff K > 0:
 *   m_star = floor( (K L / 2 pi)^2 (1 + 2^-40) ),  Q as above  (integer compare, D:R8).
 * v: HOST pointer to |Q| strictly positive weights v(k) in canonical order, or NULL
 * for v == 1.  The handle owns all device workspaces (phasor tables, rho, partial sums, minimizer
 * state).  *out receives the handle.  Errors: SHD_EINVAL, SHD_ENOMEM, SHD_ECUDA.
 */
int shd_create(int d, long N, double L, double K, const double* v, shd_ctx** out);

/* Same, with the integer shell cutoff n.n <= m_star given directly (no FP compare, D:R8). */
int shd_create_shell(int d, long N, double L, long m_star, const double* v, shd_ctx** out);

/*
 * The same with the caller's own wavevector set ("anisotropic exclusion regions"; SURVEY.md 8(f)
 * NEXT-4): n (HOST, M*d ints, row-major (k,a)) lists M distinct non-zero integer vectors, each in the half
 * space of D:R7 (first non-zero component positive); k = 2 pi n / L.  The given order is the canonical
 * order of this handle (v, shd_get_k, shd_get_rho, argmax).  Limits: |n_a| <= 2000 for d >= 2 (|n_1| <= 128
 * for d >= 3, |n_2| <= 32 for d = 4), n <= 2e6 for d = 1.  Errors: SHD_EINVAL (bad argument, vector outside the half space,
 * duplicate), SHD_ENOMEM, SHD_ECUDA.
 */
int shd_create_table(int d, long N, double L, long M, const int* n, const double* v, shd_ctx** out);

void shd_destroy(shd_ctx* h);

/* Use CUDA stream `cuda_stream` (a cudaStream_t) for all later work; default is stream 0. */
int shd_set_stream(shd_ctx* h, void* cuda_stream);

/* |Q| = M, the number of independent constraints. */
long shd_num_k(const shd_ctx* h);

/* Copy the integer vectors n of Q to HOST n_out[|Q|*d], row-major (k, a), canonical order. */
int shd_get_k(const shd_ctx* h, int* n_out);

/*
 * One energy + gradient evaluation (Eq. 4, 2, 6; "2 calculations, each with M N terms").
 *   pos_hi, pos_lo : DEVICE, d*N doubles each (in).
 *   phi            : HOST, phi[0] = hi, phi[1] = lo (out).
 *   grad_hi, grad_lo: DEVICE, d*N doubles each (out); both NULL to skip the gradient pass.
 * Side effect: rho(k) of these positions stays in the handle (shd_get_rho), as do S_max and
 * its argmax (shd_last_smax).
 */
int shd_energy_grad(shd_ctx* h, const double* pos_hi, const double* pos_lo,
                    double phi[2], double* grad_hi, double* grad_lo);

/*
 * The same evaluation for a caller whose data lives in HOST memory: pos_hi, pos_lo (in) and
 * grad_hi, grad_lo (out, both NULL to skip the gradient) are HOST pointers to d*N doubles each
 * (pinned memory makes the copies faster but is not required).  The library copies the positions
 * to a device staging buffer it owns, runs shd_energy_grad, and copies the gradient back; the call
 * returns when the results are in host memory.
 */
int shd_energy_grad_host(shd_ctx* h, const double* pos_hi, const double* pos_lo,
                         double phi[2], double* grad_hi, double* grad_lo);

/* S_max (Eq. 1) of the given positions: smax[0..1] = (hi, lo) on the HOST, *argmax_k = index
 * into the canonical order (may be NULL).  Runs the rho pass and the reduction only. */
int shd_smax(shd_ctx* h, const double* pos_hi, const double* pos_lo, double smax[2], long* argmax_k);

/* S_max / argmax of the LAST evaluation on this handle (no device work besides a 32-byte copy). */
int shd_last_smax(shd_ctx* h, double smax[2], long* argmax_k);

/* rho(k) of the LAST evaluation: four DEVICE arrays of |Q| doubles each, canonical order. */
int shd_get_rho(shd_ctx* h, double* re_hi, double* re_lo, double* im_hi, double* im_lo);

/*
 * "Tunable precision".  limbs = 3 (default): the products of the two O(N M) sums carry ~98 bits
 * (double-double results; BASELINE.json's tolerances).  limbs = 2: "fast" evaluations for the early part of a
 * quench (precision ladder): the phasor and rho operands are used at 44 bits
 * (two exact limbs), half the FMAs; per-term error ~2^-45, i.e. |rho| to ~3e-14 sqrt(N), enough to drive
 * S_max to ~1e-22.  limbs = 1: operands at 22 bits (one exact limb), one sixth of the FMAs, per-term error
 * ~2^-23: the first decades of a quench (S_max down to ~1e-10).  Everything else (phasor tables, reductions,
 * minimizer algebra) stays double-double.  On the INT8 engines (shd_set_engine) the same three levels select
 * the 13, 7 or 4 most significant base-256 digits of the operands (102, 54, 30 bits; 91, 28, 10 digit pairs).
 * Applies to every later call on the handle.  Errors: SHD_EINVAL (limbs not 1, 2 or 3).
 */
int shd_set_precision(shd_ctx* h, int limbs);

/*
 * Engine of the rho pass (step a2).  0 (default): exact FP64 limb contraction on the FP64 matrix instruction
 * (k_rho.cu).  1: exact digit-sliced contraction on the INT8 tensor cores (tcgen05.mma.kind::i8, k_rho8.cu):
 * operands as 13 balanced base-256 digits of trunc(x 2^102), the 91 digit pairs with i + l >= 12, s32
 * accumulators in tensor memory (at most 8192 particles per CTA, so they are exact), the same double-double
 * result within the same tolerances.  2: the gradient pass too (k_grad8.cu).  shd_set_precision selects the
 * number of digits on these engines.  Allocates the digit tables on first use.  Errors: SHD_EINVAL (engine not
 * 0, 1 or 2; engine 2 with more than 5024 entries in the last-axis table: its s32 sums would not be exact),
 * SHD_ENOMEM, SHD_ECUDA.
 */
int shd_set_engine(shd_ctx* h, int rho_engine);

/*
 * Structure factor of the LAST evaluation on this handle (Eq. 3): S(k) = |rho(k)|^2 / N for every k
 * of the handle's Q, canonical order, into S_out (DEVICE, |Q| doubles; may be NULL), and
 * dev2 (HOST, (hi, lo)) = sum_{k in Q} (S(k) - 1)^2 in double-double, the lattice sum behind the order
 * metric tau of Eq. 7:  tau = K^d V / N^2 * 2 * dev2  for a handle whose Q reaches far enough
 * beyond K that S has decayed to 1 (the factor 2 counts -k; V = L^d; D = 1/K).  Create a second handle
 * with a larger cutoff for this (S(k > K) and tau are SURVEY.md 8(f) NEXT-3; FP64 would suffice there,
 * the dd kernels are simply reused).  Synchronises the stream.
 */
int shd_structure_factor(shd_ctx* h, double* S_out, double dev2[2]);

typedef struct {
    int    kind;        /* 0 = L-BFGS (D:R12); 1 = FIRE                               */
    int    history;     /* L-BFGS pairs kept (1..32); 0 = default 10                          */
    double smax_tol;    /* stop when S_max < smax_tol (D:R13); e.g. 1e-30                     */
    long   max_evals;   /* stop after this many energy+gradient evaluations                   */
    int    poll_every;  /* host reads the device status word every this many iterations (>=1) */
    double fire_dt0;    /* FIRE only: initial time step (dt_max = 10 dt0); 0 = default
                           0.1 / (k_max sqrt(2 N max v)): dt_max is half the explicit stability bound */
    int    resume;      /* FIRE only: 1 = continue the previous call on this handle (same positions
                           buffer content as it left): keep velocities, dt, alpha; 0 = fresh start    */
} shd_min_opts;

typedef struct {
    long   iters, evals;
    double phi[2], smax[2];
    int    status;      /* SHD_OK, SHD_ESTALL, SHD_EMAXEVAL, SHD_ENAN */
} shd_min_report;

/*
 * Quench: minimise Phi from pos (DEVICE, in/out, d*N doubles each) until S_max < smax_tol.
 * The whole iteration (evaluations, dd vector algebra, line search decisions) runs on the device;
 * the host only polls a status word every poll_every iterations.  Re-entrant: call again to
 * continue (L-BFGS restarts its history; FIRE keeps velocities, dt and alpha when opts->resume = 1).
 * kind 0: L-BFGS with Armijo backtracking (D:R12); the caller's buffer ends at the last accepted point.
 * kind 1: FIRE (ref.[37]) with the published default parameters, unit masses, semi-implicit Euler;
 *         report->iters counts MD steps; there is no step rejection, the buffer ends at the last point
 *         evaluated.  Returns report->status.
 */
int shd_minimize(shd_ctx* h, double* pos_hi, double* pos_lo, const shd_min_opts* opts,
                 shd_min_report* report);

/* Text of the last error on this handle (never NULL). */
const char* shd_last_error(const shd_ctx* h);

/* Per-kernel device timing: with on != 0 every later shd_energy_grad / shd_smax records CUDA events on
 * the handle's stream around its launch groups; read the durations with shd_stat(h, 20..24). */
int shd_set_timing(shd_ctx* h, int on);

/* Introspection used by bench.py / tests (host scalars):
 *   what = 0 / 12: DFMAs the rho / gradient pass launches (padding included),
 *   what = 1: kernel launches of the last call, 2: padded (p,q) cell count of the rho pass,
 *   3: valid cell count, 4: bytes of device workspace, 5: particle splits of the rho pass,
 *   6: (p,q) tiles, 7: P, 8: Qn, 9: padded particle count, 10: particle blocks of the gradient
 *   pass, 11: q-steps walked by one gradient block,
 *   20..24: milliseconds of the last call's launch groups (needs shd_set_timing):
 *           20 phasor tables (a1), 21 rho pass (a2), 22 finish (a3), 23 gradient operand, 24 gradient pass (a4). */
double shd_stat(const shd_ctx* h, int what);

/*
 * Measured FP64-pipe issue rate of the current device, the denominator of the "alu" roofline
 * (DESIGN.md "roofline").  kind = 0: dependent-DFMA chains, 1: DADD chains (8 per
 * thread, all SMs), 2: chains of the FP64 matrix instruction DMMA.8x8x4 (8 per warp; counted as 8 FMAs
 * per thread and instruction), the instruction the rho and gradient passes issue; runs for about
 * `seconds` (0 < seconds <= 10).  HOST out: instr_per_s[0] = best
 * launch, instr_per_s[1] = mean over the run (sustained), in thread-level FP64 instructions per
 * second.  Errors: SHD_EINVAL, SHD_ENOMEM, SHD_ECUDA.  Needs no handle.
 */
int shd_fp64_peak(int kind, double seconds, double instr_per_s[2]);

/*
 * INT8 tensor-core probe (an exact digit-sliced contraction on tcgen05.mma.kind::i8 would
 * replace the FP64 limb FMAs).  HOST out: *mismatches = wrong entries of a 128 x 64 x 128 s8 x s8 -> s32 product
 * computed by the 5th-generation tensor core (operands in shared memory, accumulator in TMEM) against the
 * integer product on the host (0 = exact); *tops = measured issue rate of M=128, N=256, K=32 instructions on
 * all SMs in tera-operations per second (2 per multiply-accumulate).  Needs no handle.
 */
int shd_i8_probe(double* tops, long* mismatches);

#ifdef __cplusplus
}
#endif
#endif /* SHD_H */
