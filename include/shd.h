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
#define SHD_ESTOPPED -7   /* shd_minimize: stopped by the caller's poll callback (report written)  */

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
 * Engine of the two O(N M) passes (steps a2, a4).
 *   2: both on the INT8 tensor cores (tcgen05.mma.kind::i8; k_rho8.cu, k_grad8.cu): operands as 13 balanced base-256
 *      digits of trunc(x 2^102), the 91 digit pairs with i + l >= 12, s32 accumulators in tensor memory (exact: at most
 *      8192 particles per CTA in the rho pass, at most 5024 last-axis entries in the gradient pass), the gradient pass's
 *      final contraction in exact integer arithmetic; the same double-double results within the same tolerances.
 *   1: the rho pass on the INT8 tensor cores, the gradient pass on the FP64 limbs.
 *   0: exact FP64 limb contraction on the FP64 matrix instruction (k_rho.cu, k_grad.cu).
 *  -1: the library's own choice, which is also what shd_create* starts with: engine 2 when the last-axis table has at
 *      most 5024 entries and one evaluation is at least 5e7 pair-terms, engine 0 otherwise (tiny systems are
 *      launch-bound either way).
 * shd_set_precision selects the number of digits on the INT8 engines.  The tables of an engine are allocated on first
 * use and those of the engine left behind are freed.  Errors: SHD_EINVAL (engine not -1..2; engine 2 with more than 5024
 * entries in the last-axis table; no particle split keeps the s32 sums exact: the handle's engine is then unchanged),
 * SHD_ENOMEM, SHD_ECUDA.
 */
int shd_set_engine(shd_ctx* h, int rho_engine);

/*
 * Bounded workspace (the paper's N = 2 x 10^6 at chi = 0.2 ... 0.4, needs 260 GB of
 * phasor tables at once).  The per-particle tables are built for one CHUNK of particles at a time: pass 1 (rho) chunk
 * by chunk into running double-double sums, pass 2 (gradient) chunk by chunk again.  A chunk is a whole number of the
 * rho pass's particle splits and the running sums continue the same left fold over the splits, so every result is
 * bit-identical to the single-chunk evaluation whatever the cap.  bytes = cap on the tables of this handle; 0 (default)
 * = what the device has free when they are first allocated.  Errors: SHD_ENOMEM at the next evaluation when even one
 * split does not fit.
 */
int shd_set_workspace(shd_ctx* h, unsigned long bytes);

/*
 * Particle sharding over GPUs: this handle evaluates N particles (its shard: pos_*, grad_* hold
 * those only) of a system of N_total; rank / world = its position.  One exchange step per evaluation: the running sums
 * of the shard's contributions to rho (a few MB) are all-gathered as bytes in rank order and added in that order on
 * every GPU (a double-double add is not an ncclSum); the gradient pass is local.  S_max is normalised by N_total.
 * Two ways to drive it:
 *   - shd_comm_init: the library owns an NCCL communicator (unique id from shd_comm_unique_id on rank 0, broadcast by
 *     the caller, e.g. torch.distributed); shd_energy_grad / shd_smax / shd_minimize then run as on one GPU, the
 *     minimizers exchanging their few double-double dot products the same way (no host decision per iteration, all
 *     ranks take bit-identical decisions);
 *   - or the split calls below, with the caller doing the all-gather (any transport; this is also how several
 *     shards are driven from one process on one GPU).
 * Errors: SHD_EINVAL.
 */
int shd_set_shard(shd_ctx* h, long N_total, int rank, int world);
/* 128 bytes (HOST out) identifying a new NCCL communicator; call on one rank, hand the bytes to all.  SHD_ECUDA when NCCL
 * cannot be loaded (libnccl.so.2 is resolved at run time). */
int shd_comm_unique_id(void* id128);
/* Collective over the world of shd_set_shard: every rank calls it with the same 128 bytes. */
int shd_comm_init(shd_ctx* h, const void* id128);
/* Size in bytes of a shard's partial (the same on every rank: tiles x 4 sums x 1024 cells x (hi, lo)). */
unsigned long shd_partial_bytes(const shd_ctx* h);
/* Pass 1 of a shard: partial_out (DEVICE, shd_partial_bytes(h) bytes, caller-owned) receives the running sums of the
 * shard's contributions to rho; synchronises the stream. */
int shd_rho_partial(shd_ctx* h, const double* pos_hi, const double* pos_lo, void* partial_out);
/* gathered (DEVICE): nparts partials in rank order, back to back -> rho, Phi (HOST phi[2]), S_max on this handle. */
int shd_rho_finish(shd_ctx* h, const void* gathered, int nparts, double phi[2]);
/* Pass 2 of a shard: the gradient of its own particles (DEVICE, d*N doubles each) from the rho of shd_rho_finish. */
int shd_grad_local(shd_ctx* h, const double* pos_hi, const double* pos_lo, double* grad_hi, double* grad_lo);

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

/*
 * shd_structure_factor for callers that must not allocate (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the same two kernels and the same fixed reduction tree, so S_out and dev2 are
 * bit-identical to shd_structure_factor's, but the per-block partial sums live in a file-scope device array of the
 * library instead of a cudaMalloc'ed buffer.  The call makes no cudaMalloc / cudaFree and calls no allocating library
 * routine; it enqueues two kernels on the handle's stream.
 *   input : the rho(k) of the LAST evaluation on this handle (as shd_structure_factor);
 *   S_out : DEVICE, |Q| doubles, may be NULL;   dev2 : DEVICE, 2 doubles (hi, lo) -- note: device, not host;
 *   wait  : nonzero = cudaStreamSynchronize before returning; 0 = return once enqueued (read the outputs after the
 *           handle's stream has been synchronised).
 * Limit: |Q| <= SHD_NOALLOC_MAX_Q (the array holds 2 doubles per 256 wavevectors: 256 KiB of device memory that EVERY
 * GPU which loads libshd.so holds until the process exits).  A handle with more wavevectors gets SHD_EINVAL and a message
 * naming the limit; use shd_structure_factor there.  The handle's device must be the current device (checked, SHD_EINVAL).
 * The first call on each device resolves the array's device address (cudaGetSymbolAddress: no allocation by this
 * library, but the CUDA runtime may load the module then) -- make one call per device before a capture.
 * ALL calls on a device share the one array.  It keeps the last call's contents; nothing has to start at zero (every
 * element the second kernel reads was written by the first kernel of the same call).  Two calls whose kernels overlap
 * on the GPU (different handles = different streams, or two host threads) RACE on it: serialise them.
 * Errors: SHD_EINVAL, SHD_ECUDA.
 */
#define SHD_NOALLOC_MAX_Q 4194304L
int shd_structure_factor_noalloc(shd_ctx* h, double* S_out, double* dev2, int wait);

/*
 * Radially averaged structure factor of the LAST evaluation (Fig. 2a, Fig. S1a: S against |k|, beyond K when
 * the handle's cutoff reaches there).  |k|^2 = (2 pi / L)^2 n.n, so a radial bin is a range of the integer n.n: bin b
 * holds the wavevectors with edges[b] <= n.n < edges[b+1] (HOST, nbins + 1 strictly ascending longs; index work only,
 * no floating-point compare).  HOST out: count[b] = members of bin b, S_mean (hi, lo)[b] = their mean S(k) in
 * double-double, 0 for an empty bin (the half shell stands for the whole shell: S(-k) = S(k)).
 * Errors: SHD_EINVAL, SHD_ENOMEM, SHD_ECUDA.  Synchronises the stream.
 */
int shd_structure_factor_shells(shd_ctx* h, long nbins, const long* edges, long* count, double* S_mean_hi, double* S_mean_lo);
/* The distinct values of n.n in the handle's Q, ascending (HOST, shd_num_shells(h) longs): with edges = these values
 * followed by (the last + 1), shd_structure_factor_shells returns one bin per shell, the finest radial resolution. */
long shd_num_shells(const shd_ctx* h);
int shd_get_shells(const shd_ctx* h, long* nn_out);

/*
 * Order metric tau of Eq. 7 from the LAST evaluation on this handle with D = 1/K, as the lattice sum over +-Q:
 * tau = K^d V / N^2 * 2 * sum_{k in Q} (S(k) - 1)^2  (V = L^d), HOST (hi, lo).  The handle's own cutoff must reach far
 * enough beyond K that S(k) has decayed to 1.  Errors: SHD_EINVAL, SHD_ECUDA.
 */
int shd_tau(shd_ctx* h, double K, double tau[2]);

typedef struct {
    long   iters, evals;
    double phi[2], smax[2];
    int    status;      /* SHD_OK, SHD_ESTALL, SHD_EMAXEVAL, SHD_ENAN, SHD_ESTOPPED */
} shd_min_report;

/* Host callback of shd_minimize, called after every poll (every poll_every iterations; the device is idle): report =
 * the state so far (status = SHD_OK while running).  Return non-zero to stop (SHD_ESTOPPED).  shd_get_trace and
 * shd_minimize_snapshot may be called from inside it (periodic log / checkpoint); nothing else on this handle. */
typedef int (*shd_poll_fn)(const shd_min_report* report, void* user);

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
    double ladder_tol[2]; /* precision ladder ("tunable precision"): evaluate with ONE limb
                           (4 digits on the INT8 engines) until S_max < ladder_tol[0], with TWO limbs (7 digits) until
                           S_max < ladder_tol[1], then at the handle's precision (shd_set_precision) down to smax_tol.
                           0 = rung not used.  The device decides when a rung ends; the minimizer state (L-BFGS pairs,
                           FIRE velocities) is kept across rungs, the first evaluation of a rung refreshes Phi and the
                           gradient at the current point.  A line-search stall on a lower rung moves on to the next. */
    shd_poll_fn on_poll;  /* optional host callback after every poll (NULL = none) */
    void*  on_poll_user;
} shd_min_opts;

/* One record per evaluation of the last shd_minimize call, written by the device-side control kernel into a ring and
 * collected by the host at every poll. */
typedef struct {
    long   iters, evals;   /* accepted iterations / evaluations so far (both cumulative over the call) */
    double phi, smax;      /* Phi and S_max of THIS evaluation (the trial point) */
    double gnorm;          /* |grad|_2 of this evaluation */
    double step;           /* L-BFGS: step length t of the trial; FIRE: dt */
    int    limbs;          /* precision of the evaluation (shd_set_precision levels; the ladder's rung) */
    int    accepted;       /* L-BFGS: Armijo accepted; FIRE: P > 0 */
} shd_trace_rec;

/*
 * Quench: minimise Phi from pos (DEVICE, in/out, d*N doubles each) until S_max < smax_tol.
 * The whole iteration (evaluations, dd vector algebra, line search decisions) runs on the device;
 * the host only polls a status word every poll_every iterations.  Re-entrant: call again to
 * continue (L-BFGS restarts its history; FIRE keeps velocities, dt and alpha when opts->resume = 1).
 * kind 0: L-BFGS with Armijo backtracking (D:R12); the caller's buffer ends at the last accepted point.
 * kind 1: FIRE (ref.[37]) with the published default parameters, unit masses, semi-implicit Euler;
 *         report->iters counts MD steps; there is no step rejection, the buffer ends at the last point
 *         evaluated -- except on SHD_ENAN after at least one step, where it is restored to the last point with a
 *         finite Phi (a too large fire_dt0 must not destroy the caller's state).  Returns report->status.
 */
int shd_minimize(shd_ctx* h, double* pos_hi, double* pos_lo, const shd_min_opts* opts,
                 shd_min_report* report);

/* Records first .. first + max - 1 of the last shd_minimize call's trace into out (HOST); returns how many were
 * copied (0 when first is past the end; the trace keeps at most 2^22 records). */
long shd_get_trace(shd_ctx* h, long first, long max, shd_trace_rec* out);

/* During (from the poll callback) or after shd_minimize: the minimizer's current best point into pos_hi / pos_lo
 * (DEVICE, d*N doubles each): L-BFGS: the last accepted point; FIRE: the current point.  Errors: SHD_EINVAL when no
 * minimizer has run on this handle. */
int shd_minimize_snapshot(shd_ctx* h, double* pos_hi, double* pos_lo);

/* Text of the last error on this handle (never NULL). */
const char* shd_last_error(const shd_ctx* h);

#ifdef __cplusplus
}
#endif
#endif /* SHD_H */
