// shd_internal.h -- handle layout and device data layouts shared by the kernels of libshd.so.
//
// Decomposition: every k in Q is written once as
//   exp(i k.r_j) = A_j[p] * B_j[q]^sigma ,  sigma = +1 (B) or -1 (conj B),
// with per-particle tables A_j[0..P), B_j[0..Qn) of complex dd phasors built from per-axis
// integer-power recurrences:
//   d=1: n = S p + sigma q,          A[p] = (z^S)^p,          B[q] = z^q       (q <= S/2)
//   d=2: n = (p, sigma q),           A[p] = z0^p,             B[q] = z1^q
//   d=3: n = (n0(p), n1(p), sigma q) A[p] = z0^n0 z1^n1,      B[q] = z2^q
//   d=4: n = (n0, n1, n2, sigma q)(p) A[p] = z0^n0 z1^n1 z2^n2, B[q] = z3^q
// so that rho(+/-)[p,q] = sum_j A_j[p] B_j[q]^(+/-) is a contraction over particles (rho pass) and
// the gradient is a contraction over q followed by one over p (gradient pass).
//
// Each real operand x (|x| <= 1) is stored as three "limbs" (x0, x1, x2):
//   x0  = x rounded to a multiple of 2^-W0,  x1 = (x - x0) rounded to a multiple of 2^-(W0+W1),  W0 = W1 = 22,
//   x2  = x - x0 - x1 (a free double);   x12 = x1 + x2 is formed in registers,
// and a product-accumulate  acc += x*y  is the 6 FMAs
//   L0 += x0 y0 ;  L1 += x0 y1 + x1 y0 ;  L2 += x0 y2 + x2 y0 + x12 y12
// where L0 and L1 are EXACT (all partial sums representable: L0 in units of 2^-44 below 2^9, L1 in
// units of 2^-66 below 2^-13) for bursts of <= 512 products, and L2 carries the terms below 2^-44 in
// plain FP64 (error ~2^-98 per term).  Bursts are folded
// into ordinary double-double accumulators with TwoSum.
//
// The FMAs are issued as FP64 matrix instructions (mma.sync m8n8k4, SASS DMMA.8x8x4: 256 FMAs per
// warp instruction on the same FP64 pipe and at the same peak rate as DFMA, measured), with the
// contraction index (particles in the rho pass, q in the gradient pass) as the k dimension.  The
// tables are therefore stored "fragment-major": groups of 4 consecutive contraction indices, and
// inside a group  [limb 3][entry 32][index-in-group 4][re,im]  so that the 32 lanes of a warp
// (entry = lane/4, index = lane%4) read one contiguous 512-byte run with LDS.128.
#pragma once
#include "../../include/shd.h"
#include <cuda_runtime.h>
#include <cstddef>
#include <string>
#include <vector>

constexpr int SHD_PT = 32;          // A-entries (p) per tile
constexpr int SHD_QT = 32;          // B-entries (q) per tile
constexpr int SHD_NPS = 8;          // particles per rho-pass pipeline stage (2 groups of 4)
constexpr int SHD_RHO_STAGES = 6;   // TMA pipeline depth, rho pass
constexpr int SHD_BURST = 512;      // products per exact burst (see header comment)
constexpr int SHD_QCH = 4;          // q per gradient-pass pipeline stage (1 group of 4)
constexpr int SHD_GRAD_STAGES = 4;  // TMA pipeline depth, gradient pass
constexpr int SHD_JT = 64;          // particles per gradient-pass block
constexpr int SHD_PG = 16;          // p per gradient-pass block
constexpr int SHD_W0 = 22;          // limb widths (bits)
constexpr int SHD_W1 = 22;
constexpr int SHD_NLIMB = 3;
constexpr int SHD_I8_DIGITS = 13;   // balanced base-256 digits of trunc(x 2^102) (INT8 tensor-core rho pass, k_rho8.cu)
constexpr int SHD_I8_PT = 64;       // p per tile of that pass
constexpr int SHD_I8_QT = 16;       // q per tile
constexpr int SHD_I8_MAXN = 8192;   // particles per CTA: 13 pairs x 8192 x 2^14 < 2^31 keeps the s32 sums exact
constexpr int SHD_GROUP_DOUBLES = SHD_NLIMB * 32 * 4 * 2;   // one (block, group of 4) slab of A / B: 6 KB
constexpr int SHD_GGROUP_DOUBLES = 2 * SHD_GROUP_DOUBLES;   // gradient operands: 6 planes (Bg: b, q b; C: C1, C2)

// launch groups timed by shd_set_timing: tables (a1), rho (a2), finish (a3), ctable, grad (a4)
constexpr int SHD_NKERN = 5;

// device scalars (one small struct in device memory, mirrored in pinned host memory)
struct shd_scalars {
    double phi[2];
    double smax[2];       // max |rho|^2 / N
    double maxvs;         // max v^2 |rho|^2   (scale of the gradient operand)
    double cscale;        // 2^-e applied to the C table
    long long argmax;
    int nonfinite;
    int pad;
    // SM clock inside the tensor kernels: cycles (clock64) and nanoseconds (globaltimer) of the issuing thread of CTA 0,
    // [0..1] k_rho8, [2..3] k_grad8 of the last evaluation (the clock under tensor load is well below what nvidia-smi
    // shows between kernels; bench.py states the roofline at this clock too)
    long long clk[4];
};

struct shd_minstate;      // L-BFGS workspace (shd_min.cu)
struct shd_firestate;     // FIRE workspace (shd_fire.cu)

struct shd_comm;          // NCCL plumbing of a sharded handle (shd_comm.cu)

struct shd_ctx {
    int d = 0;
    long N = 0;                // particles this handle evaluates (its shard of the system)
    long Nsys = 0;             // particles of the whole system (= N unless sharded, shd_set_shard): S_max = max |rho|^2 / Nsys
    int rank = 0, world = 1;   // position of the shard
    int sms = 148;             // SMs of the device
    // Bounded workspace: the per-particle tables hold one CHUNK of particles = spc whole splits of the rho pass, so the
    // reduction tree (left fold over the splits, k_finish1) is the same for every chunk size: results are bit-identical.
    long unit = 0;             // particles per split of the current engine's rho pass
    int spc = 0;               // splits per chunk
    int nchunk = 1;            // chunks per evaluation
    long Nc = 0;               // particles per chunk = spc * unit
    size_t ws_cap = 0;         // cap on the per-particle tables in bytes (shd_set_workspace); 0 = what the device has free
    bool tables_valid = false; // device tables allocated for the current (engine, chunk) setting
    int engine_auto = 1;       // engine chosen by the library (shd_create*) rather than by shd_set_engine
    double *d_xrun = nullptr;  // running sums of the fold over chunks / the shard's partial: [ntiles][4][1024] (hi, lo)
    double *d_xall = nullptr;  // sharded: the ranks' partials gathered in rank order [world][ntiles][4][1024] (hi, lo)
    shd_comm *comm = nullptr;
    bool grad_tables_ready = false;   // one chunk: the table build of the rho pass also wrote the gradient pass's tables
    size_t table_bytes = 0;           // bytes held by the tables of the current (engine, chunk) setting
    void (*timing_mark)(shd_ctx*, int) = nullptr;   // set around a timed evaluation (shd_set_timing)
    std::vector<int> cell_kp, cell_km;              // host copies of the (p, q) -> k maps
    void *d_trace = nullptr;
    std::vector<shd_trace_rec> trace; // trace of the last shd_minimize call, collected at every poll (shd_get_trace)
    int last_min_kind = -1;           // minimizer of the last shd_minimize call (shd_minimize_snapshot)
    double L = 0;
    long m_star = 0;
    long M = 0;
    int rho_engine = 0;        // 0: FP64 limbs on DMMA (k_rho.cu); 1: s8 digits on tcgen05 (k_rho8.cu); shd_set_engine
    int nlimb = 3;             // 3: double-double products; 2: "fast" 44-bit operands (shd_set_precision)
    // decomposition
    int P = 0, Qn = 0, npb = 0, nqb = 0;
    int S1d = 0;               // d == 1: n = S1d * p + sigma q
    int qscale_log2 = 0;       // q * B is stored as q * B * 2^-qscale_log2
    long Npad = 0;             // particle slots of the FP64 engine's tables (one chunk): spc * chunks_per_split * NPS
    int nsplit = 0;
    long chunks_per_split = 0;
    int ntiles = 0;
    long njb = 0;              // ceil(N / 32)
    long njb64 = 0;            // ceil(Nc / 64): particle blocks of the gradient pass in one chunk
    int npb16 = 0;             // ceil(P / 16): p-blocks of the gradient pass
    int nsteps = 0;            // gradient pass: steps (16 p x 4 q) in the step list
    int nseg = 0;              // gradient pass: equal segments of the step list (work units per particle block)
    int Qpad = 0;              // nqb * 32
    long valid_cells = 0;
    long grad_qsteps = 0;      // 4 * nsteps: q-steps walked by the gradient pass over all 16-p blocks
    // host copies
    std::vector<int> nvec;     // M * d
    std::vector<double> v;     // M (empty = all ones)
    std::vector<int> pn0, pn1, pn2; // exponent of z0 (and z1 for d>=3, z2 for d=4) of A entry p
    // device: setup tables
    int *d_pn0 = nullptr, *d_pn1 = nullptr, *d_pn2 = nullptr;
    int *d_wT = nullptr;       // [3][P padded]: integer weight of Im(conj(A) T) for axis a
    int *d_cell_kp = nullptr, *d_cell_km = nullptr;   // [npb*32][Qpad] -> k or -1
    int *d_tile_pb = nullptr, *d_tile_qb = nullptr;   // [ntiles]
    int *d_tile_wmap = nullptr;                       // [ntiles][9]: unit of consumer warp w (or -1), active warps
    double tile_weight = 0;                           // sum over tiles of their relative duration (1 or ~0.6)
    int *d_steps = nullptr;    // [nsteps] int2: x = C slab index pb16 * (Qpad/4) + qg, y = qg | flags << 16
                               //   (flag 1: last step of a block: fold the limb burst, contract with A)
    double *d_v = nullptr;     // [M]
    // device: per-evaluation data
    double *d_A = nullptr;     // [npb][Npad/4][3 limbs][32 p][4 j][2]
    double *d_B = nullptr;     // [nqb][Npad/4][3 limbs][32 q][4 j][2]
    double *d_Bg = nullptr;    // [2 njb64][Qpad/4][3 limbs of b][32 j][4 q][2]
    double *d_C = nullptr;     // [npb16][Qpad/4][16 planes: C1, C2, D1 = q C2, D2 = -q C1, each limbs + (x1+x2)][16 p][4 q][2]
    double *d_gpart = nullptr; // [nseg][d][N] (hi, lo): partial gradients of the segments
    // INT8 rho pass (allocated by shd_set_engine(h, 1))
    signed char *d_A8 = nullptr;   // [npb64][nk8][13 digits][128 rows (p, re/im) x 32 particles, core-matrix layout]
    signed char *d_B8 = nullptr;   // [nqb16][nk8][13 digits][ 32 rows (q, re/im) x 32 particles]
    int *d_tile8_pb = nullptr, *d_tile8_qb = nullptr;
    int ntiles8 = 0, nsplit8 = 0, ksteps8 = 0, npb64 = 0, nqb16 = 0;
    long nk8 = 0;                  // spc * ksteps8: K-steps (32 particles) in the digit tables (one chunk)
    size_t part_doubles = 0;       // capacity of d_part
    // INT8 gradient pass (shd_set_engine(h, 2))
    signed char *d_Bg8 = nullptr;  // [njb128][nkq8][13][128 rows (particle) x 32 K (q%16, re/im)]
    signed char *d_W8 = nullptr;   // [npb8][nkq8][13][32 rows (p%8, out) x 32 K]
    void *d_Afix = nullptr;        // [npb8 * 8][njb128 * 128][re, im]: trunc(a 2^102) as sign-magnitude 128-bit integers
    int *d_steps8 = nullptr;       // int2: x = pb8 * nkq8 + kstep, y = kstep | block-end << 16
    int nsteps8 = 0, nseg8 = 0, npb8 = 0, nkq8 = 0;
    long njb128 = 0;
    size_t gpart_doubles = 0;      // capacity of d_gpart
    double *d_part = nullptr;  // [nsplit][ntiles][4][1024][2]
    double *d_rho = nullptr;   // [4][M]: re_hi, re_lo, im_hi, im_lo
    double *d_blockred = nullptr;   // per-block partials of the finish kernel
    int nfinish_blocks = 0;
    shd_scalars *d_scal = nullptr;
    shd_scalars *h_scal = nullptr;  // pinned
    size_t workspace_bytes = 0;
    cudaStream_t stream = 0;
    cudaStream_t gstream = nullptr;   // the minimizers' own (capturable) stream, slots.cuh
    cudaEvent_t gevent = nullptr;
    const int* d_skip = nullptr;    // device flag: when non-NULL and *d_skip != 0 every kernel of the
                                    // evaluation path returns at once (set by the minimizer when done)
    shd_minstate *min = nullptr;
    shd_firestate *fire = nullptr;
    std::string err;
    int last_launches = 0;
    // optional per-kernel device timing (shd_set_timing): events around each launch group
    bool timing = false;
    cudaEvent_t ev[SHD_NKERN + 1] = {};
    bool ev_used[SHD_NKERN + 1] = {};
    float kern_ms[SHD_NKERN] = {};
    // staging buffer of shd_energy_grad_host (device): positions (hi, lo) then gradient (hi, lo)
    double *d_hpos = nullptr;
};

// kernels / launchers (each returns the cudaError of its launches)
cudaError_t shd_launch_tables(shd_ctx* h, const double* pos_hi, const double* pos_lo, long j_first, int what);
cudaError_t shd_launch_rho(shd_ctx* h, int nsplits);      // the rho pass over nsplits splits of the chunk in the tables
cudaError_t shd_launch_rho8(shd_ctx* h, int nsplits);
cudaError_t shd_rho8_configure();
cudaError_t shd_grad8_configure();
cudaError_t shd_launch_grad8_main(shd_ctx* h, long nc);
cudaError_t shd_launch_fold(shd_ctx* h, const double* part, int nparts, const double* xin, double* xout, bool fin);
cudaError_t shd_launch_ctable(shd_ctx* h);
cudaError_t shd_launch_sfactor(shd_ctx* h, double* S_out, double* scratch, double* tau2);
cudaError_t shd_launch_sfactor_shells(shd_ctx* h, long nbins, const long* d_start, const int* d_order, double* d_mean_hi, double* d_mean_lo);
cudaError_t shd_launch_grad(shd_ctx* h, long j_first, long nc, double* grad_hi, double* grad_lo);
cudaError_t shd_tables_configure();
cudaError_t shd_rho_configure();
cudaError_t shd_grad_configure();

// a shard exchanges its partial sums: more than one rank, or a communicator of one rank (the same calls on one GPU)
inline bool shd_sharded(const shd_ctx* h) { return h->world > 1 || h->comm != nullptr; }
int shd_prepare_tables(shd_ctx* h, bool with_grad);   // shd_api.cu: allocate what the current setting needs (outside any capture)
// the whole evaluation (steps a1-a4) enqueued on h->stream, chunk by chunk; grad_hi == NULL: rho pass and reduction only
cudaError_t shd_enqueue_eval(shd_ctx* h, const double* pos_hi, const double* pos_lo, double* grad_hi, double* grad_lo);
cudaError_t shd_enqueue_rho_partial(shd_ctx* h, const double* pos_hi, const double* pos_lo, bool grad_tables_too);   // -> d_xrun (or rho when not sharded)
cudaError_t shd_enqueue_rho_finish(shd_ctx* h, const double* gathered, int nparts);
cudaError_t shd_enqueue_grad(shd_ctx* h, const double* pos_hi, const double* pos_lo, double* grad_hi, double* grad_lo);
// NCCL plumbing (shd_comm.cu): all-gather of `bytes` bytes per rank on h->stream, fixed rank order
cudaError_t shd_comm_allgather(shd_ctx* h, const void* send, void* recv, size_t bytes);
void shd_comm_free(shd_ctx* h);
// minimizers (shd_min.cu, shd_fire.cu)
void shd_min_free(shd_ctx* h);
void shd_fire_free(shd_ctx* h);
