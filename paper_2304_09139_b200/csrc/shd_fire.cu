// shd_fire.cu -- step a5, second minimizer: FIRE (ref.[37] P:152), the paper's own choice, on the
// device in double-double.  The paper restates none of FIRE's parameters (D:R12): this is the published
// algorithm with its published defaults (N_min 5, f_inc 1.1, f_dec 0.5, alpha_start 0.1, f_alpha 0.99,
// dt_max = 10 dt0), unit masses, F = -grad Phi, semi-implicit Euler.
//
// Like the L-BFGS (shd_min.cu) the host only enqueues identical slots and polls a status word:
//   slot = [ evaluation at x (a1-a4), gradient into g ]
//          k_fire_dots    : per-block dd partials of  g.v,  v.v,  g.g
//          k_fire_control : one warp: fixed-order sums, P = -g.v, the FIRE decisions (mixing
//                           coefficients, dt, alpha, counters), the stop rule S_max < smax_tol
//          k_fire_update  : v <- a v - b g;  v <- v - dt g;  x <- x + dt v   (all dd, x in place)
// No host decision per step; every reduction has a fixed tree (bit-reproducible, no atomics).
#include "../../include/shd.h"
#include "dd.cuh"
#include "shd_internal.h"
#include "slots.cuh"

#include <cmath>
#include <cstring>
#include <utility>
#include <vector>

constexpr int FIRE_THREADS = 256;
constexpr int FIRE_EPT = 4;

struct shd_firectrl {
    int done;            // 0 running, 1 finished in this slot, 2 idle
    int status, since, pad;
    long long steps, evals, max_evals;
    double phi[2], smax[2];
    double smax_tol;
    double dt[2], dt_max[2], alpha[2];   // dd: the step control is part of the arithmetic that is compared
    double a[2], b[2];   // this step's mixing: v <- a v - b g   (a = b = 0: v <- 0)
    long long ring_n;    // trace records written so far
    int ring_cap, limbs;
};

struct shd_firestate {
    long n = 0;
    int nblk = 0;
    double *v = nullptr, *g = nullptr;     // [2][n] (hi plane, lo plane)
    double *partial = nullptr;             // [nblk][3][2]
    double *rank_part = nullptr, *rank_all = nullptr;   // sharded: [3][2] and [world][3][2]
    shd_firectrl *d_ctrl = nullptr, *h_ctrl = nullptr;
    double *xprev = nullptr;               // [2][n]: the point before the last move (restored on SHD_ENAN)
    double *pos_hi = nullptr, *pos_lo = nullptr;   // the caller's buffer of the running call (shd_minimize_snapshot)
    shd_trace_rec *d_ring = nullptr, *h_ring = nullptr;
    int ring_cap = 0;
};

namespace {

__device__ __forceinline__ dd ld2(const double* base, long n, long i) { return dd{base[i], base[n + i]}; }
__device__ __forceinline__ void st2(double* base, long n, long i, dd v) { base[i] = v.h; base[n + i] = v.l; }
__device__ __forceinline__ dd warp_sum(dd v) {
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        dd o{__shfl_xor_sync(0xffffffffu, v.h, off), __shfl_xor_sync(0xffffffffu, v.l, off)};
        v = dd_add(v, o);
    }
    return v;
}

__global__ void __launch_bounds__(FIRE_THREADS) k_fire_dots(
    long n, const shd_firectrl* __restrict__ ctrl, const double* __restrict__ g, const double* __restrict__ v,
    double* __restrict__ partial)
{
    if (ctrl->done) return;
    __shared__ double red[FIRE_THREADS / 32][3][2];
    const long base = (long)blockIdx.x * (FIRE_THREADS * FIRE_EPT) + threadIdx.x;
    dd r0{0.0, 0.0}, r1{0.0, 0.0}, r2{0.0, 0.0};
#pragma unroll
    for (int e = 0; e < FIRE_EPT; e++) {
        const long i = base + (long)e * FIRE_THREADS;
        if (i < n) {
            const dd gi = ld2(g, n, i), vi = ld2(v, n, i);
            r0 = dd_add(r0, dd_mul(gi, vi));
            r1 = dd_add(r1, dd_mul(vi, vi));
            r2 = dd_add(r2, dd_mul(gi, gi));
        }
    }
    r0 = warp_sum(r0); r1 = warp_sum(r1); r2 = warp_sum(r2);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) {
        red[w][0][0] = r0.h; red[w][0][1] = r0.l;
        red[w][1][0] = r1.h; red[w][1][1] = r1.l;
        red[w][2][0] = r2.h; red[w][2][1] = r2.l;
    }
    __syncthreads();
    if (threadIdx.x < 3) {
        dd s{0.0, 0.0};
        for (int k = 0; k < FIRE_THREADS / 32; k++) s = dd_add(s, dd{red[k][threadIdx.x][0], red[k][threadIdx.x][1]});
        double* o = partial + ((size_t)blockIdx.x * 3 + threadIdx.x) * 2;
        o[0] = s.h; o[1] = s.l;
    }
}

// this rank's three sums over its blocks, in the tree k_fire_control uses (lane l adds blocks l, l+32, ...; butterfly),
// so that one rank gives exactly the unsharded result
__global__ void __launch_bounds__(32) k_fire_rank_sum(int nblk, const shd_firectrl* __restrict__ c, const double* __restrict__ partial,
                                                      double* __restrict__ out)
{
    if (c->done) return;
    const int lane = threadIdx.x;
#pragma unroll
    for (int r = 0; r < 3; r++) {
        dd s{0.0, 0.0};
        for (int k = lane; k < nblk; k += 32) {
            const double* o = partial + ((size_t)k * 3 + r) * 2;
            s = dd_add(s, dd{o[0], o[1]});
        }
        s = warp_sum(s);
        if (lane == 0) { out[2 * r] = s.h; out[2 * r + 1] = s.l; }
    }
}

__global__ void __launch_bounds__(32) k_fire_control(
    int nblk, shd_firectrl* __restrict__ c, const shd_scalars* __restrict__ scal, const double* __restrict__ partial,
    shd_trace_rec* __restrict__ ring)
{
    if (c->done) {
        if (threadIdx.x == 0) c->done = 2;
        return;
    }
    const int lane = threadIdx.x;
    // fixed-order sums: lane l adds blocks l, l+32, ...; then the butterfly
    dd D[3];
#pragma unroll
    for (int r = 0; r < 3; r++) {
        dd s{0.0, 0.0};
        for (int k = lane; k < nblk; k += 32) {
            const double* o = partial + ((size_t)k * 3 + r) * 2;
            s = dd_add(s, dd{o[0], o[1]});
        }
        D[r] = warp_sum(s);
    }
    if (lane != 0) return;
    const double f_inc = 1.1, f_dec = 0.5, alpha_start = 0.1, f_alpha = 0.99;   // the doubles nearest to these
    const int n_min = 5;
    long long evals = c->evals + 1;
    int done = 0, status = SHD_OK, since = c->since;
    dd dt{c->dt[0], c->dt[1]}, alpha{c->alpha[0], c->alpha[1]}, a{0.0, 0.0}, b{0.0, 0.0};
    c->phi[0] = scal->phi[0]; c->phi[1] = scal->phi[1];
    c->smax[0] = scal->smax[0]; c->smax[1] = scal->smax[1];
    if (scal->nonfinite) { done = 1; status = SHD_ENAN; }
    else if (dd_less(dd{scal->smax[0], scal->smax[1]}, dd{c->smax_tol, 0.0})) { done = 1; status = SHD_OK; }
    else if (evals >= c->max_evals) { done = 1; status = SHD_EMAXEVAL; }
    else {
        const dd P = dd_neg(D[0]), vv = D[1], ff = D[2];
        if (dd_less(dd{0.0, 0.0}, P)) {
            a = dd_sub(dd{1.0, 0.0}, alpha);
            b = ff.h > 0.0 ? dd_mul(alpha, dd_sqrt(dd_div(vv, ff))) : dd{0.0, 0.0};
            if (since > n_min) {
                dt = dd_mul_d(dt, f_inc);
                const dd mx{c->dt_max[0], c->dt_max[1]};
                if (dd_less(mx, dt)) dt = mx;
                alpha = dd_mul_d(alpha, f_alpha);
            }
            since++;
        } else {
            dt = dd_mul_d(dt, f_dec); alpha = dd{alpha_start, 0.0}; since = 0;
        }
        c->steps++;
    }
    if (ring && c->ring_cap > 0) {               // one trace record per evaluation
        shd_trace_rec& r = ring[c->ring_n % c->ring_cap];
        r.iters = (long)c->steps; r.evals = (long)evals;
        r.phi = scal->phi[0]; r.smax = scal->smax[0];
        r.gnorm = sqrt(fmax(D[2].h, 0.0));
        r.step = c->dt[0]; r.limbs = c->limbs; r.accepted = (a.h != 0.0 || b.h != 0.0) ? 1 : 0;
        c->ring_n++;
    }
    c->evals = evals;
    c->since = since;
    c->dt[0] = dt.h; c->dt[1] = dt.l; c->alpha[0] = alpha.h; c->alpha[1] = alpha.l;
    c->a[0] = a.h; c->a[1] = a.l; c->b[0] = b.h; c->b[1] = b.l;
    c->status = status;
    c->done = done;
}

__global__ void __launch_bounds__(FIRE_THREADS) k_fire_update(
    long n, const shd_firectrl* __restrict__ c, double* __restrict__ x_hi, double* __restrict__ x_lo,
    const double* __restrict__ g, double* __restrict__ v, double* __restrict__ xprev)
{
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (c->done) {
        // Phi went non-finite after at least one move (a too large time step): the caller gets the last point with a
        // finite Phi back, at rest, instead of the diverged one
        if (c->done == 1 && c->status == SHD_ENAN && c->steps > 0 && i < n) {
            x_hi[i] = xprev[i]; x_lo[i] = xprev[n + i];
            v[i] = 0.0; v[n + i] = 0.0;
        }
        return;
    }
    if (i >= n) return;
    xprev[i] = x_hi[i]; xprev[n + i] = x_lo[i];
    const dd gi = ld2(g, n, i);
    dd vi = ld2(v, n, i);
    const dd a{c->a[0], c->a[1]}, b{c->b[0], c->b[1]}, dt{c->dt[0], c->dt[1]};
    vi = dd_sub(dd_mul(vi, a), dd_mul(gi, b));                 // mixing (or v <- 0)
    vi = dd_sub(vi, dd_mul(gi, dt));                           // v <- v + dt F
    st2(v, n, i, vi);
    const dd xn = dd_add(dd{x_hi[i], x_lo[i]}, dd_mul(vi, dt));
    x_hi[i] = xn.h; x_lo[i] = xn.l;
}

#define CUF(call)                                                                        \
    do {                                                                                 \
        cudaError_t e_ = (call);                                                         \
        if (e_ != cudaSuccess) {                                                         \
            h->err = std::string(#call) + ": " + cudaGetErrorString(e_);                 \
            h->d_skip = nullptr;                                                         \
            return e_ == cudaErrorMemoryAllocation ? SHD_ENOMEM : SHD_ECUDA;             \
        }                                                                                \
    } while (0)

int fire_alloc(shd_ctx* h) {
    if (h->fire) return SHD_OK;
    shd_firestate* s = h->fire = new shd_firestate();
    s->n = (long)h->d * h->N;
    s->nblk = (int)((s->n + FIRE_THREADS * FIRE_EPT - 1) / (FIRE_THREADS * FIRE_EPT));
    const size_t v = (size_t)2 * s->n * sizeof(double);
    CUF(cudaMalloc((void**)&s->v, v));
    CUF(cudaMalloc((void**)&s->g, v));
    CUF(cudaMalloc((void**)&s->xprev, v));
    CUF(cudaMalloc((void**)&s->partial, (size_t)s->nblk * 3 * 2 * sizeof(double)));
    if (shd_sharded(h)) {
        CUF(cudaMalloc((void**)&s->rank_part, 3 * 2 * sizeof(double)));
        CUF(cudaMalloc((void**)&s->rank_all, (size_t)h->world * 3 * 2 * sizeof(double)));
    }
    CUF(cudaMalloc((void**)&s->d_ctrl, sizeof(shd_firectrl)));
    CUF(cudaMallocHost((void**)&s->h_ctrl, sizeof(shd_firectrl)));
    std::memset(s->h_ctrl, 0, sizeof(shd_firectrl));
    h->workspace_bytes += 3 * v;
    return SHD_OK;
}

}  // namespace

void shd_fire_free(shd_ctx* h) {
    shd_firestate* s = h->fire;
    if (!s) return;
    cudaFree(s->v); cudaFree(s->g); cudaFree(s->partial); cudaFree(s->d_ctrl); cudaFree(s->rank_part); cudaFree(s->rank_all);
    cudaFree(s->xprev); cudaFree(s->d_ring);
    if (s->h_ring) cudaFreeHost(s->h_ring);
    if (s->h_ctrl) cudaFreeHost(s->h_ctrl);
    delete s;
    h->fire = nullptr;
}

std::vector<std::pair<int, double>> shd_ladder_rungs(const shd_ctx* h, const shd_min_opts* o);      // shd_min.cu
bool shd_after_poll(shd_ctx* h, const shd_trace_rec* d_ring, shd_trace_rec* h_ring, int ring_cap, long long ring_n,
                    long long& ring_seen, const shd_min_opts* opts, const shd_min_report& rep);

int shd_fire_snapshot(shd_ctx* h, double* pos_hi, double* pos_lo) {
    shd_firestate* s = h->fire;
    if (!s || !s->pos_hi) { h->err = "shd_minimize_snapshot: no minimizer has run on this handle"; return SHD_EINVAL; }
    const size_t b = (size_t)s->n * sizeof(double);
    cudaStream_t st = h->gstream ? h->gstream : h->stream;
    CUF(cudaMemcpyAsync(pos_hi, s->pos_hi, b, cudaMemcpyDeviceToDevice, st));
    CUF(cudaMemcpyAsync(pos_lo, s->pos_lo, b, cudaMemcpyDeviceToDevice, st));
    CUF(cudaStreamSynchronize(st));
    return SHD_OK;
}

// kind == 1 of shd_minimize (shd_min.cu dispatches here)
int shd_fire_run(shd_ctx* h, double* pos_hi, double* pos_lo, const shd_min_opts* opts, shd_min_report* report) {
    if (!(opts->smax_tol >= 0.0) || opts->max_evals < 1 || opts->poll_every < 1 || !(opts->fire_dt0 >= 0.0) ||
        !std::isfinite(opts->fire_dt0)) {
        h->err = "bad smax_tol / max_evals / poll_every / fire_dt0";
        return SHD_EINVAL;
    }
    const bool cont = opts->resume != 0 && h->fire && h->fire->h_ctrl->dt[0] > 0.0;
    int rc = fire_alloc(h);
    if (rc) return rc;
    if ((rc = shd_prepare_tables(h, true))) return rc;
    shd_firestate* s = h->fire;
    const long n = s->n;
    cudaStream_t st = h->stream;
    s->pos_hi = pos_hi; s->pos_lo = pos_lo;
    if (s->ring_cap < opts->poll_every) {
        cudaFree(s->d_ring);
        if (s->h_ring) cudaFreeHost(s->h_ring);
        s->d_ring = nullptr; s->h_ring = nullptr;
        s->ring_cap = opts->poll_every;
        CUF(cudaMalloc((void**)&s->d_ring, sizeof(shd_trace_rec) * s->ring_cap));
        CUF(cudaMallocHost((void**)&s->h_ring, sizeof(shd_trace_rec) * s->ring_cap));
    }
    // default time step: the stiffest collective mode of Phi = sum v |rho|^2 has curvature ~ 2 N v k_max^2,
    // explicit integration is stable for dt < 2 / (k_max sqrt(2 N v)); dt_max = 10 dt0 sits at half of it
    double vmax = 1.0;
    for (double x : h->v) vmax = x > vmax ? x : vmax;
    const double kmax = 2.0 * 3.14159265358979323846 * std::sqrt((double)h->m_star) / h->L;
    const double dt0 = opts->fire_dt0 > 0.0 ? opts->fire_dt0 : 0.1 / (kmax * std::sqrt(2.0 * (double)h->Nsys * vmax));
    shd_firectrl* c = s->h_ctrl;
    if (cont) {                        // explicit re-entry: keep velocities, dt, alpha, counters
        const shd_firectrl keep = *c;
        std::memset(c, 0, sizeof(*c));
        c->since = keep.since;
        for (int i = 0; i < 2; i++) { c->dt[i] = keep.dt[i]; c->alpha[i] = keep.alpha[i]; c->dt_max[i] = keep.dt_max[i]; }
    } else {
        CUF(cudaMemsetAsync(s->v, 0, (size_t)2 * n * sizeof(double), st));
        std::memset(c, 0, sizeof(*c));
        c->dt[0] = dt0; c->dt_max[0] = 10.0 * dt0; c->alpha[0] = 0.1;     // 10 dt0 rounded to double, as the oracle
    }
    c->max_evals = opts->max_evals;
    c->ring_cap = s->ring_cap;
    const unsigned ublk = (unsigned)((n + FIRE_THREADS - 1) / FIRE_THREADS);
    auto slot = [&]() -> cudaError_t {
        cudaError_t e;
        cudaStream_t q = h->stream;          // the capture stream while shd_run_slots is recording
        if ((e = shd_enqueue_eval(h, pos_hi, pos_lo, s->g, s->g + n)) != cudaSuccess) return e;
        k_fire_dots<<<s->nblk, FIRE_THREADS, 0, q>>>(n, s->d_ctrl, s->g, s->v, s->partial);
        if (shd_sharded(h)) {        // sharded vectors: rank sums, all-gathered as bytes, added in rank order (shd_min.cu)
            k_fire_rank_sum<<<1, 32, 0, q>>>(s->nblk, s->d_ctrl, s->partial, s->rank_part);
            if ((e = shd_comm_allgather(h, s->rank_part, s->rank_all, 3 * 16)) != cudaSuccess) return e;
            k_fire_control<<<1, 32, 0, q>>>(h->world, s->d_ctrl, h->d_scal, s->rank_all, s->d_ring);
        } else
            k_fire_control<<<1, 32, 0, q>>>(s->nblk, s->d_ctrl, h->d_scal, s->partial, s->d_ring);
        k_fire_update<<<ublk, FIRE_THREADS, 0, q>>>(n, s->d_ctrl, pos_hi, pos_lo, s->g, s->v, s->xprev);
        h->last_launches += 3;
        return cudaGetLastError();
    };
    // the rungs of the precision ladder (shd_min.cu): velocities, dt and alpha carry over from rung to rung
    const std::vector<std::pair<int, double>> rungs = shd_ladder_rungs(h, opts);
    const int nlimb_user = h->nlimb;
    long long ring_seen = 0;
    bool stopped = false;
    for (size_t r = 0; r < rungs.size(); r++) {
        h->nlimb = rungs[r].first;
        c->done = 0; c->status = SHD_OK;
        c->smax_tol = rungs[r].second;
        c->limbs = rungs[r].first;
        cudaError_t ce = cudaMemcpyAsync(s->d_ctrl, c, sizeof(shd_firectrl), cudaMemcpyHostToDevice, st);
        if (ce == cudaSuccess) {
            h->d_skip = &s->d_ctrl->done;
            ce = shd_run_slots(h, opts->poll_every, slot, c, s->d_ctrl, sizeof(shd_firectrl), &c->done, [&]() -> bool {
                shd_min_report rp;
                rp.iters = (long)c->steps; rp.evals = (long)c->evals;
                rp.phi[0] = c->phi[0]; rp.phi[1] = c->phi[1]; rp.smax[0] = c->smax[0]; rp.smax[1] = c->smax[1];
                rp.status = c->done ? c->status : SHD_OK;
                stopped = shd_after_poll(h, s->d_ring, s->h_ring, s->ring_cap, c->ring_n, ring_seen, opts, rp) && !c->done;
                return stopped;
            });
            h->d_skip = nullptr;
        }
        if (ce != cudaSuccess) { h->nlimb = nlimb_user; CUF(ce); }
        if (stopped) { c->status = SHD_ESTOPPED; break; }
        if (r + 1 == rungs.size() || c->status != SHD_OK) break;
    }
    h->nlimb = nlimb_user;
    report->iters = (long)c->steps;
    report->evals = (long)c->evals;
    report->phi[0] = c->phi[0]; report->phi[1] = c->phi[1];
    report->smax[0] = c->smax[0]; report->smax[1] = c->smax[1];
    report->status = c->status;
    if (c->status == SHD_ENAN) h->err = "shd_minimize (FIRE): non-finite Phi (the buffer holds the last point with a finite Phi)";
    else if (c->status == SHD_EMAXEVAL) h->err = "shd_minimize (FIRE): max_evals reached";
    else if (c->status == SHD_ESTOPPED) h->err = "shd_minimize (FIRE): stopped by the poll callback";
    return c->status;
}
