// shd_min.cu -- step a5: the quench as an on-device L-BFGS (D:R12) in double-double.
//
// The host only enqueues identical "slots" and polls a status word every poll_every slots; every
// decision (Armijo acceptance, history update, convergence, stall) is taken on the device:
//   slot = [ evaluation at the trial point x_t (a1-a4, predicated on ctrl->done) ]
//          k_min_dots    : s = x_t - x, y = g_t - g into the scratch history slot, and the dots of
//                          {s, y, g_t} with every basis vector {S[.], Y[.], g_t} (per-block partials)
//          k_min_control : one block: fixed-order sum of the partials, Armijo test, Gram-matrix
//                          update, two-loop recursion in COEFFICIENT space (the direction is
//                          p = -sum_l delta_l b_l over the 2m+1 basis vectors, so the 4m dependent
//                          dot/axpy sweeps of the textbook recursion become O(m^2) scalar dd work)
//          k_min_update  : x = x_t, g = g_t on acceptance; p = -sum delta_l b_l; x_t = x + t p.
// All vector algebra is dd (dd.cuh); reductions use fixed trees (bit-reproducible, no atomics).
#include "../../include/shd.h"
#include "dd.cuh"
#include "shd_internal.h"
#include "slots.cuh"

#include <algorithm>
#include <cstring>
#include <utility>
#include <vector>

int shd_fire_run(shd_ctx* h, double* pos_hi, double* pos_lo, const shd_min_opts* opts, shd_min_report* report);
std::vector<std::pair<int, double>> shd_ladder_rungs(const shd_ctx* h, const shd_min_opts* o);

constexpr int MIN_MAXHIST = 32;
constexpr int MIN_NBS = 2 * (MIN_MAXHIST + 1) + 1;   // basis stride of the Gram matrix
constexpr int MIN_EPT = 4;                           // elements per thread in k_min_dots
constexpr int MIN_THREADS = 256;
constexpr int MIN_MAX_LS = 40;                       // halvings before SHD_ESTALL

struct shd_minctrl {
    int done;            // 0 running, 1 finished in this slot (k_min_update still restores x_t), 2 idle
    int status, first, accepted;
    long long iters, evals, max_evals;
    int ls_fails, nhist, scratch, m;
    int hist[MIN_MAXHIST];          // physical slot of pair i, 0 = oldest
    double phi[2], smax[2], gp[2], t[2];
    double smax_tol;
    double gamma;        // last H0 scaling s.y / y.y (persists across calls: first step of a continued quench)
    double delta[MIN_NBS][2];
    long long ring_n;    // trace records written so far (ring index = ring_n % ring_cap)
    int ring_cap, limbs;
};

struct shd_minstate {
    int m = 0;
    long n = 0;
    int nblk = 0;
    double *x = nullptr, *g = nullptr, *gt = nullptr, *p = nullptr;   // [2][n] (hi plane, lo plane)
    double *S = nullptr, *Y = nullptr;                                 // [m+1][2][n]
    double *partial = nullptr;                                         // [nblk][NB][3][2]
    double *rank_part = nullptr, *rank_all = nullptr;                  // sharded: [NB][3][2] and [world][NB][3][2]
    double *G = nullptr;                                               // [MIN_NBS][MIN_NBS][2]
    shd_minctrl *d_ctrl = nullptr, *h_ctrl = nullptr;
    shd_trace_rec *d_ring = nullptr, *h_ring = nullptr;                // device trace ring (poll_every records) and its pinned mirror
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

__global__ void __launch_bounds__(MIN_THREADS) k_min_dots(
    long n, int m, const shd_minctrl* __restrict__ ctrl, const double* __restrict__ xt_hi,
    const double* __restrict__ xt_lo, const double* __restrict__ x, const double* __restrict__ gt,
    const double* __restrict__ g, double* __restrict__ S, double* __restrict__ Y,
    double* __restrict__ partial)
{
    if (ctrl->done) return;
    __shared__ double red[MIN_THREADS / 32][3][2];
    const int scr = ctrl->scratch, m1 = m + 1, NB = 2 * m1 + 1;
    const long base = (long)blockIdx.x * (MIN_THREADS * MIN_EPT) + threadIdx.x;
    dd sn[MIN_EPT], yn[MIN_EPT], gn[MIN_EPT];
#pragma unroll
    for (int e = 0; e < MIN_EPT; e++) {
        long i = base + (long)e * MIN_THREADS;
        if (i < n) {
            gn[e] = ld2(gt, n, i);
            sn[e] = dd_sub(dd{xt_hi[i], xt_lo[i]}, ld2(x, n, i));
            yn[e] = dd_sub(gn[e], ld2(g, n, i));
            st2(S + (size_t)scr * 2 * n, n, i, sn[e]);
            st2(Y + (size_t)scr * 2 * n, n, i, yn[e]);
        } else {
            gn[e] = sn[e] = yn[e] = dd{0.0, 0.0};
        }
    }
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    for (int b = 0; b < NB; b++) {
        dd r0{0.0, 0.0}, r1{0.0, 0.0}, r2{0.0, 0.0};
#pragma unroll
        for (int e = 0; e < MIN_EPT; e++) {
            long i = base + (long)e * MIN_THREADS;
            dd vb{0.0, 0.0};
            if (i < n) {
                if (b == scr) vb = sn[e];
                else if (b == m1 + scr) vb = yn[e];
                else if (b == 2 * m1) vb = gn[e];
                else if (b < m1) vb = ld2(S + (size_t)b * 2 * n, n, i);
                else vb = ld2(Y + (size_t)(b - m1) * 2 * n, n, i);
            }
            r0 = dd_add(r0, dd_mul(sn[e], vb));
            r1 = dd_add(r1, dd_mul(yn[e], vb));
            r2 = dd_add(r2, dd_mul(gn[e], vb));
        }
        r0 = warp_sum(r0); r1 = warp_sum(r1); r2 = warp_sum(r2);
        __syncthreads();
        if (l == 0) {
            red[w][0][0] = r0.h; red[w][0][1] = r0.l;
            red[w][1][0] = r1.h; red[w][1][1] = r1.l;
            red[w][2][0] = r2.h; red[w][2][1] = r2.l;
        }
        __syncthreads();
        if (threadIdx.x < 3) {
            dd s{0.0, 0.0};
            for (int k = 0; k < MIN_THREADS / 32; k++) s = dd_add(s, dd{red[k][threadIdx.x][0], red[k][threadIdx.x][1]});
            double* o = partial + (((size_t)blockIdx.x * NB + b) * 3 + threadIdx.x) * 2;
            o[0] = s.h; o[1] = s.l;
        }
    }
}

// out[q] = sum over this rank's blocks of partial[block][q] (dd, fixed order); nq quantities of (hi, lo)
__global__ void __launch_bounds__(64) k_rank_sum(int nblk, int nq, const double* __restrict__ partial, double* __restrict__ out,
                                                 const int* __restrict__ done)
{
    if (*done) return;
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= nq) return;
    dd s{0.0, 0.0};
    for (int k = 0; k < nblk; k++) s = dd_add(s, dd{partial[((size_t)k * nq + q) * 2], partial[((size_t)k * nq + q) * 2 + 1]});
    out[2 * q] = s.h;
    out[2 * q + 1] = s.l;
}

// sum_l delta[l] * G[l][c] over the basis, lanes in parallel, identical result in every lane
__device__ dd gram_dot(const dd* delta, const double* G, int NB, int c) {
    const int lane = threadIdx.x & 31;
    dd s{0.0, 0.0};
    for (int l = lane; l < NB; l += 32) {
        dd d = delta[l];
        if (d.h != 0.0) {
            const double* e = G + ((size_t)l * MIN_NBS + c) * 2;
            s = dd_add(s, dd_mul(d, dd{e[0], e[1]}));
        }
    }
    s = warp_sum(s);
    return dd{__shfl_sync(0xffffffffu, s.h, 0), __shfl_sync(0xffffffffu, s.l, 0)};
}

__global__ void __launch_bounds__(MIN_THREADS) k_min_control(
    int nblk, shd_minctrl* __restrict__ c, const shd_scalars* __restrict__ scal, const double* __restrict__ partial,
    double* __restrict__ G, shd_trace_rec* __restrict__ ring)
{
    if (c->done) {
        if (threadIdx.x == 0) c->done = 2;
        return;
    }
    __shared__ dd D[3 * MIN_NBS];
    __shared__ dd delta[MIN_NBS];
    __shared__ dd alpha[MIN_MAXHIST];
    const int m = c->m, m1 = m + 1, NB = 2 * m1 + 1, gidx = 2 * m1;
    for (int q = threadIdx.x; q < 3 * NB; q += blockDim.x) {
        const int b = q / 3, r = q % 3;
        dd s{0.0, 0.0};
        for (int k = 0; k < nblk; k++) {
            const double* o = partial + (((size_t)k * NB + b) * 3 + r) * 2;
            s = dd_add(s, dd{o[0], o[1]});
        }
        D[r * MIN_NBS + b] = s;
    }
    __syncthreads();
    if (threadIdx.x >= 32) return;
    const int lane = threadIdx.x;
    // ---- every lane of warp 0 runs the same scalar logic; lanes share the basis loops
    const dd phi_t{scal->phi[0], scal->phi[1]}, smax_t{scal->smax[0], scal->smax[1]};
    const bool bad = scal->nonfinite != 0;
    const int first = c->first, scr = c->scratch;
    long long evals = c->evals + 1;
    int done = 0, status = SHD_OK, accepted = 0;
    dd t{c->t[0], c->t[1]}, gp{c->gp[0], c->gp[1]}, phi{c->phi[0], c->phi[1]};
    int nh = c->nhist, ls_fails = c->ls_fails;
    if (first) {
        if (bad) { done = 1; status = SHD_ENAN; }
        else accepted = 1;
    } else if (!bad) {
        dd rhs = dd_add(phi, dd_mul(dd_mul_d(t, 1e-4), gp));        // Armijo, c1 = 1e-4
        accepted = !dd_less(rhs, phi_t);
    }
    if (accepted) {
        int new_scr = scr;
        if (!first) {
            const dd sy = D[0 * MIN_NBS + m1 + scr];
            if (sy.h > 0.0) {                                       // curvature condition, else skip the pair
                for (int b = lane; b < NB; b += 32) {
                    dd vs = D[0 * MIN_NBS + b], vy = D[1 * MIN_NBS + b];
                    double* e;
                    e = G + ((size_t)scr * MIN_NBS + b) * 2; e[0] = vs.h; e[1] = vs.l;
                    e = G + ((size_t)b * MIN_NBS + scr) * 2; e[0] = vs.h; e[1] = vs.l;
                    e = G + ((size_t)(m1 + scr) * MIN_NBS + b) * 2; e[0] = vy.h; e[1] = vy.l;
                    e = G + ((size_t)b * MIN_NBS + m1 + scr) * 2; e[0] = vy.h; e[1] = vy.l;
                }
                __syncwarp();
                if (nh == m) {                                      // evict the oldest pair
                    new_scr = c->hist[0];
                    __syncwarp();
                    if (lane == 0) {
                        for (int i = 0; i + 1 < m; i++) c->hist[i] = c->hist[i + 1];
                        c->hist[m - 1] = scr;
                    }
                } else {
                    if (lane == 0) c->hist[nh] = scr;
                    nh++;
                    new_scr = nh;                                   // slots 0..nh-1 are in use in order
                }
                __syncwarp();
            }
        }
        for (int b = lane; b < NB; b += 32) {                       // row / column of g
            dd v = D[2 * MIN_NBS + b];
            double* e;
            e = G + ((size_t)gidx * MIN_NBS + b) * 2; e[0] = v.h; e[1] = v.l;
            e = G + ((size_t)b * MIN_NBS + gidx) * 2; e[0] = v.h; e[1] = v.l;
        }
        __syncwarp();
        __threadfence_block();
        phi = phi_t;
        ls_fails = 0;
        if (lane == 0) {
            if (!first) c->iters++;
            c->smax[0] = smax_t.h; c->smax[1] = smax_t.l;
            c->scratch = new_scr;
        }
        if (dd_less(smax_t, dd{c->smax_tol, 0.0})) {
            done = 1; status = SHD_OK;
        } else {
            // two-loop recursion on coefficients: q = sum_l delta_l b_l, starting from q = g
            for (int b = lane; b < MIN_NBS; b += 32) delta[b] = dd{0.0, 0.0};
            __syncwarp();
            if (lane == 0) delta[gidx] = dd{1.0, 0.0};
            __syncwarp();
            for (int i = nh - 1; i >= 0; i--) {
                const int s = c->hist[i];
                const double* e = G + ((size_t)s * MIN_NBS + m1 + s) * 2;
                dd a = dd_div(gram_dot(delta, G, NB, s), dd{e[0], e[1]});
                if (lane == 0) { alpha[i] = a; delta[m1 + s] = dd_sub(delta[m1 + s], a); }
                __syncwarp();
            }
            if (nh > 0) {
                const int s = c->hist[nh - 1];
                const double* e1 = G + ((size_t)s * MIN_NBS + m1 + s) * 2;
                const double* e2 = G + ((size_t)(m1 + s) * MIN_NBS + m1 + s) * 2;
                dd gamma = dd_div(dd{e1[0], e1[1]}, dd{e2[0], e2[1]});
                if (lane == 0) c->gamma = gamma.h;
                for (int b = lane; b < NB; b += 32) delta[b] = dd_mul(delta[b], gamma);
                __syncwarp();
            }
            for (int i = 0; i < nh; i++) {
                const int s = c->hist[i];
                const double* e = G + ((size_t)s * MIN_NBS + m1 + s) * 2;
                dd beta = dd_div(gram_dot(delta, G, NB, m1 + s), dd{e[0], e[1]});
                if (lane == 0) delta[s] = dd_add(delta[s], dd_sub(alpha[i], beta));
                __syncwarp();
            }
            gp = dd_neg(gram_dot(delta, G, NB, gidx));
            const dd gg = D[2 * MIN_NBS + gidx];
            if (!(gp.h < 0.0) || !isfinite(gp.h)) {                 // not a descent direction: restart
                nh = 0;
                for (int b = lane; b < MIN_NBS; b += 32) delta[b] = dd{0.0, 0.0};
                __syncwarp();
                if (lane == 0) { delta[gidx] = dd{1.0, 0.0}; c->scratch = 0; }
                __syncwarp();
                gp = dd_neg(gg);
            }
            if (nh == 0) {
                // no curvature information: a continued quench reuses the last H0 scaling, a fresh one
                // takes the first step length 1 / |g| (capped at 1)
                const double gam = c->gamma;
                if (gam > 0.0 && isfinite(gam)) t = dd{gam, 0.0};
                else t = (gg.h > 1.0) ? dd_div(dd{1.0, 0.0}, dd_sqrt(gg)) : dd{1.0, 0.0};
            } else {
                t = dd{1.0, 0.0};
            }
            if (gg.h == 0.0) { done = 1; status = SHD_OK; }          // exact stationary point
            for (int b = lane; b < MIN_NBS; b += 32) { c->delta[b][0] = delta[b].h; c->delta[b][1] = delta[b].l; }
        }
    } else if (!done) {
        ls_fails++;
        t = dd_scale2(t, 0.5);
        if (ls_fails > MIN_MAX_LS) { done = 1; status = SHD_ESTALL; }
    }
    if (!done && evals >= c->max_evals) { done = 1; status = SHD_EMAXEVAL; }
    __syncwarp();
    if (lane == 0) {
        if (ring && c->ring_cap > 0) {           // one trace record per evaluation (collected by the host at every poll)
            shd_trace_rec& r = ring[c->ring_n % c->ring_cap];
            r.iters = (long)c->iters; r.evals = (long)evals;
            r.phi = phi_t.h; r.smax = smax_t.h;
            r.gnorm = sqrt(fmax(D[2 * MIN_NBS + gidx].h, 0.0));
            r.step = c->t[0]; r.limbs = c->limbs; r.accepted = accepted;
            c->ring_n++;
        }
        c->evals = evals;
        c->first = 0;
        c->accepted = accepted;
        c->nhist = nh;
        c->ls_fails = ls_fails;
        c->t[0] = t.h; c->t[1] = t.l;
        c->gp[0] = gp.h; c->gp[1] = gp.l;
        c->phi[0] = phi.h; c->phi[1] = phi.l;
        c->status = status;
        c->done = done;
    }
}

__global__ void __launch_bounds__(MIN_THREADS) k_min_update(
    long n, int m, const shd_minctrl* __restrict__ c, double* __restrict__ xt_hi, double* __restrict__ xt_lo,
    double* __restrict__ x, const double* __restrict__ gt, double* __restrict__ g, double* __restrict__ p,
    const double* __restrict__ S, const double* __restrict__ Y)
{
    const int done = c->done;
    if (done == 2) return;
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int acc = c->accepted, m1 = m + 1;
    dd xi, gi;
    if (acc) {
        xi = dd{xt_hi[i], xt_lo[i]};
        gi = ld2(gt, n, i);
        st2(x, n, i, xi);
        st2(g, n, i, gi);
    } else {
        xi = ld2(x, n, i);
    }
    if (done) {                       // finished: the caller's buffer holds the last accepted point
        if (c->status != SHD_ENAN) { xt_hi[i] = xi.h; xt_lo[i] = xi.l; }   // (ENAN: start point untouched)
        return;
    }
    dd pi;
    if (acc) {
        dd q = dd_mul(dd{c->delta[2 * m1][0], c->delta[2 * m1][1]}, gi);
        for (int b = 0; b < 2 * m1; b++) {
            dd dl{c->delta[b][0], c->delta[b][1]};
            if (dl.h == 0.0) continue;
            dd vb = b < m1 ? ld2(S + (size_t)b * 2 * n, n, i) : ld2(Y + (size_t)(b - m1) * 2 * n, n, i);
            q = dd_add(q, dd_mul(dl, vb));
        }
        pi = dd_neg(q);
        st2(p, n, i, pi);
    } else {
        pi = ld2(p, n, i);
    }
    dd xn = dd_add(xi, dd_mul(dd{c->t[0], c->t[1]}, pi));
    xt_hi[i] = xn.h; xt_lo[i] = xn.l;
}

int min_fail(shd_ctx* h, int code, const char* msg) { h->err = msg; return code; }

#define CUM(call)                                                                        \
    do {                                                                                 \
        cudaError_t e_ = (call);                                                         \
        if (e_ != cudaSuccess) {                                                         \
            h->err = std::string(#call) + ": " + cudaGetErrorString(e_);                 \
            h->d_skip = nullptr;                                                         \
            return e_ == cudaErrorMemoryAllocation ? SHD_ENOMEM : SHD_ECUDA;             \
        }                                                                                \
    } while (0)

int min_alloc(shd_ctx* h, int m) {
    shd_minstate* s = h->min;
    const long n = (long)h->d * h->N;
    if (s && s->m == m) return SHD_OK;
    shd_min_free(h);
    s = h->min = new shd_minstate();
    s->m = m; s->n = n;
    s->nblk = (int)((n + MIN_THREADS * MIN_EPT - 1) / (MIN_THREADS * MIN_EPT));
    const size_t v = (size_t)2 * n * sizeof(double), NB = 2 * (m + 1) + 1;
    CUM(cudaMalloc((void**)&s->x, v)); CUM(cudaMalloc((void**)&s->g, v));
    CUM(cudaMalloc((void**)&s->gt, v)); CUM(cudaMalloc((void**)&s->p, v));
    CUM(cudaMalloc((void**)&s->S, v * (m + 1))); CUM(cudaMalloc((void**)&s->Y, v * (m + 1)));
    CUM(cudaMalloc((void**)&s->partial, (size_t)s->nblk * NB * 3 * 2 * sizeof(double)));
    CUM(cudaMalloc((void**)&s->G, (size_t)MIN_NBS * MIN_NBS * 2 * sizeof(double)));
    if (shd_sharded(h)) {
        CUM(cudaMalloc((void**)&s->rank_part, NB * 3 * 2 * sizeof(double)));
        CUM(cudaMalloc((void**)&s->rank_all, (size_t)h->world * NB * 3 * 2 * sizeof(double)));
    }
    CUM(cudaMalloc((void**)&s->d_ctrl, sizeof(shd_minctrl)));
    CUM(cudaMallocHost((void**)&s->h_ctrl, sizeof(shd_minctrl)));
    std::memset(s->h_ctrl, 0, sizeof(shd_minctrl));
    h->workspace_bytes += v * (4 + 2 * (m + 1));
    return SHD_OK;
}

}  // namespace

void shd_min_free(shd_ctx* h) {
    shd_minstate* s = h->min;
    if (!s) return;
    cudaFree(s->x); cudaFree(s->g); cudaFree(s->gt); cudaFree(s->p); cudaFree(s->S); cudaFree(s->Y);
    cudaFree(s->partial); cudaFree(s->G); cudaFree(s->d_ctrl); cudaFree(s->rank_part); cudaFree(s->rank_all);
    cudaFree(s->d_ring);
    if (s->h_ring) cudaFreeHost(s->h_ring);
    if (s->h_ctrl) cudaFreeHost(s->h_ctrl);
    delete s;
    h->min = nullptr;
}

// rungs of the precision ladder: (limbs, stop below this S_max); the last rung is the handle's own precision down to tol
std::vector<std::pair<int, double>> shd_ladder_rungs(const shd_ctx* h, const shd_min_opts* o) {
    std::vector<std::pair<int, double>> r;
    const double l0 = o->ladder_tol[0], l1 = o->ladder_tol[1];
    if (h->nlimb > 1 && l0 > 0.0 && l0 > std::max(l1, o->smax_tol)) r.push_back({1, l0});
    if (h->nlimb > 2 && l1 > 0.0 && l1 > o->smax_tol) r.push_back({2, l1});
    r.push_back({h->nlimb, o->smax_tol});
    return r;
}

// host side of a poll: new trace records from the device ring into h->trace, then the caller's callback
bool shd_after_poll(shd_ctx* h, const shd_trace_rec* d_ring, shd_trace_rec* h_ring, int ring_cap, long long ring_n,
                    long long& ring_seen, const shd_min_opts* opts, const shd_min_report& rep) {
    if (d_ring && ring_n > ring_seen) {
        if (cudaMemcpyAsync(h_ring, d_ring, sizeof(shd_trace_rec) * ring_cap, cudaMemcpyDeviceToHost, h->stream) == cudaSuccess &&
            cudaStreamSynchronize(h->stream) == cudaSuccess) {
            for (long long i = std::max(ring_seen, ring_n - ring_cap); i < ring_n; i++)
                if (h->trace.size() < ((size_t)1 << 22)) h->trace.push_back(h_ring[i % ring_cap]);
        }
        ring_seen = ring_n;
    }
    return opts->on_poll && opts->on_poll(&rep, opts->on_poll_user) != 0;
}

extern "C" long shd_get_trace(shd_ctx* h, long first, long max, shd_trace_rec* out) {
    if (!h || !out || first < 0 || max < 1 || (size_t)first >= h->trace.size()) return 0;
    const long n = (long)std::min<size_t>((size_t)max, h->trace.size() - (size_t)first);
    std::memcpy(out, h->trace.data() + first, sizeof(shd_trace_rec) * (size_t)n);
    return n;
}

int shd_fire_snapshot(shd_ctx* h, double* pos_hi, double* pos_lo);

extern "C" int shd_minimize_snapshot(shd_ctx* h, double* pos_hi, double* pos_lo) {
    if (!h) return SHD_EINVAL;
    if (!pos_hi || !pos_lo) return min_fail(h, SHD_EINVAL, "NULL pointer");
    if (h->last_min_kind == 1) return shd_fire_snapshot(h, pos_hi, pos_lo);
    if (h->last_min_kind != 0 || !h->min) return min_fail(h, SHD_EINVAL, "shd_minimize_snapshot: no minimizer has run on this handle");
    const size_t b = (size_t)h->min->n * sizeof(double);
    cudaStream_t st = h->gstream ? h->gstream : h->stream;      // (from the poll callback: the minimizers' own stream)
    CUM(cudaMemcpyAsync(pos_hi, h->min->x, b, cudaMemcpyDeviceToDevice, st));
    CUM(cudaMemcpyAsync(pos_lo, h->min->x + h->min->n, b, cudaMemcpyDeviceToDevice, st));
    CUM(cudaStreamSynchronize(st));
    return SHD_OK;
}

extern "C" int shd_minimize(shd_ctx* h, double* pos_hi, double* pos_lo, const shd_min_opts* opts,
                            shd_min_report* report) {
    if (!h) return SHD_EINVAL;
    if (!pos_hi || !pos_lo || !opts || !report) return min_fail(h, SHD_EINVAL, "NULL pointer");
    if (!(opts->ladder_tol[0] >= 0.0) || !(opts->ladder_tol[1] >= 0.0)) return min_fail(h, SHD_EINVAL, "bad ladder_tol");
    h->trace.clear();
    if (opts->kind == 1) { h->last_min_kind = 1; return shd_fire_run(h, pos_hi, pos_lo, opts, report); }
    if (opts->kind != 0) return min_fail(h, SHD_EINVAL, "shd_minimize: kind must be 0 (L-BFGS) or 1 (FIRE)");
    const int m = opts->history == 0 ? 10 : opts->history;
    if (m < 1 || m > MIN_MAXHIST) return min_fail(h, SHD_EINVAL, "history must be in 1..32");
    if (!(opts->smax_tol >= 0.0) || opts->max_evals < 1 || opts->poll_every < 1)
        return min_fail(h, SHD_EINVAL, "bad smax_tol / max_evals / poll_every");
    int rc = min_alloc(h, m);
    if (rc) return rc;
    if ((rc = shd_prepare_tables(h, true))) return rc;
    h->last_min_kind = 0;
    shd_minstate* s = h->min;
    const long n = s->n;
    const size_t v = (size_t)2 * n * sizeof(double);
    cudaStream_t st = h->stream;
    if (s->ring_cap < opts->poll_every) {
        cudaFree(s->d_ring);
        if (s->h_ring) cudaFreeHost(s->h_ring);
        s->d_ring = nullptr; s->h_ring = nullptr;
        s->ring_cap = opts->poll_every;
        CUM(cudaMalloc((void**)&s->d_ring, sizeof(shd_trace_rec) * s->ring_cap));
        CUM(cudaMallocHost((void**)&s->h_ring, sizeof(shd_trace_rec) * s->ring_cap));
    }
    CUM(cudaMemsetAsync(s->x, 0, v, st)); CUM(cudaMemsetAsync(s->g, 0, v, st));
    CUM(cudaMemsetAsync(s->p, 0, v, st));
    CUM(cudaMemsetAsync(s->S, 0, v * (m + 1), st)); CUM(cudaMemsetAsync(s->Y, 0, v * (m + 1), st));
    CUM(cudaMemsetAsync(s->G, 0, (size_t)MIN_NBS * MIN_NBS * 2 * sizeof(double), st));
    const double gamma_prev = s->h_ctrl->gamma;      // 0 on a fresh state (min_alloc zeroes it)
    std::memset(s->h_ctrl, 0, sizeof(shd_minctrl));
    s->h_ctrl->gamma = gamma_prev;
    s->h_ctrl->m = m;
    s->h_ctrl->max_evals = opts->max_evals;
    s->h_ctrl->ring_cap = s->ring_cap;
    const unsigned ublk = (unsigned)((n + MIN_THREADS - 1) / MIN_THREADS);
    auto slot = [&]() -> cudaError_t {
        cudaError_t e;
        cudaStream_t q = h->stream;          // the capture stream while shd_run_slots is recording
        if ((e = shd_enqueue_eval(h, pos_hi, pos_lo, s->gt, s->gt + n)) != cudaSuccess) return e;
        k_min_dots<<<s->nblk, MIN_THREADS, 0, q>>>(n, m, s->d_ctrl, pos_hi, pos_lo, s->x, s->gt, s->g,
                                                   s->S, s->Y, s->partial);
        if (shd_sharded(h)) {
            // sharded vectors: this rank's sums of its block partials, all-gathered as bytes, added in rank order by
            // k_min_control on every rank (identical decisions everywhere: Phi, S_max and the dots are bit-identical)
            const int nq = 3 * (2 * (m + 1) + 1);
            k_rank_sum<<<(nq + 63) / 64, 64, 0, q>>>(s->nblk, nq, s->partial, s->rank_part, &s->d_ctrl->done);
            if ((e = shd_comm_allgather(h, s->rank_part, s->rank_all, (size_t)nq * 16)) != cudaSuccess) return e;
            k_min_control<<<1, MIN_THREADS, 0, q>>>(h->world, s->d_ctrl, h->d_scal, s->rank_all, s->G, s->d_ring);
        } else
            k_min_control<<<1, MIN_THREADS, 0, q>>>(s->nblk, s->d_ctrl, h->d_scal, s->partial, s->G, s->d_ring);
        k_min_update<<<ublk, MIN_THREADS, 0, q>>>(n, m, s->d_ctrl, pos_hi, pos_lo, s->x, s->gt, s->g,
                                                  s->p, s->S, s->Y);
        h->last_launches += 3;
        return cudaGetLastError();
    };
    // ---- the rungs of the precision ladder (one rung when opts->ladder_tol is zero): the device decides when a rung
    // ends (S_max below its threshold, or the line search stalls at the rung's precision floor); the pairs, the Gram
    // matrix and the counters carry over, the first slot of a rung re-evaluates Phi and the gradient at the current point
    const std::vector<std::pair<int, double>> rungs = shd_ladder_rungs(h, opts);
    const int nlimb_user = h->nlimb;
    shd_minctrl* c = s->h_ctrl;
    long long ring_seen = 0;
    bool stopped = false;
    for (size_t r = 0; r < rungs.size(); r++) {
        h->nlimb = rungs[r].first;
        c->done = 0; c->status = SHD_OK; c->first = 1; c->accepted = 0; c->ls_fails = 0;
        c->t[0] = 1.0; c->t[1] = 0.0;
        c->smax_tol = rungs[r].second;
        c->limbs = rungs[r].first;
        cudaError_t ce = cudaMemcpyAsync(s->d_ctrl, c, sizeof(shd_minctrl), cudaMemcpyHostToDevice, st);
        if (ce == cudaSuccess) {
            h->d_skip = &s->d_ctrl->done;
            ce = shd_run_slots(h, opts->poll_every, slot, c, s->d_ctrl, sizeof(shd_minctrl), &c->done, [&]() -> bool {
                shd_min_report rp;
                rp.iters = (long)c->iters; rp.evals = (long)c->evals;
                rp.phi[0] = c->phi[0]; rp.phi[1] = c->phi[1]; rp.smax[0] = c->smax[0]; rp.smax[1] = c->smax[1];
                rp.status = c->done ? c->status : SHD_OK;
                stopped = shd_after_poll(h, s->d_ring, s->h_ring, s->ring_cap, c->ring_n, ring_seen, opts, rp) && !c->done;
                return stopped;
            });
            h->d_skip = nullptr;
        }
        if (ce != cudaSuccess) { h->nlimb = nlimb_user; CUM(ce); }
        if (stopped) {
            // the caller's buffer holds a trial point: put the last accepted one back (k_min_update's exit path)
            c->done = 1; c->status = SHD_ESTOPPED; c->accepted = 0;
            CUM(cudaMemcpyAsync(s->d_ctrl, c, sizeof(shd_minctrl), cudaMemcpyHostToDevice, st));
            k_min_update<<<ublk, MIN_THREADS, 0, st>>>(n, m, s->d_ctrl, pos_hi, pos_lo, s->x, s->gt, s->g, s->p, s->S, s->Y);
            CUM(cudaStreamSynchronize(st));
            break;
        }
        if (r + 1 == rungs.size() || !(c->status == SHD_OK || c->status == SHD_ESTALL)) break;
    }
    h->nlimb = nlimb_user;
    report->iters = (long)c->iters;
    report->evals = (long)c->evals;
    report->phi[0] = c->phi[0]; report->phi[1] = c->phi[1];
    report->smax[0] = c->smax[0]; report->smax[1] = c->smax[1];
    report->status = c->status;
    if (c->status == SHD_ENAN) h->err = "shd_minimize: non-finite Phi at the starting point";
    else if (c->status == SHD_ESTALL) h->err = "shd_minimize: line search found no decrease";
    else if (c->status == SHD_EMAXEVAL) h->err = "shd_minimize: max_evals reached";
    else if (c->status == SHD_ESTOPPED) h->err = "shd_minimize: stopped by the poll callback";
    return c->status;
}
