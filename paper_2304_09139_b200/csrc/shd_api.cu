// shd_api.cu -- the C-ABI of include/shd.h: host-side setup (step a0: enumeration of Q, the
// outer-product decomposition, tile lists) and the launch sequences of the hot path.
#include "../../include/shd_bench.h"
#include "shd_internal.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <functional>
#include <map>
#include <new>
#include <utility>

namespace {

int fail(shd_ctx* h, int code, const std::string& msg) {
    if (h) h->err = msg;
    return code;
}
#define CU(call)                                                                         \
    do {                                                                                 \
        cudaError_t e_ = (call);                                                         \
        if (e_ != cudaSuccess) {                                                         \
            h->err = std::string(#call) + ": " + cudaGetErrorString(e_);                 \
            (void)cudaGetLastError();   /* a failed cudaMalloc must not poison the next launch check */ \
            return e_ == cudaErrorMemoryAllocation ? SHD_ENOMEM : SHD_ECUDA;             \
        }                                                                                \
    } while (0)

long isqrt_floor(long m) {
    long r = (long)std::floor(std::sqrt((double)m));
    while ((r + 1) * (r + 1) <= m) r++;
    while (r * r > m) r--;
    return r;
}

// a0: canonical half-space set Q (D:R6-R8): lexicographic, first non-zero component > 0
void enumerate_Q(int d, long m_star, std::vector<int>& out) {
    long R = isqrt_floor(m_star);
    out.clear();
    if (d == 1) {
        for (long n = 1; n <= R; n++) out.push_back((int)n);
    } else if (d == 2) {
        for (long a = 0; a <= R; a++) {
            long r1 = isqrt_floor(m_star - a * a);
            for (long b = (a == 0 ? 1 : -r1); b <= r1; b++) { out.push_back((int)a); out.push_back((int)b); }
        }
    } else {
        for (long a = 0; a <= R; a++) {
            long r1 = isqrt_floor(m_star - a * a);
            for (long b = (a == 0 ? 0 : -r1); b <= r1; b++) {
                long r2 = isqrt_floor(m_star - a * a - b * b);
                long c0 = (a == 0 && b == 0) ? 1 : -r2;
                for (long c = c0; c <= r2; c++) { out.push_back((int)a); out.push_back((int)b); out.push_back((int)c); }
            }
        }
    }
}

// d = 4 ("d = 1-4"): same order (lexicographic, n0 slowest), by filtering the cube
void enumerate_Q4(long m_star, std::vector<int>& out) {
    const long R = isqrt_floor(m_star);
    out.clear();
    for (long a = 0; a <= R; a++)
        for (long b = -R; b <= R; b++)
            for (long c = -R; c <= R; c++)
                for (long e = -R; e <= R; e++) {
                    if (a * a + b * b + c * c + e * e > m_star) continue;
                    const long first = a != 0 ? a : (b != 0 ? b : (c != 0 ? c : e));
                    if (first <= 0) continue;
                    out.push_back((int)a); out.push_back((int)b); out.push_back((int)c); out.push_back((int)e);
                }
}

template <class T>
int upload(shd_ctx* h, T** dst, const std::vector<T>& src) {
    size_t bytes = std::max<size_t>(src.size(), 1) * sizeof(T);
    CU(cudaMalloc((void**)dst, bytes));
    h->workspace_bytes += bytes;
    if (!src.empty()) CU(cudaMemcpy(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice));
    return SHD_OK;
}
int dalloc_zero(shd_ctx* h, double** dst, size_t ndoubles) {
    size_t bytes = std::max<size_t>(ndoubles, 1) * sizeof(double);
    CU(cudaMalloc((void**)dst, bytes));
    h->workspace_bytes += bytes;
    CU(cudaMemset(*dst, 0, bytes));
    return SHD_OK;
}

int build(shd_ctx* h, const double* v) {
    const int d = h->d;
    const long m_star = h->m_star;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)
        return fail(h, SHD_ECUDA, "no CUDA device: libshd has no CPU fallback");
    if (h->nvec.empty()) {                                     // else: the caller's table (shd_create_table)
        if (d == 4) enumerate_Q4(m_star, h->nvec); else enumerate_Q(d, m_star, h->nvec);
    }
    h->M = (long)h->nvec.size() / d;
    if (h->M < 1) return fail(h, SHD_EINVAL, "empty Q");
    if (v) {
        h->v.assign(v, v + h->M);
        for (double x : h->v)
            if (!(x > 0.0) || !std::isfinite(x)) return fail(h, SHD_EINVAL, "v(k) must be positive and finite");
    }
    // ---- outer-product decomposition, derived from the set itself (so that any half-space table works)
    std::map<std::vector<int>, int> index;
    long R0 = 0, Rlast = 0;
    for (long k = 0; k < h->M; k++) {
        std::vector<int> n(h->nvec.begin() + k * d, h->nvec.begin() + (k + 1) * d);
        int first = 0;
        for (int a = 0; a < d && first == 0; a++) first = n[a];
        if (first <= 0) return fail(h, SHD_EINVAL, "wavevector table: every n must be non-zero with its first non-zero component positive (half space, D:R7)");
        if (!index.emplace(n, (int)k).second) return fail(h, SHD_EINVAL, "wavevector table: duplicate n");
        R0 = std::max<long>(R0, n[0]);
        Rlast = std::max<long>(Rlast, std::abs(n[d - 1]));
        for (int a = 0; a < d; a++)
            if (std::abs((long)n[a]) > (d == 1 ? 2000000L : 2000L)) return fail(h, SHD_EINVAL, "wavevector table: |n_a| too large");
    }
    std::vector<std::vector<int>> wT(3);
    if (d == 1) {
        const long R = R0;
        int S = 2;
        while ((double)S * S < 2.0 * (double)R) S *= 2;
        h->S1d = S;
        h->Qn = S / 2 + 1;
        h->P = (int)((R + S / 2 - 1) / S) + 1;
        for (int p = 0; p < h->P; p++) { h->pn0.push_back(p); h->pn1.push_back(0); }
    } else if (d == 2) {
        h->P = (int)R0 + 1;
        h->Qn = (int)Rlast + 1;
        for (int p = 0; p < h->P; p++) { h->pn0.push_back(p); h->pn1.push_back(0); }
    } else {
        // A entries = the distinct prefixes (n0, n1) of the set, lexicographic (n0 ascending: k_tables walks
        // the powers of z0 forward)
        // (d = 4: prefixes (n0, n1, n2))
        std::map<std::vector<int>, int> prefixes;
        for (long k = 0; k < h->M; k++)
            prefixes.emplace(std::vector<int>(h->nvec.begin() + k * d, h->nvec.begin() + k * d + d - 1), 0);
        for (auto& pr : prefixes) {
            if (std::abs(pr.first[1]) > 128) return fail(h, SHD_EINVAL, "d >= 3 supports |n_1| <= 128");
            if (d == 4 && std::abs(pr.first[2]) > 32) return fail(h, SHD_EINVAL, "d = 4 supports |n_2| <= 32");
            h->pn0.push_back(pr.first[0]); h->pn1.push_back(pr.first[1]);
            h->pn2.push_back(d == 4 ? pr.first[2] : 0);
        }
        h->P = (int)h->pn0.size();
        h->Qn = (int)Rlast + 1;
    }
    h->npb = (h->P + 31) / 32;
    h->nqb = (h->Qn + 31) / 32;
    h->Qpad = h->nqb * 32;
    const int Ppad = h->npb * 32;
    h->qscale_log2 = 0;
    while ((1 << h->qscale_log2) < std::max(h->Qn - 1, 1)) h->qscale_log2++;
    for (int a = 0; a < 3; a++) wT[a].assign(Ppad, 0);
    for (int p = 0; p < h->P; p++) {
        if (d == 1) wT[0][p] = h->S1d * p;
        else if (d == 2) wT[0][p] = h->pn0[p];
        else { wT[0][p] = h->pn0[p]; wT[1][p] = h->pn1[p]; if (d == 4) wT[2][p] = h->pn2[p]; }
    }
    std::vector<int> kp((size_t)Ppad * h->Qpad, -1), km((size_t)Ppad * h->Qpad, -1);
    long found = 0;
    for (int p = 0; p < h->P; p++)
        for (int q = 0; q < h->Qn; q++)
            for (int sg = 1; sg >= -1; sg -= 2) {
                if (q == 0 && sg < 0) continue;
                std::vector<int> n(d);
                if (d == 1) n[0] = h->S1d * p + sg * q;
                else if (d == 2) { n[0] = h->pn0[p]; n[1] = sg * q; }
                else if (d == 3) { n[0] = h->pn0[p]; n[1] = h->pn1[p]; n[2] = sg * q; }
                else { n[0] = h->pn0[p]; n[1] = h->pn1[p]; n[2] = h->pn2[p]; n[3] = sg * q; }
                if (d == 1 && q == h->S1d / 2 && sg < 0) continue;   // S p - S/2 is (p-1, +S/2)
                auto it = index.find(n);
                if (it == index.end()) continue;
                int& slot = (sg > 0 ? kp : km)[(size_t)p * h->Qpad + q];
                if (slot >= 0) return fail(h, SHD_EINVAL, "internal: duplicate cell");
                slot = it->second;
                found++;
            }
    if (found != h->M) return fail(h, SHD_EINVAL, "internal: decomposition does not cover Q");
    // ---- tiles and q-chunk counts
    std::vector<int> tile_pb, tile_qb, tile_wmap;
    h->tile_weight = 0.0;
    h->valid_cells = 0;
    for (int pb = 0; pb < h->npb; pb++)
        for (int qb = 0; qb < h->nqb; qb++) {
            bool any = false;
            for (int pi = 0; pi < 32; pi++)
                for (int qi = 0; qi < 32; qi++) {
                    size_t c = (size_t)(pb * 32 + pi) * h->Qpad + qb * 32 + qi;
                    if (kp[c] >= 0 || km[c] >= 0) {
                        any = true;
                        h->valid_cells++;
                    }
                }
            if (any) {
                tile_pb.push_back(pb); tile_qb.push_back(qb);
                // units (8 p x 16 q) with a valid cell -> consumer warps; <= 4 of them: one per scheduler
                int valid_unit[8], nv = 0;
                for (int u = 0; u < 8; u++) {
                    bool uv = false;
                    for (int pi = 0; pi < 8 && !uv; pi++)
                        for (int qi = 0; qi < 16 && !uv; qi++) {
                            size_t c = (size_t)(pb * 32 + (u >> 1) * 8 + pi) * h->Qpad + qb * 32 + (u & 1) * 16 + qi;
                            uv = kp[c] >= 0 || km[c] >= 0;
                        }
                    if (uv) valid_unit[nv++] = u;
                }
                int wmap[9];
                for (int w = 0; w < 8; w++) wmap[w] = -1;
                if (nv <= 4) for (int i = 0; i < nv; i++) wmap[i] = valid_unit[i];
                else for (int i = 0; i < nv; i++) wmap[valid_unit[i]] = valid_unit[i];
                wmap[8] = nv;
                tile_wmap.insert(tile_wmap.end(), wmap, wmap + 9);
                h->tile_weight += nv <= 4 ? 0.6 : 1.0;      // one warp per scheduler: ~half the time
            }
        }
    h->ntiles = (int)tile_pb.size();
    // ---- gradient pass: step list over blocks of 16 p (q-groups up to the last valid cell of the block)
    h->npb16 = (h->P + SHD_PG - 1) / SHD_PG;
    std::vector<int> steps;
    const int fold_every = SHD_BURST / 8;        // 2 products per q and L0 accumulator, 4 q per step
    for (int pb = 0; pb < h->npb16; pb++) {
        int nq = 0;
        for (int pi = 0; pi < SHD_PG; pi++)
            for (int q = 0; q < h->Qpad; q++) {
                size_t c = (size_t)(pb * SHD_PG + pi) * h->Qpad + q;
                if (kp[c] >= 0 || km[c] >= 0) nq = std::max(nq, q / SHD_QCH + 1);
            }
        for (int qg = 0; qg < nq; qg++) {
            // flag 1: end of a block: after <= 64 steps (one exact burst) or at the block's last q-group
            // (the p-contraction is linear in T, so a long q-range may be contracted in pieces)
            int flags = ((qg + 1) % fold_every == 0 || qg == nq - 1) ? 1 : 0;
            steps.push_back(pb * (h->Qpad / 4) + qg);
            steps.push_back(qg | (flags << 16));
        }
    }
    h->nsteps = (int)steps.size() / 2;
    h->grad_qsteps = (long)h->nsteps * SHD_QCH;
    // ---- particle splits of the rho pass: minimise (waves of CTAs) x (chunks per CTA)
    cudaDeviceProp prop;
    int dev = 0;
    cudaGetDevice(&dev);
    if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return fail(h, SHD_ECUDA, "cudaGetDeviceProperties failed");
    const long sms = prop.multiProcessorCount;
    h->sms = (int)sms;
    const long nchunks = (h->N + SHD_NPS - 1) / SHD_NPS;
    // CTAs are dispatched in blockIdx order (split-major, tile-minor) to the first free SM; a tile with
    // <= 4 valid units takes ~0.6 of a full tile's time.  Simulate that list schedule for every split count.
    double best_cost = -1.0;
    {
        std::vector<double> tw(h->ntiles);
        for (int t = 0; t < h->ntiles; t++) tw[t] = tile_wmap[(size_t)t * 9 + 8] <= 4 ? 0.6 : 1.0;
        std::vector<double> sm_free((size_t)sms);
        for (long ns = 1; ns <= std::min<long>(256, nchunks); ns++) {
            const long cps = (nchunks + ns - 1) / ns;
            std::fill(sm_free.begin(), sm_free.end(), 0.0);
            std::make_heap(sm_free.begin(), sm_free.end(), std::greater<double>());
            double makespan = 0.0;
            for (long b = 0; b < (long)h->ntiles * ns; b++) {
                std::pop_heap(sm_free.begin(), sm_free.end(), std::greater<double>());
                double& slot = sm_free.back();
                slot += tw[b % h->ntiles] * (double)cps + 2.0;        // +2: per-CTA prologue/epilogue
                makespan = std::max(makespan, slot);
                std::push_heap(sm_free.begin(), sm_free.end(), std::greater<double>());
            }
            // k_finish1 sums ns partials per cell: measured ~0.015 chunk-times per (split, tile)
            const double cost = makespan + 0.015 * (double)ns * (double)h->ntiles;
            if (best_cost < 0.0 || cost < best_cost) { best_cost = cost; h->nsplit = (int)ns; h->chunks_per_split = cps; }
        }
    }
    h->njb = (h->N + 31) / 32;
    // ---- segments of the gradient pass: minimise (waves of CTAs) x (steps per CTA)
    {
        double best = -1.0;
        h->nseg = 1;
        const long njb64 = (h->N + SHD_JT - 1) / SHD_JT;
        for (int ns = 1; ns <= std::min(16, h->nsteps); ns++) {
            long waves = (njb64 * ns + sms - 1) / sms;
            double cost = (double)waves * ((double)((h->nsteps + ns - 1) / ns) + 4.0);   // +4: prologue, epilogue, partial write
            if (best < 0.0 || cost < best) { best = cost; h->nseg = ns; }
        }
    }
    // ---- device memory that does not depend on the engine or on the chunk size
    int rc;
    if ((rc = upload(h, &h->d_pn0, h->pn0))) return rc;
    if ((rc = upload(h, &h->d_pn1, h->pn1))) return rc;
    if ((rc = upload(h, &h->d_pn2, h->pn2))) return rc;
    std::vector<int> wflat;
    for (int a = 0; a < 3; a++) wflat.insert(wflat.end(), wT[a].begin(), wT[a].end());
    if ((rc = upload(h, &h->d_wT, wflat))) return rc;
    if ((rc = upload(h, &h->d_cell_kp, kp))) return rc;
    if ((rc = upload(h, &h->d_cell_km, km))) return rc;
    if ((rc = upload(h, &h->d_tile_pb, tile_pb))) return rc;
    if ((rc = upload(h, &h->d_tile_qb, tile_qb))) return rc;
    if ((rc = upload(h, &h->d_tile_wmap, tile_wmap))) return rc;
    if ((rc = upload(h, &h->d_steps, steps))) return rc;
    if (!h->v.empty()) { if ((rc = upload(h, &h->d_v, h->v))) return rc; }
    if ((rc = dalloc_zero(h, &h->d_rho, (size_t)4 * h->M))) return rc;
    CU(cudaMalloc((void**)&h->d_scal, sizeof(shd_scalars)));
    CU(cudaMemset(h->d_scal, 0, sizeof(shd_scalars)));
    CU(cudaMallocHost((void**)&h->h_scal, sizeof(shd_scalars)));
    std::memset(h->h_scal, 0, sizeof(shd_scalars));
    h->cell_kp.swap(kp);
    h->cell_km.swap(km);
    CU(shd_tables_configure());
    CU(shd_rho_configure());
    CU(shd_grad_configure());
    return SHD_OK;
}

// ---- INT8 engines: tile list and particle splits of the rho pass (k_rho8.cu), step list of the gradient pass
// (k_grad8.cu).  Host work and small uploads only; the digit tables are allocated by shd_prepare_tables.
int plan_engine8(shd_ctx* h, int engine) {
    cudaDeviceProp prop;
    int dev = 0;
    cudaGetDevice(&dev);
    CU(cudaGetDeviceProperties(&prop, dev));
    const long sms = prop.multiProcessorCount;
    const std::vector<int>&kp = h->cell_kp, &km = h->cell_km;
    int rc;
    if (engine == 2 && !h->d_steps8) {
        // step list over blocks of 8 p (K-steps of 16 q up to the block's last valid cell)
        h->npb8 = (h->P + 7) / 8;
        h->nkq8 = h->Qpad / 16;
        std::vector<int> steps;
        for (int pb = 0; pb < h->npb8; pb++) {
            int nk = 0;
            for (int pi = 0; pi < 8; pi++) {
                const int p = pb * 8 + pi;
                if (p >= h->npb * 32) continue;
                for (int q = 0; q < h->Qpad; q++)
                    if (kp[(size_t)p * h->Qpad + q] >= 0 || km[(size_t)p * h->Qpad + q] >= 0) nk = std::max(nk, q / 16 + 1);
            }
            for (int k = 0; k < nk; k++) {
                steps.push_back(pb * h->nkq8 + k);
                steps.push_back(k | ((k == nk - 1 ? 1 : 0) << 16));
            }
        }
        h->nsteps8 = (int)steps.size() / 2;
        double best = -1.0;
        h->nseg8 = 1;
        const long njb128 = (h->N + 127) / 128;
        // at least two segments: the CTAs of one particle block then stream the same digit slabs side by side (L2).
        // The kernel is persistent (one CTA per SM walks the units round-robin), so a unit costs its steps plus about one
        // block's epilogue (1.5 step-times), not a CTA prologue: finer segments balance small systems (cfg3: 79 particle
        // blocks on 148 SMs) at the price of one more partial gradient per segment for k_gradsum to add (0.05 each).
        for (int ns = std::min(2, h->nsteps8); ns <= std::min(32, h->nsteps8); ns++) {
            const long rounds = (njb128 * ns + sms - 1) / sms;
            const double cost = (double)rounds * ((double)((h->nsteps8 + ns - 1) / ns) + 1.5) + 0.05 * ns;
            if (best < 0.0 || cost < best) { best = cost; h->nseg8 = ns; }
        }
        if ((rc = upload(h, &h->d_steps8, steps))) return rc;
        CU(shd_grad8_configure());
    }
    if (engine >= 1 && !h->d_tile8_pb) {
        h->npb64 = (h->P + SHD_I8_PT - 1) / SHD_I8_PT;
        h->nqb16 = (h->Qn + SHD_I8_QT - 1) / SHD_I8_QT;
        std::vector<int> tpb, tqb;
        for (int pb = 0; pb < h->npb64; pb++)
            for (int qb = 0; qb < h->nqb16; qb++) {
                bool any = false;
                for (int pi = 0; pi < SHD_I8_PT && !any; pi++)
                    for (int qi = 0; qi < SHD_I8_QT && !any; qi++) {
                        const int p = pb * SHD_I8_PT + pi, q = qb * SHD_I8_QT + qi;
                        if (p < h->npb * 32 && q < h->Qpad) any = kp[(size_t)p * h->Qpad + q] >= 0 || km[(size_t)p * h->Qpad + q] >= 0;
                    }
                if (any) { tpb.push_back(pb); tqb.push_back(qb); }
            }
        h->ntiles8 = (int)tpb.size();
        // particle splits: at most SHD_I8_MAXN particles per CTA (exact s32 sums); minimise waves x (K-steps + epilogue)
        const long nk = (h->N + 31) / 32;
        double best = -1.0;
        h->nsplit8 = 0;
        for (long ns = (h->N + SHD_I8_MAXN - 1) / SHD_I8_MAXN; ns <= std::max<long>(std::min<long>(512, nk), (h->N + SHD_I8_MAXN - 1) / SHD_I8_MAXN); ns++) {
            const long per = (nk + ns - 1) / ns, waves = ((long)h->ntiles8 * ns + sms - 1) / sms;
            const double cost = (double)waves * ((double)per + 8.0) + 0.004 * (double)ns * h->ntiles8;
            if (best < 0.0 || cost < best) { best = cost; h->nsplit8 = (int)ns; h->ksteps8 = (int)per; }
        }
        if (h->nsplit8 < 1 || (long)h->ksteps8 * 32 > SHD_I8_MAXN)
            return fail(h, SHD_EINVAL, "shd_set_engine: no particle split keeps the s32 digit sums of the INT8 rho pass exact");
        if ((rc = upload(h, &h->d_tile8_pb, tpb))) return rc;
        if ((rc = upload(h, &h->d_tile8_qb, tqb))) return rc;
        CU(shd_rho8_configure());
    }
    return SHD_OK;
}

void free_tables(shd_ctx* h) {
    cudaFree(h->d_A); cudaFree(h->d_B); cudaFree(h->d_Bg); cudaFree(h->d_A8); cudaFree(h->d_B8); cudaFree(h->d_Bg8);
    cudaFree(h->d_Afix); cudaFree(h->d_W8); cudaFree(h->d_C); cudaFree(h->d_part); cudaFree(h->d_gpart);
    cudaFree(h->d_blockred); cudaFree(h->d_xrun); cudaFree(h->d_xall);
    h->d_A = h->d_B = h->d_Bg = h->d_C = h->d_part = h->d_gpart = h->d_blockred = h->d_xrun = h->d_xall = nullptr;
    h->d_A8 = h->d_B8 = h->d_Bg8 = h->d_W8 = nullptr;
    h->d_Afix = nullptr;
    h->workspace_bytes -= h->table_bytes;
    h->table_bytes = 0;
    h->tables_valid = false;
    h->grad_tables_ready = false;
}

// bytes of per-particle tables (both passes) and of rho-pass partials per split for the current engine
void table_footprint(const shd_ctx* h, double& per_particle, double& per_split, double& fixed) {
    const int e = h->rho_engine;
    const double limbA = (double)h->npb * 1536.0, limbB = (double)h->nqb * 1536.0, limbBg = (double)h->Qpad * 48.0;
    const double a8 = (double)h->npb64 * 1664.0, b8 = (double)h->nqb16 * 416.0, bg8 = (double)h->nkq8 * 416.0;
    const double afix = (double)h->npb8 * 8 * 32.0;
    const int ntiles = e >= 1 ? h->ntiles8 : h->ntiles;
    if (e == 0) per_particle = limbA + limbB + limbBg + (double)h->nseg * h->d * 16.0;
    else if (e == 1) per_particle = a8 + b8 + limbA + limbBg + (double)h->nseg * h->d * 16.0;
    else per_particle = a8 + b8 + bg8 + afix + 4.0 * h->nseg8 * h->d * 16.0;
    per_split = (double)ntiles * 65536.0;
    fixed = 3.0 * ntiles * 65536.0 + (double)h->npb16 * (h->Qpad / 4) * 16384.0 + (double)h->npb8 * h->nkq8 * SHD_I8_DIGITS * 1024.0;
}

// chunk size for the current engine: as many whole splits as the workspace cap (or the free device memory) holds
int choose_chunks(shd_ctx* h) {
    const int e = h->rho_engine;
    const long nsplit_total = e >= 1 ? h->nsplit8 : h->nsplit;
    h->unit = e >= 1 ? (long)h->ksteps8 * 32 : h->chunks_per_split * SHD_NPS;
    double pp, ps, fx;
    table_footprint(h, pp, ps, fx);
    double cap = (double)h->ws_cap;
    if (h->ws_cap == 0) {
        size_t fr = 0, tot = 0;
        CU(cudaMemGetInfo(&fr, &tot));
        cap = 0.92 * (double)fr;
    }
    const double per_split_all = pp * (double)h->unit + ps;
    long m = (long)std::floor((cap - fx) / per_split_all);
    if (m < 1) return fail(h, SHD_ENOMEM, "workspace cap (or free device memory) below the tables of one particle split");
    m = std::min(m, nsplit_total);
    h->nchunk = (int)((nsplit_total + m - 1) / m);
    h->spc = (int)((nsplit_total + h->nchunk - 1) / h->nchunk);          // balanced chunks
    h->nchunk = (int)((nsplit_total + h->spc - 1) / h->spc);
    h->Nc = (long)h->spc * h->unit;
    h->Npad = e == 0 ? h->Nc : ((h->Nc + 7) / 8) * 8;                    // FP64 limb tables (engine 1: A limbs and Bg of the gradient pass)
    h->nk8 = e >= 1 ? (long)h->spc * h->ksteps8 : 0;
    h->njb64 = (h->Nc + SHD_JT - 1) / SHD_JT;
    h->njb128 = e == 2 ? (h->Nc + 127) / 128 : 0;
    return SHD_OK;
}

}  // namespace

// Device tables of the current (engine, chunk) setting, allocated on first use (outside any stream capture) and freed
// when the setting changes: a handle driven on the INT8 engines never holds the FP64 limb tables and vice versa.
int shd_prepare_tables(shd_ctx* h, bool with_grad) {
    int rc;
    const int e = h->rho_engine;
    if (!h->tables_valid) {
        free_tables(h);
        if ((rc = choose_chunks(h))) return rc;
        const size_t before = h->workspace_bytes;
        const int ntiles = e >= 1 ? h->ntiles8 : h->ntiles;
        const size_t xdoubles = (size_t)ntiles * 4 * 1024 * 2;
        if (e == 0 || e == 1) {
            if (e == 0 && (rc = dalloc_zero(h, &h->d_B, (size_t)h->nqb * (h->Npad / 4) * SHD_GROUP_DOUBLES))) return rc;
        }
        if (e >= 1) {
            const size_t a8 = (size_t)h->npb64 * h->nk8 * SHD_I8_DIGITS * (SHD_I8_PT * 2 * 32);
            const size_t b8 = (size_t)h->nqb16 * h->nk8 * SHD_I8_DIGITS * (SHD_I8_QT * 2 * 32);
            CU(cudaMalloc((void**)&h->d_A8, a8));
            CU(cudaMalloc((void**)&h->d_B8, b8));
            CU(cudaMemset(h->d_A8, 0, a8));
            CU(cudaMemset(h->d_B8, 0, b8));
            h->workspace_bytes += a8 + b8;
        }
        if (e == 0 && (rc = dalloc_zero(h, &h->d_A, (size_t)h->npb * (h->Npad / 4) * SHD_GROUP_DOUBLES))) return rc;
        if ((rc = dalloc_zero(h, &h->d_part, (size_t)h->spc * xdoubles))) return rc;
        if ((rc = dalloc_zero(h, &h->d_blockred, (size_t)(((long)ntiles * 1024 + 255) / 256) * 8))) return rc;
        if (h->nchunk > 1 || shd_sharded(h))
            if ((rc = dalloc_zero(h, &h->d_xrun, xdoubles))) return rc;
        if (shd_sharded(h))
            if ((rc = dalloc_zero(h, &h->d_xall, (size_t)h->world * xdoubles))) return rc;
        h->table_bytes += h->workspace_bytes - before;
        h->tables_valid = true;
    }
    if (with_grad && !h->d_gpart) {
        const size_t before = h->workspace_bytes;
        if (e == 2) {
            const size_t g8 = (size_t)h->njb128 * h->nkq8 * SHD_I8_DIGITS * 4096;
            const size_t w8 = (size_t)h->npb8 * h->nkq8 * SHD_I8_DIGITS * 1024;
            const size_t af = (size_t)h->npb8 * 8 * (size_t)h->njb128 * 128 * 32;
            CU(cudaMalloc(&h->d_Afix, af));
            CU(cudaMemset(h->d_Afix, 0, af));
            CU(cudaMalloc((void**)&h->d_Bg8, g8));
            CU(cudaMemset(h->d_Bg8, 0, g8));
            CU(cudaMalloc((void**)&h->d_W8, w8));
            CU(cudaMemset(h->d_W8, 0, w8));
            h->workspace_bytes += g8 + w8 + af;
            if ((rc = dalloc_zero(h, &h->d_gpart, (size_t)4 * h->nseg8 * h->d * h->Nc * 2))) return rc;
        } else {
            if (e == 1 && (rc = dalloc_zero(h, &h->d_A, (size_t)h->npb * (h->Npad / 4) * SHD_GROUP_DOUBLES))) return rc;
            if ((rc = dalloc_zero(h, &h->d_Bg, (size_t)(2 * h->njb64) * (h->Qpad / 4) * SHD_GROUP_DOUBLES))) return rc;
            if ((rc = dalloc_zero(h, &h->d_C, (size_t)h->npb16 * (h->Qpad / 4) * (16 * SHD_PG * 4 * 2)))) return rc;
            if ((rc = dalloc_zero(h, &h->d_gpart, (size_t)h->nseg * h->d * h->Nc * 2))) return rc;
        }
        h->table_bytes += h->workspace_bytes - before;
    }
    return SHD_OK;
}

// ---- the evaluation, enqueued on h->stream (also inside the minimizers' captured slots)
cudaError_t shd_enqueue_rho_partial(shd_ctx* h, const double* pos_hi, const double* pos_lo, bool grad_tables_too)
{
    const int e = h->rho_engine;
    const long nsplit_total = e >= 1 ? h->nsplit8 : h->nsplit;
    const bool both = h->nchunk == 1 && grad_tables_too;      // one chunk: one table build serves both passes
    // (Building the gradient pass's tables on a side stream beside k_rho8 was tried and is slower, 4.73 against 4.45 ms at
    // cfg4: k_tables is bound by its FP64 recurrences, not by its writes -- the rho tables alone take 0.65 of its 0.73 ms --
    // and FP64 all but stalls beside a tensor stream, so the second launch repeats the recurrences and then waits.)
    cudaError_t err;
    for (int c = 0; c < h->nchunk; c++) {
        const long j0 = (long)c * h->Nc;
        const int ns = (int)std::min<long>(h->spc, nsplit_total - (long)c * h->spc);
        const bool last = c == h->nchunk - 1;
        if ((err = shd_launch_tables(h, pos_hi, pos_lo, j0, both ? 3 : 1)) != cudaSuccess) return err;
        if (c == 0 && h->timing_mark) h->timing_mark(h, 1);
        if ((err = shd_launch_rho(h, ns)) != cudaSuccess) return err;
        if (last && h->timing_mark) h->timing_mark(h, 2);
        const bool fin = last && !shd_sharded(h);
        if ((err = shd_launch_fold(h, h->d_part, ns, c > 0 ? h->d_xrun : nullptr, fin ? nullptr : h->d_xrun, fin)) != cudaSuccess) return err;
    }
    h->grad_tables_ready = both;
    return cudaSuccess;
}

cudaError_t shd_enqueue_rho_finish(shd_ctx* h, const double* gathered, int nparts)
{
    return shd_launch_fold(h, gathered, nparts, nullptr, nullptr, true);
}

cudaError_t shd_enqueue_grad(shd_ctx* h, const double* pos_hi, const double* pos_lo, double* grad_hi, double* grad_lo)
{
    cudaError_t err;
    if ((err = shd_launch_ctable(h)) != cudaSuccess) return err;
    if (h->timing_mark) h->timing_mark(h, 4);
    for (int c = 0; c < h->nchunk; c++) {
        const long j0 = (long)c * h->Nc;
        const long nc = std::min<long>(h->Nc, h->N - j0);
        if (nc <= 0) break;
        if (!h->grad_tables_ready)
            if ((err = shd_launch_tables(h, pos_hi, pos_lo, j0, 2)) != cudaSuccess) return err;
        if ((err = shd_launch_grad(h, j0, nc, grad_hi, grad_lo)) != cudaSuccess) return err;
    }
    h->grad_tables_ready = false;          // the caller may move the particles before the next call
    return cudaSuccess;
}

cudaError_t shd_enqueue_eval(shd_ctx* h, const double* pos_hi, const double* pos_lo, double* grad_hi, double* grad_lo)
{
    cudaError_t err;
    h->last_launches = 0;
    if (h->timing_mark) h->timing_mark(h, 0);
    if ((err = shd_enqueue_rho_partial(h, pos_hi, pos_lo, grad_hi != nullptr)) != cudaSuccess) return err;
    if (shd_sharded(h)) {
        const int ntiles = h->rho_engine >= 1 ? h->ntiles8 : h->ntiles;
        if ((err = shd_comm_allgather(h, h->d_xrun, h->d_xall, (size_t)ntiles * 4 * 1024 * 16)) != cudaSuccess) return err;
        if ((err = shd_enqueue_rho_finish(h, h->d_xall, h->world)) != cudaSuccess) return err;
    }
    if (h->timing_mark) h->timing_mark(h, 3);
    if (grad_hi) {
        if ((err = shd_enqueue_grad(h, pos_hi, pos_lo, grad_hi, grad_lo)) != cudaSuccess) return err;
        if (h->timing_mark) h->timing_mark(h, 5);
    }
    return cudaSuccess;
}

namespace {

// The engine a fresh handle starts on: both O(N M) passes on the INT8 tensor cores (engine 2) where they pay off --
// a last-axis table short enough for exact s32 sums and enough pair-terms to amortise the digit tables (measured on
// B200: cfg2, 8e7 pair-terms, 0.23 ms against 0.44 ms; cfg3, d = 3 with an 18-entry last axis, 0.61 against 0.95 ms;
// cfg1, 9e3 pair-terms, is launch-bound either way) -- else the FP64 limb engine.  shd_set_engine overrides.
void auto_engine(shd_ctx* h) {
    h->engine_auto = 1;
    const bool fits8 = (long)h->Qpad * 2 * SHD_I8_DIGITS * 16384 < (1L << 31);
    const bool pays = (double)h->N * (double)h->M >= 5e7;
    if (fits8 && pays && plan_engine8(h, 2) == SHD_OK) h->rho_engine = 2;
    else { h->rho_engine = 0; h->err.clear(); }
}

// table != nullptr: the caller's half-space set (M vectors, row-major) instead of the shell n.n <= m_star
int create_common(int d, long N, double L, long m_star, const double* v, shd_ctx** out,
                  const int* table = nullptr, long M = 0) {
    if (!out) return SHD_EINVAL;
    *out = nullptr;
    if (d < 1 || d > 4 || N < 1 || !(L > 0.0) || !std::isfinite(L)) return SHD_EINVAL;
    if (table) {
        if (M < 1 || M > 50000000L) return SHD_EINVAL;
    } else {
        if (m_star < 1) return SHD_EINVAL;
        if (d == 1 && m_star > (long)4e12) return SHD_EINVAL;
        if (d >= 2 && m_star > (long)4e6) return SHD_EINVAL;
        if (d == 4 && m_star > 32 * 32) return SHD_EINVAL;
    }
    shd_ctx* h = new (std::nothrow) shd_ctx();
    if (!h) return SHD_ENOMEM;
    h->d = d; h->N = N; h->Nsys = N; h->L = L; h->m_star = m_star;
    if (table) {
        h->nvec.assign(table, table + M * d);
        h->m_star = 0;
        for (long k = 0; k < M; k++) {
            long nn = 0;
            for (int a = 0; a < d; a++) nn += (long)table[k * d + a] * table[k * d + a];
            h->m_star = std::max(h->m_star, nn);       // largest |n|^2 (k_max of the FIRE default time step)
        }
    }
    int rc;
    try {
        rc = build(h, v);
        if (rc == SHD_OK) auto_engine(h);
    } catch (const std::bad_alloc&) {
        rc = SHD_ENOMEM;
        h->err = "host allocation failed";
    }
    *out = h;            // returned even on error so that shd_last_error() can be read; caller destroys
    return rc;
}

// event i is recorded BEFORE launch group i; event SHD_NKERN after the last group
void mark(shd_ctx* h, int i) {
    if (!h->timing) return;
    if (cudaEventRecord(h->ev[i], h->stream) == cudaSuccess) h->ev_used[i] = true;
}
int collect_timing(shd_ctx* h) {      // after the stream has been synchronised
    if (!h->timing) return SHD_OK;
    for (int i = 0; i < SHD_NKERN; i++) {
        h->kern_ms[i] = 0.f;
        if (!h->ev_used[i]) continue;
        int nxt = i + 1;
        while (nxt <= SHD_NKERN && !h->ev_used[nxt]) nxt++;
        if (nxt > SHD_NKERN) continue;
        CU(cudaEventElapsedTime(&h->kern_ms[i], h->ev[i], h->ev[nxt]));
    }
    return SHD_OK;
}
int fetch_scalars(shd_ctx* h) {
    CU(cudaMemcpyAsync(h->h_scal, h->d_scal, sizeof(shd_scalars), cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    return SHD_OK;
}
int run_eval(shd_ctx* h, const double* pos_hi, const double* pos_lo, double* grad_hi, double* grad_lo) {
    int rc = shd_prepare_tables(h, grad_hi != nullptr);
    if (rc) return rc;
    for (int i = 0; i <= SHD_NKERN; i++) h->ev_used[i] = false;
    h->timing_mark = h->timing ? mark : nullptr;
    cudaError_t e = shd_enqueue_eval(h, pos_hi, pos_lo, grad_hi, grad_lo);
    h->timing_mark = nullptr;
    CU(e);
    if ((rc = fetch_scalars(h))) return rc;
    return collect_timing(h);
}

}  // namespace

extern "C" {

int shd_create_shell(int d, long N, double L, long m_star, const double* v, shd_ctx** out) {
    return create_common(d, N, L, m_star, v, out);
}

int shd_create_table(int d, long N, double L, long M, const int* n, const double* v, shd_ctx** out) {
    if (!n) { if (out) *out = nullptr; return SHD_EINVAL; }
    return create_common(d, N, L, 0, v, out, n, M);
}

int shd_create(int d, long N, double L, double K, const double* v, shd_ctx** out) {
    if (!(K > 0.0) || !std::isfinite(K) || !(L > 0.0) || !std::isfinite(L)) { if (out) *out = nullptr; return SHD_EINVAL; }
    double x = K * L / (2.0 * 3.14159265358979323846);
    double m = std::floor(x * x * (1.0 + std::ldexp(1.0, -40)));
    if (!(m >= 1.0) || m > 4e12) { if (out) *out = nullptr; return SHD_EINVAL; }
    return create_common(d, N, L, (long)m, v, out);
}

void shd_destroy(shd_ctx* h) {
    if (!h) return;
    shd_min_free(h);
    shd_fire_free(h);
    shd_comm_free(h);
    free_tables(h);
    cudaFree(h->d_pn0); cudaFree(h->d_pn1); cudaFree(h->d_pn2); cudaFree(h->d_wT); cudaFree(h->d_cell_kp); cudaFree(h->d_cell_km);
    cudaFree(h->d_tile_pb); cudaFree(h->d_tile_qb); cudaFree(h->d_tile_wmap); cudaFree(h->d_steps); cudaFree(h->d_v);
    cudaFree(h->d_rho); cudaFree(h->d_scal); cudaFree(h->d_hpos);
    cudaFree(h->d_tile8_pb); cudaFree(h->d_tile8_qb); cudaFree(h->d_steps8); cudaFree(h->d_trace);
    for (int i = 0; i <= SHD_NKERN; i++) if (h->ev[i]) cudaEventDestroy(h->ev[i]);
    if (h->h_scal) cudaFreeHost(h->h_scal);
    if (h->gevent) cudaEventDestroy(h->gevent);
    if (h->gstream) cudaStreamDestroy(h->gstream);
    delete h;
}

int shd_set_stream(shd_ctx* h, void* cuda_stream) {
    if (!h) return SHD_EINVAL;
    h->stream = (cudaStream_t)cuda_stream;
    return SHD_OK;
}

long shd_num_k(const shd_ctx* h) { return h ? h->M : 0; }

int shd_get_k(const shd_ctx* h, int* n_out) {
    if (!h || !n_out) return SHD_EINVAL;
    std::memcpy(n_out, h->nvec.data(), h->nvec.size() * sizeof(int));
    return SHD_OK;
}

int shd_energy_grad(shd_ctx* h, const double* pos_hi, const double* pos_lo, double phi[2],
                    double* grad_hi, double* grad_lo) {
    if (!h) return SHD_EINVAL;
    if (!pos_hi || !pos_lo || !phi) return fail(h, SHD_EINVAL, "NULL pointer");
    if ((grad_hi == nullptr) != (grad_lo == nullptr)) return fail(h, SHD_EINVAL, "grad_hi and grad_lo must both be given or both NULL");
    int rc = run_eval(h, pos_hi, pos_lo, grad_hi, grad_lo);
    if (rc) return rc;
    phi[0] = h->h_scal->phi[0];
    phi[1] = h->h_scal->phi[1];
    if (h->h_scal->nonfinite) return fail(h, SHD_ENAN, "non-finite Phi (non-finite positions?)");
    return SHD_OK;
}

int shd_energy_grad_host(shd_ctx* h, const double* pos_hi, const double* pos_lo, double phi[2],
                         double* grad_hi, double* grad_lo) {
    if (!h) return SHD_EINVAL;
    if (!pos_hi || !pos_lo || !phi) return fail(h, SHD_EINVAL, "NULL pointer");
    if ((grad_hi == nullptr) != (grad_lo == nullptr)) return fail(h, SHD_EINVAL, "grad_hi and grad_lo must both be given or both NULL");
    const size_t n = (size_t)h->d * h->N, b = n * sizeof(double);
    if (!h->d_hpos) {                       // one allocation: positions (hi, lo) and gradient (hi, lo)
        CU(cudaMalloc((void**)&h->d_hpos, 4 * b));
        h->workspace_bytes += 4 * b;
    }
    double* d_hgrad = h->d_hpos + 2 * n;
    CU(cudaMemcpyAsync(h->d_hpos, pos_hi, b, cudaMemcpyHostToDevice, h->stream));
    CU(cudaMemcpyAsync(h->d_hpos + n, pos_lo, b, cudaMemcpyHostToDevice, h->stream));
    const bool want_grad = grad_hi != nullptr;
    int rc = shd_energy_grad(h, h->d_hpos, h->d_hpos + n, phi, want_grad ? d_hgrad : nullptr,
                             want_grad ? d_hgrad + n : nullptr);
    if (rc) return rc;
    if (want_grad) {
        CU(cudaMemcpyAsync(grad_hi, d_hgrad, b, cudaMemcpyDeviceToHost, h->stream));
        CU(cudaMemcpyAsync(grad_lo, d_hgrad + n, b, cudaMemcpyDeviceToHost, h->stream));
        CU(cudaStreamSynchronize(h->stream));
    }
    return SHD_OK;
}

int shd_set_timing(shd_ctx* h, int on) {
    if (!h) return SHD_EINVAL;
    if (on && !h->ev[0])
        for (int i = 0; i <= SHD_NKERN; i++) CU(cudaEventCreate(&h->ev[i]));
    h->timing = on != 0;
    return SHD_OK;
}

int shd_smax(shd_ctx* h, const double* pos_hi, const double* pos_lo, double smax[2], long* argmax_k) {
    if (!h) return SHD_EINVAL;
    if (!pos_hi || !pos_lo || !smax) return fail(h, SHD_EINVAL, "NULL pointer");
    int rc = run_eval(h, pos_hi, pos_lo, nullptr, nullptr);
    if (rc) return rc;
    smax[0] = h->h_scal->smax[0];
    smax[1] = h->h_scal->smax[1];
    if (argmax_k) *argmax_k = (long)h->h_scal->argmax;
    if (h->h_scal->nonfinite) return fail(h, SHD_ENAN, "non-finite S_max");
    return SHD_OK;
}

int shd_last_smax(shd_ctx* h, double smax[2], long* argmax_k) {
    if (!h || !smax) return SHD_EINVAL;
    int rc = fetch_scalars(h);
    if (rc) return rc;
    smax[0] = h->h_scal->smax[0];
    smax[1] = h->h_scal->smax[1];
    if (argmax_k) *argmax_k = (long)h->h_scal->argmax;
    return SHD_OK;
}

int shd_get_rho(shd_ctx* h, double* re_hi, double* re_lo, double* im_hi, double* im_lo) {
    if (!h) return SHD_EINVAL;
    if (!re_hi || !re_lo || !im_hi || !im_lo) return fail(h, SHD_EINVAL, "NULL pointer");
    size_t b = (size_t)h->M * sizeof(double);
    CU(cudaMemcpyAsync(re_hi, h->d_rho, b, cudaMemcpyDeviceToDevice, h->stream));
    CU(cudaMemcpyAsync(re_lo, h->d_rho + h->M, b, cudaMemcpyDeviceToDevice, h->stream));
    CU(cudaMemcpyAsync(im_hi, h->d_rho + 2 * h->M, b, cudaMemcpyDeviceToDevice, h->stream));
    CU(cudaMemcpyAsync(im_lo, h->d_rho + 3 * h->M, b, cudaMemcpyDeviceToDevice, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    return SHD_OK;
}

int shd_set_precision(shd_ctx* h, int limbs) {
    if (!h) return SHD_EINVAL;
    if (limbs < 1 || limbs > 3) return fail(h, SHD_EINVAL, "shd_set_precision: limbs must be 1, 2 or 3");
    h->nlimb = limbs;
    return SHD_OK;
}

int shd_set_engine(shd_ctx* h, int rho_engine) {
    if (!h) return SHD_EINVAL;
    if (rho_engine == -1) {                      // back to the library's own choice
        const int before = h->rho_engine;
        auto_engine(h);
        if (h->rho_engine != before) h->tables_valid = false;
        return SHD_OK;
    }
    if (rho_engine < 0 || rho_engine > 2) return fail(h, SHD_EINVAL, "shd_set_engine: engine must be -1 (auto), 0, 1 or 2");
    // exactness of the s32 digit sums of the gradient pass: 13 pairs x 2 Qpad products x 2^14 must stay below 2^31
    if (rho_engine == 2 && (long)h->Qpad * 2 * SHD_I8_DIGITS * 16384 >= (1L << 31))
        return fail(h, SHD_EINVAL, "shd_set_engine: last-axis table too long for the INT8 gradient pass (Qn <= 5024)");
    if (rho_engine >= 1) {
        int rc = plan_engine8(h, rho_engine);    // the handle's engine is unchanged when this fails
        if (rc) return rc;
    }
    if (rho_engine != h->rho_engine) h->tables_valid = false;
    h->rho_engine = rho_engine;
    h->engine_auto = 0;
    return SHD_OK;
}

int shd_set_workspace(shd_ctx* h, size_t bytes) {
    if (!h) return SHD_EINVAL;
    h->ws_cap = bytes;
    h->tables_valid = false;
    return SHD_OK;
}

int shd_set_shard(shd_ctx* h, long N_total, int rank, int world) {
    if (!h) return SHD_EINVAL;
    if (world < 1 || rank < 0 || rank >= world || N_total < h->N) return fail(h, SHD_EINVAL, "shd_set_shard: bad rank / world / N_total");
    h->Nsys = N_total;
    h->rank = rank;
    h->world = world;
    h->tables_valid = false;
    return SHD_OK;
}

unsigned long shd_partial_bytes(const shd_ctx* h) {
    if (!h) return 0;
    return (unsigned long)(h->rho_engine >= 1 ? h->ntiles8 : h->ntiles) * 4 * 1024 * 16;
}

int shd_rho_partial(shd_ctx* h, const double* pos_hi, const double* pos_lo, void* partial_out) {
    if (!h) return SHD_EINVAL;
    if (!pos_hi || !pos_lo || !partial_out) return fail(h, SHD_EINVAL, "NULL pointer");
    if (!shd_sharded(h)) return fail(h, SHD_EINVAL, "shd_rho_partial: the handle is not a shard (shd_set_shard)");
    int rc = shd_prepare_tables(h, false);
    if (rc) return rc;
    h->last_launches = 0;
    CU(shd_enqueue_rho_partial(h, pos_hi, pos_lo, false));
    CU(cudaMemcpyAsync(partial_out, h->d_xrun, shd_partial_bytes(h), cudaMemcpyDeviceToDevice, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    return SHD_OK;
}

int shd_rho_finish(shd_ctx* h, const void* gathered, int nparts, double phi[2]) {
    if (!h) return SHD_EINVAL;
    if (!gathered || nparts < 1 || !phi) return fail(h, SHD_EINVAL, "shd_rho_finish: bad argument");
    if (!h->tables_valid) return fail(h, SHD_EINVAL, "shd_rho_finish: call shd_rho_partial first");
    CU(shd_enqueue_rho_finish(h, (const double*)gathered, nparts));
    int rc = fetch_scalars(h);
    if (rc) return rc;
    phi[0] = h->h_scal->phi[0];
    phi[1] = h->h_scal->phi[1];
    if (h->h_scal->nonfinite) return fail(h, SHD_ENAN, "non-finite Phi (non-finite positions?)");
    return SHD_OK;
}

int shd_grad_local(shd_ctx* h, const double* pos_hi, const double* pos_lo, double* grad_hi, double* grad_lo) {
    if (!h) return SHD_EINVAL;
    if (!pos_hi || !pos_lo || !grad_hi || !grad_lo) return fail(h, SHD_EINVAL, "NULL pointer");
    int rc = shd_prepare_tables(h, true);
    if (rc) return rc;
    CU(shd_enqueue_grad(h, pos_hi, pos_lo, grad_hi, grad_lo));
    CU(cudaStreamSynchronize(h->stream));
    return SHD_OK;
}

int shd_structure_factor(shd_ctx* h, double* S_out, double dev2[2]) {
    if (!h) return SHD_EINVAL;
    if (!dev2) return fail(h, SHD_EINVAL, "NULL pointer");
    const size_t nb = (size_t)((h->M + 255) / 256);
    double* scratch = nullptr;
    CU(cudaMalloc((void**)&scratch, (2 * nb + 2) * sizeof(double)));
    cudaError_t e = shd_launch_sfactor(h, S_out, scratch, scratch + 2 * nb);
    if (e == cudaSuccess) e = cudaMemcpyAsync(dev2, scratch + 2 * nb, 2 * sizeof(double), cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    cudaFree(scratch);
    CU(e);
    return SHD_OK;
}

// distinct values of n.n in Q, ascending (the finest radial bins: one per shell)
static std::vector<long> shells_of(const shd_ctx* h) {
    std::vector<long> nn((size_t)h->M);
    for (long k = 0; k < h->M; k++) {
        long v = 0;
        for (int a = 0; a < h->d; a++) v += (long)h->nvec[k * h->d + a] * h->nvec[k * h->d + a];
        nn[(size_t)k] = v;
    }
    std::sort(nn.begin(), nn.end());
    nn.erase(std::unique(nn.begin(), nn.end()), nn.end());
    return nn;
}

long shd_num_shells(const shd_ctx* h) { return h ? (long)shells_of(h).size() : 0; }

int shd_get_shells(const shd_ctx* h, long* nn_out) {
    if (!h || !nn_out) return SHD_EINVAL;
    const std::vector<long> nn = shells_of(h);
    std::memcpy(nn_out, nn.data(), nn.size() * sizeof(long));
    return SHD_OK;
}

int shd_structure_factor_shells(shd_ctx* h, long nbins, const long* edges, long* count, double* S_mean_hi, double* S_mean_lo) {
    if (!h) return SHD_EINVAL;
    if (nbins < 1 || !edges || !count || !S_mean_hi || !S_mean_lo) return fail(h, SHD_EINVAL, "shd_structure_factor_shells: bad argument");
    for (long b = 0; b < nbins; b++)
        if (!(edges[b] < edges[b + 1])) return fail(h, SHD_EINVAL, "shd_structure_factor_shells: edges must be strictly ascending");
    // index work on the host (exact integers): the wavevectors of each bin, ascending k inside a bin
    std::vector<long> start((size_t)nbins + 1, 0);
    std::vector<int> bin((size_t)h->M);
    for (long k = 0; k < h->M; k++) {
        long nn = 0;
        for (int a = 0; a < h->d; a++) nn += (long)h->nvec[k * h->d + a] * h->nvec[k * h->d + a];
        const long b = (long)(std::upper_bound(edges, edges + nbins + 1, nn) - edges) - 1;      // edges[b] <= nn < edges[b+1]
        bin[k] = (b >= 0 && b < nbins) ? (int)b : -1;
        if (bin[k] >= 0) start[(size_t)b + 1]++;
    }
    for (long b = 0; b < nbins; b++) { count[b] = start[(size_t)b + 1]; start[(size_t)b + 1] += start[(size_t)b]; }
    std::vector<int> order((size_t)std::max<long>(start[(size_t)nbins], 1));
    std::vector<long> fill(start.begin(), start.end() - 1);
    for (long k = 0; k < h->M; k++)
        if (bin[k] >= 0) order[(size_t)fill[(size_t)bin[k]]++] = (int)k;
    long* d_start = nullptr;
    int* d_order = nullptr;
    double* d_mean = nullptr;
    cudaError_t e = cudaMalloc((void**)&d_start, start.size() * sizeof(long));
    if (e == cudaSuccess) e = cudaMalloc((void**)&d_order, order.size() * sizeof(int));
    if (e == cudaSuccess) e = cudaMalloc((void**)&d_mean, (size_t)2 * nbins * sizeof(double));
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_start, start.data(), start.size() * sizeof(long), cudaMemcpyHostToDevice, h->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_order, order.data(), order.size() * sizeof(int), cudaMemcpyHostToDevice, h->stream);
    if (e == cudaSuccess) e = shd_launch_sfactor_shells(h, nbins, d_start, d_order, d_mean, d_mean + nbins);
    if (e == cudaSuccess) e = cudaMemcpyAsync(S_mean_hi, d_mean, (size_t)nbins * sizeof(double), cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(S_mean_lo, d_mean + nbins, (size_t)nbins * sizeof(double), cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    cudaFree(d_start); cudaFree(d_order); cudaFree(d_mean);
    CU(e);
    return SHD_OK;
}

int shd_tau(shd_ctx* h, double K, double tau[2]) {
    if (!h) return SHD_EINVAL;
    if (!tau || !(K > 0.0) || !std::isfinite(K)) return fail(h, SHD_EINVAL, "shd_tau: bad argument");
    double dev2[2];
    int rc = shd_structure_factor(h, nullptr, dev2);
    if (rc) return rc;
    // tau = K^d V / N^2 * 2 * dev2 (Eq. 7 P:81 as a lattice sum, D = 1/K): prefactor in long double, product error-free
    long double pref = 2.0L;
    for (int a = 0; a < h->d; a++) pref *= (long double)K * (long double)h->L;
    pref /= (long double)h->Nsys * (long double)h->Nsys;
    const double ph = (double)pref, pl = (double)(pref - (long double)ph);
    const double p = dev2[0] * ph, e = std::fma(dev2[0], ph, -p) + (dev2[0] * pl + dev2[1] * ph);
    tau[0] = p + e;
    tau[1] = e - (tau[0] - p);
    return SHD_OK;
}

const char* shd_last_error(const shd_ctx* h) { return h ? h->err.c_str() : "NULL handle"; }

double shd_stat(const shd_ctx* h, int what) {
    if (!h) return 0.0;
    const double cells_rho = (double)h->ntiles * 1024.0;
    switch (what) {
        case 0: return cells_rho * (double)h->nsplit * h->chunks_per_split * SHD_NPS * 24.0;   // DFMAs launched by the rho pass (padded, 3 limbs)
        case 12: return (double)((h->N + SHD_JT - 1) / SHD_JT) * SHD_JT * (double)h->grad_qsteps * SHD_PG * 48.0;   // ... by the gradient pass
        case 1: return (double)h->last_launches;
        case 2: return cells_rho;
        case 3: return (double)h->valid_cells;
        case 4: return (double)h->workspace_bytes;
        case 5: return (double)h->nsplit;
        case 6: return (double)h->ntiles;
        case 7: return (double)h->P;
        case 8: return (double)h->Qn;
        case 9: return (double)h->Npad;
        case 10: return (double)h->njb;
        case 11: return (double)h->grad_qsteps;
        case 13: return (double)h->nseg;
        case 14: return (double)h->ntiles8;
        case 15: return (double)h->nsplit8;
        case 16: return (double)h->rho_engine;
        case 17: return (double)h->nseg8;
        case 18: return (double)h->nsteps8;
        case 19: return (double)h->nchunk;
        case 25: return (double)h->Nc;
        case 26: return (double)h->table_bytes;
        case 27: return (double)h->engine_auto;
        // SM clock in MHz inside the tensor kernels of the last evaluation whose scalars were fetched (shd_internal.h)
        case 28: return h->h_scal && h->h_scal->clk[1] > 0 ? 1e3 * (double)h->h_scal->clk[0] / (double)h->h_scal->clk[1] : 0.0;
        case 29: return h->h_scal && h->h_scal->clk[3] > 0 ? 1e3 * (double)h->h_scal->clk[2] / (double)h->h_scal->clk[3] : 0.0;
        case 20: case 21: case 22: case 23: case 24: return (double)h->kern_ms[what - 20];
        default: return 0.0;
    }
}

}  // extern "C"
