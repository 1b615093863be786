// Matrix-free Newton direction in ONE kernel (SURVEY 8(a) rows a2, a3 at d > 128).
//
//   H Delta = -g,   H q = (tau/sigma) q + sigma sum_i P_i q,   P_i of reading 1.
//
// A launch per conjugate-gradient iteration (HVP over the active list, its two-level reduction, the CG update: four
// dependent kernels for a few hundred active rows) made this the largest part of the config-3 solve.  Here
//  1. gather: the active rows are normalised ONCE per Newton step into a compact |A| x d matrix W (w_i = b_i / ||b_i||,
//     b_i = c_i - c + v_i / sigma; rows of branch B1 are stored as zeros: their P_i = I goes through the count n1);
//  2. solve: a persistent grid of up to one CTA per SM runs the WHOLE CG loop.  Per iteration and CTA: y_k = <w_k, p_1>
//     and the partial z = sum_k (p_0 - rho_k y_k) w_k over its block of rows (W is L2-resident), then three grid-wide
//     barriers separate the fixed-order reductions (z over the CTAs per column slice, <p, Hp>, ||res||^2).  Every CTA
//     keeps its own copy of p in shared memory and forms the next p = res + beta p redundantly, so no fourth barrier.
// Only as many CTAs as there is work for take part (64 KB of W each); a 5-ball reduced problem runs on one CTA with
// no grid barrier at all.
//
// Grid barrier: monotone arrival counter in global memory (zeroed by the launcher), one atomicAdd per CTA and barrier.
// The grid never exceeds the SM count and a CTA needs less than the shared memory of one SM, so all CTAs are
// co-resident (nothing else runs on the stream); a watchdog turns a barrier that does not complete within ~1 s
// into an error flag instead of a hang.
//
// Determinism: static row -> CTA -> warp assignment; partials of CTAs, warps and lanes are added in index order.
#include <string.h>

#include "meb_internal.cuh"
#include "meb_ctrl.cuh"

namespace {

constexpr int CG_THREADS = 256;
constexpr int CG_WARPS = CG_THREADS / 32;

struct CgArgs {
    const void* C; int64_t ld; int prec;
    const int32_t* v_slot; const void* V; int64_t ldv;      // resolved through dyn (graph side)
    const MebDyn* dyn;
    const int32_t* slot2[2]; const void* V2[2];
    const double* x;                       // (r, c) of the accepted point, raw units
    const int32_t* list; const int32_t* count;
    const double* rec_rho;
    int32_t d, dpad;
    double* W; int64_t wc_cap;             // [wc_cap][dpad] normalised rows
    double* rho_c;                         // [wc_cap] rho_k (0 for a B1 row)
    double* zpart;                         // [grid][dpad] per-CTA partial of z
    double* spart;                         // [3][grid] per-CTA partials: sum y, <p, Hp>, ||res||^2
    unsigned int* bar;                     // [2]: arrival counter, error flag
    int32_t rper_cap;                      // rows a CTA can be given (size of its coefficient array)
    int32_t full_vec;                      // 1: every CTA keeps res and delta whole in shared memory and updates them
                                           // redundantly (same order, same bits): no third barrier per iteration
    int32_t wcache_cap;                    // doubles of shared memory behind the coefficients: the CTA's block of W is
                                           // copied there once per solve when it fits (every CG iteration reads it twice)
    SolverDev* S; SolverVecs v;
};

// TEAM = 32: a warp per active row (rows of a few KB); TEAM = CG_THREADS: the whole CTA per row (long rows: one
// warp would walk 1e4 columns in 300 dependent-latency steps).  Two passes over the row (the second one hits L1/L2):
// first ||b||^2 with nothing but loads in the loop, then the normalised row is written.
template <typename T, int TEAM>
__global__ void __launch_bounds__(CG_THREADS) cg_gather_kernel(const CgArgs a) {
    __shared__ double red[CG_WARPS];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int tt = TEAM == 32 ? lane : (int)threadIdx.x;
    const int n = *a.count < a.wc_cap ? *a.count : (int)a.wc_cap;
    const int cur = a.dyn->cur;
    const bool hm = a.dyn->has_mult != 0;
    const int32_t* slotp = hm ? a.slot2[cur] : nullptr;
    const T* __restrict__ V = static_cast<const T*>(hm ? a.V2[cur] : nullptr);
    const T* __restrict__ C = static_cast<const T*>(a.C);
    const T inv_sig = T(1) / (T)a.dyn->sigma_raw;
    const double* __restrict__ cx = a.x + 1;
    const int d = a.d;
    constexpr int TPB = CG_THREADS / TEAM;
    const int nteams = gridDim.x * TPB;
    for (int k = blockIdx.x * TPB + (TEAM == 32 ? warp : 0); k < n; k += nteams) {
        const int i = a.list[k];
        const double rho = a.rec_rho[i];
        double* __restrict__ wrow = a.W + (size_t)k * a.dpad;
        if (rho > 1.5) {                                   // B1: P_i = I (counted in n1), no rank-one part
            for (int j = tt; j < a.dpad; j += TEAM) wrow[j] = 0.0;
            if (tt == 0) a.rho_c[k] = 0.0;
            continue;
        }
        const T* __restrict__ rowp = C + (int64_t)i * a.ld;
        const int slot = slotp ? slotp[i] : -1;
        const T* __restrict__ vrow = slot >= 0 ? V + (int64_t)slot * a.ldv : nullptr;
        double nb2 = 0.0, nb2b = 0.0;
        if (vrow) {
#pragma unroll 4
            for (int j = tt; j < d; j += TEAM) {
                const double bd = (double)fma(vrow[j], inv_sig, rowp[j] - (T)cx[j]);
                nb2 = fma(bd, bd, nb2);
            }
        } else {
            int j = tt;
#pragma unroll 1
            for (; j + 7 * TEAM < d; j += 8 * TEAM) {
                double bd[8];
#pragma unroll
                for (int u = 0; u < 8; ++u) bd[u] = (double)(rowp[j + u * TEAM] - (T)cx[j + u * TEAM]);
#pragma unroll
                for (int u = 0; u < 8; u += 2) { nb2 = fma(bd[u], bd[u], nb2); nb2b = fma(bd[u + 1], bd[u + 1], nb2b); }
            }
            for (; j < d; j += TEAM) { const double bd = (double)(rowp[j] - (T)cx[j]); nb2 = fma(bd, bd, nb2); }
            nb2 += nb2b;
        }
        nb2 = warp_sum(nb2);
        if (TEAM != 32) {                                  // warps of the CTA in index order
            __syncthreads();
            if (lane == 0) red[warp] = nb2;
            __syncthreads();
            nb2 = 0.0;
#pragma unroll
            for (int w = 0; w < CG_WARPS; ++w) nb2 += red[w];
        }
        const double inv = 1.0 / sqrt(nb2);                // B3: nb > |a| >= 0
#pragma unroll 4
        for (int j = tt; j < a.dpad; j += TEAM) {
            double wv = 0.0;
            if (j < d) {
                T bq = rowp[j] - (T)cx[j];
                if (vrow) bq = fma(vrow[j], inv_sig, bq);
                wv = (double)bq * inv;
            }
            wrow[j] = wv;
        }
        if (tt == 0) a.rho_c[k] = rho;
    }
}

// all threads of the CTA call it; returns false if the watchdog fired (the caller leaves the loop)
__device__ __forceinline__ bool grid_barrier(unsigned int* bar, unsigned int target) {
    __shared__ int ok_s;
    __syncthreads();                                         // the CTA's writes happen before thread 0's release
    if (threadIdx.x == 0) {
        // arrive: release (cumulative over the CTA's writes through the barrier above); wait: acquire loads, which
        // also drop this SM's stale L1 lines before the others read what the other CTAs wrote
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(bar) : "memory");
        int ok = 1;
        long long spins = 0;
        for (;;) {
            unsigned int v;
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(bar) : "memory");
            if (v >= target) break;
            if (*reinterpret_cast<volatile unsigned int*>(&bar[1]) != 0u) { ok = 0; break; }
            if (++spins > 2000000000LL) { atomicExch(&bar[1], 1u); ok = 0; break; }
        }
        ok_s = ok;
    }
    __syncthreads();
    return ok_s != 0;
}

__device__ __forceinline__ double cta_sum(double v, double* red) {
    v = warp_sum(v);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
#pragma unroll
    for (int w = 0; w < CG_WARPS; ++w) t += red[w];
    return t;
}

__global__ void __launch_bounds__(CG_THREADS, 1) cg_solve_kernel(const CgArgs a) {
    extern __shared__ __align__(16) double cg_sm[];          // p_s[dpad + 8], coef_s[rper_cap]
    __shared__ double red[CG_WARPS];
    __shared__ double ysum_w[CG_WARPS];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    SolverDev* S = a.S;
    const int d = a.d, n1d = d + 1, dpad = a.dpad;
    const int n = *a.count < a.wc_cap ? *a.count : (int)a.wc_cap;
    // CTAs that take part: 64 KB of W each
    long long want = ((long long)n * dpad * 8 + 65535) / 65536;
    const int G = (int)(want < 1 ? 1 : (want > (long long)gridDim.x ? (long long)gridDim.x : want));
    const int b = blockIdx.x;
    if (b >= G) return;
    double* p_s = cg_sm;                    // p_s[0] = p_0, p_s[1 + j] = p_1[j]
    const bool full = a.full_vec != 0;
    double* res_s = cg_sm + (dpad + 8);     // [dpad + 8] (full only)
    double* del_s = res_s + (dpad + 8);     // [dpad + 8] (full only)
    double* coef_s = cg_sm + (full ? 3 : 1) * (dpad + 8);    // [rper_cap] coefficients of my rows
    const double sigma = a.dyn->sigma_raw, tau = a.dyn->tau_eff;
    const double tos = tau / sigma;
    const double Ls = S->L;
    const double nB1 = a.v.ev[MEB_EV_N_B1], nB3 = a.v.ev[MEB_EV_N_B3], srho = a.v.ev[MEB_EV_SUM_RHO];
    const double diag0 = tos + sigma * (nB1 + 0.5 * nB3);
    const double diag1 = tos + sigma * (nB1 + 0.5 * (nB3 + srho));
    // my block of rows and my slice of the (d+1) vector entries
    const int rper = (n + G - 1) / G;
    if (rper > a.rper_cap) {                // cannot happen for n <= wc_cap (the launcher sized rper_cap for it)
        if (b == 0 && tid == 0) { S->chol_info = -2; S->cg_go = 0; }
        return;
    }
    const int r0 = b * rper, r1 = (r0 + rper < n) ? r0 + rper : n;
    // my block of W: in shared memory when it fits, else where the gather left it (L2)
    const double* Wl = a.W + (size_t)r0 * dpad;
    if (r1 > r0 && (long long)(r1 - r0) * dpad <= (long long)a.wcache_cap) {
        double* wc = coef_s + ((a.rper_cap + 1) & ~1);
        const double2* src = reinterpret_cast<const double2*>(Wl);      // rows start at multiples of 64 bytes
        double2* dst = reinterpret_cast<double2*>(wc);
        const int n2 = (r1 - r0) * (dpad / 2);
#pragma unroll 4
        for (int q = tid; q < n2; q += CG_THREADS) dst[q] = src[q];
        Wl = wc;
    }
    const int cper = ((n1d + G - 1) / G + 3) & ~3;
    const int c0 = b * cper, c1 = (c0 + cper < n1d) ? c0 + cper : n1d;
    double* zp = a.zpart + (size_t)b * dpad;
    double* sp_y = a.spart, *sp_pHp = a.spart + gridDim.x, *sp_rr = a.spart + 2 * gridDim.x;
    // start: delta = 0, res = p = -g (written by the controller), rr = ||g||^2, tolerance: S->cg_tol
    for (int j = tid; j < n1d; j += CG_THREADS) p_s[j] = a.v.p[j];
    if (full)
        for (int j = tid; j < n1d; j += CG_THREADS) { res_s[j] = a.v.res[j]; del_s[j] = 0.0; }
    double rr = S->cg_rr;
    const double tol = S->cg_tol;
    const int itmax = S->cg_max;
    unsigned int bars = 0;
    int it = 0;
    bool ok = true;
    __syncthreads();
    while (it < itmax && sqrt(rr) > tol) {
        // ---- phase A over my rows (warp per row): y_k = <w_k, p_1>, coef_k = p_0 - rho_k y_k ----
        // (a B1 row is stored as zeros: y = 0 and coef w = 0 whatever coef is)
        const double q0 = p_s[0];
        double ys = 0.0;
        if (d >= 2048) {
            // long rows (a CTA holds one or two of them): all threads on one row, four loads in flight per thread
            for (int k = r0; k < r1; ++k) {
                const double* __restrict__ wrow = Wl + (size_t)(k - r0) * dpad;
                double y0 = 0.0, y1 = 0.0, y2 = 0.0, y3 = 0.0;
                int j = tid;
                for (; j + 3 * CG_THREADS < d; j += 4 * CG_THREADS) {
                    const double w0 = wrow[j], w1 = wrow[j + CG_THREADS], w2 = wrow[j + 2 * CG_THREADS], w3 = wrow[j + 3 * CG_THREADS];
                    y0 = fma(w0, p_s[1 + j], y0); y1 = fma(w1, p_s[1 + j + CG_THREADS], y1);
                    y2 = fma(w2, p_s[1 + j + 2 * CG_THREADS], y2); y3 = fma(w3, p_s[1 + j + 3 * CG_THREADS], y3);
                }
                for (; j < d; j += CG_THREADS) y0 = fma(wrow[j], p_s[1 + j], y0);
                const double y = cta_sum((y0 + y1) + (y2 + y3), red);
                if (tid == 0) coef_s[k - r0] = q0 - a.rho_c[k] * y;
                if (warp == 0) ys += y;                      // counted once (warp 0's slot below)
            }
        } else {
            for (int k = r0 + warp; k < r1; k += CG_WARPS) {
                const double* __restrict__ wrow = Wl + (size_t)(k - r0) * dpad;
                double y0 = 0.0, y1 = 0.0;
                int j = lane;
                for (; j + 96 < d; j += 128) {
                    const double w0 = wrow[j], w1 = wrow[j + 32], w2 = wrow[j + 64], w3 = wrow[j + 96];
                    y0 = fma(w0, p_s[1 + j], y0); y1 = fma(w1, p_s[1 + j + 32], y1);
                    y0 = fma(w2, p_s[1 + j + 64], y0); y1 = fma(w3, p_s[1 + j + 96], y1);
                }
                for (; j < d; j += 32) y0 = fma(wrow[j], p_s[1 + j], y0);
                const double y = warp_sum(y0 + y1);
                if (lane == 0) coef_s[k - r0] = q0 - a.rho_c[k] * y;
                ys += y;
            }
        }
        if (lane == 0) ysum_w[warp] = ys;
        __syncthreads();
        // ---- phase B (thread per column): z_j = sum_k coef_k W[k][j], rows in index order ----
        {
            const double* __restrict__ Wr = Wl;
            double* __restrict__ zpr = zp;
            int j = tid;
            for (; j + 3 * CG_THREADS < d; j += 4 * CG_THREADS) {     // four columns per thread and sweep: loads first
                double z0 = 0.0, z1 = 0.0, z2 = 0.0, z3 = 0.0;
                for (int k = r0; k < r1; ++k) {
                    const double ck = coef_s[k - r0];
                    const double* wk = Wr + (size_t)(k - r0) * dpad + j;
                    const double w0 = wk[0], w1 = wk[CG_THREADS], w2 = wk[2 * CG_THREADS], w3 = wk[3 * CG_THREADS];
                    z0 = fma(ck, w0, z0); z1 = fma(ck, w1, z1); z2 = fma(ck, w2, z2); z3 = fma(ck, w3, z3);
                }
                zpr[j] = z0; zpr[j + CG_THREADS] = z1; zpr[j + 2 * CG_THREADS] = z2; zpr[j + 3 * CG_THREADS] = z3;
            }
            for (; j < d; j += CG_THREADS) {
                double z = 0.0;
                for (int k = r0; k < r1; ++k) z = fma(coef_s[k - r0], Wr[(size_t)(k - r0) * dpad + j], z);
                zpr[j] = z;
            }
        }
        if (tid == 0) { double t = 0.0; for (int w = 0; w < CG_WARPS; ++w) t += ysum_w[w]; sp_y[b] = t; }
        if (G > 1) { bars += G; ok = grid_barrier(a.bar, bars); if (!ok) break; } else __syncthreads();
        // ---- my slice of Hp (raw units), <p, Hp> partial ----
        double pHp = 0.0;
#pragma unroll 2
        for (int e = c0 + tid; e < c1; e += CG_THREADS) {
            double hp;
            if (e == 0) {
                double sy = 0.0;
                for (int bb = 0; bb < G; ++bb) sy += sp_y[bb];
                hp = diag0 * q0 + 0.5 * sigma * sy;
            } else {
                double s = 0.0;
                for (int bb = 0; bb < G; ++bb) s += a.zpart[(size_t)bb * dpad + (e - 1)];
                hp = diag1 * p_s[e] + 0.5 * sigma * s;
            }
            hp *= Ls;                                        // H~ = L H_raw (normalised units)
            a.v.Hp[e] = hp;
            pHp = fma(p_s[e], hp, pHp);
        }
        pHp = cta_sum(pHp, red);
        if (tid == 0) sp_pHp[b] = pHp;
        if (G > 1) { bars += G; ok = grid_barrier(a.bar, bars); if (!ok) break; } else __syncthreads();
        double tot = 0.0;
        for (int bb = 0; bb < G; ++bb) tot += sp_pHp[bb];
        const double alpha = rr / tot;
        double rrn = 0.0;
        if (full) {
            // every CTA updates the WHOLE residual and direction sum from the Hp slices the others published before
            // the barrier above: ||res||^2 and the next p follow without another exchange
            const double* hpv = a.v.Hp;
#pragma unroll 4
            for (int e = tid; e < n1d; e += CG_THREADS) {
                del_s[e] = fma(alpha, p_s[e], del_s[e]);
                const double rj = fma(-alpha, hpv[e], res_s[e]);
                res_s[e] = rj;
                rrn = fma(rj, rj, rrn);
            }
            const double rr_new = cta_sum(rrn, red);
            const double beta = rr_new / rr;
#pragma unroll 4
            for (int e = tid; e < n1d; e += CG_THREADS) p_s[e] = fma(beta, p_s[e], res_s[e]);
            rr = rr_new;
            ++it;
            __syncthreads();
            continue;
        }
        {
            double* __restrict__ dl = a.v.delta; double* __restrict__ rs = a.v.res; const double* __restrict__ hpv = a.v.Hp;
#pragma unroll 4
            for (int e = c0 + tid; e < c1; e += CG_THREADS) {
                dl[e] = fma(alpha, p_s[e], dl[e]);
                const double rj = fma(-alpha, hpv[e], rs[e]);
                rs[e] = rj;
                rrn = fma(rj, rj, rrn);
            }
        }
        rrn = cta_sum(rrn, red);
        if (tid == 0) sp_rr[b] = rrn;
        if (G > 1) { bars += G; ok = grid_barrier(a.bar, bars); if (!ok) break; } else __syncthreads();
        double rr_new = 0.0;
        for (int bb = 0; bb < G; ++bb) rr_new += sp_rr[bb];
        const double beta = rr_new / rr;
        {
            const double* __restrict__ rs = a.v.res;
            int j = tid;
            for (; j + 3 * CG_THREADS < n1d; j += 4 * CG_THREADS) {
                const double r0v = rs[j], r1v = rs[j + CG_THREADS], r2v = rs[j + 2 * CG_THREADS], r3v = rs[j + 3 * CG_THREADS];
                p_s[j] = fma(beta, p_s[j], r0v); p_s[j + CG_THREADS] = fma(beta, p_s[j + CG_THREADS], r1v);
                p_s[j + 2 * CG_THREADS] = fma(beta, p_s[j + 2 * CG_THREADS], r2v);
                p_s[j + 3 * CG_THREADS] = fma(beta, p_s[j + 3 * CG_THREADS], r3v);
            }
            for (; j < n1d; j += CG_THREADS) p_s[j] = fma(beta, p_s[j], rs[j]);
        }
        rr = rr_new;
        ++it;
        __syncthreads();
    }
    if (full && b == 0)
        for (int e = tid; e < n1d; e += CG_THREADS) { a.v.delta[e] = del_s[e]; a.v.res[e] = res_s[e]; }
    if (b == 0 && tid == 0) {
        S->cg_rr = rr;
        S->cg_it = it;
        S->cg_total += it;
        S->cg_go = 0;
        if (!ok) S->chol_info = -1;
    }
}

}  // namespace


// The Newton direction of the matrix-free path for at most wc_cap active rows: gather + persistent CG.
// v.delta / v.res / v.p were initialised by the controller (delta = 0, res = p = -g).
int meb_launch_cg(meb_ctx* ctx, const EvalCall& c, double* W, int64_t wc_cap, double* rho_c, unsigned int* bar) {
    const GraphSide* gs = c.gs;
    if (!gs || !gs->S || !gs->v) return MEB_E_ARG;
    CgArgs a;
    memset(&a, 0, sizeof(a));
    a.C = c.C; a.ld = c.ld; a.prec = c.prec; a.ldv = c.ldv; a.dyn = gs->dyn;
    for (int b = 0; b < 2; ++b) { a.slot2[b] = gs->slot2[b]; a.V2[b] = gs->V2[b]; }
    a.x = c.x; a.list = ctx->list; a.count = ctx->count_dev; a.rec_rho = ctx->rec_rho;
    a.d = c.d; a.dpad = (c.d + 7) / 8 * 8;
    a.W = W; a.wc_cap = wc_cap; a.rho_c = rho_c;
    a.zpart = ctx->part_vec; a.spart = ctx->part_sc; a.bar = bar;
    a.S = gs->S; a.v = *gs->v;
    int grid = ctx->sm_count > 0 ? ctx->sm_count : 148;
    if ((int64_t)grid > ctx->vec_rows) grid = (int)ctx->vec_rows;
    if (3 * grid > 1024) grid = 341;
    // no more CTAs than the rows can use
    const int64_t by_rows = (wc_cap * a.dpad * 8 + 65535) / 65536;
    if (by_rows < grid) grid = (int)(by_rows < 1 ? 1 : by_rows);
    const int ggrid = (int)((wc_cap + CG_WARPS - 1) / CG_WARPS < 4 * grid ? ((wc_cap + CG_WARPS - 1) / CG_WARPS) : 4 * grid);
    MEB_CUDA_OK(ctx, cudaMemsetAsync(bar, 0, 2 * sizeof(unsigned int), ctx->stream));
    ctx->launches++;
    if (c.d >= 2048) {                                       // CTA per row
        const int gg = (int)(wc_cap < 4 * grid ? wc_cap : 4 * grid);
        if (c.prec == MEB_FP64) cg_gather_kernel<double, CG_THREADS><<<gg < 1 ? 1 : gg, CG_THREADS, 0, ctx->stream>>>(a);
        else cg_gather_kernel<float, CG_THREADS><<<gg < 1 ? 1 : gg, CG_THREADS, 0, ctx->stream>>>(a);
    } else if (c.prec == MEB_FP64) cg_gather_kernel<double, 32><<<ggrid < 1 ? 1 : ggrid, CG_THREADS, 0, ctx->stream>>>(a);
    else cg_gather_kernel<float, 32><<<ggrid < 1 ? 1 : ggrid, CG_THREADS, 0, ctx->stream>>>(a);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    // rows per CTA: 64 KB of W while CTAs are left, wc_cap / grid once all of them take part
    a.rper_cap = (int32_t)(65536 / ((size_t)a.dpad * 8) + 2);
    if ((wc_cap + grid - 1) / grid + 1 > a.rper_cap) a.rper_cap = (int32_t)((wc_cap + grid - 1) / grid + 1);
    size_t base = ((size_t)a.dpad + 8 + (size_t)a.rper_cap + 8) * sizeof(double);
    if (base > 200 * 1024) return MEB_E_CAPACITY;
    a.full_vec = (base + 2 * ((size_t)a.dpad + 8) * sizeof(double) + 65536 <= 200 * 1024) ? 1 : 0;
    if (a.full_vec) base += 2 * ((size_t)a.dpad + 8) * sizeof(double);
    size_t wcache = 65536 + (size_t)a.dpad * 8;               // a CTA's block: 64 KB, rounded up to whole rows
    if (base + wcache > 200 * 1024) wcache = 200 * 1024 - base;
    a.wcache_cap = (int32_t)(wcache / sizeof(double));
    const size_t smem = base + wcache;
    MEB_CUDA_OK(ctx, cudaFuncSetAttribute(cg_solve_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    ctx->launches++;
    cg_solve_kernel<<<grid, CG_THREADS, smem, ctx->stream>>>(a);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}
