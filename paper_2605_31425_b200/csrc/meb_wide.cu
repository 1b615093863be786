// One-CLUSTER ripALM for problems with FEW balls and LONG rows (m <= 256, 126 < d, FP64): the reduced problem of the
// mixed-precision method when the screening keeps a handful of balls of a high-dimensional instance
// (config 5: 5 of 200,000 balls at d = 10^4).  Such a problem is a few hundred KB, L2-resident, and as a graph of grid
// kernels every evaluation costs ~10 dependent launches of one-CTA kernels that walk (d+1)-vectors (4.8 ms for the
// 5-ball problem of config 5); one CTA alone cannot pull the rows out of L2 fast enough either (5.3 ms, measured).
// Here ONE thread-block cluster of 8 CTAs x 512 threads runs the whole phase -- Algorithm 1 with
// Algorithm 2 inside -- with no launch in the loop:
//
//   columns      CTA c of the cluster owns a contiguous slice of the d columns of every row (C, V, W, the vectors);
//   evaluation   a team of warps per ball sums its slice of ||b_i||^2 (and <e,v>, ||e||^2, ||v||^2 for a ball with
//                v_i); the per-CTA sums are exchanged through distributed shared memory (each CTA reads the eight
//                records in rank order: same bits everywhere); every CTA then runs the scalar epilogue (branch of
//                P:L115, multiplier, KKT terms) of all balls redundantly, so lam_i, rho_i, the branch and the active
//                set are known cluster-wide without a second exchange;
//   gradient     thread per column of the slice: sum over the active balls, in index order, of lam_i b_ij;
//   controller   CTA 0 alone, the same device functions as the graph path (meb_ctrl.cuh) on the full vectors (global
//                memory); the others wait at a cluster barrier and copy the new state from CTA 0's shared memory;
//   Newton       matrix-free: slice of w_k = b_k / ||b_k|| (||b_k|| is known from the evaluation), then
//                conjugate gradients with y_k = <w_k, p_1> (slice sums exchanged), z = sum_k coef_k w_k (thread per
//                column), <p, Hp> and ||res||^2 exchanged: three cluster barriers per iteration;
//   update       (u, v) <- sigma Pi(z) (eq. (6)), every CTA its slice of the new rows.
//
// Exchange records are double-buffered (a CTA can be at most one barrier ahead of a reader).  Deterministic: static
// assignment of columns, balls and warps; partial sums are added in warp order, then in rank order.
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <cooperative_groups.h>

#include "meb_ctrl.cuh"
#include "meb_internal.cuh"
#include "meb_rowops.cuh"

namespace cg = cooperative_groups;

namespace {

constexpr int WD_THREADS = 512;
constexpr int WD_WARPS = WD_THREADS / 32;
constexpr int WD_M_MAX = 256;
constexpr int WD_NC = 8;                 // CTAs of the cluster (portable maximum)
constexpr int WD_MB = 4;                 // balls (evaluation) / rows (CG) summed together by the column threads
constexpr int WD_REC = 4 * WD_M_MAX + 8; // doubles of an exchange record: four sums per ball, then a few scalars

struct WideArgs {
    const double* C; int64_t ld; const double* R;
    int32_t m, d; int64_t ldv;
    double* U2[2]; int32_t* slot2[2]; double* V2[2];
    SolverDev* S; SolverVecs v;
    double* W; int32_t dpad;         // [m][dpad] normalised active rows of the current Newton step (global, L2)
    long long* prof;                 // nullable: cycles of CTA 0 per section (MEB_TUNING builds, MEB_TRACE)
};

// sum of v over the CTA: lanes by an xor tree, warps in index order
__device__ __forceinline__ double wd_block_sum(double v, double* red) {
    v = warp_sum(v);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
#pragma unroll
    for (int w = 0; w < WD_WARPS; ++w) t += red[w];
    return t;
}

// Every CTA has written the first `count` doubles of its record xrec[buf]; afterwards xsum[t] = sum over the ranks, in
// rank order, of their xrec[buf][t] -- the same bits in every CTA.
__device__ __forceinline__ void wd_exchange(cg::cluster_group& cluster, double* xrec, int buf, int count, double* xsum) {
    cluster.sync();                                          // records complete (release / acquire, cluster scope)
    double* mine = xrec + (size_t)buf * WD_REC;
    for (int t = threadIdx.x; t < count; t += WD_THREADS) {
        double s = 0.0;
#pragma unroll
        for (int r = 0; r < WD_NC; ++r) s += cluster.map_shared_rank(mine, r)[t];
        xsum[t] = s;
    }
    __syncthreads();
}

__global__ void __launch_bounds__(WD_THREADS, 1) wide_solve_kernel(const WideArgs a) {
    cg::cluster_group cluster = cg::this_cluster();
    const int rank = (int)cluster.block_rank();
    extern __shared__ __align__(16) double wd_sm[];
    __shared__ __align__(16) SolverDev sS;
    __shared__ double ev_s[MEB_EVAL_NSCALARS];
    __shared__ double sm[104];
    __shared__ double red[WD_WARPS];
    __shared__ double wred[WD_WARPS][MEB_NPART];
    __shared__ int wcnt[WD_M_MAX / 32];
    __shared__ int nact_s;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int m = a.m, d = a.d, n = d + 1, dpad = a.dpad;
    const int mc = (m + 7) & ~7;
    // my slice of the columns, and of the (d+1)-vectors (entry 0 = r belongs to rank 0, entry 1 + j to column j)
    const int wcol = ((d + WD_NC - 1) / WD_NC + 7) & ~7;
    const int lo = min(d, rank * wcol), hi = min(d, lo + wcol);
    const int elo = rank == 0 ? 0 : 1 + lo, ehi = 1 + hi;
    // ---- shared memory carve-up (doubles) ----
    double* cs = wd_sm;                                      // [wcol + 8] centre slice; p slice during the Newton solve
    double* xrec = cs + wcol + 8;                            // [2][WD_REC]
    double* xsum = xrec + 2 * WD_REC;                        // [WD_REC]
    double* wpart = xsum + WD_REC;                           // [WD_WARPS][4 * WD_MB] per-warp sums of a chunk
    double* lam_r = wpart + WD_WARPS * 4 * WD_MB;            // [mc] records of the last evaluation: lam_i, rho_i, t_i
    double* rho_r = lam_r + mc;
    double* t_r = rho_r + mc;
    double* nb_s = t_r + mc;                                 // ||b_i||
    double* coef_s = nb_s + mc;                              // CG: coefficient of active row k
    double* rho_s = coef_s + mc;                             // rho of active row k (0: branch B1, stored as zeros)
    int* list_s = reinterpret_cast<int*>(rho_s + mc);        // [mc] ascending active balls
    int* slot_s = list_s + mc;                               // [mc]
    int* pos_s = slot_s + mc;                                // [mc] position of ball i in the list (-1: not active)
    unsigned char* act = reinterpret_cast<unsigned char*>(pos_s + mc);   // [mc]

    {   // working copy of the solver state
        const unsigned long long* src = reinterpret_cast<const unsigned long long*>(a.S);
        unsigned long long* dst = reinterpret_cast<unsigned long long*>(&sS);
        for (int q = tid; q < (int)(sizeof(SolverDev) / 8); q += WD_THREADS) dst[q] = src[q];
    }
    __syncthreads();
    StreamArgs sa;                                           // only the fields the row epilogue touches
    sa.rec_lam = lam_r; sa.rec_rho = rho_r; sa.rec_t = t_r;
    sa.t_out = nullptr; sa.lam_out = nullptr;
    int buf = 0;
    long long tmark = clock64();
    auto lap = [&](int k) { if (a.prof && rank == 0 && tid == 0) { const long long t = clock64(); a.prof[k] += t - tmark; tmark = t; } };
    auto publish_state = [&]() {                             // CTA 0 ran the controller: everyone takes its state
        cluster.sync();
        if (rank != 0) {
            const unsigned long long* src = reinterpret_cast<const unsigned long long*>(cluster.map_shared_rank(&sS, 0));
            unsigned long long* dst = reinterpret_cast<unsigned long long*>(&sS);
            for (int q = tid; q < (int)(sizeof(SolverDev) / 8); q += WD_THREADS) dst[q] = src[q];
        }
        __syncthreads();
    };

    for (;;) {
        // =================================== evaluation at v.x_raw ===================================
        const double sigma = sS.dyn.sigma_raw, tau = sS.dyn.tau_eff;
        const bool hm = sS.dyn.has_mult != 0;
        const int cur = sS.dyn.cur;
        const double* U = hm ? a.U2[cur] : nullptr;
        const int32_t* slotp = hm ? a.slot2[cur] : nullptr;
        const double* V = hm ? a.V2[cur] : nullptr;
        for (int j = lo + tid; j < hi; j += WD_THREADS) cs[j - lo] = a.v.x_raw[1 + j];
        const double r = a.v.x_raw[0];
        const double inv_sig = 1.0 / sigma;
        __syncthreads();
        // slice sums of every ball: thread per column, WD_MB balls at a time (all their loads in flight together),
        // lanes by an xor tree, warps in index order
        for (int i = tid; i < m; i += WD_THREADS) slot_s[i] = slotp ? slotp[i] : -1;
        __syncthreads();
        for (int i0 = 0; i0 < m; i0 += WD_MB) {
            double q4[WD_MB][4];
#pragma unroll
            for (int u = 0; u < WD_MB; ++u) { q4[u][0] = 0.0; q4[u][1] = 0.0; q4[u][2] = 0.0; q4[u][3] = 0.0; }
            for (int j = lo + tid; j < hi; j += WD_THREADS) {
                const double cj = cs[j - lo];
                double cv[WD_MB], vq[WD_MB];
#pragma unroll
                for (int u = 0; u < WD_MB; ++u) {
                    const int i = i0 + u;
                    const int slot = i < m ? slot_s[i] : -1;
                    cv[u] = i < m ? a.C[(int64_t)i * a.ld + j] : cj;
                    vq[u] = slot >= 0 ? V[(int64_t)slot * a.ldv + j] : 0.0;
                }
#pragma unroll
                for (int u = 0; u < WD_MB; ++u) {
                    const double e0 = cv[u] - cj;
                    const double b0 = fma(vq[u], inv_sig, e0);           // = e0 for a ball without v_i
                    q4[u][0] = fma(b0, b0, q4[u][0]); q4[u][1] = fma(e0, e0, q4[u][1]);
                    q4[u][2] = fma(e0, vq[u], q4[u][2]); q4[u][3] = fma(vq[u], vq[u], q4[u][3]);
                }
            }
#pragma unroll
            for (int u = 0; u < WD_MB; ++u)
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const double t = warp_sum(q4[u][q]);
                    if (lane == 0) wpart[(size_t)warp * (4 * WD_MB) + 4 * u + q] = t;
                }
            __syncthreads();
            if (tid < 4 * WD_MB && i0 + tid / 4 < m) {
                double t = 0.0;
#pragma unroll
                for (int w = 0; w < WD_WARPS; ++w) t += wpart[(size_t)w * (4 * WD_MB) + tid];
                xrec[(size_t)buf * WD_REC + 4 * i0 + tid] = t;
            }
            __syncthreads();
        }
        lap(0);
        wd_exchange(cluster, xrec, buf, 4 * m, xsum);
        buf ^= 1;
        lap(1);
        // ---- scalar epilogue of every ball, redundantly in every CTA (thread per ball) ----
        Acc acc;
        if (tid < mc) {
            bool flag = false;
            if (tid < m) {
                const int i = tid;
                const int slot = slotp ? slotp[i] : -1;
                const double ui = U ? U[i] : 0.0;
                const double ri = a.R ? a.R[i] : 0.0;
                double mylam;
                flag = row_epilogue_core<double, OP_EVAL>(sa, i, true, slot >= 0, xsum[4 * i], xsum[4 * i + 1], xsum[4 * i + 2],
                                                          xsum[4 * i + 3], r, sigma, ri, ui, acc, mylam);
                if (!flag) lam_r[i] = 0.0;
                slot_s[i] = slot;
                nb_s[i] = sqrt(xsum[4 * i]);
            }
            act[tid] = flag ? 1 : 0;
        }
        {   // lanes of a warp (xor tree), then warps in index order
            const double r0 = warp_sum(acc.s0), r1 = warp_sum(acc.s1), r2 = warp_sum(acc.s2);
            const double r3 = warp_sum((double)acc.n0), r4 = warp_sum((double)acc.n1);
            const double r5 = warp_max(acc.m0), r6 = warp_max(acc.m1), r7 = warp_max(acc.m2), r8 = warp_sum(acc.s3);
            if (lane == 0) {
                wred[warp][0] = r0; wred[warp][1] = r1; wred[warp][2] = r2; wred[warp][3] = r3; wred[warp][4] = r4;
                wred[warp][5] = r5; wred[warp][6] = r6; wred[warp][7] = r7; wred[warp][8] = r8;
            }
        }
        __syncthreads();
        // ---- gradient (thread per column of my slice, active balls in index order) ----
        const double tos = tau / sigma;
        double nv2 = 0.0, dx2 = 0.0, dummy = 0.0;
        for (int j = lo + tid; j < hi; j += WD_THREADS) {
            const double cj = cs[j - lo];
            double s = 0.0;
            for (int i0 = 0; i0 < m; i0 += WD_MB) {          // loads of four balls together; lam = 0 adds exactly zero
                double cv[WD_MB], vq[WD_MB], lm[WD_MB];
#pragma unroll
                for (int u = 0; u < WD_MB; ++u) {
                    const int i = i0 + u;
                    const bool on = i < m && act[i];         // CTA-uniform
                    const int slot = on ? slot_s[i] : -1;
                    lm[u] = on ? lam_r[i] : 0.0;
                    cv[u] = on ? a.C[(int64_t)i * a.ld + j] : cj;
                    vq[u] = slot >= 0 ? V[(int64_t)slot * a.ldv + j] : 0.0;
                }
#pragma unroll
                for (int u = 0; u < WD_MB; ++u) s = fma(lm[u], fma(vq[u], inv_sig, cv[u] - cj), s);
            }
            const double sv = sigma * s;
            const double dx = a.v.x_raw[1 + j] - a.v.xbar_raw[1 + j];
            a.v.grad_t[1 + j] = -sv + tos * dx;
            nv2 = fma(sv, sv, nv2);
            dx2 = fma(dx, dx, dx2);
        }
        ctrl_block_sum3(nv2, dx2, dummy, sm);
        lap(2);
        if (tid == 0) { double* xr = xrec + (size_t)buf * WD_REC; xr[0] = nv2; xr[1] = dx2; }
        wd_exchange(cluster, xrec, buf, 2, xsum);            // (also: every slice of grad_t is in global memory now)
        buf ^= 1;
        if (tid == 0) {
            nv2 = xsum[0]; dx2 = xsum[1];
            double sc[9];
            for (int k = 0; k < 9; ++k) sc[k] = wred[0][k];
            for (int w = 1; w < WD_WARPS; ++w) {
                sc[0] += wred[w][0]; sc[1] += wred[w][1]; sc[2] += wred[w][2]; sc[3] += wred[w][3];
                sc[4] += wred[w][4]; sc[8] += wred[w][8];
                sc[5] = fmax(sc[5], wred[w][5]); sc[6] = fmax(sc[6], wred[w][6]); sc[7] = fmax(sc[7], wred[w][7]);
            }
            const double dx0 = a.v.x_raw[0] - a.v.xbar_raw[0];
            const double dxx = dx2 + dx0 * dx0;
            if (rank == 0) a.v.grad_t[0] = 1.0 - sc[1] + tos * dx0;
            ev_s[MEB_EV_PSI] = a.v.x_raw[0] + 0.5 * sigma * sc[0] + 0.5 * tos * dxx;
            ev_s[MEB_EV_SUM_UPLUS] = sc[1];
            ev_s[MEB_EV_SUM_PROJ2] = sc[0];
            ev_s[MEB_EV_SUM_DMULT2] = sc[2];
            ev_s[MEB_EV_N_B1] = sc[3];
            ev_s[MEB_EV_N_B3] = sc[4];
            ev_s[MEB_EV_MAX_PFEAS] = sc[5];
            ev_s[MEB_EV_MAX_COMPL] = sc[6];
            ev_s[MEB_EV_MAX_DFEAS] = sc[7];
            ev_s[MEB_EV_SUM_RHO] = sc[8];
            ev_s[MEB_EV_NORM_SUM_VPLUS] = sqrt(nv2);
            ev_s[MEB_EV_N_ACTIVE] = sc[3] + sc[4];
            ev_s[12] = dxx; ev_s[13] = 0.0; ev_s[14] = 0.0; ev_s[15] = 0.0;
        }
        __syncthreads();
        // =================================== controller (CTA 0) ======================================
        lap(3);
        if (rank == 0) ctrl_after_eval_body(&sS, a.v, ev_s, sm);
        lap(4);
        publish_state();
        lap(5);
        if (sS.done) break;
        if (sS.action == ACT_TRIAL) continue;

        // ---- ascending list of the active balls of the accepted pass (every CTA builds the same list) ----
        {
            int c = 0, flagged = 0;
            if (tid < WD_M_MAX) {                            // thread per ball: warps 0..7
                flagged = (tid < m && act[tid]) ? 1 : 0;
                const unsigned bits = __ballot_sync(MEB_FULL_MASK, flagged);
                c = __popc(bits & ((1u << lane) - 1u));
                if (lane == 0) wcnt[warp] = __popc(bits);
            }
            __syncthreads();
            if (tid < WD_M_MAX) {
                int pre = 0;
                for (int w = 0; w < warp; ++w) pre += wcnt[w];
                if (flagged) list_s[pre + c] = tid;
                if (tid < m) pos_s[tid] = flagged ? pre + c : -1;
            }
            if (tid == 0) {
                int tot = 0;
                for (int w = 0; w < WD_M_MAX / 32; ++w) tot += wcnt[w];
                nact_s = tot;
            }
            __syncthreads();
        }
        const int nact = nact_s;

        if (sS.action == ACT_NEWTON) {
            // ================= Newton direction, matrix-free (P_i: reading 1) ==================
            // H q = (tau/sigma) q + sigma sum_i P_i q.  The controller has set delta = 0, res = p = -g, cg_rr = ||g||^2
            // and the tolerance (reading 5).  Rows of branch B1 (P_i = I) are stored as zeros: they go through n1.
            // my slice of w_k = b_k / ||b_k||: thread per column, four rows at a time (coef_s holds 1 / ||b_k|| here)
            for (int k = tid; k < nact; k += WD_THREADS) {
                const int i = list_s[k];
                const double rho = rho_r[i];
                rho_s[k] = rho > 1.5 ? 0.0 : rho;
                coef_s[k] = rho > 1.5 ? 0.0 : 1.0 / nb_s[i];             // B3: nb > |a| >= 0
            }
            __syncthreads();
            for (int j = lo + tid; j < hi; j += WD_THREADS) {
                const double cj = cs[j - lo];
                for (int k0 = 0; k0 < nact; k0 += WD_MB) {
                    double cv[WD_MB], vq[WD_MB];
#pragma unroll
                    for (int u = 0; u < WD_MB; ++u) {
                        const int k = k0 + u;
                        const int i = k < nact ? list_s[k] : -1;
                        const int slot = i >= 0 ? slot_s[i] : -1;
                        cv[u] = i >= 0 ? a.C[(int64_t)i * a.ld + j] : cj;
                        vq[u] = slot >= 0 ? V[(int64_t)slot * a.ldv + j] : 0.0;
                    }
#pragma unroll
                    for (int u = 0; u < WD_MB; ++u)
                        if (k0 + u < nact) a.W[(size_t)(k0 + u) * dpad + j] = fma(vq[u], inv_sig, cv[u] - cj) * coef_s[k0 + u];
                }
            }
            __syncthreads();                                 // my slice of W is complete (only this CTA reads it)
            lap(6);
            double* p_s = cs;                                // the centre is not needed until the next evaluation
            for (int e = elo + tid; e < ehi; e += WD_THREADS) p_s[e - elo] = a.v.p[e];
            const double Ls = sS.L;
            const double nB1 = ev_s[MEB_EV_N_B1], nB3 = ev_s[MEB_EV_N_B3], srho = ev_s[MEB_EV_SUM_RHO];
            const double diag0 = tos + sigma * (nB1 + 0.5 * nB3);
            const double diag1 = tos + sigma * (nB1 + 0.5 * (nB3 + srho));
            double rr = sS.cg_rr;
            const double tol = sS.cg_tol;
            const int itmax = sS.cg_max;
            int cgit = 0;
            __syncthreads();
            while (cgit < itmax && sqrt(rr) > tol) {
                // ---- y_k = <w_k, p_1>: slice sums by teams, exchanged; p_0 travels with rank 0's record ----
                double* xr = xrec + (size_t)buf * WD_REC;
                for (int k0 = 0; k0 < nact; k0 += 2 * WD_MB) {           // thread per column, eight rows at a time
                    double y8[2 * WD_MB];
#pragma unroll
                    for (int u = 0; u < 2 * WD_MB; ++u) y8[u] = 0.0;
                    for (int j = lo + tid; j < hi; j += WD_THREADS) {
                        const double pj = p_s[1 + j - elo];
                        double wv[2 * WD_MB];
#pragma unroll
                        for (int u = 0; u < 2 * WD_MB; ++u) wv[u] = (k0 + u < nact) ? a.W[(size_t)(k0 + u) * dpad + j] : 0.0;
#pragma unroll
                        for (int u = 0; u < 2 * WD_MB; ++u) y8[u] = fma(wv[u], pj, y8[u]);
                    }
#pragma unroll
                    for (int u = 0; u < 2 * WD_MB; ++u) {
                        const double t = warp_sum(y8[u]);
                        if (lane == 0) wpart[(size_t)warp * (2 * WD_MB) + u] = t;
                    }
                    __syncthreads();
                    if (tid < 2 * WD_MB && k0 + tid < nact) {
                        double t = 0.0;
#pragma unroll
                        for (int w = 0; w < WD_WARPS; ++w) t += wpart[(size_t)w * (2 * WD_MB) + tid];
                        xr[k0 + tid] = t;
                    }
                    __syncthreads();
                }
                if (tid == 0) xr[nact] = rank == 0 ? p_s[0] : 0.0;
                wd_exchange(cluster, xrec, buf, nact + 1, xsum);
                buf ^= 1;
                const double q0 = xsum[nact];
                for (int k = tid; k < nact; k += WD_THREADS) coef_s[k] = q0 - rho_s[k] * xsum[k];
                double sy = 0.0;
                for (int k = 0; k < nact; ++k) sy += xsum[k];            // (every thread: same order, same bits)
                __syncthreads();
                // ---- my entries of Hp (normalised units: H~ = L H_raw), <p, Hp> ----
                double pHp = 0.0;
                for (int e = elo + tid; e < ehi; e += WD_THREADS) {
                    double hp;
                    const double pe = p_s[e - elo];
                    if (e == 0) {
                        hp = diag0 * q0 + 0.5 * sigma * sy;
                    } else {
                        double z = 0.0;
                        for (int k = 0; k < nact; ++k) z = fma(coef_s[k], a.W[(size_t)k * dpad + (e - 1)], z);
                        hp = diag1 * pe + 0.5 * sigma * z;
                    }
                    hp *= Ls;
                    a.v.Hp[e] = hp;
                    pHp = fma(pe, hp, pHp);
                }
                pHp = wd_block_sum(pHp, red);
                if (tid == 0) xrec[(size_t)buf * WD_REC] = pHp;
                wd_exchange(cluster, xrec, buf, 1, xsum);
                buf ^= 1;
                const double alpha = rr / xsum[0];
                double rrn = 0.0;
                for (int e = elo + tid; e < ehi; e += WD_THREADS) {      // (the same thread wrote Hp[e])
                    a.v.delta[e] = fma(alpha, p_s[e - elo], a.v.delta[e]);
                    const double rj = fma(-alpha, a.v.Hp[e], a.v.res[e]);
                    a.v.res[e] = rj;
                    rrn = fma(rj, rj, rrn);
                }
                rrn = wd_block_sum(rrn, red);
                if (tid == 0) xrec[(size_t)buf * WD_REC] = rrn;
                wd_exchange(cluster, xrec, buf, 1, xsum);
                buf ^= 1;
                rrn = xsum[0];
                const double beta = rrn / rr;
                for (int e = elo + tid; e < ehi; e += WD_THREADS) p_s[e - elo] = fma(beta, p_s[e - elo], a.v.res[e]);
                rr = rrn;
                ++cgit;
                __syncthreads();
            }
            if (tid == 0) { sS.cg_rr = rr; sS.cg_it = cgit; sS.cg_total += cgit; sS.cg_go = 0; }
            lap(7);
            cluster.sync();                                  // every slice of delta is in global memory
            if (rank == 0) meb_ctrl_after_newton_dev(&sS, a.v, a.v.delta, n);
            lap(8);
            publish_state();
            lap(9);
        } else {
            // ================= multiplier update (eq. (6)) and outer-iteration bookkeeping ===============
            const int nxt = hm ? 1 - cur : 0;
            double* Un = a.U2[nxt];
            int32_t* sn = a.slot2[nxt];
            double* Vn = a.V2[nxt];
            if (rank == 0)
                for (int i = tid; i < m; i += WD_THREADS) {
                    const int k = pos_s[i];
                    Un[i] = k >= 0 ? sigma * t_r[i] : 0.0;
                    sn[i] = k;
                }
            // my slice of v_k = sigma lam_k b_k: thread per column, four rows at a time
            for (int j = lo + tid; j < hi; j += WD_THREADS) {
                const double cj = cs[j - lo];
                for (int k0 = 0; k0 < nact; k0 += WD_MB) {
                    double cv[WD_MB], vq[WD_MB], sl[WD_MB];
#pragma unroll
                    for (int u = 0; u < WD_MB; ++u) {
                        const int k = k0 + u;
                        const int i = k < nact ? list_s[k] : -1;
                        const int slot = i >= 0 ? slot_s[i] : -1;
                        sl[u] = i >= 0 ? sigma * lam_r[i] : 0.0;
                        cv[u] = i >= 0 ? a.C[(int64_t)i * a.ld + j] : cj;
                        vq[u] = slot >= 0 ? V[(int64_t)slot * a.ldv + j] : 0.0;
                    }
#pragma unroll
                    for (int u = 0; u < WD_MB; ++u)
                        if (k0 + u < nact) Vn[(int64_t)(k0 + u) * a.ldv + j] = sl[u] * fma(vq[u], inv_sig, cv[u] - cj);
                }
            }
            cluster.sync();                                  // the new multipliers are complete
            lap(10);
            if (rank == 0) meb_ctrl_after_update_dev(&sS, a.v, (long long)nact);
            publish_state();
            lap(11);
            if (sS.done) break;
        }
    }
    __syncthreads();
    if (rank == 0) {   // state back to global memory
        const unsigned long long* src = reinterpret_cast<const unsigned long long*>(&sS);
        unsigned long long* dst = reinterpret_cast<unsigned long long*>(a.S);
        for (int q = tid; q < (int)(sizeof(SolverDev) / 8); q += WD_THREADS) dst[q] = src[q];
    }
    cluster.sync();                                          // nobody leaves while its shared memory may still be read
}

size_t wide_smem_bytes(int m, int d) {
    const int mc = (m + 7) & ~7;
    const int wcol = ((d + WD_NC - 1) / WD_NC + 7) & ~7;
    const size_t doubles = (size_t)wcol + 8 + 3 * (size_t)WD_REC + (size_t)WD_WARPS * 4 * WD_MB + 6 * (size_t)mc;
    return doubles * sizeof(double) + 3 * (size_t)mc * sizeof(int) + (size_t)mc + 64;
}

}  // namespace

// FP64 problems with at most 256 balls and rows too long for the dense Newton path: one cluster runs the phase --
// if the device can place such a cluster at all (asked once per shape class; a partitioned or busy GPU may not).
bool meb_wide_applicable(int prec, int64_t m, int32_t d) {
    if (!(prec == MEB_FP64 && m >= 1 && m <= WD_M_MAX && d > 126)) return false;
    const size_t smem = wide_smem_bytes((int)m, d);
    if (smem > 200 * 1024) return false;
    if (cudaFuncSetAttribute(wide_solve_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3(WD_NC, 1, 1);
    cfg.blockDim = dim3(WD_THREADS, 1, 1);
    cfg.dynamicSmemBytes = smem;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = WD_NC; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    int nclusters = 0;
    if (cudaOccupancyMaxActiveClusters(&nclusters, wide_solve_kernel, &cfg) != cudaSuccess) { cudaGetLastError(); return false; }
    return nclusters >= 1;
}

// W: device buffer of at least m * dpad doubles (dpad = d rounded up to 8).  V pools must hold m rows each.
int meb_launch_wide_solve(meb_ctx* ctx, const void* C, int64_t ld, const void* R, int64_t m, int32_t d, int64_t ldv,
                          void* const U2[2], int32_t* const slot2[2], void* const V2[2], SolverDev* S,
                          const SolverVecs& v, double* W) {
    if (!meb_wide_applicable(MEB_FP64, m, d) || !W) return MEB_E_CAPACITY;
    WideArgs a;
    memset(&a, 0, sizeof(a));
    a.C = (const double*)C; a.ld = ld; a.R = (const double*)R; a.m = (int32_t)m; a.d = d; a.ldv = ldv;
    for (int b = 0; b < 2; ++b) { a.U2[b] = (double*)U2[b]; a.slot2[b] = slot2[b]; a.V2[b] = (double*)V2[b]; }
    a.S = S; a.v = v; a.W = W; a.dpad = (d + 7) / 8 * 8;
    long long* prof = nullptr;
#ifdef MEB_TUNING
    if (getenv("MEB_TRACE")) { cudaMalloc(&prof, 16 * sizeof(long long)); cudaMemset(prof, 0, 16 * sizeof(long long)); }
#endif
    a.prof = prof;
    const size_t smem = wide_smem_bytes((int)m, d);
    MEB_CUDA_OK(ctx, cudaFuncSetAttribute(wide_solve_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3(WD_NC, 1, 1);
    cfg.blockDim = dim3(WD_THREADS, 1, 1);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = ctx->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = WD_NC; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    ctx->launches++;
    MEB_CUDA_OK(ctx, cudaLaunchKernelEx(&cfg, wide_solve_kernel, a));
    if (prof) {
        long long h[16];
        cudaMemcpy(h, prof, sizeof(h), cudaMemcpyDeviceToHost);
        fprintf(stderr, "[meb trace] wide solver cycles: sums %lld xchg %lld epi+grad %lld xchg2 %lld ctrl_eval %lld publish %lld | "
                        "list+gather %lld cg %lld after_newton %lld publish %lld | update %lld after_update %lld\n",
                h[0], h[1], h[2], h[3], h[4], h[5], h[6], h[7], h[8], h[9], h[10], h[11]);
        cudaFree(prof);
    }
    return MEB_OK;
}
