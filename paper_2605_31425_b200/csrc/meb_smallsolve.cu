// Single-CTA ripALM for SMALL problems (m <= 4096 balls, d <= 128, FP64): the reduced problem of the
// mixed-precision method and any small instance.  Such problems are L2-resident and
// launch-bound: a pass over 145 balls is ~1 us of work, while a graph iteration costs ~10 kernel nodes.
// Here ONE persistent CTA of 256 threads runs the whole phase -- Algorithm 1 with
// Algorithm 2 inside -- with no launch and no grid-wide synchronisation in the loop:
//
//   evaluation   warp per ball: b_i = c_i - c + v_i/sigma (lanes over columns, kept in registers),
//                shuffle reduction, the shared scalar epilogue (branch of P:L115, multiplier, KKT terms),
//                lam_i b_i added to per-warp register accumulators for the active balls;
//   controller   the same device functions as the graph path (meb_ctrl.cuh) on a shared-memory state;
//   Newton       H = (tau/sigma) I + sigma sum_i P_i (P_i: reading 1) accumulated straight into
//                the register tiles of the LDL^T solver (meb_ldlt.cuh) from shared tiles of normalised
//                active rows -- the matrix never exists in memory;
//   update       (u, v) <- sigma Pi(z) (eq. (6)) into the other multiplier buffer.
//
// Deterministic: static ball -> warp assignment, warps and tiles combined in index order.
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <vector>

#include "meb_ctrl.cuh"
#include "meb_internal.cuh"
#include "meb_ldlt.cuh"
#include "meb_rowops.cuh"

namespace {

constexpr int SM_THREADS = 256;
constexpr int SM_WARPS = 8;
constexpr int SM_RB = 32;            // active rows per Hessian tile
constexpr int SM_MAXCOL = 4;         // columns per lane: d <= 128

struct SmallArgs {
    const double* C; int64_t ld; const double* R;
    int32_t m, d; int64_t ldv;
    double* U2[2]; int32_t* slot2[2]; double* V2[2];
    double* rec_lam; double* rec_rho; double* rec_t;
    SolverDev* S; SolverVecs v;
    int32_t m_cap;                   // capacity of the shared index list / flags
    long long* prof;                 // nullable: cycles per section (eval, finalize, ctrl, list, hessian, ldlt, update), MEB_TRACE
};

template <int BS>
__device__ __forceinline__ void small_solve_body(const SmallArgs& a) {
    constexpr int DP = 16 * BS;                          // padded matrix order (>= n + 1)
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ __align__(16) SolverDev sS;
    __shared__ double ev_s[MEB_EVAL_NSCALARS];
    __shared__ double sm[104];
    __shared__ double wred[SM_WARPS][MEB_NPART];
    __shared__ int bad;
    __shared__ int nact_s;
    __shared__ int wcnt[SM_WARPS];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tx = tid & 15, ty = tid >> 4;
    const int m = a.m, d = a.d, n = d + 1;
    // ---- shared memory carve-up ----
    double* Lm = reinterpret_cast<double*>(smem_raw);
    double* cs = Lm + LdltShape<BS>::smem_doubles(n);    // centre c (d values)
    double* ws = cs + DP;                                // [SM_RB][DP] normalised active rows, index 0 = 1
    double* rho_t = ws + SM_RB * DP;                     // [SM_RB]
    double* vecp = rho_t + SM_RB;                        // [SM_WARPS][DP] per-warp sum of lam_i b_i
    int* list_s = reinterpret_cast<int*>(vecp + SM_WARPS * DP);      // [m_cap]
    unsigned char* act = reinterpret_cast<unsigned char*>(list_s + a.m_cap);   // [m_cap]

    {   // working copy of the solver state
        const unsigned long long* src = reinterpret_cast<const unsigned long long*>(a.S);
        unsigned long long* dst = reinterpret_cast<unsigned long long*>(&sS);
        for (int q = tid; q < (int)(sizeof(SolverDev) / 8); q += SM_THREADS) dst[q] = src[q];
    }
    __syncthreads();
    StreamArgs sa;                                       // only the fields the row epilogue touches
    sa.rec_lam = a.rec_lam; sa.rec_rho = a.rec_rho; sa.rec_t = a.rec_t;
    sa.t_out = nullptr; sa.lam_out = nullptr;

    long long tmark = clock64();
    auto lap = [&](int k) { if (a.prof && tid == 0) { const long long t = clock64(); a.prof[k] += t - tmark; tmark = t; } };
    for (;;) {
        // =================================== evaluation at v.x_raw ===================================
        const double sigma = sS.dyn.sigma_raw, tau = sS.dyn.tau_eff;
        const bool hm = sS.dyn.has_mult != 0;
        const int cur = sS.dyn.cur;
        const double* U = hm ? a.U2[cur] : nullptr;
        const int32_t* slotp = hm ? a.slot2[cur] : nullptr;
        const double* V = hm ? a.V2[cur] : nullptr;
        for (int j = tid; j < DP; j += SM_THREADS) cs[j] = j < d ? a.v.x_raw[1 + j] : 0.0;
        const double r = a.v.x_raw[0];
        const double inv_sig = 1.0 / sigma;
        __syncthreads();
        Acc acc;
        double vacc[SM_MAXCOL];
#pragma unroll
        for (int q = 0; q < SM_MAXCOL; ++q) vacc[q] = 0.0;
        // THREAD per ball: a thread walks its own row (d independent loads in flight, lines shared through
        // L1), so the latency of the L2-resident data is paid once per pass, not once per ball, and every
        // thread runs the scalar epilogue of its ball in parallel.
        for (int i = tid; i < m; i += SM_THREADS) {
            const double* rowp = a.C + (int64_t)i * a.ld;
            const int slot = slotp ? slotp[i] : -1;
            const double ui = U ? U[i] : 0.0;
            const double ri = a.R ? a.R[i] : 0.0;
            double nb2 = 0.0, ne2 = 0.0, evd = 0.0, vv = 0.0;
            if (slot < 0) {
                double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
                int j = 0;
                for (; j + 4 <= d; j += 4) {
                    const double e0 = rowp[j] - cs[j], e1 = rowp[j + 1] - cs[j + 1];
                    const double e2 = rowp[j + 2] - cs[j + 2], e3 = rowp[j + 3] - cs[j + 3];
                    s0 = fma(e0, e0, s0); s1 = fma(e1, e1, s1); s2 = fma(e2, e2, s2); s3 = fma(e3, e3, s3);
                }
                for (; j < d; ++j) { const double e = rowp[j] - cs[j]; s0 = fma(e, e, s0); }
                nb2 = (s0 + s1) + (s2 + s3);
            } else {
                const double* vrow = V + (int64_t)slot * a.ldv;
#pragma unroll 4
                for (int j = 0; j < d; ++j) {
                    const double e = rowp[j] - cs[j];
                    const double vj = vrow[j];
                    const double bj = fma(vj, inv_sig, e);
                    nb2 = fma(bj, bj, nb2); ne2 = fma(e, e, ne2); evd = fma(e, vj, evd); vv = fma(vj, vj, vv);
                }
            }
            double mylam;
            const bool flag = row_epilogue_core<double, OP_EVAL>(sa, i, true, slot >= 0, nb2, ne2, evd, vv, r, sigma, ri, ui,
                                                                 acc, mylam);
            act[i] = flag ? 1 : 0;
        }
        __syncthreads();
        // gradient vector part: warp per ACTIVE ball, lanes over the columns (lam_i from the records)
        for (int i = warp; i < m; i += SM_WARPS) {
            if (!act[i]) continue;
            const double lam = a.rec_lam[i];
            const int slot = slotp ? slotp[i] : -1;
            const double* rowp = a.C + (int64_t)i * a.ld;
            const double* vrow = slot >= 0 ? V + (int64_t)slot * a.ldv : nullptr;
#pragma unroll
            for (int q = 0; q < SM_MAXCOL; ++q) {
                const int j = lane + 32 * q;
                if (j < d) {
                    double bj = rowp[j] - cs[j];
                    if (vrow) bj = fma(vrow[j], inv_sig, bj);
                    vacc[q] = fma(lam, bj, vacc[q]);
                }
            }
        }
        lap(0);
        // ---- per-warp partials -> block, fixed order ----
#pragma unroll
        for (int q = 0; q < SM_MAXCOL; ++q) {
            const int j = lane + 32 * q;
            if (j < DP) vecp[warp * DP + j] = vacc[q];
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
        // ---- finalize: psi, gradient, KKT terms (reading 13) ----
        const double tos = tau / sigma;
        double nv2 = 0.0, dx2 = 0.0, dummy = 0.0;
        for (int j = tid; j < d; j += SM_THREADS) {
            double s = 0.0;
#pragma unroll
            for (int w = 0; w < SM_WARPS; ++w) s += vecp[w * DP + j];
            const double sv = sigma * s;
            const double dx = a.v.x_raw[1 + j] - a.v.xbar_raw[1 + j];
            a.v.grad_t[1 + j] = -sv + tos * dx;
            nv2 = fma(sv, sv, nv2);
            dx2 = fma(dx, dx, dx2);
        }
        ctrl_block_sum3(nv2, dx2, dummy, sm);
        if (tid == 0) {
            double sc[9];
            for (int k = 0; k < 9; ++k) sc[k] = wred[0][k];
            for (int w = 1; w < SM_WARPS; ++w) {
                sc[0] += wred[w][0]; sc[1] += wred[w][1]; sc[2] += wred[w][2]; sc[3] += wred[w][3];
                sc[4] += wred[w][4]; sc[8] += wred[w][8];
                sc[5] = fmax(sc[5], wred[w][5]); sc[6] = fmax(sc[6], wred[w][6]); sc[7] = fmax(sc[7], wred[w][7]);
            }
            const double dx0 = a.v.x_raw[0] - a.v.xbar_raw[0];
            const double dxx = dx2 + dx0 * dx0;
            a.v.grad_t[0] = 1.0 - sc[1] + tos * dx0;
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
        lap(1);
        // =================================== controller ==============================================
        ctrl_after_eval_body(&sS, a.v, ev_s, sm);
        __syncthreads();
        lap(2);
        if (sS.done) break;
        if (sS.action == ACT_TRIAL) continue;

        // ---- ascending list of the active balls of the accepted pass (both branches need it) ----
        {
            const int per = (m + SM_THREADS - 1) / SM_THREADS;
            const int i0 = tid * per, i1 = min(m, i0 + per);
            int c = 0;
            for (int i = i0; i < i1; ++i) c += act[i];
            int incl = c;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(MEB_FULL_MASK, incl, o);
                if (lane >= o) incl += t;
            }
            if (lane == 31) wcnt[warp] = incl;
            __syncthreads();
            int pre = 0, tot = 0;
#pragma unroll
            for (int w = 0; w < SM_WARPS; ++w) { if (w < warp) pre += wcnt[w]; tot += wcnt[w]; }
            int pos = pre + incl - c;
            for (int i = i0; i < i1; ++i) if (act[i]) list_s[pos++] = i;
            if (tid == 0) nact_s = tot;
            __syncthreads();
        }
        const int nact = nact_s;
        lap(3);

        if (sS.action == ACT_NEWTON) {
            // ================= Newton direction: H in registers, LDL^T, first Armijo trial ============
            const double Ls = sS.L;
            double acc_h[BS][BS];
#pragma unroll
            for (int ii = 0; ii < BS; ++ii)
#pragma unroll
                for (int jj = 0; jj < BS; ++jj) acc_h[ii][jj] = 0.0;
            for (int t0 = 0; t0 < nact; t0 += SM_RB) {
                __syncthreads();
                for (int rr = warp; rr < SM_RB; rr += SM_WARPS) {        // stage normalised rows of the tile
                    const int k = t0 + rr;
                    double rho = 0.0;
                    bool use = false;
                    int i = 0;
                    if (k < nact) { i = list_s[k]; rho = a.rec_rho[i]; use = rho < 1.5; }   // B1: P_i = I, no outer product
                    double bq[SM_MAXCOL];
                    double nb2 = 0.0;
                    if (use) {
                        const double* rowp = a.C + (int64_t)i * a.ld;
                        const int slot = slotp ? slotp[i] : -1;
                        const double* vrow = slot >= 0 ? V + (int64_t)slot * a.ldv : nullptr;
#pragma unroll
                        for (int q = 0; q < SM_MAXCOL; ++q) {
                            const int j = lane + 32 * q;
                            double bj = 0.0;
                            if (j < d) {
                                bj = rowp[j] - cs[j];
                                if (vrow) bj = fma(vrow[j], inv_sig, bj);
                            }
                            bq[q] = bj;
                            nb2 = fma(bj, bj, nb2);
                        }
                        nb2 = warp_sum(nb2);
                    }
                    const double inv = use ? 1.0 / sqrt(nb2) : 0.0;
                    double* wrow = ws + rr * DP;
                    for (int j = lane; j < DP; j += 32) wrow[j] = 0.0;
                    __syncwarp();
                    if (use) {
#pragma unroll
                        for (int q = 0; q < SM_MAXCOL; ++q) {
                            const int j = lane + 32 * q;
                            if (j < d) wrow[1 + j] = bq[q] * inv;        // matrix index 1 + j  <->  column j of c
                        }
                        if (lane == 0) wrow[0] = 1.0;                    // index 0 <-> r
                    }
                    if (lane == 0) rho_t[rr] = use ? rho : 0.0;
                }
                __syncthreads();
#pragma unroll 2
                for (int rr = 0; rr < SM_RB; ++rr) {
                    const double* w = ws + rr * DP;
                    const double w0 = w[0];                              // 1 for a B3 row of the tile, else 0
                    const double cr = -0.5 * sigma * Ls * rho_t[rr];
                    const double c0 = 0.5 * sigma * Ls * w0;
                    double wi[BS], wj[BS];
#pragma unroll
                    for (int q = 0; q < BS; ++q) { wi[q] = w[ty + 16 * q]; wj[q] = w[tx + 16 * q]; }
                    const double wj0 = (tx == 0) ? 0.0 : wj[0];          // column 0 gets no rho-weighted term
#pragma unroll
                    for (int ii = 0; ii < BS; ++ii) {
                        const double ci = cr * wi[ii];
#pragma unroll
                        for (int jj = 0; jj <= ii; ++jj) acc_h[ii][jj] = fma(ci, jj == 0 ? wj0 : wj[jj], acc_h[ii][jj]);
                        if (tx == 0) acc_h[ii][0] = fma(c0, wi[ii], acc_h[ii][0]);   // 1/2 sigma [n3; s] in column 0
                    }
                }
            }
            // constants of H (SURVEY 8(a) row a2'), the right-hand side row, zeros elsewhere
            const double n1 = ev_s[MEB_EV_N_B1], n3 = ev_s[MEB_EV_N_B3], srho = ev_s[MEB_EV_SUM_RHO];
            const double d0 = Ls * (tau / sigma + sigma * n1);
            const double d1 = Ls * (tau / sigma + sigma * (n1 + 0.5 * (n3 + srho)));
#pragma unroll
            for (int ii = 0; ii < BS; ++ii)
#pragma unroll
                for (int jj = 0; jj < BS; ++jj) {
                    const int i = ty + 16 * ii, j = tx + 16 * jj;
                    double hv = acc_h[ii][jj];
                    if (jj > ii || j > i || j >= n || i > n) hv = 0.0;
                    else if (i == n) hv = -a.v.g[j];
                    else if (i == j) hv += (i == 0) ? d0 : d1;
                    acc_h[ii][jj] = hv;
                }
            lap(4);
            const double* z = meb_ldlt_solve_regs<BS>(acc_h, n, Lm, &bad);
            for (int e = tid; e < n; e += SM_THREADS) a.v.delta[e] = z[e];
            if (tid == 0) sS.chol_info = bad;
            meb_ctrl_after_newton_dev(&sS, a.v, z, n);
            __syncthreads();
            lap(5);
        } else {
            // ================= multiplier update (eq. (6)) and outer-iteration bookkeeping ===============
            const int nxt = hm ? 1 - cur : 0;
            double* Un = a.U2[nxt];
            int32_t* sn = a.slot2[nxt];
            double* Vn = a.V2[nxt];
            for (int i = tid; i < m; i += SM_THREADS) { Un[i] = 0.0; sn[i] = -1; }
            __syncthreads();
            for (int k = warp; k < nact; k += SM_WARPS) {
                const int i = list_s[k];
                const double* rowp = a.C + (int64_t)i * a.ld;
                const int slot = slotp ? slotp[i] : -1;
                const double* vrow = slot >= 0 ? V + (int64_t)slot * a.ldv : nullptr;
                const double sl = sigma * a.rec_lam[i];
                double* vout = Vn + (int64_t)k * a.ldv;
                for (int j = lane; j < d; j += 32) {
                    double bj = rowp[j] - cs[j];
                    if (vrow) bj = fma(vrow[j], inv_sig, bj);
                    vout[j] = sl * bj;
                }
                if (lane == 0) { Un[i] = sigma * a.rec_t[i]; sn[i] = k; }
            }
            __syncthreads();
            meb_ctrl_after_update_dev(&sS, a.v, (long long)nact);
            __syncthreads();
            lap(6);
            if (sS.done) break;
        }
    }
    __syncthreads();
    {   // state back to global memory
        const unsigned long long* src = reinterpret_cast<const unsigned long long*>(&sS);
        unsigned long long* dst = reinterpret_cast<unsigned long long*>(a.S);
        for (int q = tid; q < (int)(sizeof(SolverDev) / 8); q += SM_THREADS) dst[q] = src[q];
    }
}

template <int BS>
__global__ void __launch_bounds__(SM_THREADS) small_solve_kernel(const SmallArgs a) {
    small_solve_body<BS>(a);
}

// ---- batched solves: one CTA per independent instance ----------------------------
// Instance k owns rows row0 .. row0 + m - 1 of the shared centre / radius arrays and its own state.
struct BatchInst {
    SmallArgs a;
    double* c0;              // [d] = a.v.off
    double* out;             // [d + 4]: centre, radius, KKT residual, status, L
    int32_t sample_rows;
    double sigma0;
};

// a0 for one instance (readings 3, 16): c0 = mean of a strided row sample, L = max_i(||c_i - c0|| + r_i),
// validation, then the start of Algorithm 1 (x~ = (1, 0), (alpha, beta) = x~, multipliers 0).
__global__ void __launch_bounds__(SM_THREADS) batch_setup_kernel(const BatchInst* insts, const SolverDev* tmpl) {
    const BatchInst in = insts[blockIdx.x];
    const SmallArgs& a = in.a;
    __shared__ double red[SM_WARPS];
    __shared__ int badn[SM_WARPS];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int m = a.m, d = a.d, n = d + 1;
    {   // state = the template (constants of the run)
        const unsigned long long* src = reinterpret_cast<const unsigned long long*>(tmpl);
        unsigned long long* dst = reinterpret_cast<unsigned long long*>(a.S);
        for (int q = tid; q < (int)(sizeof(SolverDev) / 8); q += SM_THREADS) dst[q] = src[q];
    }
    const int S = m < in.sample_rows ? m : in.sample_rows;
    for (int j = tid; j < d; j += SM_THREADS) {
        double s = 0.0;
        for (int k = 0; k < S; ++k) s += a.C[(((int64_t)k * m) / S) * a.ld + j];
        in.c0[j] = s / (double)S;
    }
    __syncthreads();
    double best = 0.0;
    int bad = 0;
    for (int i = warp; i < m; i += SM_WARPS) {           // warp per ball
        const double* rowp = a.C + (int64_t)i * a.ld;
        double s = 0.0, f = 0.0;
        for (int j = lane; j < d; j += 32) { const double e = rowp[j] - in.c0[j]; s = fma(e, e, s); f = fma(rowp[j], 0.0, f); }
        s = warp_sum(s); f = warp_sum(f);
        const double ri = a.R ? a.R[i] : 0.0;
        if (!(f == 0.0) || !(ri >= 0.0) || !(ri < 1.79e308)) bad++;
        best = fmax(best, sqrt(s) + ri);
    }
    if (lane == 0) { red[warp] = best; badn[warp] = bad; }
    __syncthreads();
    double L = 0.0; int nbad = 0;
    for (int w = 0; w < SM_WARPS; ++w) { L = fmax(L, red[w]); nbad += badn[w]; }
    for (int j = tid; j < n; j += SM_THREADS) { const double x0 = j == 0 ? 1.0 : 0.0; a.v.xn[j] = x0; a.v.ab[j] = x0; }
    __syncthreads();
    if (tid == 0) {
        a.S->L = L;
        a.S->vcap[0] = m; a.S->vcap[1] = m;
    }
    __syncthreads();
    // every ball is the point c0 up to the rounding of the coordinates (reading 16): nothing to iterate on
    double cmax = 0.0;
    for (int j = 0; j < d; ++j) cmax = fmax(cmax, fabs(in.c0[j]));
    const bool degenerate = nbad > 0 || !(L > 1e-14 * cmax) || !(L < 1.79e308);
    if (!degenerate) meb_ctrl_init_dev(a.S, a.v, in.sigma0, 0, 0);
    __syncthreads();
    if (tid == 0) {
        in.out[d + 3] = L;
        if (degenerate) {                                 // nothing to iterate on: bad input, or every ball is the point c0
            a.S->done = 1;
            a.S->status = ST_CONVERGED;
            a.S->kkt = 0.0;
            in.out[d + 2] = nbad > 0 ? (double)MEB_E_INPUT : (double)MEB_OK;
        } else {
            in.out[d + 2] = 1e9;                          // overwritten by the final kernel
        }
    }
}

template <int BS>
__global__ void __launch_bounds__(SM_THREADS) small_solve_batch_kernel(const BatchInst* insts) {
    const SmallArgs a = insts[blockIdx.x].a;
    if (a.S->done) return;                                // uniform: decided by the set-up kernel
    small_solve_body<BS>(a);
}

// Result of one instance (step 7 of SURVEY 8(c)): c = c0 + L c~, r = max_i(||c - c_i|| + r_i), the smallest
// feasible radius for that centre.
__global__ void __launch_bounds__(SM_THREADS) batch_final_kernel(const BatchInst* insts) {
    const BatchInst in = insts[blockIdx.x];
    const SmallArgs& a = in.a;
    __shared__ double cs[128];
    __shared__ double red[SM_WARPS];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int m = a.m, d = a.d;
    const bool bad = in.out[d + 2] == (double)MEB_E_INPUT;
    const double L = a.S->L;
    for (int j = tid; j < d; j += SM_THREADS) { cs[j] = in.c0[j] + (L > 0.0 ? L * a.v.xn[1 + j] : 0.0); in.out[j] = cs[j]; }
    __syncthreads();
    double best = 0.0;
    for (int i = warp; i < m; i += SM_WARPS) {
        const double* rowp = a.C + (int64_t)i * a.ld;
        double s = 0.0;
        for (int j = lane; j < d; j += 32) { const double e = rowp[j] - cs[j]; s = fma(e, e, s); }
        s = warp_sum(s);
        best = fmax(best, sqrt(s) + (a.R ? a.R[i] : 0.0));
    }
    if (lane == 0) red[warp] = best;
    __syncthreads();
    if (tid == 0) {
        double r = 0.0;
        for (int w = 0; w < SM_WARPS; ++w) r = fmax(r, red[w]);
        in.out[d] = r;
        in.out[d + 1] = a.S->kkt;
        if (!bad) in.out[d + 2] = (a.S->status == ST_CONVERGED) ? (double)MEB_OK : (double)MEB_W_NOT_CONVERGED;
    }
}

template <int BS>
size_t small_smem(int n, int m_cap) {
    constexpr int DP = 16 * BS;
    return (LdltShape<BS>::smem_doubles(n) + DP + (size_t)SM_RB * DP + SM_RB + (size_t)SM_WARPS * DP) * sizeof(double) +
           (size_t)m_cap * sizeof(int) + (size_t)m_cap + 16;
}

}  // namespace

// The single-CTA solver handles FP64 problems with m <= 4096, d <= 128 whose V pools hold m rows each.
bool meb_small_applicable(int prec, int64_t m, int32_t d) {
    return prec == MEB_FP64 && m <= 4096 && d <= 126 && d >= 1;
}

int meb_launch_small_solve(meb_ctx* ctx, const void* C, int64_t ld, const void* R, int64_t m, int32_t d, int64_t ldv,
                           void* const U2[2], int32_t* const slot2[2], void* const V2[2], SolverDev* S,
                           const SolverVecs& v) {
    SmallArgs a;
    memset(&a, 0, sizeof(a));
    a.C = (const double*)C; a.ld = ld; a.R = (const double*)R; a.m = (int32_t)m; a.d = d; a.ldv = ldv;
    for (int b = 0; b < 2; ++b) { a.U2[b] = (double*)U2[b]; a.slot2[b] = slot2[b]; a.V2[b] = (double*)V2[b]; }
    a.rec_lam = ctx->rec_lam; a.rec_rho = ctx->rec_rho; a.rec_t = ctx->rec_t;
    a.S = S; a.v = v;
    a.m_cap = (int32_t)((m + 15) / 16 * 16);
    long long* prof = nullptr;
#ifdef MEB_TUNING
    if (getenv("MEB_TRACE")) { cudaMalloc(&prof, 8 * sizeof(long long)); cudaMemset(prof, 0, 8 * sizeof(long long)); }
#endif
    a.prof = prof;
    const int n = d + 1;
    const int bs = (n + 1 + 15) / 16;
#define MEB_SMALL_CASE(B)                                                                                         \
    case B: {                                                                                                     \
        const size_t smem = small_smem<B>(n, a.m_cap);                                                            \
        if (smem > 225 * 1024) return MEB_E_CAPACITY;                                                             \
        MEB_CUDA_OK(ctx, cudaFuncSetAttribute(small_solve_kernel<B>, cudaFuncAttributeMaxDynamicSharedMemorySize, \
                                              (int)smem));                                                        \
        ctx->launches++;                                                                                          \
        small_solve_kernel<B><<<1, SM_THREADS, smem, ctx->stream>>>(a);                                           \
        break;                                                                                                    \
    }
    switch (bs) {
        MEB_SMALL_CASE(1) MEB_SMALL_CASE(2) MEB_SMALL_CASE(3) MEB_SMALL_CASE(4)
        MEB_SMALL_CASE(5) MEB_SMALL_CASE(6) MEB_SMALL_CASE(7) MEB_SMALL_CASE(8)
        default: return MEB_E_CAPACITY;
    }
#undef MEB_SMALL_CASE
    MEB_CUDA_OK(ctx, cudaGetLastError());
    if (prof) {
        long long h[8];
        cudaMemcpy(h, prof, sizeof(h), cudaMemcpyDeviceToHost);
        fprintf(stderr, "[meb trace] small solver cycles: eval %lld finalize %lld ctrl %lld list %lld hessian %lld ldlt %lld update %lld\n",
                h[0], h[1], h[2], h[3], h[4], h[5], h[6]);
        cudaFree(prof);
    }
    return MEB_OK;
}

// ---- C-ABI: batched solves ---------------------------------------------------------------------------
namespace {
constexpr int OWN_BATCH = 20;          // slot of meb_ctx::own used by meb_solve_batch (OWN_BATCH_RESERVED in meb_solver.cu)

int batch_reserve(meb_ctx* ctx, size_t bytes) {
    if (ctx->own_bytes[OWN_BATCH] >= bytes) return MEB_OK;
    if (ctx->own[OWN_BATCH]) { cudaFree(ctx->own[OWN_BATCH]); ctx->own[OWN_BATCH] = nullptr; ctx->own_bytes[OWN_BATCH] = 0; }
    const size_t want = bytes + bytes / 4;
    if (cudaMalloc(&ctx->own[OWN_BATCH], want) != cudaSuccess) { cudaGetLastError(); return MEB_E_ALLOC; }
    ctx->own_bytes[OWN_BATCH] = want;
    return MEB_OK;
}
}  // namespace

extern "C" int meb_solve_batch(meb_ctx* ctx, int32_t nprob, const int64_t* h_row_offsets, int32_t d,
                               const double* centers, int64_t ld, const double* radii, double tol,
                               const meb_params* h_params, double* h_centers_out, double* h_radii_out,
                               int32_t* h_status_out, double* h_kkt_out) {
    if (!ctx || nprob < 1 || !h_row_offsets || !centers || !h_centers_out || !h_radii_out || d < 1 || ld < d)
        return MEB_E_ARG;
    if (!(tol > 0.0)) return MEB_E_ARG;
    meb_params par;
    if (h_params) par = *h_params; else meb_default_params(&par);
    if (!(par.rho >= 0.0 && par.rho < 1.0) || !(par.sigma0 > 0.0) || !(par.tau > 0.0) || !(par.kappa >= 1.0) ||
        par.sample_rows < 1)
        return MEB_E_ARG;
    int64_t m_maxi = 0;
    for (int k = 0; k < nprob; ++k) {
        const int64_t mk = h_row_offsets[k + 1] - h_row_offsets[k];
        if (mk < 1 || h_row_offsets[k] < 0) return MEB_E_ARG;
        if (!meb_small_applicable(MEB_FP64, mk, d)) return MEB_E_CAPACITY;    // m_k <= 4096, d <= 126
        if (mk > m_maxi) m_maxi = mk;
    }
    const int64_t row_base = h_row_offsets[0];
    const int64_t rows = h_row_offsets[nprob] - row_base;
    const int n = d + 1;
    const size_t nv = ((size_t)n + 7) / 8 * 8;
    const int64_t ldv = ((int64_t)d + 1) / 2 * 2;
    const size_t vec_doubles = 15 * nv + 2 * MEB_EVAL_NSCALARS;
    const size_t out_doubles = ((size_t)d + 4 + 7) / 8 * 8;
    // one block of device memory, carved up (all pieces 16-byte aligned)
    auto al = [](size_t b) { return (b + 255) / 256 * 256; };
    size_t off = 0;
    const size_t o_inst = off; off += al((size_t)nprob * sizeof(BatchInst));
    const size_t o_tmpl = off; off += al(sizeof(SolverDev));
    const size_t o_S = off;    off += al((size_t)nprob * sizeof(SolverDev));
    const size_t o_vec = off;  off += al((size_t)nprob * vec_doubles * sizeof(double));
    const size_t o_out = off;  off += al((size_t)nprob * out_doubles * sizeof(double));
    size_t o_U[2], o_sl[2], o_V[2];
    for (int b = 0; b < 2; ++b) {
        o_U[b] = off;  off += al((size_t)rows * sizeof(double));
        o_sl[b] = off; off += al((size_t)rows * sizeof(int32_t));
        o_V[b] = off;  off += al((size_t)rows * ldv * sizeof(double));
    }
    const size_t o_rec = off;  off += al((size_t)3 * rows * sizeof(double));
    int rc = batch_reserve(ctx, off);
    if (rc) return rc;
    unsigned char* base = (unsigned char*)ctx->own[OWN_BATCH];

    std::vector<BatchInst> hi((size_t)nprob);
    for (int k = 0; k < nprob; ++k) {
        BatchInst& in = hi[(size_t)k];
        memset(&in, 0, sizeof(in));
        const int64_t r0 = h_row_offsets[k], mk = h_row_offsets[k + 1] - r0, q0 = r0 - row_base;
        SmallArgs& a = in.a;
        a.C = centers + r0 * ld; a.ld = ld; a.R = radii ? radii + r0 : nullptr;
        a.m = (int32_t)mk; a.d = d; a.ldv = ldv;
        for (int b = 0; b < 2; ++b) {
            a.U2[b] = (double*)(base + o_U[b]) + q0;
            a.slot2[b] = (int32_t*)(base + o_sl[b]) + q0;
            a.V2[b] = (double*)(base + o_V[b]) + q0 * ldv;
        }
        double* rec = (double*)(base + o_rec);
        a.rec_lam = rec + q0 - 0; a.rec_rho = rec + rows + q0; a.rec_t = rec + 2 * rows + q0;
        // the records and multiplier arrays are indexed by the ball's index INSIDE the instance
        a.S = (SolverDev*)(base + o_S) + k;
        double* vb = (double*)(base + o_vec) + (size_t)k * vec_doubles;
        double** vecs[] = {&a.v.xn, &a.v.xbar, &a.v.ab, &a.v.delta, &a.v.g, &a.v.xt, &a.v.x_raw, &a.v.xbar_raw,
                           &a.v.off, &a.v.grad_t, &a.v.res, &a.v.p, &a.v.Hp, &a.v.xbest};
        for (size_t i = 0; i < 14; ++i) *vecs[i] = vb + i * nv;
        a.v.dir_raw = vb + 14 * nv;
        a.v.ev_t = vb + 15 * nv;
        a.v.ev = a.v.ev_t + MEB_EVAL_NSCALARS;
        a.m_cap = (int32_t)((m_maxi + 15) / 16 * 16);
        a.prof = nullptr;
        in.c0 = a.v.off;
        in.out = (double*)(base + o_out) + (size_t)k * out_doubles;
        in.sample_rows = par.sample_rows;
        in.sigma0 = par.sigma0;
    }
    SolverDev ht;
    memset(&ht, 0, sizeof(ht));
    ht.L = 1.0; ht.tol = 0.1 * tol; ht.tol_accept = tol;      // KKT test at tol/10 as in meb_solve (reading 7)
    ht.rho = par.rho; ht.tau = par.tau; ht.kappa = par.kappa; ht.sigma_max = par.sigma_max; ht.armijo_mu = par.armijo_mu;
    ht.shrink_min = (par.armijo_shrink_min > 0.0 && par.armijo_shrink_min <= 0.5) ? par.armijo_shrink_min : 0.5;
    ht.slope_floor = 2e-15; ht.abort_margin = 0.0; ht.stall_max = 6;
    ht.n = n; ht.d = d; ht.inner_max = par.inner_max; ht.outer_max = par.outer_max; ht.armijo_max = par.armijo_max_halvings;
    ht.cg_max = par.cg_max; ht.dense = 1; ht.use_off = 1; ht.in_graph = 0;
    ht.eval_cap = 4 * par.outer_max * (par.inner_max + 2);
    ht.multi_max = 0; ht.pred_margin = 1e-6; ht.ag_outer = 0; ht.lowprec = 0; ht.m_rows = 0;
    MEB_CUDA_OK(ctx, cudaMemcpyAsync(base + o_inst, hi.data(), (size_t)nprob * sizeof(BatchInst), cudaMemcpyHostToDevice, ctx->stream));
    MEB_CUDA_OK(ctx, cudaMemcpyAsync(base + o_tmpl, &ht, sizeof(ht), cudaMemcpyHostToDevice, ctx->stream));
    const BatchInst* dinst = (const BatchInst*)(base + o_inst);
    ctx->launches++;
    batch_setup_kernel<<<nprob, SM_THREADS, 0, ctx->stream>>>(dinst, (const SolverDev*)(base + o_tmpl));
    MEB_CUDA_OK(ctx, cudaGetLastError());
    const int bs = (n + 1 + 15) / 16;
    const int m_cap = (int)((m_maxi + 15) / 16 * 16);
#define MEB_BATCH_CASE(B)                                                                                              \
    case B: {                                                                                                          \
        const size_t smem = small_smem<B>(n, m_cap);                                                                   \
        if (smem > 225 * 1024) return MEB_E_CAPACITY;                                                                  \
        MEB_CUDA_OK(ctx, cudaFuncSetAttribute(small_solve_batch_kernel<B>, cudaFuncAttributeMaxDynamicSharedMemorySize, \
                                              (int)smem));                                                             \
        ctx->launches++;                                                                                               \
        small_solve_batch_kernel<B><<<nprob, SM_THREADS, smem, ctx->stream>>>(dinst);                                  \
        break;                                                                                                         \
    }
    switch (bs) {
        MEB_BATCH_CASE(1) MEB_BATCH_CASE(2) MEB_BATCH_CASE(3) MEB_BATCH_CASE(4)
        MEB_BATCH_CASE(5) MEB_BATCH_CASE(6) MEB_BATCH_CASE(7) MEB_BATCH_CASE(8)
        default: return MEB_E_CAPACITY;
    }
#undef MEB_BATCH_CASE
    MEB_CUDA_OK(ctx, cudaGetLastError());
    ctx->launches++;
    batch_final_kernel<<<nprob, SM_THREADS, 0, ctx->stream>>>(dinst);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    std::vector<double> ho((size_t)nprob * out_doubles);
    MEB_CUDA_OK(ctx, cudaMemcpyAsync(ho.data(), base + o_out, ho.size() * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    MEB_CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
    int worst = MEB_OK;
    for (int k = 0; k < nprob; ++k) {
        const double* o = ho.data() + (size_t)k * out_doubles;
        memcpy(h_centers_out + (size_t)k * d, o, (size_t)d * sizeof(double));
        h_radii_out[k] = o[d];
        const int stt = (int)o[d + 2];
        if (h_status_out) h_status_out[k] = stt;
        if (h_kkt_out) h_kkt_out[k] = o[d + 1];
        if (stt < 0) worst = stt;
        else if (stt > 0 && worst >= 0) worst = stt;
    }
    return worst;
}
