// Device-resident state of Algorithm 1 (ripALM) and Algorithm 2 (semismooth Newton,
// P:L220-242), and the single-CTA controller steps that advance it inside a CUDA graph WHILE loop.
// No host round trip happens between the evaluations of a phase: the controllers decide on the
// device what runs next (another Armijo trial, a Newton solve, a multiplier update) by setting the
// graph's conditional handles.
//
// Units (reading 3): the (d+1)-sized state lives in normalised units x~ = (r/L, (c - off)/L); the
// streaming kernels run on the raw data with x_raw = (L r~, off + L c~), sigma_raw = sigma/L,
// tau_eff = tau/L^2.  g and the multipliers are the same in both unit systems, psi~ = psi_raw/L.
#pragma once
#include "meb_internal.cuh"

enum { PH_FIRST = 0,      // first evaluation of an outer iteration (Alg. 2 lines 3-4): always accepted
       PH_ARMIJO = 1,     // evaluation of an Armijo trial point x + eta*Delta (Alg. 2 line 9)
       PH_REEVAL = 2,     // re-evaluation at x before a multiplier update (records of the last pass are stale)
       PH_AG_Y = 3,       // accelerated gradient (reading 20): evaluation at the extrapolated point y
       PH_AG_X = 4 };     //   evaluation at the candidate x+ = y - grad Psi(y) / Lip (backtracking on Lip)
enum { ACT_TRIAL = 0, ACT_NEWTON = 1, ACT_UPDATE = 2, ACT_DONE = 3 };
enum { ST_RUNNING = 0, ST_CONVERGED = 1, ST_OUTER_CAP = 2, ST_NEED_CAPACITY = 3, ST_CHOL_FAILED = 4, ST_STALLED = 5 };

struct SolverDev {
    // ---- constants of the phase (written by the host before the graph is launched) ----
    double L, tol, rho, tau, kappa, sigma_max, armijo_mu, shrink_min;
    double slope_floor;           // Newton decrement below slope_floor |Psi|: Psi cannot resolve the predicted decrease (reading 6)
    int32_t n, d, inner_max, outer_max, armijo_max, cg_max, dense, use_off;
    int64_t vcap[2];              // rows available in the two V pools
    // ---- dynamic ----
    MebDyn dyn;                   // what the streaming kernels read: sigma_raw, tau_eff, cur, has_mult
    double sigma;                 // normalised sigma_k
    double eta, psi_cur, slope;
    int32_t phase, action, outer, inner, ls, done, status, stalled;
    int32_t newton_total, cg_total, evals, chol_info;
    double kkt, terms[5];
    int64_t n_support;
    double cg_rr, cg_tol;
    int32_t cg_it, cg_go;
    // ---- in-graph timing of the evaluation passes (globaltimer, ns) ----
    unsigned long long pass_ns;
    long long pass_count;
    unsigned long long vrow_reads;  // sum over the evaluation passes that ran to the end (the ones pass_ns / pass_count
                                    // cover) of the V rows they read: one per ball with a slot, i.e. n_support
    // ---- conditional handles of the solve graph ----
    cudaGraphConditionalHandle h_while, h_newton, h_update, h_cg;
    cudaGraphConditionalHandle h_cgp;   // matrix-free Newton solve in one persistent kernel (meb_cg.cu)
    long long wc_cap;                   // active rows the gathered matrix W of that kernel can hold
    int32_t cg_mode;                    // 1: persistent kernel, 0: one launch per CG iteration (more active rows than W holds)
    int32_t screen_valid;               // 1: the last evaluation pass ran at the current x (its fused screening mask is the
                                        // retain rule at x); cleared by every pass at another point and by a fall-back to xbest
    double tol_accept, best_kkt, best_terms[5];   // best outer iterate so far (reading 18)
    double abort_margin;          // relative slack of MebDyn::s0_abort (rounding of the partial sums); 0: early stop off
    int32_t aborted, pad3;        // Armijo trials cut short
    int32_t stall_max;            // outer iterations without halving the best KKT residual before the phase stops (reading 18)
    int32_t stall_count, tiny;    // tiny: the last Newton direction had a decrement below the floor
    uint32_t pass_hist[48], act_hist[48];   // MEB_TRACE: ns and active balls of the first evaluation passes
    int32_t in_graph, eval_cap;   // eval_cap: hard bound on the evaluations of a phase (a runaway loop cannot hang the GPU)
    // ---- multi-trial Armijo (DESIGN reading 19) ----
    int32_t multi_max;            // predictions asked of every trial pass (meb_params.armijo_multi, <= MEB_MULTI_MAX); 0: off
    int32_t pred_n;               // predictions the last pass delivered (written by the finalize kernel)
    double pred_s[MEB_MULTI_MAX]; // sum_i ||Pi(z_i)||^2 at x + eta 2^-k Delta, k = 1..pred_n (lower bounds if the pass was cut)
    int32_t skipped, ag_total;    // step sizes never evaluated; accelerated-gradient iterations
    double pred_margin;           // relative slack of the predicted sums (rounding of the expansion), like abort_margin
    // ---- accelerated-gradient inner solver (DESIGN reading 20) ----
    int32_t ag_outer;             // outer iterations k < ag_outer use it instead of semismooth Newton
    int32_t ag_it;                // iterations of the current inner solve
    double ag_t, ag_Lip;          // momentum parameter t_j, current estimate of the Lipschitz constant of grad Psi
    double ag_psi_y, ag_gg_y;     // Psi(y), ||grad Psi(y)||^2 of the extrapolated point
    int32_t ag_bt, ag_inner_max;  // doublings of Lip at the current y; iteration cap of one inner solve
    long long m_rows;             // balls of this phase's problem
    int32_t lowprec, pad_lp;      // 1: low-precision run: it only has to deliver (r_hat, c_hat) for the screening
};

// (d+1)-vectors of the state, each of length nv = n rounded up to 8, in one device array
struct SolverVecs {
    double *xn, *xbar, *ab, *delta, *g, *xt, *x_raw, *xbar_raw, *off, *grad_t, *res, *p, *Hp, *xbest;
    double *dir_raw;             // L * delta: the direction in raw units, read by the evaluation kernels (multi-trial)
    double *ev_t, *ev;           // [MEB_EVAL_NSCALARS] scalars of the trial / accepted evaluation
};

// arguments of the evaluation-finalize kernel (meb_small.cu)
struct FinalizeArgs {
    const double* part; int grid;                 // per-CTA scalar partials of the streaming kernel
    const double* part_vec; int nvec; int tpb;    // per-CTA vector partials; tpb > 0: written by the active-list
    int dpad;                                     //   kernel (only CTAs b < ceil(count/tpb) hold data); 0: all nvec
    const int32_t* count;
    const double* x; const double* xbar;
    double sigma, tau; int d;
    double* out; double* grad;
    const MebDyn* dyn;                            // nullable: overrides sigma, tau
    SolverDev* S; SolverVecs v;                   // nullable: controller step of the solve graph
    const double* multi_part;                     // nullable: per-CTA partials of the predicted step sizes [grid][MEB_MULTI_MAX]
    // strides (in doubles) between consecutive partials; 0 = the packed layouts MEB_NPART / dpad / MEB_MULTI_MAX.
    // A sharded solve hands in the records gathered from the ranks (one record of rec_stride doubles per rank).
    int part_stride, vec_stride, multi_stride;
};

__device__ __forceinline__ double ctrl_block_sum(double v, double* sm) {
    v = warp_sum(v);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
    const int nw = (blockDim.x + 31) >> 5;
    for (int w = 0; w < nw; ++w) t += sm[w];
    return t;
}

// three block-wide sums with one pair of barriers (fixed order: warp xor tree, then warps in index order)
__device__ __forceinline__ void ctrl_block_sum3(double& a, double& b, double& c, double* sm) {
    a = warp_sum(a); b = warp_sum(b); c = warp_sum(c);
    __syncthreads();
    const int w = threadIdx.x >> 5;
    if ((threadIdx.x & 31) == 0) { sm[w] = a; sm[32 + w] = b; sm[64 + w] = c; }
    __syncthreads();
    const int nw = (blockDim.x + 31) >> 5;
    double ta = 0.0, tb = 0.0, tc = 0.0;
    for (int q = 0; q < nw; ++q) { ta += sm[q]; tb += sm[32 + q]; tc += sm[64 + q]; }
    a = ta; b = tb; c = tc;
}

// x_raw = (L r~, off + L c~)
__device__ __forceinline__ void ctrl_to_raw(const SolverDev* S, const SolverVecs& v, const double* xn_, double* out) {
    for (int j = threadIdx.x; j < S->n; j += blockDim.x)
        out[j] = (j == 0) ? S->L * xn_[0] : ((S->use_off ? v.off[j - 1] : 0.0) + S->L * xn_[j]);
}

// Start of a phase (Alg. 1 line 1): xbar = x, trial point = x, counters cleared.  xn and ab were
// written before (by the host, by a set-up kernel, or by the previous phase).  Any CTA size.
__device__ inline void meb_ctrl_init_dev(SolverDev* S, const SolverVecs v, double sigma0, int cur, int has_mult) {
    const int n = S->n;
    _Pragma("unroll 4")
    for (int j = threadIdx.x; j < n; j += blockDim.x) v.xbar[j] = v.xn[j];
    ctrl_to_raw(S, v, v.xn, v.x_raw);
    __syncthreads();
    _Pragma("unroll 4")
    for (int j = threadIdx.x; j < n; j += blockDim.x) v.xbar_raw[j] = v.x_raw[j];
    if (threadIdx.x == 0) {
        S->sigma = sigma0;
        S->dyn.sigma_raw = sigma0 / S->L;
        S->dyn.tau_eff = S->tau / (S->L * S->L);
        S->dyn.cur = cur;
        S->dyn.has_mult = has_mult;
        S->phase = PH_FIRST; S->action = ACT_TRIAL;
        S->outer = 0; S->inner = 0; S->ls = 0; S->done = 0; S->status = ST_RUNNING; S->stalled = 0;
        S->newton_total = 0; S->cg_total = 0; S->evals = 0; S->chol_info = 0;
        S->kkt = 1e300; S->n_support = 0; S->best_kkt = 1e300; S->stall_count = 0; S->tiny = 0; S->aborted = 0;
        S->dyn.s0_abort = 1e300; S->dyn.multi_n = 0; S->pred_n = 0; S->skipped = 0; S->ag_total = 0; S->ag_it = 0;
        S->ag_t = 1.0; S->ag_Lip = 1.0; S->ag_bt = 0;
        S->pass_ns = 0ull; S->pass_count = 0; S->vrow_reads = 0ull;
        S->eta = 1.0; S->psi_cur = 0.0; S->slope = 0.0;
        S->cg_go = 0; S->cg_it = 0;
    }
}

__device__ __forceinline__ void ctrl_set_handles(const SolverDev* S) {
    if (!S->in_graph) return;
    cudaGraphSetConditional(S->h_while, S->done ? 0u : 1u);
    cudaGraphSetConditional(S->h_newton, (!S->done && S->action == ACT_NEWTON) ? 1u : 0u);
    cudaGraphSetConditional(S->h_update, (!S->done && S->action == ACT_UPDATE) ? 1u : 0u);
    if (!S->dense) {
        const bool go = !S->done && S->action == ACT_NEWTON && S->cg_go;
        cudaGraphSetConditional(S->h_cgp, (go && S->cg_mode == 1) ? 1u : 0u);
        cudaGraphSetConditional(S->h_cg, (go && S->cg_mode == 0) ? 1u : 0u);
    }
}

// Thread 0: arm the early stop (MebDyn::s0_abort) for the Armijo trial with normalised radius rt and
// dx2t = ||x_t - xbar||^2, or disarm it (trial = false).  In normalised units
//   Psi~(x_t) = r~_t + (sigma / 2 L^2) S0 + (tau / 2 sigma) dx2t,   S0 = sum_i ||Pi(z_i)||^2 on the raw data,
// so Psi~(x_t) > Psi~(x) -- which fails the Armijo test and the last-trial test alike -- as soon as
// S0 > 2 L^2 (Psi~(x) - r~_t - (tau / 2 sigma) dx2t) / sigma.
__device__ __forceinline__ void ctrl_arm_abort(SolverDev* S, bool trial, double rt, double dx2t) {
    double thr = 1e300;
    if (trial && S->abort_margin > 0.0) {
        const double room = S->psi_cur - rt - 0.5 * (S->tau / S->sigma) * dx2t;
        if (room > 0.0) thr = 2.0 * S->L * S->L * room / S->sigma * (1.0 + S->abort_margin);
    }
    S->dyn.s0_abort = thr;
    if (!trial) S->dyn.multi_n = 0;
}

// Thread 0: the trial pass at step eta (after `ls` shortenings) also predicts the next halvings eta 2^-k
// (MebDyn::multi_*): as many as asked for and as the halving budget still allows.  dir_r, dir_c2: Delta r and
// ||Delta c||^2 in raw units.
__device__ __forceinline__ void ctrl_arm_multi(SolverDev* S, double eta, int ls, double dir_r, double dir_c2) {
    int nm = S->multi_max;
    if (nm > S->armijo_max - ls) nm = S->armijo_max - ls;
    if (nm < 0 || S->shrink_min != 0.5 || S->tiny) nm = 0;
    S->dyn.multi_n = nm;
    double f = 1.0;
    for (int k = 0; k < MEB_MULTI_MAX; ++k) { f *= 0.5; S->dyn.multi_gamma[k] = eta * (1.0 - f); }
    S->dyn.dir_r = dir_r;
    S->dyn.dir_c2 = dir_c2;
    S->dyn.dir_c = sqrt(dir_c2);
}

// relative KKT residual (reading 7) from the scalars of an evaluation
__device__ __forceinline__ double ctrl_rel_kkt(const double* ev, double r_raw, double* terms) {
    terms[0] = fabs(1.0 - ev[MEB_EV_SUM_UPLUS]);
    terms[1] = ev[MEB_EV_NORM_SUM_VPLUS];
    terms[2] = ev[MEB_EV_MAX_PFEAS] / (1.0 + r_raw);
    terms[3] = ev[MEB_EV_MAX_DFEAS];
    terms[4] = ev[MEB_EV_MAX_COMPL] / (1.0 + r_raw);
    double k = 0.0;
    for (int i = 0; i < 5; ++i) k = fmax(k, terms[i]);
    return k;
}

// Runs in the single CTA of the evaluation-finalize kernel, after ev_t / grad_t of the pass at
// x_raw have been written: Armijo test (reading 4), stopping tests (5) and KKT (P:L133-135,
// L244, reading 6), choice of the next action.  All threads of the CTA call it.
// S is a SHARED-MEMORY copy of the state (loaded by the caller); it is written back to Sg at the end.
// ev_s: the scalars of this evaluation in shared memory (the caller also wrote them to v.ev_t).
__device__ inline void ctrl_after_eval_body(SolverDev* S, const SolverVecs v, const double* ev_s, double* sm);
__device__ inline void ctrl_after_eval(SolverDev* Sg, SolverDev* S, const SolverVecs v, const double* ev_s,
                                       double* sm) {
    ctrl_after_eval_body(S, v, ev_s, sm);
    __syncthreads();
    const unsigned long long* src = reinterpret_cast<const unsigned long long*>(S);
    unsigned long long* dst = reinterpret_cast<unsigned long long*>(Sg);
    for (int q = threadIdx.x; q < (int)(sizeof(SolverDev) / 8); q += blockDim.x) dst[q] = src[q];
}
__device__ inline void ctrl_after_eval_body(SolverDev* S, const SolverVecs v, const double* ev_s, double* sm) {
    __syncthreads();
    if (threadIdx.x == 0) S->screen_valid = 0;              // (set below if this pass becomes the evaluation at x)
    double* __restrict__ xn_ = v.xn;
    double* __restrict__ xbar_ = v.xbar;
    double* __restrict__ ab_ = v.ab;
    double* __restrict__ delta_ = v.delta;
    double* __restrict__ g_ = v.g;
    double* __restrict__ xt_ = v.xt;
    double* __restrict__ x_raw_ = v.x_raw;
    double* __restrict__ off_ = v.off;
    double* __restrict__ grad_t_ = v.grad_t;
    double* __restrict__ res_ = v.res;
    double* __restrict__ p_ = v.p;
    double* __restrict__ Hp_ = v.Hp;
    const int n = S->n;
    const int phase = S->phase;
    const double Ls = S->L;
    const bool use_off = S->use_off != 0;
    const double psi_t = ev_s[MEB_EV_PSI] / Ls;
    bool accept = true, stalled = false;
    // ---- accelerated gradient inner solver (outer iterations k < ag_outer, reading 20) ----
    // y lives in v.p, grad Psi(y) in v.res, the previous iterate in v.Hp (the CG vectors are idle in this mode).
    if (phase == PH_AG_Y) {
        // the pass evaluated Psi and its gradient at y = v.xt: candidate x+ = y - grad Psi(y) / Lip
        double gg = 0.0;
        const double il = 1.0 / S->ag_Lip;
        _Pragma("unroll 4")
        for (int j = threadIdx.x; j < n; j += blockDim.x) {
            const double gj = grad_t_[j], yj = xt_[j];
            res_[j] = gj; p_[j] = yj;
            gg = fma(gj, gj, gg);
            const double xj = fma(-il, gj, yj);
            xt_[j] = xj;
            x_raw_[j] = (j == 0) ? Ls * xj : ((use_off ? off_[j - 1] : 0.0) + Ls * xj);
        }
        gg = ctrl_block_sum(gg, sm);
        if (threadIdx.x == 0) {
            S->ag_psi_y = psi_t; S->ag_gg_y = gg; S->ag_bt = 0;
            S->phase = PH_AG_X; S->action = ACT_TRIAL; S->evals++;
            ctrl_arm_abort(S, false, 0.0, 0.0);
            if (S->evals >= S->eval_cap) { S->done = 1; S->status = ST_OUTER_CAP; }
            ctrl_set_handles(S);
        }
        return;
    }
    if (phase == PH_AG_X && !(psi_t <= S->ag_psi_y - 0.5 * S->ag_gg_y / S->ag_Lip)) {
        // sufficient decrease failed: Lip <- 2 Lip and a shorter step from the same y; after 60 doublings give up
        // and re-evaluate at x (the records of this pass are not those of x)
        const bool giveup = S->ag_bt >= 60;
        const double il = 1.0 / (2.0 * S->ag_Lip);
        _Pragma("unroll 4")
        for (int j = threadIdx.x; j < n; j += blockDim.x) {
            const double xj = giveup ? xn_[j] : fma(-il, res_[j], p_[j]);
            xt_[j] = xj;
            x_raw_[j] = (j == 0) ? Ls * xj : ((use_off ? off_[j - 1] : 0.0) + Ls * xj);
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            if (giveup) S->phase = PH_REEVAL; else { S->ag_Lip *= 2.0; S->ag_bt++; }
            S->action = ACT_TRIAL; S->evals++;
            ctrl_arm_abort(S, false, 0.0, 0.0);
            if (S->evals >= S->eval_cap) { S->done = 1; S->status = ST_OUTER_CAP; }
            ctrl_set_handles(S);
        }
        return;
    }
    if (phase == PH_ARMIJO) {
        if (!(psi_t <= S->psi_cur + S->armijo_mu * S->eta * S->slope)) {
            if (S->ls >= S->armijo_max || S->tiny) {
                stalled = true;
                accept = psi_t <= S->psi_cur;          // last trial did not increase Psi: take it
            } else {
                accept = false;
            }
        }
    }
    if (!accept) {
        // rejected trial: either halve the step (next trial x + eta Delta) or, when the halvings are
        // exhausted, re-evaluate at x (the records of this pass are not those of x)
        // shortened step: eta / 2, except after a trial so far off that the parabola through Psi(x),
        // Psi'(x; Delta) = slope and Psi(x + eta Delta) has its minimiser below shrink_min * eta: then the
        // trials in between are skipped (shrink_min = 1/2: plain halving; 1/8 keeps eta on the halving grid); reading 4
        double eta = 0.0;
        int skip = 0;
        if (!stalled) {
            const double den = psi_t - S->psi_cur - S->slope * S->eta;      // > 0 whenever the Armijo test fails
            const double fq = -0.5 * S->slope * S->eta / den;
            eta = ((fq < S->shrink_min) ? S->shrink_min : 0.5) * S->eta;    // a NaN trial value halves
            // Multi-trial (reading 19): the pass also summed ||Pi(z_i)||^2 at eta/2, eta/4, ... (lower bounds if it
            // was cut short).  Psi~(x + e Delta) = r~ + (sigma / 2 L^2) S + (tau / 2 sigma) ||x + e Delta - xbar||^2;
            // a halving whose bound already fails the Armijo test is skipped: it would be rejected when evaluated,
            // so the step that is finally accepted is the one plain halving accepts.
            const int np = S->pred_n;
            if (np > 0) {
                double A = 0.0, B = 0.0, D = 0.0;
                _Pragma("unroll 4")
                for (int j = threadIdx.x; j < n; j += blockDim.x) {
                    const double w = xn_[j] - xbar_[j], dj = delta_[j];
                    A = fma(w, w, A); B = fma(w, dj, B); D = fma(dj, dj, D);
                }
                ctrl_block_sum3(A, B, D, sm);
                const double cs = 0.5 * S->sigma / (Ls * Ls) * (1.0 - S->pred_margin);
                const double cp = 0.5 * S->tau / S->sigma;
                double ek = S->eta;
                for (int k = 0; k < np; ++k) {
                    ek *= 0.5;
                    if (S->ls + 1 + skip >= S->armijo_max) break;             // the last allowed halving is always evaluated
                    const double lb = xn_[0] + ek * delta_[0] + cs * S->pred_s[k] + cp * (A + ek * (2.0 * B + ek * D));
                    if (lb > S->psi_cur + S->armijo_mu * ek * S->slope) ++skip; else break;
                }
                for (int q = 0; q < skip; ++q) eta *= 0.5;
            }
        }
        double dx2t = 0.0;
        _Pragma("unroll 4")
        for (int j = threadIdx.x; j < n; j += blockDim.x) {
            const double xj = xn_[j] + eta * delta_[j];
            xt_[j] = xj;
            x_raw_[j] = (j == 0) ? Ls * xj : ((use_off ? off_[j - 1] : 0.0) + Ls * xj);
            const double dxb = xj - xbar_[j];
            dx2t = fma(dxb, dxb, dx2t);
        }
        dx2t = ctrl_block_sum(dx2t, sm);
        __syncthreads();
        if (threadIdx.x == 0) {
            ctrl_arm_abort(S, !stalled, xn_[0] + eta * delta_[0], dx2t);
            if (stalled) { S->phase = PH_REEVAL; } else {
                S->eta = eta; S->ls += 1 + skip; S->skipped += skip;
                ctrl_arm_multi(S, eta, S->ls, S->dyn.dir_r, S->dyn.dir_c2);
            }
            S->action = ACT_TRIAL; S->evals++;
            if (S->evals >= S->eval_cap) { S->done = 1; S->status = ST_OUTER_CAP; }
            ctrl_set_handles(S);
        }
        return;
    }
    // ---- accepted: the pass becomes the evaluation at x; condition (5) in the same sweep:
    //      2 sigma |<(alpha,beta) - x, g>| + sigma^2 ||g||^2 <= rho (sum ||dmult||^2 + tau ||x - xbar||^2)
    double agx = 0.0, gg = 0.0, dx2 = 0.0, dotr = 0.0;
    const bool take_xt = phase == PH_ARMIJO || phase == PH_AG_X;
    const bool agmode = S->outer < S->ag_outer;
    _Pragma("unroll 4")
    for (int j = threadIdx.x; j < n; j += blockDim.x) {
        const double xj = take_xt ? xt_[j] : xn_[j];
        const double gj = grad_t_[j];
        const double abj = ab_[j], xbj = xbar_[j];
        if (agmode) {                                   // previous iterate, and <grad Psi(y), x+ - x> for the restart test
            const double xp = xn_[j];
            Hp_[j] = xp;
            if (phase == PH_AG_X) dotr = fma(res_[j], xj - xp, dotr);
        }
        if (take_xt) xn_[j] = xj;
        g_[j] = gj;
        agx = fma(abj - xj, gj, agx);
        gg = fma(gj, gj, gg);
        const double dx = xj - xbj;
        dx2 = fma(dx, dx, dx2);
        if (j == 0) sm[96] = xj;                       // r~ for the KKT normalisation
    }
    if (threadIdx.x < MEB_EVAL_NSCALARS) v.ev[threadIdx.x] = ev_s[threadIdx.x];
    ctrl_block_sum3(agx, gg, dx2, sm);
    if (agmode && phase == PH_AG_X) dotr = ctrl_block_sum(dotr, sm);        // (touches sm[0..31] only)
    if (threadIdx.x == 0) {
        sm[97] = 0.0;                                   // AG continuation: 0 none, 1 step from y = x, 2 extrapolate (sm[98] = beta)
        S->screen_valid = 1;                            // the pass ran at what is now x
        S->evals++;
        S->psi_cur = psi_t;
        double terms[5];
        const double kkt = ctrl_rel_kkt(ev_s, Ls * sm[96], terms);
        S->kkt = kkt;
        for (int i = 0; i < 5; ++i) S->terms[i] = terms[i];
        const double sg = S->sigma;
        const double lhs = 2.0 * sg * fabs(agx) + sg * sg * gg;
        const double rhs = S->rho * (ev_s[MEB_EV_SUM_DMULT2] + S->tau * dx2);
        const bool exit_inner = (phase == PH_REEVAL) || stalled || (phase == PH_ARMIJO && S->tiny) || lhs <= rhs || kkt <= S->tol ||
                                S->inner >= (agmode ? S->ag_inner_max : S->inner_max);
        if (exit_inner) {
            S->action = ACT_UPDATE;
        } else if (agmode) {
            // next accelerated-gradient iteration (reading 20)
            S->action = ACT_TRIAL;
            S->inner++; S->ag_total++;
            ctrl_arm_abort(S, false, 0.0, 0.0);
            double beta = 0.0;
            if (phase == PH_AG_X && !(dotr > 0.0)) {        // momentum, unless the gradient restart fires
                const double t = S->ag_t;
                const double tn = 0.5 * (1.0 + sqrt(1.0 + 4.0 * t * t));
                beta = (t - 1.0) / tn;
                S->ag_t = tn;
            } else {
                S->ag_t = 1.0;
                if (phase != PH_AG_X)                       // first iteration of this inner solve: ||H|| <= tau/sigma + sigma |A|
                    S->ag_Lip = S->tau / sg + sg * fmax(1.0, ev_s[MEB_EV_N_ACTIVE]);
            }
            if (beta > 0.0) { sm[97] = 2.0; sm[98] = beta; S->phase = PH_AG_Y; }
            else {                                          // y = x: this pass IS the evaluation at y
                sm[97] = 1.0; S->ag_psi_y = psi_t; S->ag_gg_y = gg; S->ag_bt = 0; S->phase = PH_AG_X;
            }
        } else {
            S->action = ACT_NEWTON;
            S->inner++;
            S->newton_total++;
            // CG start (matrix-free path): delta = 0, res = p = -g, stop at min(0.1, ||g||) ||g||  (reading 5)
            const double gn = sqrt(gg);
            S->cg_rr = gg;
            S->cg_tol = fmin(0.1, gn) * gn;
            S->cg_it = 0;
            S->cg_go = (gn > S->cg_tol && S->cg_max > 0) ? 1 : 0;
            S->cg_mode = ((long long)ev_s[MEB_EV_N_ACTIVE] <= S->wc_cap) ? 1 : 0;
        }
        if (S->evals >= S->eval_cap) { S->done = 1; S->status = ST_OUTER_CAP; }
        ctrl_set_handles(S);
    }
    __syncthreads();
    if (sm[97] != 0.0) {                                    // accelerated gradient: the next point to evaluate
        const bool extrap = sm[97] == 2.0;
        const double beta = sm[98], il = 1.0 / S->ag_Lip;
        _Pragma("unroll 4")
        for (int j = threadIdx.x; j < n; j += blockDim.x) {
            const double xj = xn_[j];
            double tj;
            if (extrap) tj = fma(beta, xj - Hp_[j], xj);                      // y = x+ + beta (x+ - x)
            else { const double gj = grad_t_[j]; res_[j] = gj; p_[j] = xj; tj = fma(-il, gj, xj); }
            xt_[j] = tj;
            x_raw_[j] = (j == 0) ? Ls * tj : ((use_off ? off_[j - 1] : 0.0) + Ls * tj);
        }
    } else if (S->action == ACT_NEWTON && !S->dense)
        _Pragma("unroll 4")
        for (int j = threadIdx.x; j < n; j += blockDim.x) {
            const double gj = grad_t_[j];
            delta_[j] = 0.0;
            res_[j] = -gj;
            p_[j] = -gj;
        }
}

// Controller step after a Newton solve (Alg. 2 line 9): slope <g, Delta>, first Armijo trial x + Delta.
// z: Delta (n doubles, shared or global).  S may live in global or shared memory.  Any CTA size (whole warps).
__device__ inline void meb_ctrl_after_newton_dev(SolverDev* S, const SolverVecs v, const double* z, int n) {
    double* __restrict__ xn_ = v.xn;
    double* __restrict__ xbar_ = v.xbar;
    double* __restrict__ g_ = v.g;
    double* __restrict__ xt_ = v.xt;
    double* __restrict__ x_raw_ = v.x_raw;
    double* __restrict__ off_ = v.off;
    double* __restrict__ dir_raw_ = v.dir_raw;
    __shared__ double red[32], red2[32];
    const int tid = threadIdx.x;
    const double Ls = S->L;
    const bool use_off = S->use_off != 0;
    __shared__ double red3[32];
    double sl = 0.0, dx2t = 0.0, dc2 = 0.0;
    for (int j = tid; j < n; j += blockDim.x) {
        const double dj = z[j];
        sl = fma(g_[j], dj, sl);
        const double xj = xn_[j] + dj;
        xt_[j] = xj;
        x_raw_[j] = (j == 0) ? Ls * xj : ((use_off ? off_[j - 1] : 0.0) + Ls * xj);
        dir_raw_[j] = Ls * dj;
        const double dxb = xj - xbar_[j];
        dx2t = fma(dxb, dxb, dx2t);
        if (j > 0) dc2 = fma(dj, dj, dc2);
    }
    sl = warp_sum(sl);
    dx2t = warp_sum(dx2t);
    dc2 = warp_sum(dc2);
    if ((tid & 31) == 0) { red[tid >> 5] = sl; red2[tid >> 5] = dx2t; red3[tid >> 5] = dc2; }
    __syncthreads();
    if (tid == 0) {
        double t = 0.0, t2 = 0.0, t3 = 0.0;
        const int nw = (blockDim.x + 31) >> 5;
        for (int w = 0; w < nw; ++w) { t += red[w]; t2 += red2[w]; t3 += red3[w]; }
        ctrl_arm_abort(S, true, xn_[0] + z[0], t2);
        S->slope = t; S->eta = 1.0; S->ls = 0; S->phase = PH_ARMIJO; S->action = ACT_TRIAL;
        S->tiny = (-t <= S->slope_floor * fabs(S->psi_cur)) ? 1 : 0;
        ctrl_arm_multi(S, 1.0, 0, Ls * z[0], Ls * Ls * t3);
    }
}

// After (U+, V+) of the accepted point were written into the other multiplier buffer (eq. (6)):
// capacity check, buffer flip, (alpha, beta) update, KKT test, best-iterate / stall
// logic (reading 18), sigma update, start of the next outer iteration.  Every thread of the CTA
// calls it; S may live in global or shared memory; nact = number of active balls of the accepted pass.
__device__ inline void meb_ctrl_after_update_dev(SolverDev* S, const SolverVecs v, long long nact) {
    double* __restrict__ xn_ = v.xn;
    double* __restrict__ xbar_ = v.xbar;
    double* __restrict__ ab_ = v.ab;
    double* __restrict__ g_ = v.g;
    double* __restrict__ x_raw_ = v.x_raw;
    double* __restrict__ xbar_raw_ = v.xbar_raw;
    double* __restrict__ off_ = v.off;
    double* __restrict__ xbest_ = v.xbest;
    const int n = S->n;
    const int nxt = S->dyn.has_mult ? 1 - S->dyn.cur : 0;
    const bool fits = nact <= S->vcap[nxt];
    __syncthreads();
    if (!fits) {                                    // host grows the pool and relaunches; x is re-evaluated
        ctrl_to_raw(S, v, v.xn, v.x_raw);
        if (threadIdx.x == 0) {
            S->n_support = nact;
            ctrl_arm_abort(S, false, 0.0, 0.0);
            S->phase = PH_REEVAL; S->action = ACT_DONE; S->done = 1; S->status = ST_NEED_CAPACITY;
            ctrl_set_handles(S);
        }
        return;
    }
    // ---- decisions (every thread computes the same from the state as it was on entry) ----
    const double sg = S->sigma;
    const double kkt = S->kkt;
    const int outer1 = S->outer + 1;
    const bool improved = kkt < S->best_kkt;                     // best iterate so far (returned if the run stalls)
    const int stall = (kkt < 0.5 * S->best_kkt) ? 0 : S->stall_count + 1;
    const double best = improved ? kkt : S->best_kkt;
    int status = ST_RUNNING;
    if (kkt <= S->tol) status = ST_CONVERGED;
    else if (stall >= 3 && best <= S->tol_accept) status = ST_CONVERGED;     // floor of the arithmetic (reading 18)
    else if (stall >= S->stall_max) status = ST_STALLED;
    // reading 17: a low-precision run whose support is a large part of ALL balls (degenerate: co-spherical points)
    // cannot resolve multipliers of size 1/|support| and will not reach tol_lo (config 4: its third outer iteration
    // alone spends 60 passes on line searches in rounding noise): two outer iterations give the (r_hat, c_hat) the
    // screening needs.  The a-posteriori check makes the result independent of this.
    else if (S->lowprec && outer1 >= 2 && 10.0 * v.ev[MEB_EV_N_ACTIVE] > (double)S->m_rows) status = ST_STALLED;
    else if (outer1 >= S->outer_max) status = (best <= S->tol_accept) ? ST_CONVERGED : ST_OUTER_CAP;
    const bool take_best = status != ST_RUNNING && !improved && kkt > S->tol;
    __syncthreads();
    _Pragma("unroll 4")
    for (int j = threadIdx.x; j < n; j += blockDim.x) {
        const double xj = xn_[j];
        ab_[j] -= sg * g_[j];
        if (improved) xbest_[j] = xj;
        const double xo = take_best ? xbest_[j] : xj;
        if (take_best) xn_[j] = xo;
        xbar_[j] = xo;
        const double xr = (j == 0) ? S->L * xo : ((S->use_off ? off_[j - 1] : 0.0) + S->L * xo);
        x_raw_[j] = xr;
        xbar_raw_[j] = xr;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        S->dyn.cur = nxt;
        S->dyn.has_mult = 1;
        S->outer = outer1;
        S->n_support = nact;
        S->stall_count = stall;
        if (improved) { S->best_kkt = kkt; for (int i = 0; i < 5; ++i) S->best_terms[i] = S->terms[i]; }
        if (status != ST_RUNNING) {
            S->done = 1; S->status = status;
            if (take_best) { S->screen_valid = 0; S->kkt = S->best_kkt; for (int i = 0; i < 5; ++i) S->terms[i] = S->best_terms[i]; }
        } else {
            const double s2 = fmin(S->sigma_max, S->kappa * sg);
            S->sigma = s2;
            S->dyn.sigma_raw = s2 / S->L;
        }
        S->inner = 0;
        ctrl_arm_abort(S, false, 0.0, 0.0);
        S->phase = PH_FIRST;
        S->action = S->done ? ACT_DONE : ACT_TRIAL;
        ctrl_set_handles(S);
    }
}
