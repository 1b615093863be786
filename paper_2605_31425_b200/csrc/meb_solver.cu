// meb_solve: Algorithm 1, Algorithm 2 and the mixed-precision reduction
// loop of Section 4.2, sequencing the kernels of this library.
//
// Units (reading 3): the (d+1)-sized state x~ = (r/L, (c - c0)/L), (alpha, beta), sigma, tau live in
// normalised units; the kernels run on the RAW data with x_raw = (L r~, off + L c~),
// sigma_raw = sigma/L, tau_eff = tau/L^2.  Then the multipliers and g are unchanged,
// psi~ = psi_raw/L and H~ = L H_raw, so no scaled copy of C is ever made.
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <vector>

#include "meb_internal.cuh"

#define SM_EV 0
#define SM_AUX 16
#define SM_X 32

namespace {

enum { OWN_U0 = 0, OWN_U1, OWN_S0, OWN_S1, OWN_V0, OWN_V1, OWN_C32, OWN_R32, OWN_IDX, OWN_CRED, OWN_RRED,
       OWN_KEPT, OWN_STATE, OWN_HOSTC, OWN_HOSTR, OWN_SPARE };

int own_reserve(meb_ctx* ctx, int slot, size_t bytes) {
    if (ctx->own_bytes[slot] >= bytes && ctx->own[slot]) return MEB_OK;
    if (ctx->own[slot]) { cudaFree(ctx->own[slot]); ctx->own[slot] = nullptr; ctx->own_bytes[slot] = 0; }
    const size_t want = bytes < 256 ? 256 : bytes;
    cudaError_t e = cudaMalloc(&ctx->own[slot], want);
    if (e != cudaSuccess) { cudaGetLastError(); ctx->last_cuda_error = (int)e; return MEB_E_ALLOC; }
    ctx->own_bytes[slot] = want;
    return MEB_OK;
}

struct Problem {                   // one ripALM run: data + double-buffered multipliers
    int prec; int64_t m; int32_t d;
    const void* C; int64_t ld; const void* R;
    void* U[2]; int32_t* slot[2]; void* V[2]; int64_t ldv; int64_t vcap[2];
    int own_v[2];                  // own[] slots holding the V pools
    int cur; bool has_mult;
    const double* off;             // host: raw offset of the centre (c0 for raw data, nullptr for the centred shadow)
    bool full;                     // streams all m rows (for the pass statistics)
};

struct Solver {
    meb_ctx* ctx; meb_params par; meb_stats* st;
    int32_t d; double L;
    double* dx; double* dxbar; double* dq; double* dHq; double* dgrad;   // device (d+1)
    double* dH; double* ddelta;                                         // device (d+1)^2, (d+1): dense Newton system
    std::vector<double> hx, hxbar;
    double bytes;
};

size_t esz(int prec) { return prec == MEB_FP64 ? 8 : 4; }

int sync_stream(meb_ctx* ctx) { MEB_CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream)); return MEB_OK; }

int upload(meb_ctx* ctx, double* dst, const double* src, size_t n) {
    // staged through pinned memory so that the copy is truly asynchronous and ordered on the stream
    MEB_CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
    double* stage = ctx->h_pinned + ctx->h_pinned_len / 2;      // second half of the pinned mirror
    memcpy(stage, src, n * sizeof(double));
    MEB_CUDA_OK(ctx, cudaMemcpyAsync(dst, stage, n * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
    return MEB_OK;
}

// x_raw = (L r~, off + L c~)
void to_raw(const Solver& S, const Problem& P, const std::vector<double>& xn, std::vector<double>& xr) {
    xr.resize(S.d + 1);
    xr[0] = S.L * xn[0];
    for (int j = 0; j < S.d; ++j) xr[1 + j] = (P.off ? P.off[j] : 0.0) + S.L * xn[1 + j];
}

struct Ev { double s[MEB_EVAL_NSCALARS]; std::vector<double> g; double psi_n; };

EvalCall make_call(const Solver& S, const Problem& P, double sigma) {
    EvalCall c;
    c.gs = nullptr;
    c.prec = P.prec; c.m = P.m; c.d = P.d; c.C = P.C; c.ld = P.ld; c.R = P.R;
    c.U = P.has_mult ? P.U[P.cur] : nullptr;
    c.v_slot = P.has_mult ? P.slot[P.cur] : nullptr;
    c.V = P.has_mult ? P.V[P.cur] : nullptr;
    c.ldv = P.ldv;
    c.x = S.dx; c.xbar = S.dxbar; c.sigma = sigma / S.L; c.tau = S.par.tau / (S.L * S.L);
    return c;
}

void count_pass(Solver& S, const Problem& P) {
    if (!P.full) S.st->passes_reduced++;
    else if (P.prec == MEB_FP64) S.st->passes_fp64_full++;
    else S.st->passes_fp32_full++;
    S.bytes += S.ctx->last_pass_bytes;
}

// evaluate at normalised x; want_grad = false gives psi and the scalars only (Armijo trials)
int evaluate(Solver& S, const Problem& P, const std::vector<double>& xn, double sigma, bool want_grad, Ev& ev) {
    meb_ctx* ctx = S.ctx;
    std::vector<double> xr;
    to_raw(S, P, xn, xr);
    int rc = upload(ctx, S.dx, xr.data(), S.d + 1);
    if (rc) return rc;
    EvalCall c = make_call(S, P, sigma);
    ctx->cur_class = !P.full ? MEB_PASS_EVAL_REDUCED : (P.prec == MEB_FP64 ? MEB_PASS_EVAL_FP64 : MEB_PASS_EVAL_FP32);
    want_grad = true;
    rc = meb_eval_internal(ctx, c, ctx->small + SM_EV, S.dgrad, nullptr, nullptr);
    if (rc) return rc;
    count_pass(S, P);
    MEB_CUDA_OK(ctx, cudaMemcpyAsync(ctx->h_pinned, ctx->small + SM_EV, MEB_EVAL_NSCALARS * sizeof(double),
                                     cudaMemcpyDeviceToHost, ctx->stream));
    if (want_grad)
        MEB_CUDA_OK(ctx, cudaMemcpyAsync(ctx->h_pinned + 16, S.dgrad, (S.d + 1) * sizeof(double),
                                         cudaMemcpyDeviceToHost, ctx->stream));
    rc = sync_stream(ctx);
    if (rc) return rc;
    memcpy(ev.s, ctx->h_pinned, sizeof(ev.s));
    ev.psi_n = ev.s[MEB_EV_PSI] / S.L;
    if (want_grad) ev.g.assign(ctx->h_pinned + 16, ctx->h_pinned + 16 + S.d + 1);
    return MEB_OK;
}

double rel_kkt(const Ev& ev, double r_raw, double terms[5]) {   // P:L307-311, reading 7
    terms[0] = fabs(1.0 - ev.s[MEB_EV_SUM_UPLUS]);
    terms[1] = ev.s[MEB_EV_NORM_SUM_VPLUS];
    terms[2] = ev.s[MEB_EV_MAX_PFEAS] / (1.0 + r_raw);
    terms[3] = ev.s[MEB_EV_MAX_DFEAS];
    terms[4] = ev.s[MEB_EV_MAX_COMPL] / (1.0 + r_raw);
    double k = 0.0;
    for (int i = 0; i < 5; ++i) k = fmax(k, terms[i]);
    return k;
}

double dot(const std::vector<double>& a, const std::vector<double>& b) {
    double s = 0.0;
    for (size_t i = 0; i < a.size(); ++i) s += a[i] * b[i];
    return s;
}

// H~ q = L * H_raw q through the active-list kernel (records of the evaluation at the current x)
int apply_H(Solver& S, const Problem& P, double sigma, const std::vector<double>& q, std::vector<double>& Hq) {
    meb_ctx* ctx = S.ctx;
    int rc = upload(ctx, S.dq, q.data(), S.d + 1);
    if (rc) return rc;
    EvalCall c = make_call(S, P, sigma);
    rc = meb_hvp_from_records(ctx, c, ctx->small + SM_EV, S.dq, S.dHq);
    if (rc) return rc;
    MEB_CUDA_OK(ctx, cudaMemcpyAsync(ctx->h_pinned + 16, S.dHq, (S.d + 1) * sizeof(double),
                                     cudaMemcpyDeviceToHost, ctx->stream));
    rc = sync_stream(ctx);
    if (rc) return rc;
    Hq.resize(S.d + 1);
    for (int j = 0; j <= S.d; ++j) Hq[j] = S.L * ctx->h_pinned[16 + j];
    return MEB_OK;
}

// Newton direction by conjugate gradients (reading 5)
int newton_cg(Solver& S, const Problem& P, double sigma, const std::vector<double>& g, std::vector<double>& delta) {
    const int n = S.d + 1;
    const double gn = sqrt(dot(g, g));
    const double tol = fmin(0.1, gn) * gn;
    delta.assign(n, 0.0);
    std::vector<double> res(n), p(n), Hp;
    for (int j = 0; j < n; ++j) { res[j] = -g[j]; p[j] = res[j]; }
    double rr = dot(res, res);
    for (int it = 0; it < S.par.cg_max; ++it) {
        if (sqrt(rr) <= tol) break;
        int rc = apply_H(S, P, sigma, p, Hp);
        if (rc) return rc;
        S.st->cg_iters++;
        const double alpha = rr / dot(p, Hp);
        for (int j = 0; j < n; ++j) { delta[j] += alpha * p[j]; res[j] -= alpha * Hp[j]; }
        const double rr_new = dot(res, res);
        const double beta = rr_new / rr;
        for (int j = 0; j < n; ++j) p[j] = res[j] + beta * p[j];
        rr = rr_new;
    }
    return MEB_OK;
}

// Newton direction by dense assembly + Cholesky on the device (moderate d)
int newton_dense(Solver& S, const Problem& P, double sigma, std::vector<double>& delta) {
    meb_ctx* ctx = S.ctx;
    const int n = S.d + 1;
    EvalCall c = make_call(S, P, sigma);
    int rc = meb_dense_from_records(ctx, c, ctx->small + SM_EV, S.dH);
    if (rc) return rc;
    rc = meb_chol_solve(ctx, S.dH, S.dgrad, n, S.L, S.ddelta, nullptr);      // H~ = L H_raw
    if (rc) return rc;
    MEB_CUDA_OK(ctx, cudaMemcpyAsync(ctx->h_pinned + 16, S.ddelta, n * sizeof(double), cudaMemcpyDeviceToHost,
                                     ctx->stream));
    rc = sync_stream(ctx);
    if (rc) return rc;
    delta.assign(ctx->h_pinned + 16, ctx->h_pinned + 16 + n);
    return MEB_OK;
}

// (U, V) <- (U+, V+) from the records of the evaluation at the accepted point (eq. (6))
int update_multipliers(Solver& S, Problem& P, double sigma, const Ev& ev) {
    meb_ctx* ctx = S.ctx;
    const int nxt = P.has_mult ? 1 - P.cur : 0;
    const int64_t nact = (int64_t)ev.s[MEB_EV_N_ACTIVE];
    if (P.vcap[nxt] < nact || !P.V[nxt]) {
        if (P.own_v[nxt] < 0) return MEB_E_CAPACITY;
        const int64_t cap = nact + nact / 2 + 64;
        int rc = own_reserve(ctx, P.own_v[nxt], (size_t)cap * P.ldv * esz(P.prec));
        if (rc) return rc;
        P.V[nxt] = ctx->own[P.own_v[nxt]];
        P.vcap[nxt] = (int64_t)(ctx->own_bytes[P.own_v[nxt]] / ((size_t)P.ldv * esz(P.prec)));
    }
    int rc = P.prec == MEB_FP64 ? meb_fill_f64(ctx, (double*)P.U[nxt], P.m, 0.0)
                                : meb_fill_f32(ctx, (float*)P.U[nxt], P.m, 0.f);
    if (rc) return rc;
    rc = meb_fill_i32(ctx, P.slot[nxt], P.m, -1);
    if (rc) return rc;
    EvalCall c = make_call(S, P, sigma);
    rc = meb_ensure_list(ctx, P.m);
    if (rc) return rc;
    ActiveArgs a;
    memset(&a, 0, sizeof(a));
    a.C = c.C; a.ld = c.ld; a.U = c.U; a.v_slot = c.v_slot; a.V = c.V; a.ldv = c.ldv; a.x = c.x; a.d = c.d;
    a.dpad = (c.d + 7) / 8 * 8; a.sigma = c.sigma; a.list = ctx->list; a.count = ctx->count_dev;
    a.rec_lam = ctx->rec_lam; a.rec_rho = ctx->rec_rho; a.rec_t = ctx->rec_t;
    a.part_vec = ctx->part_vec; a.part_sc = ctx->part_sc;
    a.U_out = P.U[nxt]; a.slot_out = P.slot[nxt]; a.V_out = P.V[nxt]; a.ldv_out = P.ldv; a.cap_rows = P.vcap[nxt];
    int nvec = 0;
    rc = meb_launch_active(ctx, MODE_WRITEV, P.prec, a, &nvec);
    if (rc) return rc;
    P.cur = nxt;
    P.has_mult = true;
    return MEB_OK;
}

// Algorithm 1 with Algorithm 2 inside.  xn / ab are the normalised x and (alpha, beta), in/out.
int ripalm(Solver& S, Problem& P, std::vector<double>& xn, std::vector<double>& ab, double tol, bool* converged,
           double* kkt_out, double terms_out[5]) {
    const meb_params& par = S.par;
    meb_ctx* ctx = S.ctx;
    const int n = S.d + 1;
    double sigma = par.sigma0;
    const double tau = par.tau;
    *converged = false;
    Ev ev, evt;
    std::vector<double> xbar, delta, xt(n), xr;
    double terms[5];
    for (int k = 0; k < par.outer_max; ++k) {
        xbar = xn;                                                    // (r^k, c^k)
        to_raw(S, P, xbar, xr);
        int rc = upload(ctx, S.dxbar, xr.data(), n);
        if (rc) return rc;
        rc = evaluate(S, P, xn, sigma, true, ev);                     // Alg. 2 lines 3-4
        if (rc) return rc;
        bool records_current = true;
        for (int j = 0; j < par.inner_max; ++j) {
            const double kkt = rel_kkt(ev, S.L * xn[0], terms);
            // relative-type stopping condition (5), on the tentative quantities
            double agx = 0.0, dx2 = 0.0;
            for (int i = 0; i < n; ++i) {
                agx += (ab[i] - xn[i]) * ev.g[i];
                dx2 += (xn[i] - xbar[i]) * (xn[i] - xbar[i]);
            }
            const double lhs = 2.0 * sigma * fabs(agx) + sigma * sigma * dot(ev.g, ev.g);
            const double rhs = par.rho * (ev.s[MEB_EV_SUM_DMULT2] + tau * dx2);
            if (lhs <= rhs) break;                                    // Alg. 2 line 5
            if (kkt <= tol) break;                                    // reading 6
            rc = (S.d <= par.dense_d_max && S.d <= 128) ? newton_dense(S, P, sigma, delta)
                                                        : newton_cg(S, P, sigma, ev.g, delta);   // Alg. 2 line 8
            if (rc) return rc;
            S.st->newton_iters++;
            const double slope = dot(ev.g, delta);
            double eta = 1.0;
            bool accepted = false;
            for (int ls = 0; ls <= par.armijo_max_halvings; ++ls) {   // Armijo, P:L212 / reading 4
                for (int i = 0; i < n; ++i) xt[i] = xn[i] + eta * delta[i];
                rc = evaluate(S, P, xt, sigma, false, evt);
                if (rc) return rc;
                if (evt.psi_n <= ev.psi_n + par.armijo_mu * eta * slope) { accepted = true; break; }
                eta *= 0.5;
            }
            if (!accepted) {
                if (evt.psi_n <= ev.psi_n) {                          // last trial did not increase Psi: take it
                    xn = xt;
                    ev = evt;
                } else {
                    records_current = false;
                }
                break;                                                // stalled
            }
            xn = xt;
            ev = evt;                                                 // the accepted trial is the next evaluation
        }
        if (!records_current) {                                       // rare: re-evaluate at x for the update
            rc = evaluate(S, P, xn, sigma, true, ev);
            if (rc) return rc;
        }
        rc = update_multipliers(S, P, sigma, ev);                     // eq. (6)
        if (rc) return rc;
        for (int i = 0; i < n; ++i) ab[i] -= sigma * ev.g[i];
        S.st->outer_iters++;
        const double kkt = rel_kkt(ev, S.L * xn[0], terms);
        *kkt_out = kkt;
        memcpy(terms_out, terms, sizeof(terms));
        S.st->n_support = (int64_t)ev.s[MEB_EV_N_ACTIVE];
        if (kkt <= tol) { *converged = true; break; }
        sigma = fmin(par.sigma_max, par.kappa * sigma);               // P:L175, reading 3
    }
    return MEB_OK;
}

int setup_multipliers(meb_ctx* ctx, Problem& P, int ownU0, int ownS0, int ownV0) {
    for (int b = 0; b < 2; ++b) {
        int rc = own_reserve(ctx, ownU0 + b, (size_t)P.m * esz(P.prec));
        if (rc) return rc;
        rc = own_reserve(ctx, ownS0 + b, (size_t)P.m * sizeof(int32_t));
        if (rc) return rc;
        P.U[b] = ctx->own[ownU0 + b];
        P.slot[b] = (int32_t*)ctx->own[ownS0 + b];
        P.own_v[b] = ownV0 + b;
        P.V[b] = ctx->own[ownV0 + b];
        P.vcap[b] = P.V[b] ? (int64_t)(ctx->own_bytes[ownV0 + b] / ((size_t)P.ldv * esz(P.prec))) : 0;
    }
    P.cur = 0;
    P.has_mult = false;
    return MEB_OK;
}

}  // namespace

extern "C" int meb_solve(meb_ctx* ctx, int64_t m, int32_t d, const double* centers, int64_t ld,
                         const double* radii, double tol, int precision_mode, const meb_params* h_params,
                         double* h_center_out, double* h_radius_out, meb_stats* h_stats) {
    if (!ctx || !centers || !h_center_out || !h_radius_out || m < 1 || d < 1 || ld < d) return MEB_E_ARG;
    if (!(tol > 0.0) || (precision_mode != MEB_MODE_FP64 && precision_mode != MEB_MODE_MIXED)) return MEB_E_ARG;
    if (m > ctx->m_max || d > ctx->d_max) return MEB_E_CAPACITY;
    meb_stats local_stats;
    meb_stats* st = h_stats ? h_stats : &local_stats;
    memset(st, 0, sizeof(*st));
    Solver S;
    S.ctx = ctx; S.st = st; S.d = d; S.bytes = 0.0;
    if (h_params) S.par = *h_params; else meb_default_params(&S.par);
    if (!(S.par.rho >= 0.0 && S.par.rho < 1.0) || !(S.par.sigma0 > 0.0) || !(S.par.tau > 0.0) ||
        !(S.par.kappa >= 1.0) || S.par.sample_rows < 1)
        return MEB_E_ARG;
    const int n = d + 1;
    const bool timing_was = ctx->time_passes;
    ctx->evn = 0;
    ctx->ev_record = true;
    const int64_t launches0 = ctx->launches;
    cudaEvent_t e_start, e_mid, e_hi, e_end;
    MEB_CUDA_OK(ctx, cudaEventCreate(&e_start));
    MEB_CUDA_OK(ctx, cudaEventCreate(&e_mid));
    MEB_CUDA_OK(ctx, cudaEventCreate(&e_hi));
    MEB_CUDA_OK(ctx, cudaEventCreate(&e_end));
    int rc = MEB_OK;
    std::vector<double> c0(d), xn(n, 0.0), ab, creturn(d);
    bool converged = false;
    double kkt = INFINITY, terms[5] = {0, 0, 0, 0, 0};
    Problem P;
    memset(&P, 0, sizeof(P));
    do {
        MEB_CUDA_OK(ctx, cudaEventRecord(e_start, ctx->stream));
        // ---- state vectors on the device ----
        const size_t nH = (d <= 128) ? (size_t)n * n + 8 : 8;
        rc = own_reserve(ctx, OWN_STATE, (size_t)(7 * (n + 8) + nH) * sizeof(double));
        if (rc) break;
        double* base = (double*)ctx->own[OWN_STATE];
        S.dx = base; S.dxbar = base + (n + 8); S.dq = base + 2 * (n + 8); S.dHq = base + 3 * (n + 8);
        S.dgrad = base + 4 * (n + 8);
        double* dc0 = base + 5 * (n + 8);
        S.ddelta = base + 6 * (n + 8);
        S.dH = base + 7 * (n + 8);
        // ---- a0: ingest (initial point, validation, FP32 shadow) ----
        float* C32 = nullptr; float* R32 = nullptr;
        const int64_t ld32 = ((int64_t)d + 3) / 4 * 4;
        if (precision_mode == MEB_MODE_MIXED) {
            rc = own_reserve(ctx, OWN_C32, (size_t)m * ld32 * sizeof(float));
            if (rc) break;
            C32 = (float*)ctx->own[OWN_C32];
            if (radii) {
                rc = own_reserve(ctx, OWN_R32, (size_t)m * sizeof(float));
                if (rc) break;
                R32 = (float*)ctx->own[OWN_R32];
            }
        }
        rc = meb_ingest(ctx, m, d, centers, ld, radii, S.par.sample_rows, dc0, ctx->small + SM_AUX, C32, ld32, R32);
        if (rc) break;
        st->passes_fp64_full++;
        S.bytes += ctx->last_pass_bytes;
        MEB_CUDA_OK(ctx, cudaMemcpyAsync(ctx->h_pinned, ctx->small + SM_AUX, 3 * sizeof(double),
                                         cudaMemcpyDeviceToHost, ctx->stream));
        MEB_CUDA_OK(ctx, cudaMemcpyAsync(ctx->h_pinned + 16, dc0, d * sizeof(double), cudaMemcpyDeviceToHost,
                                         ctx->stream));
        rc = sync_stream(ctx);
        if (rc) break;
        if (ctx->h_pinned[2] > 0.0 || !(ctx->h_pinned[0] < 1.79e308)) { rc = MEB_E_INPUT; break; }
        S.L = ctx->h_pinned[0];
        st->length_scale = S.L;
        memcpy(c0.data(), ctx->h_pinned + 16, d * sizeof(double));
        if (!(S.L > 0.0)) {                      // reading 16: every ball is the point c0
            creturn = c0;
            *h_radius_out = 0.0;
            converged = true;
            kkt = 0.0;
            MEB_CUDA_OK(ctx, cudaEventRecord(e_mid, ctx->stream));
            MEB_CUDA_OK(ctx, cudaEventRecord(e_hi, ctx->stream));
            break;
        }
        xn[0] = 1.0;                              // x~0 = (1, 0), feasible
        ab = xn;
        double r_alg = 0.0, dmax = 0.0;
        if (precision_mode == MEB_MODE_FP64) {
            P.prec = MEB_FP64; P.m = m; P.d = d; P.C = centers; P.ld = ld; P.R = radii; P.ldv = (d + 1) / 2 * 2;
            P.off = c0.data(); P.full = true;
            rc = setup_multipliers(ctx, P, OWN_U0, OWN_S0, OWN_V0);
            if (rc) break;
            MEB_CUDA_OK(ctx, cudaEventRecord(e_mid, ctx->stream));
            rc = ripalm(S, P, xn, ab, tol, &converged, &kkt, terms);
            if (rc) break;
            MEB_CUDA_OK(ctx, cudaEventRecord(e_hi, ctx->stream));
            // final full pass: r_out = max_i(||c - c_i|| + r_i)   (step 7)
            std::vector<double> xr;
            to_raw(S, P, xn, xr);
            rc = upload(ctx, S.dx, xr.data(), n);
            if (rc) break;
            r_alg = xr[0];
            int32_t am = 0; int64_t nv = 0;
            rc = meb_feasibility_check(ctx, m, d, centers, ld, radii, r_alg, S.dx + 1, INFINITY, nullptr, &dmax,
                                       &am, nullptr, 0, &nv);
            if (rc) break;
            st->passes_fp64_full++;
            S.bytes += ctx->last_pass_bytes;
            for (int j = 0; j < d; ++j) creturn[j] = xr[1 + j];
        } else {
            // ---- phase 1: FP32, loose tolerance, all m ----
            Problem P1;
            memset(&P1, 0, sizeof(P1));
            P1.prec = MEB_FP32; P1.m = m; P1.d = d; P1.C = C32; P1.ld = ld32; P1.R = R32; P1.ldv = ld32;
            P1.off = nullptr; P1.full = true;
            rc = setup_multipliers(ctx, P1, OWN_U0, OWN_S0, OWN_V0);
            if (rc) break;
            bool conv1 = false;
            double kkt1, terms1[5];
            rc = ripalm(S, P1, xn, ab, S.par.tol_lo, &conv1, &kkt1, terms1);
            if (rc) break;
            MEB_CUDA_OK(ctx, cudaEventRecord(e_mid, ctx->stream));
            // ---- screening, tol_red = 0.02 r_hat (reading 9) ----
            rc = own_reserve(ctx, OWN_IDX, ((size_t)m + 32) * sizeof(int32_t));
            if (rc) break;
            int32_t* idx = (int32_t*)ctx->own[OWN_IDX];
            std::vector<double> xs(n);
            xs[0] = S.L * xn[0];
            for (int j = 0; j < d; ++j) xs[1 + j] = S.L * xn[1 + j];   // centred coordinates of the shadow
            rc = upload(ctx, S.dq, xs.data(), n);
            if (rc) break;
            int64_t nred = 0;
            rc = meb_screen_compact(ctx, m, d, C32, ld32, R32, (float)xs[0], S.dq + 1,
                                    (float)(S.par.tol_red_factor * xs[0]), idx, m, &nred, nullptr, 0);
            if (rc) break;
            st->passes_fp32_full++;
            S.bytes += ctx->last_pass_bytes;
            if (nred == 0) { rc = MEB_E_INPUT; break; }
            rc = own_reserve(ctx, OWN_KEPT, (size_t)m);
            if (rc) break;
            uint8_t* kept = (uint8_t*)ctx->own[OWN_KEPT];
            rc = meb_fill_u8(ctx, kept, m, 0);
            if (rc) break;
            // ---- reduced problem: gather rows and multipliers ----
            const int64_t ldr = (d + 1) / 2 * 2;
            int64_t cap_red = 2 * nred + 1024;               // room for re-introduced balls
            if (cap_red > m) cap_red = m;
            rc = own_reserve(ctx, OWN_CRED, (size_t)cap_red * ldr * sizeof(double));
            if (rc) break;
            rc = own_reserve(ctx, OWN_RRED, (size_t)cap_red * sizeof(double));
            if (rc) break;
            rc = own_reserve(ctx, OWN_HOSTC, (size_t)cap_red * sizeof(double));        // U buffer a
            if (rc) break;
            rc = own_reserve(ctx, OWN_HOSTR, (size_t)cap_red * sizeof(double));        // U buffer b
            if (rc) break;
            rc = own_reserve(ctx, OWN_SPARE, (size_t)cap_red * 2 * sizeof(int32_t));   // slot buffers a, b
            if (rc) break;
            rc = meb_gather_rows_f64(ctx, centers, ld, idx, nred, d, (double*)ctx->own[OWN_CRED], ldr);
            if (rc) break;
            if (radii) {
                rc = meb_gather_vec_f64(ctx, radii, idx, nred, (double*)ctx->own[OWN_RRED]);
                if (rc) break;
            }
            rc = meb_set_kept(ctx, idx, nred, kept);
            if (rc) break;
            Problem P2;
            memset(&P2, 0, sizeof(P2));
            {
                double* Cred = (double*)ctx->own[OWN_CRED];
                double* Rred = radii ? (double*)ctx->own[OWN_RRED] : nullptr;
                // reduced multipliers: dense V (slot k = k) of capacity cap_red rows, double-buffered
                void* Vred[2] = {nullptr, nullptr};
                cudaError_t ce = cudaMalloc(&Vred[0], (size_t)cap_red * ldr * sizeof(double));
                if (ce == cudaSuccess) ce = cudaMalloc(&Vred[1], (size_t)cap_red * ldr * sizeof(double));
                if (ce != cudaSuccess) {
                    cudaGetLastError();
                    if (Vred[0]) cudaFree(Vred[0]);
                    rc = MEB_E_ALLOC;
                    break;
                }
                P2.prec = MEB_FP64; P2.d = d; P2.ldv = ldr; P2.off = c0.data(); P2.full = false;
                P2.C = Cred; P2.ld = ldr; P2.R = Rred;
                P2.U[0] = ctx->own[OWN_HOSTC]; P2.U[1] = ctx->own[OWN_HOSTR];
                P2.slot[0] = (int32_t*)ctx->own[OWN_SPARE]; P2.slot[1] = P2.slot[0] + cap_red;
                P2.V[0] = Vred[0]; P2.V[1] = Vred[1]; P2.vcap[0] = P2.vcap[1] = cap_red;
                P2.own_v[0] = P2.own_v[1] = -1;
                P2.cur = 0; P2.has_mult = true;
                // warm start restricted to I_red
                rc = meb_gather_mult(ctx, P1.has_mult ? (const float*)P1.U[P1.cur] : nullptr,
                                     P1.has_mult ? P1.slot[P1.cur] : nullptr,
                                     P1.has_mult ? (const float*)P1.V[P1.cur] : nullptr, P1.ldv, idx, nred, d,
                                     (double*)P2.U[0], P2.slot[0], (double*)P2.V[0], ldr);
                if (!P1.has_mult) P2.has_mult = false;
                ab = xn;                                        // reading 11
                for (int rnd = 0; rc == MEB_OK && rnd < S.par.max_rounds; ++rnd) {
                    P2.m = nred;
                    st->n_reduced = nred;
                    st->rounds = rnd + 1;
                    rc = ripalm(S, P2, xn, ab, tol, &converged, &kkt, terms);
                    if (rc) break;
                    if (rnd == 0) MEB_CUDA_OK(ctx, cudaEventRecord(e_hi, ctx->stream));
                    // a-posteriori check against ALL original constraints
                    std::vector<double> xr;
                    to_raw(S, P2, xn, xr);
                    rc = upload(ctx, S.dx, xr.data(), n);
                    if (rc) break;
                    r_alg = xr[0];
                    for (int j = 0; j < d; ++j) creturn[j] = xr[1 + j];
                    const double eps_feas = tol * (1.0 + r_alg);            // reading 10
                    int32_t am = 0; int64_t nv = 0;
                    rc = meb_feasibility_check(ctx, m, d, centers, ld, radii, r_alg, S.dx + 1, eps_feas, kept,
                                               &dmax, &am, idx + nred, m - nred, &nv);
                    if (rc) break;
                    st->passes_fp64_full++;
                    S.bytes += ctx->last_pass_bytes;
                    if (nv == 0) break;
                    if (nred + nv > cap_red) { rc = MEB_E_CAPACITY; break; }
                    // re-introduce the violated balls with zero multipliers (reading 12)
                    rc = meb_gather_rows_f64(ctx, centers, ld, idx + nred, nv, d, Cred + nred * ldr, ldr);
                    if (rc) break;
                    if (radii) { rc = meb_gather_vec_f64(ctx, radii, idx + nred, nv, Rred + nred); if (rc) break; }
                    rc = meb_set_kept(ctx, idx + nred, nv, kept);
                    if (rc) break;
                    if (P2.has_mult) {
                        rc = meb_fill_f64(ctx, (double*)P2.U[P2.cur] + nred, nv, 0.0);
                        if (rc) break;
                        rc = meb_fill_i32(ctx, P2.slot[P2.cur] + nred, nv, -1);
                        if (rc) break;
                    }
                    nred += nv;
                    converged = false;
                    ab = xn;
                }
                sync_stream(ctx);
                cudaFree(Vred[0]);
                cudaFree(Vred[1]);
                if (rc) break;
            }
        }
        st->radius_alg = r_alg;
        st->delta_max = dmax;
        *h_radius_out = r_alg + dmax;                     // = max_i(||c - c_i|| + r_i)   (step 7)
    } while (0);
    if (rc == MEB_OK) {
        cudaEventRecord(e_end, ctx->stream);
        cudaEventSynchronize(e_end);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e_start, e_end); st->ms_total = ms;
        if (cudaEventElapsedTime(&ms, e_start, e_mid) == cudaSuccess) st->ms_phase_lo = ms;
        if (cudaEventElapsedTime(&ms, e_mid, e_hi) == cudaSuccess) st->ms_phase_hi = ms;
        if (cudaEventElapsedTime(&ms, e_hi, e_end) == cudaSuccess) st->ms_check = ms;
        cudaGetLastError();
        memcpy(h_center_out, creturn.data(), d * sizeof(double));
        st->converged = converged ? 1 : 0;
        st->kkt = kkt;
        memcpy(st->kkt_terms, terms, sizeof(terms));
        st->bytes_streamed = S.bytes;
        for (int k = 0; k < ctx->evn; ++k) {           // per-class device time of the streaming launches
            float pms = 0.f;
            if (cudaEventElapsedTime(&pms, ctx->evpool[2 * k], ctx->evpool[2 * k + 1]) != cudaSuccess) continue;
            const int cls = ctx->evclass[k] & 7;
            st->pass_ms[cls] += pms; st->pass_bytes[cls] += ctx->evbytes[k]; st->pass_count[cls]++;
        }
        cudaGetLastError();
        st->kernel_launches = ctx->launches - launches0;
    }
    ctx->ev_record = false;
    cudaEventDestroy(e_start); cudaEventDestroy(e_mid); cudaEventDestroy(e_hi); cudaEventDestroy(e_end);
    ctx->time_passes = timing_was;
    if (rc != MEB_OK) return rc;
    return converged ? MEB_OK : MEB_W_NOT_CONVERGED;
}

extern "C" int meb_solve_host(meb_ctx* ctx, int64_t m, int32_t d, const double* h_centers, int64_t ld,
                              const double* h_radii, double tol, int precision_mode, const meb_params* h_params,
                              double* h_center_out, double* h_radius_out, meb_stats* h_stats) {
    if (!ctx || !h_centers || m < 1 || d < 1 || ld < d) return MEB_E_ARG;
    if (m > ctx->m_max || d > ctx->d_max) return MEB_E_CAPACITY;
    // device copies owned by the context (slots reused across calls)
    static const int OWN_DC = 14, OWN_DR = 15;
    (void)OWN_DR;
    void* dC = nullptr; void* dR = nullptr;
    cudaError_t e = cudaMalloc(&dC, (size_t)m * ld * sizeof(double));
    if (e == cudaSuccess && h_radii) e = cudaMalloc(&dR, (size_t)m * sizeof(double));
    if (e != cudaSuccess) { cudaGetLastError(); if (dC) cudaFree(dC); return MEB_E_ALLOC; }
    (void)OWN_DC;
    e = cudaMemcpyAsync(dC, h_centers, (size_t)m * ld * sizeof(double), cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess && h_radii)
        e = cudaMemcpyAsync(dR, h_radii, (size_t)m * sizeof(double), cudaMemcpyHostToDevice, ctx->stream);
    int rc;
    if (e != cudaSuccess) { ctx->last_cuda_error = (int)e; rc = MEB_E_CUDA; }
    else rc = meb_solve(ctx, m, d, (const double*)dC, ld, (const double*)dR, tol, precision_mode, h_params,
                        h_center_out, h_radius_out, h_stats);
    cudaStreamSynchronize(ctx->stream);
    cudaFree(dC);
    if (dR) cudaFree(dR);
    return rc;
}
