// meb_solve: Algorithm 1, Algorithm 2 and the mixed-precision reduction
// loop of Section 4.2, sequencing the kernels of this library.
//
// Units (reading 3): the (d+1)-sized state x~ = (r/L, (c - c0)/L), (alpha, beta), sigma, tau live in
// normalised units; the kernels run on the RAW data with x_raw = (L r~, off + L c~),
// sigma_raw = sigma/L, tau_eff = tau/L^2.  Then the multipliers and g are unchanged,
// psi~ = psi_raw/L and H~ = L H_raw, so no scaled copy of C is ever made.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <vector>

#include "meb_internal.cuh"
#include "meb_ctrl.cuh"

#define SM_EV 0
#define SM_AUX 16
#define SM_X 32

namespace {

// slots of meb_ctx::own (20 = the batch solver's block, meb_smallsolve.cu)
enum { OWN_U0 = 0, OWN_U1, OWN_S0, OWN_S1, OWN_V0, OWN_V1, OWN_C32, OWN_R32, OWN_IDX, OWN_CRED, OWN_RRED,
       OWN_KEPT, OWN_STATE, OWN_UREDA, OWN_UREDB, OWN_SREDA, OWN_VRED0, OWN_VRED1, OWN_DEVC, OWN_DEVR,
       OWN_BATCH_RESERVED, OWN_SREDB, OWN_WC, OWN_VL0, OWN_VL1, OWN_VLRED0, OWN_VLRED1 };

int own_reserve(meb_ctx* ctx, int slot, size_t bytes) {
    if (ctx->own_bytes[slot] >= bytes && ctx->own[slot]) return MEB_OK;
    if (ctx->own[slot]) { cudaFree(ctx->own[slot]); ctx->own[slot] = nullptr; ctx->own_bytes[slot] = 0; }
    const size_t want = bytes < 256 ? 256 : bytes;
    cudaError_t e = cudaMalloc(&ctx->own[slot], want);
    if (e != cudaSuccess) { cudaGetLastError(); ctx->last_cuda_error = (int)e; return MEB_E_ALLOC; }
    ctx->own_bytes[slot] = want;
    return MEB_OK;
}

// Grow own[slot] to at least `bytes`, keeping its first `keep` bytes (the reduced problem when violated balls are
// re-introduced).  The stream is drained before the old block is freed.
int own_grow_keep(meb_ctx* ctx, int slot, size_t bytes, size_t keep) {
    if (ctx->own_bytes[slot] >= bytes && ctx->own[slot]) return MEB_OK;
    void* fresh = nullptr;
    cudaError_t e = cudaMalloc(&fresh, bytes < 256 ? 256 : bytes);
    if (e != cudaSuccess) { cudaGetLastError(); ctx->last_cuda_error = (int)e; return MEB_E_ALLOC; }
    if (ctx->own[slot] && keep > 0) {
        const size_t n = keep < ctx->own_bytes[slot] ? keep : ctx->own_bytes[slot];
        e = cudaMemcpyAsync(fresh, ctx->own[slot], n, cudaMemcpyDeviceToDevice, ctx->stream);
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    if (e != cudaSuccess) { cudaFree(fresh); ctx->last_cuda_error = (int)e; return MEB_E_CUDA; }
    if (ctx->own[slot]) cudaFree(ctx->own[slot]);
    ctx->own[slot] = fresh;
    ctx->own_bytes[slot] = bytes < 256 ? 256 : bytes;
    return MEB_OK;
}

struct Problem {                   // one ripALM run: data + double-buffered multipliers
    int prec; int64_t m; int32_t d;
    const void* C; int64_t ld; const void* R;
    void* U[2]; int32_t* slot[2]; void* V[2]; int64_t ldv; int64_t vcap[2];
    int own_v[2];                  // own[] slots holding the V pools (-1: fixed capacity)
    int32_t* vlist[2]; int32_t* vcount[2];   // long rows: ascending list of the balls with a multiplier row, per buffer
    int cur; bool has_mult;
    const double* off;             // host: raw offset of the centre (c0 for raw data, nullptr for the centred shadow)
    bool full;                     // streams all m rows (for the pass statistics)
};

struct Solver {
    meb_ctx* ctx; meb_params par; meb_stats* st;
    double sigma_start;            // sigma_0 of the next phase (normalised units)
    double sigma_end;              // sigma reached by the last phase
    bool screen_arm;               // the phase about to run fuses the screening into its evaluation passes
    bool screen_valid;             // ... and its last pass ran at the iterate it returned
    int32_t d; double L;
    double* dH;                    // device (d+1)^2: dense Newton system
    double* dW; int64_t wc_cap;    // device [wc_cap][dpad] gathered active rows of the matrix-free Newton solve, then
    double* rho_c;                 //   [wc_cap] their rho, then the grid barrier's two counters
    unsigned int* cg_bar;
    SolverVecs v;                  // device (d+1)-vectors of the controller
    double bytes;
};

size_t esz(int prec) { return prec == MEB_FP64 ? 8 : 4; }

int sync_stream(meb_ctx* ctx) { MEB_CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream)); return MEB_OK; }

// x_raw = (L r~, off + L c~)
void to_raw(const Solver& S, const Problem& P, const std::vector<double>& xn, std::vector<double>& xr) {
    xr.resize(S.d + 1);
    xr[0] = S.L * xn[0];
    for (int j = 0; j < S.d; ++j) xr[1 + j] = (P.off ? P.off[j] : 0.0) + S.L * xn[1 + j];
}

int upload(meb_ctx* ctx, double* dst, const double* src, size_t n) {
    // staged through a ring of 8 pinned slots so that the copy is truly asynchronous and ordered on the stream
    // without draining it: a slot is reused only after the copy that last read it has run (its event)
    const int64_t dpad = (ctx->h_pinned_len - 256) / 12;
    const int slot = ctx->stage_next;
    ctx->stage_next = (slot + 1) & 7;
    MEB_CUDA_OK(ctx, cudaEventSynchronize(ctx->ev_stage[slot]));
    double* stage = ctx->h_pinned + 4 * dpad + 256 + (int64_t)slot * dpad;
    memcpy(stage, src, n * sizeof(double));
    MEB_CUDA_OK(ctx, cudaMemcpyAsync(dst, stage, n * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
    MEB_CUDA_OK(ctx, cudaEventRecord(ctx->ev_stage[slot], ctx->stream));
    return MEB_OK;
}

// ---- the solve graph of one phase ------------------------------------------------------------------
// WHILE (!done) { evaluation at the trial point + controller;  IF (Newton) { active list, dense H +
// LDL^T  |  CG: WHILE { H p; CG step } ; first Armijo trial };  IF (update) { active list, (U,V) <- (U+,V+),
// outer-iteration bookkeeping } }.  Everything the kernels need that changes between iterations is
// read from device memory (SolverDev / MebDyn), so the instantiated graph is launched once per phase.
struct GraphKey {
    int prec, dense; int64_t m; int32_t d; const void* C; int64_t ld; const void* R;
    void* U[2]; int32_t* slot[2]; void* V[2]; int64_t ldv; int64_t vcap[2];
    const double* dH; const double* xn;
    const int32_t* vlist[2]; int multi, ag;
    const double* dW; int64_t wc_cap;
};
struct SolveGraph {
    bool used; GraphKey key; cudaGraph_t g; cudaGraphExec_t ex;
    cudaGraphConditionalHandle h_while, h_newton, h_update, h_cg, h_cgp;
    int k_eval, k_newton, k_cg, k_update;      // kernels launched per evaluation / Newton solve / CG step / update
    double bytes_per_eval; uint64_t stamp;
};
constexpr int MAX_GRAPHS = 8;
struct GraphCache { SolveGraph e[MAX_GRAPHS]; uint64_t clock; };

}  // namespace

size_t meb_solver_dev_size() { return sizeof(SolverDev); }

void meb_free_graph_cache(meb_ctx* ctx) {
    GraphCache* gc = (GraphCache*)ctx->graph_cache;
    if (!gc) return;
    for (int i = 0; i < MAX_GRAPHS; ++i)
        if (gc->e[i].used) { cudaGraphExecDestroy(gc->e[i].ex); cudaGraphDestroy(gc->e[i].g); }
    free(gc);
    ctx->graph_cache = nullptr;
}

namespace {

GraphCache* cache_of(meb_ctx* ctx) {
    if (!ctx->graph_cache) ctx->graph_cache = calloc(1, sizeof(GraphCache));
    return (GraphCache*)ctx->graph_cache;
}

int add_conditional(meb_ctx* ctx, cudaGraph_t parent, cudaGraphConditionalHandle h, bool is_while,
                    cudaGraphNode_t* node, cudaGraph_t* body) {
    // inside a stream capture into `parent`: append a conditional node after what was captured so far
    cudaStreamCaptureStatus status;
    cudaGraph_t cg = nullptr;
    const cudaGraphNode_t* deps = nullptr;
    size_t ndeps = 0;
    MEB_CUDA_OK(ctx, cudaStreamGetCaptureInfo(ctx->stream, &status, nullptr, &cg, &deps, &ndeps));
    if (status != cudaStreamCaptureStatusActive || cg != parent) return MEB_E_CUDA;
    cudaGraphNodeParams p = {};
    p.type = cudaGraphNodeTypeConditional;
    p.conditional.handle = h;
    p.conditional.type = is_while ? cudaGraphCondTypeWhile : cudaGraphCondTypeIf;
    p.conditional.size = 1;
    MEB_CUDA_OK(ctx, cudaGraphAddNode(node, parent, deps, ndeps, &p));
    *body = p.conditional.phGraph_out[0];
    MEB_CUDA_OK(ctx, cudaStreamUpdateCaptureDependencies(ctx->stream, node, 1, cudaStreamSetCaptureDependencies));
    return MEB_OK;
}

// predictions per Armijo trial pass (meb_params.armijo_multi; -1: on for long rows only)
int multi_of(const meb_params& par, const Problem& P) {
    int n = par.armijo_multi;
    if (n < 0) n = ((size_t)P.ld * esz(P.prec) > 1024 || P.d > 256) ? MEB_MULTI_MAX : 0;
    return n > MEB_MULTI_MAX ? MEB_MULTI_MAX : n;
}

// ---- launch sequences shared by the captured graph and the stepped (host-sequenced) driver ----------
struct Seq {
    Solver* S; const Problem* P; bool dense;
    GraphSide gs; EvalCall c; SolverDev* dev;
};

void seq_init(Seq& q, Solver& S, const Problem& P, bool dense) {
    meb_ctx* ctx = S.ctx;
    q.S = &S; q.P = &P; q.dense = dense;
    q.dev = (SolverDev*)ctx->sdev;
    memset(&q.gs, 0, sizeof(q.gs));
    q.gs.dyn = &q.dev->dyn; q.gs.S = q.dev; q.gs.v = &S.v;
    for (int b = 0; b < 2; ++b) {
        q.gs.U2[b] = P.U[b]; q.gs.slot2[b] = P.slot[b]; q.gs.V2[b] = P.V[b]; q.gs.vcap2[b] = P.vcap[b];
        q.gs.vlist2[b] = P.vlist[b]; q.gs.vcount2[b] = P.vcount[b];
    }
    q.gs.multi = multi_of(S.par, P);
    memset(&q.c, 0, sizeof(q.c));
    q.c.prec = P.prec; q.c.m = P.m; q.c.d = P.d; q.c.C = P.C; q.c.ld = P.ld; q.c.R = P.R; q.c.ldv = P.ldv;
    q.c.x = S.v.x_raw; q.c.xbar = S.v.xbar_raw; q.c.sigma = 1.0; q.c.tau = 1.0; q.c.gs = &q.gs;
}

// evaluation at the trial point + controller step (Alg. 2 lines 3-7, 9)
int seq_eval(Seq& q) {
    meb_ctx* ctx = q.S->ctx;
    const Problem& P = *q.P;
    ctx->cur_class = !P.full ? MEB_PASS_EVAL_REDUCED : (P.prec == MEB_FP64 ? MEB_PASS_EVAL_FP64 : MEB_PASS_EVAL_FP32);
    return meb_eval_internal(ctx, q.c, q.S->v.ev_t, q.S->v.grad_t, nullptr, nullptr);
}
// Newton direction, dense path (Alg. 2 line 8): active list, H, LDL^T
int seq_newton_dense(Seq& q) {
    meb_ctx* ctx = q.S->ctx;
    int rc = meb_ensure_list(ctx, q.P->m);
    if (rc) return rc;
    rc = meb_dense_from_records(ctx, q.c, q.S->v.ev, q.S->dH);
    if (rc) return rc;
    return meb_chol_solve(ctx, q.S->dH, q.S->v.g, q.S->d + 1, q.S->L, q.S->v.delta, &q.dev->chol_info, q.dev, &q.S->v);
}
// the whole CG solve in one persistent kernel (at most wc_cap active rows)
int seq_cg_persistent(Seq& q) {
    return meb_launch_cg(q.S->ctx, q.c, q.S->dW, q.S->wc_cap, q.S->rho_c, q.S->cg_bar);
}
// one CG iteration of the matrix-free path: Hp = H p over the active rows, CG step
int seq_cg_body(Seq& q) {
    meb_ctx* ctx = q.S->ctx;
    int rc = meb_hvp_from_records(ctx, q.c, q.S->v.ev, q.S->v.p, q.S->v.Hp);
    if (rc) return rc;
    return meb_ctrl_cg_step(ctx, q.dev, q.S->v);
}
// multiplier update (eq. (6)) and the bookkeeping of Algorithm 1 lines 3-4
int seq_update(Seq& q) {
    meb_ctx* ctx = q.S->ctx;
    const Problem& P = *q.P;
    int rc = meb_ensure_list(ctx, P.m);
    if (rc) return rc;
    rc = meb_reset_next(ctx, P.prec, &q.dev->dyn, P.U[0], P.U[1], P.slot[0], P.slot[1], P.m);
    if (rc) return rc;
    ActiveArgs a;
    memset(&a, 0, sizeof(a));
    a.C = q.c.C; a.ld = q.c.ld; a.ldv = q.c.ldv; a.x = q.c.x; a.d = q.c.d; a.dpad = (q.c.d + 7) / 8 * 8; a.sigma = 1.0;
    a.list = ctx->list; a.count = ctx->count_dev;
    a.rec_lam = ctx->rec_lam; a.rec_rho = ctx->rec_rho; a.rec_t = ctx->rec_t;
    a.part_vec = ctx->part_vec; a.part_sc = ctx->part_sc; a.ldv_out = P.ldv;
    a.dyn = q.gs.dyn;
    for (int b = 0; b < 2; ++b) { a.U2[b] = q.gs.U2[b]; a.slot2[b] = q.gs.slot2[b]; a.V2[b] = q.gs.V2[b]; a.vcap2[b] = q.gs.vcap2[b]; }
    int nvec = 0;
    rc = meb_launch_active(ctx, MODE_WRITEV, P.prec, a, &nvec);
    if (rc) return rc;
    if (P.vlist[0]) {                 // long rows: the balls that just got a multiplier row, for the next evaluations
        rc = meb_copy_vlist(ctx, ctx->list, ctx->count_dev, q.gs.dyn, P.vlist[0], P.vlist[1], P.vcount[0], P.vcount[1], P.m);
        if (rc) return rc;
    }
    return meb_ctrl_after_update(ctx, q.dev, q.S->v, ctx->count_dev);
}

#define RC(expr) do { rc = (expr); if (rc != MEB_OK) goto fail; } while (0)
#define CU(expr) do { cudaError_t e__ = (expr); if (e__ != cudaSuccess) { ctx->last_cuda_error = (int)e__; meb_debug_cuda(ctx, __FILE__, __LINE__, (int)e__); rc = MEB_E_CUDA; goto fail; } } while (0)

int build_graph(Solver& S, const Problem& P, bool dense, SolveGraph* G) {
    meb_ctx* ctx = S.ctx;
    int rc = MEB_OK;
    bool capturing = false;
    cudaGraph_t tmp = nullptr, body = nullptr, bn = nullptr, bu = nullptr, bcg = nullptr, bcgp = nullptr;
    cudaGraphNode_t wnode, nnode, unode, cgnode, cgpnode;
    Seq q;
    seq_init(q, S, P, dense);
    bool list_after_eval = false;
    int64_t l0;
    cudaStream_t user_stream = ctx->stream;
    ctx->stream = ctx->cap_stream;                 // launches below are CAPTURED on the private stream

    CU(cudaGraphCreate(&G->g, 0));
    CU(cudaGraphConditionalHandleCreate(&G->h_while, G->g, 1, cudaGraphCondAssignDefault));
    CU(cudaGraphConditionalHandleCreate(&G->h_newton, G->g, 0, cudaGraphCondAssignDefault));
    CU(cudaGraphConditionalHandleCreate(&G->h_update, G->g, 0, cudaGraphCondAssignDefault));
    if (!dense) CU(cudaGraphConditionalHandleCreate(&G->h_cg, G->g, 0, cudaGraphCondAssignDefault));
    if (!dense) CU(cudaGraphConditionalHandleCreate(&G->h_cgp, G->g, 0, cudaGraphCondAssignDefault));
    {
        cudaGraphNodeParams p = {};
        p.type = cudaGraphNodeTypeConditional;
        p.conditional.handle = G->h_while;
        p.conditional.type = cudaGraphCondTypeWhile;
        p.conditional.size = 1;
        CU(cudaGraphAddNode(&wnode, G->g, nullptr, 0, &p));
        body = p.conditional.phGraph_out[0];
    }
    // ---- loop body: evaluation + controller, then the two conditional branches ----
    CU(cudaStreamBeginCaptureToGraph(ctx->stream, body, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed));
    capturing = true;
    l0 = ctx->launches;
    RC(seq_eval(q));
    G->k_eval = (int)(ctx->launches - l0);
    G->bytes_per_eval = ctx->last_pass_bytes;
    list_after_eval = ctx->list_valid;
    RC(add_conditional(ctx, body, G->h_newton, false, &nnode, &bn));
    RC(add_conditional(ctx, body, G->h_update, false, &unode, &bu));
    CU(cudaStreamEndCapture(ctx->stream, &tmp));
    capturing = false;
    // ---- Newton branch (Alg. 2 line 8) ----
    CU(cudaStreamBeginCaptureToGraph(ctx->stream, bn, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed));
    capturing = true;
    l0 = ctx->launches;
    ctx->list_valid = list_after_eval;
    if (dense) {
        RC(seq_newton_dense(q));
        G->k_cg = 0;
    } else {
        RC(meb_ensure_list(ctx, P.m));
        RC(add_conditional(ctx, bn, G->h_cgp, false, &cgpnode, &bcgp));
        RC(add_conditional(ctx, bn, G->h_cg, true, &cgnode, &bcg));
        RC(meb_ctrl_after_newton(ctx, q.dev, S.v));
    }
    G->k_newton = (int)(ctx->launches - l0);
    CU(cudaStreamEndCapture(ctx->stream, &tmp));
    capturing = false;
    if (!dense) {
        CU(cudaStreamBeginCaptureToGraph(ctx->stream, bcgp, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed));
        capturing = true;
        l0 = ctx->launches;
        ctx->list_valid = true;
        RC(seq_cg_persistent(q));
        G->k_newton += (int)(ctx->launches - l0);          // (counted with every Newton step; the legacy loop is rare)
        CU(cudaStreamEndCapture(ctx->stream, &tmp));
        capturing = false;
    }
    if (!dense) {
        CU(cudaStreamBeginCaptureToGraph(ctx->stream, bcg, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed));
        capturing = true;
        l0 = ctx->launches;
        ctx->list_valid = true;
        RC(seq_cg_body(q));
        G->k_cg = (int)(ctx->launches - l0);
        CU(cudaStreamEndCapture(ctx->stream, &tmp));
        capturing = false;
    }
    // ---- multiplier update branch (eq. (6), Alg. 1 lines 3-4) ----
    CU(cudaStreamBeginCaptureToGraph(ctx->stream, bu, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed));
    capturing = true;
    l0 = ctx->launches;
    ctx->list_valid = list_after_eval;
    RC(seq_update(q));
    G->k_update = (int)(ctx->launches - l0);
    CU(cudaStreamEndCapture(ctx->stream, &tmp));
    capturing = false;
    ctx->list_valid = false;
    CU(cudaGraphInstantiate(&G->ex, G->g, 0));
    ctx->stream = user_stream;
    return MEB_OK;
fail:
    if (capturing) { cudaStreamEndCapture(ctx->stream, &tmp); }
    ctx->stream = user_stream;
    cudaGetLastError();
    if (G->g) { cudaGraphDestroy(G->g); G->g = nullptr; }
    ctx->list_valid = false;
    return rc;
}
#undef RC
#undef CU

// Stepped driver (environment variable MEB_NO_GRAPH=1): the SAME kernels and controller steps, but
// sequenced by the host, which reads the controller's decision after every evaluation.  It exists so
// that profilers, which do not see inside conditional graph nodes, can list every launch of a solve.
int run_stepped(Solver& S, const Problem& P, bool dense, SolverDev* h) {
    meb_ctx* ctx = S.ctx;
    Seq q;
    seq_init(q, S, P, dense);
    SolverDev* dev = q.dev;
    int cut_seen = h->aborted;
    for (;;) {
        ctx->ev_extra_bytes = h->dyn.has_mult ? (double)h->n_support * (double)P.d * (double)esz(P.prec) : 0.0;
        int rc = seq_eval(q);
        if (rc) return rc;
        MEB_CUDA_OK(ctx, cudaMemcpyAsync(h, dev, sizeof(*h), cudaMemcpyDeviceToHost, ctx->stream));
        MEB_CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
        if (h->aborted > cut_seen && ctx->evn > 0) ctx->evcut[ctx->evn - 1] = true;   // the pass just timed was cut short
        cut_seen = h->aborted;
#ifdef MEB_TUNING
        if (getenv("MEB_TRACE") && atoi(getenv("MEB_TRACE")) >= 2) {
            double ev[MEB_EVAL_NSCALARS];
            cudaMemcpy(ev, S.v.ev_t, sizeof(ev), cudaMemcpyDeviceToHost);
            fprintf(stderr, "[meb trace]   eval %d outer %d inner %d -> action %d phase %d eta %.3g ls %d psi_t %.15g psi_cur %.15g slope %.3e kkt %.3e nact %.0f\n",
                    h->evals, h->outer, h->inner, h->action, h->phase, h->eta, h->ls, ev[MEB_EV_PSI] / h->L, h->psi_cur, h->slope, h->kkt,
                    ev[MEB_EV_N_ACTIVE]);
            if (atoi(getenv("MEB_TRACE")) >= 3) {      // per-CTA device times of the pass (globaltimer stamps)
                static double hp[2048 * MEB_NPART];
                cudaMemcpy(hp, ctx->part_scalar, sizeof(double) * 148 * MEB_NPART, cudaMemcpyDeviceToHost);
                long long t0min = 0x7fffffffffffffffLL, t1max = 0; int slow = -1;
                for (int b = 0; b < 148; ++b) {
                    long long s0, s1; memcpy(&s0, &hp[b * MEB_NPART + 10], 8); memcpy(&s1, &hp[b * MEB_NPART + 11], 8);
                    if (s0 < t0min) t0min = s0;
                    if (s1 > t1max) { t1max = s1; slow = b; }
                }
                fprintf(stderr, "[meb trace]     pass %lld ns, last CTA %d; CTA durations:", t1max - t0min, slow);
                for (int b = 0; b < 148; ++b) { long long s0, s1; memcpy(&s0, &hp[b * MEB_NPART + 10], 8); memcpy(&s1, &hp[b * MEB_NPART + 11], 8); fprintf(stderr, " %lld", s1 - s0); }
                fprintf(stderr, "\n");
            }
        }
#endif
        if (h->done) return MEB_OK;
        if (h->action == ACT_NEWTON) {
            if (dense) {
                rc = seq_newton_dense(q);
                if (rc) return rc;
            } else {
                rc = meb_ensure_list(ctx, P.m);
                if (rc) return rc;
                int go = h->cg_go;
                if (go && h->cg_mode == 1) {
                    rc = seq_cg_persistent(q);
                    if (rc) return rc;
                    go = 0;
                }
                while (go) {
                    rc = seq_cg_body(q);
                    if (rc) return rc;
                    MEB_CUDA_OK(ctx, cudaMemcpyAsync(&h->cg_go, &dev->cg_go, sizeof(int32_t), cudaMemcpyDeviceToHost,
                                                     ctx->stream));
                    MEB_CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
                    go = h->cg_go;
                }
                rc = meb_ctrl_after_newton(ctx, dev, S.v);
                if (rc) return rc;
            }
        } else if (h->action == ACT_UPDATE) {
#ifdef MEB_TUNING
            if (getenv("MEB_TRACE")) {
                double ev[MEB_EVAL_NSCALARS];
                cudaMemcpy(ev, S.v.ev, sizeof(ev), cudaMemcpyDeviceToHost);
                fprintf(stderr, "[meb trace] outer %d sigma %.3g inner %d evals %d kkt %.3e terms %.2e %.2e %.2e %.2e %.2e nB1 %.0f nB3 %.0f psi %.12g\n",
                        h->outer, h->sigma, h->inner, h->evals, h->kkt, h->terms[0], h->terms[1], h->terms[2], h->terms[3],
                        h->terms[4], ev[MEB_EV_N_B1], ev[MEB_EV_N_B3], h->psi_cur);
            }
#endif
            rc = seq_update(q);
            if (rc) return rc;
            MEB_CUDA_OK(ctx, cudaMemcpyAsync(h, dev, sizeof(*h), cudaMemcpyDeviceToHost, ctx->stream));
            MEB_CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
            if (h->done) return MEB_OK;
        }
    }
}

GraphKey make_key(const Solver& S, const Problem& P, bool dense) {
    GraphKey k;
    memset(&k, 0, sizeof(k));
    k.prec = P.prec; k.dense = dense ? 1 : 0; k.m = P.m; k.d = P.d; k.C = P.C; k.ld = P.ld; k.R = P.R;
    for (int b = 0; b < 2; ++b) { k.U[b] = P.U[b]; k.slot[b] = P.slot[b]; k.V[b] = P.V[b]; k.vcap[b] = P.vcap[b]; }
    k.ldv = P.ldv; k.dH = S.dH; k.xn = S.v.xn;
    k.vlist[0] = P.vlist[0]; k.vlist[1] = P.vlist[1];
    k.multi = S.par.armijo_multi; k.ag = S.par.ag_outer;
    k.dW = S.dW; k.wc_cap = S.wc_cap;
    return k;
}

int get_graph(Solver& S, const Problem& P, bool dense, SolveGraph** out) {
    GraphCache* gc = cache_of(S.ctx);
    if (!gc) return MEB_E_ALLOC;
    const GraphKey key = make_key(S, P, dense);
    int victim = 0;
    for (int i = 0; i < MAX_GRAPHS; ++i) {
        if (gc->e[i].used && memcmp(&gc->e[i].key, &key, sizeof(key)) == 0) {
            gc->e[i].stamp = ++gc->clock;
            *out = &gc->e[i];
            return MEB_OK;
        }
        if (!gc->e[i].used) victim = i;
    }
    if (gc->e[victim].used)
        for (int i = 0; i < MAX_GRAPHS; ++i)
            if (gc->e[i].stamp < gc->e[victim].stamp) victim = i;
    SolveGraph* G = &gc->e[victim];
    if (G->used) { cudaGraphExecDestroy(G->ex); cudaGraphDestroy(G->g); }
    memset(G, 0, sizeof(*G));
    int rc = build_graph(S, P, dense, G);
    if (rc != MEB_OK) return rc;
    G->used = true; G->key = key; G->stamp = ++gc->clock;
    *out = G;
    return MEB_OK;
}

// Grow the V pool of buffer b to at least `rows` rows (keeps nothing: only called for the buffer that
// is about to be overwritten, or before any multiplier exists).
int grow_pool(meb_ctx* ctx, Problem& P, int b, int64_t rows) {
    if (P.own_v[b] < 0) return MEB_E_CAPACITY;
    int rc = own_reserve(ctx, P.own_v[b], (size_t)rows * P.ldv * esz(P.prec));
    if (rc) return rc;
    P.V[b] = ctx->own[P.own_v[b]];
    P.vcap[b] = (int64_t)(ctx->own_bytes[P.own_v[b]] / ((size_t)P.ldv * esz(P.prec)));
    return MEB_OK;
}

// Algorithm 1 with Algorithm 2 inside, device-resident: one graph launch per phase (plus one relaunch
// whenever a V pool has to grow).  xn / ab are the normalised x and (alpha, beta), in/out (host).
int ripalm(Solver& S, Problem& P, std::vector<double>& xn, std::vector<double>& ab, double tol, double tol_accept,
           bool* converged, double* kkt_out, double terms_out[5], int outer_cap) {
    meb_ctx* ctx = S.ctx;
    const meb_params& par = S.par;
    const int n = S.d + 1;
    SolverDev* dev = (SolverDev*)ctx->sdev;
    SolverDev* h = (SolverDev*)ctx->h_sdev;
    const bool dense = S.d <= par.dense_d_max && S.d <= 128;
    *converged = false;
    // V pools: start small, grow on demand (ST_NEED_CAPACITY)
    for (int b = 0; b < 2; ++b)
        if (P.own_v[b] >= 0 && P.vcap[b] < 1024) {
            int rc = grow_pool(ctx, P, b, P.m < 4096 ? P.m : 4096);
            if (rc) return rc;
        }
    int rc = upload(ctx, S.v.xn, xn.data(), n);
    if (rc) return rc;
    {   // (alpha, beta) and the raw offset share one staged upload each
        rc = upload(ctx, S.v.ab, ab.data(), n);
        if (rc) return rc;
        if (P.off) { rc = upload(ctx, S.v.off, P.off, S.d); if (rc) return rc; }
    }
    bool first = true;
    // a sharded solve is host-stepped (the all-gather between the two levels of every reduction is the caller's
    // collective) and keeps full-size V pools, so that no rank ever stops for capacity on its own
    bool stepped = ctx->opt[MEB_OPT_STEPPED] != 0 || ctx->shard != nullptr;
    if (ctx->shard)
        for (int b = 0; b < 2; ++b)
            if (P.own_v[b] >= 0 && P.vcap[b] < P.m) { int rcg = grow_pool(ctx, P, b, P.m); if (rcg) return rcg; }
    // small problems (the reduced problem of the mixed mode, small instances): one persistent CTA runs the phase
    bool small = dense && !ctx->opt[MEB_OPT_NO_SMALL] && !ctx->shard && meb_small_applicable(P.prec, P.m, P.d);
    if (small) {
        for (int b = 0; b < 2 && small; ++b)
            if (P.vcap[b] < P.m) { if (P.own_v[b] < 0 || grow_pool(ctx, P, b, P.m) != MEB_OK) small = false; }
    }
    // few balls with long rows (the reduced problem of a high-dimensional instance): one persistent CTA too,
    // matrix-free Newton steps on the gathered rows (meb_wide.cu)
    bool wide = !small && !dense && !ctx->opt[MEB_OPT_NO_SMALL] && !ctx->shard && S.dW != nullptr && S.wc_cap >= P.m &&
                meb_wide_applicable(P.prec, P.m, P.d);
    if (wide) {
        for (int b = 0; b < 2 && wide; ++b)
            if (P.vcap[b] < P.m) { if (P.own_v[b] < 0 || grow_pool(ctx, P, b, P.m) != MEB_OK) wide = false; }
    }
    const bool one_cta = small || wide;
    if (one_cta) stepped = false;
    int64_t stepped_launches = 0;
    (void)stepped_launches;
    SolveGraph stepped_info;
    memset(&stepped_info, 0, sizeof(stepped_info));
    for (int attempt = 0; attempt < 64; ++attempt) {
        SolveGraph* G = &stepped_info;
        if (one_cta) {
            stepped_info.k_eval = 0; stepped_info.k_newton = 0; stepped_info.k_cg = 0; stepped_info.k_update = 0;
            stepped_info.bytes_per_eval = (double)P.m * (P.d * 8.0 + (P.R ? 8 : 0) + 12.0);
        } else if (!stepped) {
            rc = get_graph(S, P, dense, &G);
            if (rc) return rc;
        }
        MEB_CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));          // h is free to be rewritten
        if (first) {
            memset(h, 0, sizeof(*h));
            h->L = S.L; h->tol = tol; h->tol_accept = tol_accept; h->rho = par.rho; h->tau = par.tau; h->kappa = par.kappa;
            h->sigma_max = par.sigma_max; h->armijo_mu = par.armijo_mu;
            h->shrink_min = (par.armijo_shrink_min > 0.0 && par.armijo_shrink_min <= 0.5) ? par.armijo_shrink_min : 0.5;
            h->n = n; h->d = S.d; h->inner_max = par.inner_max; h->outer_max = outer_cap;
            h->armijo_max = par.armijo_max_halvings; h->cg_max = par.cg_max; h->dense = dense ? 1 : 0;
            h->use_off = P.off ? 1 : 0;
            if (P.prec == MEB_FP32) {      // FP32 cannot resolve steps below ~2^-12 or more than a few Newton steps (reading 17)
                if (h->armijo_max > 12) h->armijo_max = 12;
                if (h->inner_max > 20) h->inner_max = 20;
            }
            h->slope_floor = (P.prec == MEB_FP32) ? 1e-7 : 2e-15;
            h->abort_margin = ctx->opt[MEB_OPT_NO_ABORT] ? 0.0 : ((P.prec == MEB_FP32) ? 1e-3 : 1e-6);
            h->pred_margin = (P.prec == MEB_FP32) ? 1e-3 : 1e-6;
            h->m_rows = (ctx->shard && P.full) ? ctx->shard->m_global : P.m;      // (counts in v.ev are global in a sharded solve)
            h->lowprec = (P.prec == MEB_FP32 && P.full) ? 1 : 0;
            h->dyn.screen_on = (S.screen_arm && !one_cta) ? 1 : 0;
            h->dyn.screen_factor = par.tol_red_factor;
            h->multi_max = one_cta ? 0 : multi_of(par, P);
            h->ag_outer = (par.ag_outer > 0 && !one_cta) ? par.ag_outer : 0;
            h->ag_inner_max = 500;
            h->stall_max = (P.prec == MEB_FP32) ? 3 : 6;   // the FP32 run only has to deliver a warm start
#ifdef MEB_TUNING
            if (getenv("MEB_SHRINK_MIN")) h->shrink_min = atof(getenv("MEB_SHRINK_MIN"));
            if (getenv("MEB_STALL_MAX")) h->stall_max = atoi(getenv("MEB_STALL_MAX"));
            if (getenv("MEB_SLOPE_FLOOR")) h->slope_floor = atof(getenv("MEB_SLOPE_FLOOR"));
#endif
            h->eval_cap = 4 * outer_cap * (par.inner_max + 2);
        }
        h->vcap[0] = P.vcap[0]; h->vcap[1] = P.vcap[1];
        h->h_while = G->h_while; h->h_newton = G->h_newton; h->h_update = G->h_update; h->h_cg = G->h_cg;
        h->h_cgp = G->h_cgp; h->wc_cap = ctx->shard ? -1 : S.wc_cap;     // sharded: one exchange per CG iteration
        h->in_graph = (stepped || one_cta) ? 0 : 1;
        if (first) {
            MEB_CUDA_OK(ctx, cudaMemcpyAsync(dev, h, sizeof(*h), cudaMemcpyHostToDevice, ctx->stream));
            rc = meb_ctrl_init(ctx, dev, S.v, S.sigma_start, P.cur, P.has_mult ? 1 : 0);
        } else {                                                        // resume: constants that may have changed
            MEB_CUDA_OK(ctx, cudaMemcpyAsync(&dev->vcap[0], &h->vcap[0], 2 * sizeof(int64_t),
                                             cudaMemcpyHostToDevice, ctx->stream));
            MEB_CUDA_OK(ctx, cudaMemcpyAsync(&dev->h_while, &h->h_while, 5 * sizeof(cudaGraphConditionalHandle),
                                             cudaMemcpyHostToDevice, ctx->stream));
            rc = meb_ctrl_resume(ctx, dev);
        }
        if (rc) return rc;
        first = false;
        if (small) {
            rc = meb_launch_small_solve(ctx, P.C, P.ld, P.R, P.m, P.d, P.ldv, P.U, P.slot, P.V, dev, S.v);
            if (rc) return rc;
        } else if (wide) {
            rc = meb_launch_wide_solve(ctx, P.C, P.ld, P.R, P.m, P.d, P.ldv, P.U, P.slot, P.V, dev, S.v, S.dW);
            if (rc) return rc;
        } else if (stepped) {
            const int64_t l0 = ctx->launches;
            rc = run_stepped(S, P, dense, h);
            if (rc) return rc;
            stepped_info.bytes_per_eval = ctx->last_pass_bytes;
            stepped_launches += ctx->launches - l0;
        } else {
            MEB_CUDA_OK(ctx, cudaGraphLaunch(G->ex, ctx->stream));
        }
        MEB_CUDA_OK(ctx, cudaMemcpyAsync(h, dev, sizeof(*h), cudaMemcpyDeviceToHost, ctx->stream));
        MEB_CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
        // ---- statistics of this launch ----
        const int cls = !P.full ? MEB_PASS_EVAL_REDUCED : (P.prec == MEB_FP64 ? MEB_PASS_EVAL_FP64 : MEB_PASS_EVAL_FP32);
        if (h->status == ST_NEED_CAPACITY) {
            const int nxt = h->dyn.has_mult ? 1 - h->dyn.cur : 0;
            const int64_t want = h->n_support + h->n_support / 2 + 64;
            rc = grow_pool(ctx, P, nxt, want < P.m ? want : P.m);
            if (rc) return rc;
            if (!h->dyn.has_mult) { rc = grow_pool(ctx, P, 1 - nxt, want < P.m ? want : P.m); if (rc) return rc; }
            continue;
        }
        // ---- phase finished ----
#ifdef MEB_TUNING
        if (getenv("MEB_TRACE")) {
            fprintf(stderr, "[meb trace] %d of %d passes cut short; eval passes (ns / active):", h->aborted, h->evals);
            for (int q = 0; q < h->evals && q < 48; ++q) {
                if (h->act_hist[q] == 0xffffffffu) fprintf(stderr, " %u/cut", h->pass_hist[q]);
                else fprintf(stderr, " %u/%u", h->pass_hist[q], h->act_hist[q]);
            }
            fprintf(stderr, "\n");
        }
#endif
        S.st->outer_iters += h->outer;
        S.st->newton_iters += h->newton_total;
        S.st->cg_iters += h->cg_total;
        if (!P.full) S.st->passes_reduced += h->evals;
        else if (P.prec == MEB_FP64) S.st->passes_fp64_full += h->evals;
        else S.st->passes_fp32_full += h->evals;
        const double vbytes = (double)h->vrow_reads * (double)S.d * (double)esz(P.prec);   // V rows of balls with u_i > 0
        S.bytes += (double)(h->evals - h->aborted) * G->bytes_per_eval + vbytes;
        S.st->passes_cut += h->aborted;
        S.screen_valid = h->dyn.screen_on != 0 && h->screen_valid != 0 && h->status != ST_NEED_CAPACITY;
        S.st->trials_skipped += h->skipped;
        S.st->ag_iters += h->ag_total;
        S.st->pass_ms[cls] += (double)h->pass_ns * 1e-6;
        S.st->pass_bytes[cls] += (double)h->pass_count * G->bytes_per_eval + vbytes;
        S.st->pass_count[cls] += (int32_t)h->pass_count;
        if (!stepped && !one_cta)   // kernels launched by the graph: counted from the device-side iteration counters
            ctx->launches += (int64_t)h->evals * G->k_eval + (int64_t)h->newton_total * G->k_newton +
                             (int64_t)h->cg_total * G->k_cg + (int64_t)h->outer * G->k_update;
        S.st->n_support = h->n_support;
        *kkt_out = h->kkt;
        memcpy(terms_out, h->terms, 5 * sizeof(double));
        *converged = h->status == ST_CONVERGED;
        S.sigma_end = h->sigma;
        P.cur = h->dyn.cur;
        P.has_mult = h->dyn.has_mult != 0;
        // final iterate back to the host
        MEB_CUDA_OK(ctx, cudaMemcpyAsync(ctx->h_pinned, S.v.xn, n * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
        MEB_CUDA_OK(ctx, cudaMemcpyAsync(ctx->h_pinned + n, S.v.ab, n * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
        MEB_CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
        xn.assign(ctx->h_pinned, ctx->h_pinned + n);
        ab.assign(ctx->h_pinned + n, ctx->h_pinned + 2 * n);
        return MEB_OK;
    }
    return MEB_E_CAPACITY;
}

bool long_rows(const Problem& P) { return (size_t)P.ld * esz(P.prec) > 1024 || P.d > 256; }

int setup_multipliers(meb_ctx* ctx, Problem& P, int ownU0, int ownS0, int ownV0) {
    for (int b = 0; b < 2; ++b) {
        P.vlist[b] = nullptr; P.vcount[b] = nullptr;
        if (long_rows(P) && ctx->vlist) {
            int rcv = own_reserve(ctx, OWN_VL0 + b, ((size_t)P.m + 32) * sizeof(int32_t));
            if (rcv) return rcv;
            P.vlist[b] = (int32_t*)ctx->own[OWN_VL0 + b];
            P.vcount[b] = ctx->count_dev + 2 + b;
        }
    }
    if (P.vcount[0]) { cudaError_t e = cudaMemsetAsync(ctx->count_dev + 2, 0, 2 * sizeof(int32_t), ctx->stream); if (e != cudaSuccess) { ctx->last_cuda_error = (int)e; return MEB_E_CUDA; } }
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

// sharded solve: (delta_max, argmax, number of violators) of this rank -> maximum over the ranks, its GLOBAL index,
// total number of violators (the local count stays in *nv_local)
int feas_global(meb_ctx* ctx, double* dmax, int32_t* am, int64_t nv_local, int64_t* nv_total) {
    *nv_total = nv_local;
    if (!ctx->shard) return MEB_OK;
    double h3[3] = {*dmax, (double)*am, (double)nv_local};
    int rc = upload(ctx, ctx->small + SM_AUX, h3, 3);
    if (rc) return rc;
    rc = meb_shard_argmax(ctx, ctx->small + SM_AUX);
    if (rc) return rc;
    MEB_CUDA_OK(ctx, cudaMemcpyAsync(ctx->h_pinned, ctx->small + SM_AUX, 3 * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    rc = sync_stream(ctx);
    if (rc) return rc;
    *dmax = ctx->h_pinned[0]; *am = (int32_t)ctx->h_pinned[1]; *nv_total = (int64_t)ctx->h_pinned[2];
    return MEB_OK;
}

// resets the per-solve recording state of the context on every way out of meb_solve
struct SolveScope {
    meb_ctx* ctx; bool timing_was;
    explicit SolveScope(meb_ctx* c) : ctx(c), timing_was(c->time_passes) { c->evn = 0; c->ev_record = true; c->ev_extra_bytes = 0.0; }
    ~SolveScope() { ctx->ev_record = false; ctx->time_passes = timing_was; ctx->ev_extra_bytes = 0.0; }
};

// buffers of the reduced problem: rows, radii, double-buffered multipliers with a dense V (slot k = k)
struct Reduced {
    int64_t cap; int64_t ldr; int32_t d; bool radii; bool longrows;
};
int reduced_reserve(meb_ctx* ctx, Reduced& Q, int64_t cap, int64_t keep_rows) {
    const size_t row = (size_t)Q.ldr * sizeof(double);
    int rc = own_grow_keep(ctx, OWN_CRED, (size_t)cap * row, (size_t)keep_rows * row);
    if (rc == MEB_OK) rc = own_grow_keep(ctx, OWN_RRED, (size_t)cap * sizeof(double), (size_t)keep_rows * sizeof(double));
    if (rc == MEB_OK) rc = own_grow_keep(ctx, OWN_UREDA, (size_t)cap * sizeof(double), (size_t)keep_rows * sizeof(double));
    if (rc == MEB_OK) rc = own_grow_keep(ctx, OWN_UREDB, (size_t)cap * sizeof(double), (size_t)keep_rows * sizeof(double));
    if (rc == MEB_OK) rc = own_grow_keep(ctx, OWN_SREDA, (size_t)cap * sizeof(int32_t), (size_t)keep_rows * sizeof(int32_t));
    if (rc == MEB_OK) rc = own_grow_keep(ctx, OWN_SREDB, (size_t)cap * sizeof(int32_t), (size_t)keep_rows * sizeof(int32_t));
    if (rc == MEB_OK) rc = own_grow_keep(ctx, OWN_VRED0, (size_t)cap * row, (size_t)keep_rows * row);
    if (rc == MEB_OK) rc = own_grow_keep(ctx, OWN_VRED1, (size_t)cap * row, (size_t)keep_rows * row);
    if (rc == MEB_OK && Q.longrows) rc = own_grow_keep(ctx, OWN_VLRED0, ((size_t)cap + 32) * sizeof(int32_t), (size_t)keep_rows * sizeof(int32_t));
    if (rc == MEB_OK && Q.longrows) rc = own_grow_keep(ctx, OWN_VLRED1, ((size_t)cap + 32) * sizeof(int32_t), (size_t)keep_rows * sizeof(int32_t));
    if (rc == MEB_OK) Q.cap = cap;
    return rc;
}
void reduced_bind(meb_ctx* ctx, const Reduced& Q, Problem& P2) {
    P2.C = ctx->own[OWN_CRED]; P2.ld = Q.ldr; P2.R = Q.radii ? ctx->own[OWN_RRED] : nullptr;
    P2.U[0] = ctx->own[OWN_UREDA]; P2.U[1] = ctx->own[OWN_UREDB];
    P2.slot[0] = (int32_t*)ctx->own[OWN_SREDA]; P2.slot[1] = (int32_t*)ctx->own[OWN_SREDB];
    P2.V[0] = ctx->own[OWN_VRED0]; P2.V[1] = ctx->own[OWN_VRED1];
    P2.vcap[0] = P2.vcap[1] = Q.cap;
    P2.own_v[0] = P2.own_v[1] = -1;
    for (int b = 0; b < 2; ++b) {
        P2.vlist[b] = Q.longrows ? (int32_t*)ctx->own[OWN_VLRED0 + b] : nullptr;
        P2.vcount[b] = Q.longrows ? ctx->count_dev + 4 + b : nullptr;
    }
}

int solve_impl(meb_ctx* ctx, int64_t m, int32_t d, const double* centers, int64_t ld,
               const double* radii, double tol, int precision_mode, const meb_params* h_params,
               double* h_center_out, double* h_radius_out, meb_stats* h_stats) {
    if (!ctx || !centers || !h_center_out || !h_radius_out || m < 1 || d < 1 || ld < d) return MEB_E_ARG;
    if (!(tol > 0.0) || (precision_mode != MEB_MODE_FP64 && precision_mode != MEB_MODE_MIXED)) return MEB_E_ARG;
    if (m > ctx->m_max || d > ctx->d_max) return MEB_E_CAPACITY;
    meb_stats local_stats;
    meb_stats* st = h_stats ? h_stats : &local_stats;
    memset(st, 0, sizeof(*st));
    Solver S;
    S.ctx = ctx; S.st = st; S.d = d; S.bytes = 0.0; S.sigma_start = 0.0; S.sigma_end = 0.0;
    S.screen_arm = false; S.screen_valid = false;
    if (h_params) S.par = *h_params; else meb_default_params(&S.par);
    if (!(S.par.rho >= 0.0 && S.par.rho < 1.0) || !(S.par.sigma0 > 0.0) || !(S.par.tau > 0.0) ||
        !(S.par.kappa >= 1.0) || S.par.sample_rows < 1)
        return MEB_E_ARG;
    S.sigma_start = S.par.sigma0;
    const int n = d + 1;
    // The KKT test runs at tol/10: the primal-feasibility term only bounds the error of the returned
    // (feasible) radius by about tol (1 + r)/r, and the contract is a radius within tol (DESIGN reading 7).
    const double tol_kkt = 0.1 * tol;
    SolveScope scope(ctx);
    const int64_t launches0 = ctx->launches;
    cudaEvent_t e_start = ctx->ev_solve[0], e_mid = ctx->ev_solve[1], e_hi = ctx->ev_solve[2], e_end = ctx->ev_solve[3];
    bool have_mid = false, have_hi = false;
    int rc = MEB_OK;
    std::vector<double> c0(d), xn(n, 0.0), ab, creturn(d);
    bool converged = false;
    double kkt = INFINITY, terms[5] = {0, 0, 0, 0, 0};
    Problem P;
    memset(&P, 0, sizeof(P));
#define CUB(expr) { cudaError_t e__ = (expr); if (e__ != cudaSuccess) { ctx->last_cuda_error = (int)e__; meb_debug_cuda(ctx, __FILE__, __LINE__, (int)e__); rc = MEB_E_CUDA; break; } }
    do {
        CUB(cudaEventRecord(e_start, ctx->stream));
        // ---- state vectors on the device ----
        const size_t nH = (d <= 128) ? (size_t)n * n + 8 : 8;
        const size_t nv = ((size_t)n + 7) / 8 * 8;
        rc = own_reserve(ctx, OWN_STATE, (17 * nv + 2 * MEB_EVAL_NSCALARS + nH) * sizeof(double));
        if (rc) break;
        double* base = (double*)ctx->own[OWN_STATE];
        double** vecs[] = {&S.v.xn, &S.v.xbar, &S.v.ab, &S.v.delta, &S.v.g, &S.v.xt, &S.v.x_raw, &S.v.xbar_raw,
                           &S.v.off, &S.v.grad_t, &S.v.res, &S.v.p, &S.v.Hp, &S.v.xbest, &S.v.dir_raw};
        for (size_t i = 0; i < 15; ++i) *vecs[i] = base + i * nv;
        double* dc0 = base + 15 * nv;
        S.v.ev_t = base + 17 * nv;
        S.v.ev = S.v.ev_t + MEB_EVAL_NSCALARS;
        S.dH = S.v.ev + MEB_EVAL_NSCALARS;
        S.dW = nullptr; S.wc_cap = 0; S.rho_c = nullptr; S.cg_bar = nullptr;
        if (d > 128 || d > S.par.dense_d_max) {
            // matrix-free Newton path: room for the gathered active rows (up to 256 MB, L2-sized in practice)
            const size_t dpadw = ((size_t)d + 7) / 8 * 8;
            int64_t cap = (int64_t)(((size_t)256 << 20) / (dpadw * sizeof(double)));
            if (cap > m) cap = m;
            if (cap < 1) cap = 1;
            rc = own_reserve(ctx, OWN_WC, (size_t)cap * (dpadw + 1) * sizeof(double) + 64);
            if (rc) break;
            S.dW = (double*)ctx->own[OWN_WC];
            S.rho_c = S.dW + (size_t)cap * dpadw;
            S.cg_bar = (unsigned int*)(S.rho_c + cap);
            S.wc_cap = cap;
        }
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
        CUB(cudaMemcpyAsync(ctx->h_pinned, ctx->small + SM_AUX, 3 * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
        CUB(cudaMemcpyAsync(ctx->h_pinned + 16, dc0, d * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
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
            CUB(cudaEventRecord(e_mid, ctx->stream)); have_mid = true;
            rc = ripalm(S, P, xn, ab, tol_kkt, tol, &converged, &kkt, terms, S.par.outer_max);
            if (rc) break;
            CUB(cudaEventRecord(e_hi, ctx->stream)); have_hi = true;
            // final full pass: r_out = max_i(||c - c_i|| + r_i)   (step 7)
            std::vector<double> xr;
            to_raw(S, P, xn, xr);
            rc = upload(ctx, S.v.x_raw, xr.data(), n);
            if (rc) break;
            r_alg = xr[0];
            int32_t am = 0; int64_t nvl = 0;
            rc = meb_feasibility_check(ctx, m, d, centers, ld, radii, r_alg, S.v.x_raw + 1, INFINITY, nullptr, &dmax,
                                       &am, nullptr, 0, &nvl);
            if (rc) break;
            { int64_t nvt = 0; rc = feas_global(ctx, &dmax, &am, nvl, &nvt); if (rc) break; }
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
            // long rows (meb_long.cu): the evaluation passes of this run also apply the retain rule of the screening at
            // the point they evaluate, which saves the screening pass (8 GB on config 5) when the run ends at the point
            // of its last pass.  Short rows keep the separate pass: it is 1-2 % of their solve and the extra per-row work
            // in the instruction-bound tile kernel would cost as much.
            S.screen_arm = !ctx->shard && !ctx->opt[MEB_OPT_NO_FUSED_SCREEN] && meb_eval_path(ctx, MEB_FP32, C32, ld32, m, d) == PATH_LONG;
            S.screen_valid = false;
            rc = ripalm(S, P1, xn, ab, S.par.tol_lo, S.par.tol_lo, &conv1, &kkt1, terms1,
                        S.par.outer_max_lo > 0 ? S.par.outer_max_lo : S.par.outer_max);
            if (rc) break;
            CUB(cudaEventRecord(e_mid, ctx->stream)); have_mid = true;
            // ---- screening, tol_red = 0.02 r_hat (reading 9) ----
            rc = own_reserve(ctx, OWN_IDX, ((size_t)m + 32) * sizeof(int32_t));
            if (rc) break;
            int32_t* idx = (int32_t*)ctx->own[OWN_IDX];
            std::vector<double> xs(n);
            xs[0] = S.L * xn[0];
            for (int j = 0; j < d; ++j) xs[1 + j] = S.L * xn[1 + j];   // centred coordinates of the shadow
            rc = upload(ctx, S.v.xt, xs.data(), n);
            if (rc) break;
            int64_t nred = 0;
            S.screen_arm = false;
            if (S.screen_valid) {
                // the last pass of the low-precision run evaluated at (r_hat, c_hat): its mask IS the screening
                rc = meb_compact_mask(ctx, ctx->smask, m, idx, m, &nred);
                if (rc) break;
            } else {
                rc = meb_screen_compact(ctx, m, d, C32, ld32, R32, (float)xs[0], S.v.xt + 1,
                                        (float)(S.par.tol_red_factor * xs[0]), idx, m, &nred, nullptr, 0);
                if (rc) break;
                st->passes_fp32_full++;
                S.bytes += ctx->last_pass_bytes;
            }
            Problem P2;
            memset(&P2, 0, sizeof(P2));
            P2.prec = MEB_FP64; P2.d = d; P2.off = c0.data(); P2.full = false;
            if (nred == 0) {
                // nothing passed the retain rule (a useless coarse ball): keep the farthest ball, as the oracle does
                // (oracle/ripalm.py, P:L281-283 then brings back whatever is violated)
                std::vector<double> xr0;
                to_raw(S, P2, xn, xr0);
                rc = upload(ctx, S.v.x_raw, xr0.data(), n);
                if (rc) break;
                int32_t am0 = 0; int64_t nv0 = 0; double dm0 = 0.0;
                rc = meb_feasibility_check(ctx, m, d, centers, ld, radii, xr0[0], S.v.x_raw + 1, INFINITY, nullptr, &dm0,
                                           &am0, nullptr, 0, &nv0);
                if (rc) break;
                st->passes_fp64_full++;
                S.bytes += ctx->last_pass_bytes;
                rc = meb_fill_i32(ctx, idx, 1, am0);
                if (rc) break;
                nred = 1;
            }
            rc = own_reserve(ctx, OWN_KEPT, (size_t)m);
            if (rc) break;
            uint8_t* kept = (uint8_t*)ctx->own[OWN_KEPT];
            rc = meb_fill_u8(ctx, kept, m, 0);
            if (rc) break;
            // ---- reduced problem: gather rows and multipliers ----
            Reduced Q;
            Q.cap = 0; Q.ldr = (d + 1) / 2 * 2; Q.d = d; Q.radii = radii != nullptr;
            Q.longrows = ((size_t)Q.ldr * 8 > 1024 || d > 256) && ctx->vlist != nullptr;
            {
                int64_t cap_red = 2 * nred + 1024;           // room for re-introduced balls; grows on demand
                if (cap_red > m) cap_red = m;
                rc = reduced_reserve(ctx, Q, cap_red, 0);
                if (rc) break;
            }
            const int64_t ldr = Q.ldr;
            rc = meb_gather_rows_f64(ctx, centers, ld, idx, nred, d, (double*)ctx->own[OWN_CRED], ldr);
            if (rc) break;
            if (radii) {
                rc = meb_gather_vec_f64(ctx, radii, idx, nred, (double*)ctx->own[OWN_RRED]);
                if (rc) break;
            }
            rc = meb_set_kept(ctx, idx, nred, kept);
            if (rc) break;
            P2.ldv = ldr;
            reduced_bind(ctx, Q, P2);
            P2.cur = 0; P2.has_mult = true;
            // warm start restricted to I_red.  If the low-precision run did not reach its
            // tolerance (degenerate supports: reading 17) its multipliers are noise: start from zero.
            if (Q.longrows) CUB(cudaMemsetAsync(ctx->count_dev + 4, 0, 2 * sizeof(int32_t), ctx->stream));
            if (P1.has_mult && conv1) {
                rc = meb_gather_mult(ctx, (const float*)P1.U[P1.cur], P1.slot[P1.cur], (const float*)P1.V[P1.cur],
                                     P1.ldv, idx, nred, d, (double*)P2.U[0], P2.slot[0], (double*)P2.V[0], ldr);
                if (rc == MEB_OK && P2.vlist[0]) rc = meb_build_vlist(ctx, P2.slot[0], nred, P2.vlist[0], P2.vcount[0]);
            } else {
                P2.has_mult = false;
            }
            if (rc) break;
            ab = xn;                                        // reading 11
            S.sigma_start = S.par.sigma0;
            if (P2.has_mult && S.par.sigma_carry > 0.0 && S.par.sigma_carry * S.sigma_end > S.par.sigma0)
                S.sigma_start = S.par.sigma_carry * S.sigma_end;
            for (int rnd = 0; rc == MEB_OK && rnd < S.par.max_rounds; ++rnd) {
                P2.m = nred;
                st->n_reduced = nred;
                st->rounds = rnd + 1;
                rc = ripalm(S, P2, xn, ab, tol_kkt, tol, &converged, &kkt, terms, S.par.outer_max);
                if (rc) break;
                if (rnd == 0) { CUB(cudaEventRecord(e_hi, ctx->stream)); have_hi = true; }
                // a-posteriori check against ALL original constraints
                std::vector<double> xr;
                to_raw(S, P2, xn, xr);
                rc = upload(ctx, S.v.x_raw, xr.data(), n);
                if (rc) break;
                r_alg = xr[0];
                for (int j = 0; j < d; ++j) creturn[j] = xr[1 + j];
                const double eps_feas = tol_kkt * (1.0 + r_alg);        // reading 10
                int32_t am = 0; int64_t nvl = 0;
                rc = meb_feasibility_check(ctx, m, d, centers, ld, radii, r_alg, S.v.x_raw + 1, eps_feas, kept,
                                           &dmax, &am, idx + nred, m - nred, &nvl);
                if (rc) break;
                int64_t nv_total = nvl;                         // sharded: every rank re-adds its own violators, all
                rc = feas_global(ctx, &dmax, &am, nvl, &nv_total);   // ranks stop together when no rank has any
                if (rc) break;
                st->passes_fp64_full++;
                S.bytes += ctx->last_pass_bytes;
                if (nv_total == 0) break;
                if (rnd + 1 == S.par.max_rounds) { converged = false; break; }      // round cap: best iterate, not converged
                // re-introduce the violated balls with zero multipliers (reading 12); the reduced
                // buffers grow as needed and keep the rows, radii and current multipliers of the balls already there
                if (nred + nvl > Q.cap) {
                    int64_t want = 2 * (nred + nvl) + 1024;
                    if (want > m) want = m;
                    rc = reduced_reserve(ctx, Q, want, nred);
                    if (rc) break;
                    reduced_bind(ctx, Q, P2);
                }
                double* Cred = (double*)ctx->own[OWN_CRED];
                rc = meb_gather_rows_f64(ctx, centers, ld, idx + nred, nvl, d, Cred + nred * ldr, ldr);
                if (rc) break;
                if (radii) { rc = meb_gather_vec_f64(ctx, radii, idx + nred, nvl, (double*)ctx->own[OWN_RRED] + nred); if (rc) break; }
                rc = meb_set_kept(ctx, idx + nred, nvl, kept);
                if (rc) break;
                if (P2.has_mult) {
                    rc = meb_fill_f64(ctx, (double*)P2.U[P2.cur] + nred, nvl, 0.0);
                    if (rc) break;
                    rc = meb_fill_i32(ctx, P2.slot[P2.cur] + nred, nvl, -1);
                    if (rc) break;
                }
                nred += nvl;
                converged = false;
                ab = xn;
            }
            if (rc) break;
        }
        st->radius_alg = r_alg;
        st->delta_max = dmax;
        *h_radius_out = r_alg + dmax;                     // = max_i(||c - c_i|| + r_i)   (step 7)
    } while (0);
#undef CUB
    if (rc != MEB_OK) return rc;
    cudaEventRecord(e_end, ctx->stream);
    cudaEventSynchronize(e_end);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e_start, e_end); st->ms_total = ms;
    if (have_mid && cudaEventElapsedTime(&ms, e_start, e_mid) == cudaSuccess) st->ms_phase_lo = ms;
    if (have_mid && have_hi && cudaEventElapsedTime(&ms, e_mid, e_hi) == cudaSuccess) st->ms_phase_hi = ms;
    if (have_hi && cudaEventElapsedTime(&ms, e_hi, e_end) == cudaSuccess) st->ms_check = ms;
    cudaGetLastError();
    memcpy(h_center_out, creturn.data(), d * sizeof(double));
    st->converged = converged ? 1 : 0;
    st->kkt = kkt;
    memcpy(st->kkt_terms, terms, sizeof(terms));
    st->bytes_streamed = S.bytes;
    for (int k = 0; k < ctx->evn; ++k) {           // CUDA-event time of the streaming launches made outside graphs
        float pms = 0.f;
        if (ctx->evcut[k]) continue;
        if (cudaEventElapsedTime(&pms, ctx->evpool[2 * k], ctx->evpool[2 * k + 1]) != cudaSuccess) continue;
        const int cls = ctx->evclass[k] & 7;
        st->pass_ev_ms[cls] += pms; st->pass_ev_bytes[cls] += ctx->evbytes[k]; st->pass_ev_count[cls]++;
        if (cls == MEB_PASS_INGEST || cls == MEB_PASS_SCREEN || cls == MEB_PASS_FEAS) {     // never inside a graph
            st->pass_ms[cls] += pms; st->pass_bytes[cls] += ctx->evbytes[k]; st->pass_count[cls]++;
        }
    }
    cudaGetLastError();
    st->kernel_launches = ctx->launches - launches0;
    return converged ? MEB_OK : MEB_W_NOT_CONVERGED;
}

}  // namespace

extern "C" int meb_solve(meb_ctx* ctx, int64_t m, int32_t d, const double* centers, int64_t ld,
                         const double* radii, double tol, int precision_mode, const meb_params* h_params,
                         double* h_center_out, double* h_radius_out, meb_stats* h_stats) {
    if (!ctx) return MEB_E_ARG;
    ctx->shard = nullptr;
    return solve_impl(ctx, m, d, centers, ld, radii, tol, precision_mode, h_params, h_center_out, h_radius_out, h_stats);
}

extern "C" int meb_solve_sharded(meb_ctx* ctx, int32_t rank, int32_t nranks, int64_t m_local, int64_t row_offset,
                                 int64_t m_global, int32_t d, const double* centers_local, int64_t ld,
                                 const double* radii_local, double tol, int precision_mode, const meb_params* h_params,
                                 double* xchg_send, double* xchg_recv, int64_t xchg_doubles, meb_allgather_fn allgather,
                                 void* user, double* h_center_out, double* h_radius_out, meb_stats* h_stats) {
    if (!ctx || nranks < 1 || rank < 0 || rank >= nranks || m_local < 1 || row_offset < 0 || m_global < row_offset + m_local ||
        !xchg_send || !xchg_recv || (nranks > 1 && !allgather))
        return MEB_E_ARG;
    if (xchg_doubles < meb_shard_record_doubles(d)) return MEB_E_CAPACITY;
    MebShard sh;
    sh.rank = rank; sh.nranks = nranks; sh.row_offset = row_offset; sh.m_global = m_global;
    sh.send = xchg_send; sh.recv = xchg_recv; sh.rec_doubles = xchg_doubles; sh.allgather = allgather; sh.user = user;
    ctx->shard = &sh;
    const int rc = solve_impl(ctx, m_local, d, centers_local, ld, radii_local, tol, precision_mode, h_params, h_center_out,
                              h_radius_out, h_stats);
    ctx->shard = nullptr;
    return rc;
}

extern "C" int meb_solve_host(meb_ctx* ctx, int64_t m, int32_t d, const double* h_centers, int64_t ld,
                              const double* h_radii, double tol, int precision_mode, const meb_params* h_params,
                              double* h_center_out, double* h_radius_out, meb_stats* h_stats) {
    if (!ctx || !h_centers || m < 1 || d < 1 || ld < d) return MEB_E_ARG;
    if (m > ctx->m_max || d > ctx->d_max) return MEB_E_CAPACITY;
    // device copies owned by the context (reused across calls: no allocation in the steady state)
    int rc = own_reserve(ctx, OWN_DEVC, (size_t)m * ld * sizeof(double));
    if (rc == MEB_OK && h_radii) rc = own_reserve(ctx, OWN_DEVR, (size_t)m * sizeof(double));
    if (rc != MEB_OK) return rc;
    double* dC = (double*)ctx->own[OWN_DEVC];
    double* dR = h_radii ? (double*)ctx->own[OWN_DEVR] : nullptr;
    MEB_CUDA_OK(ctx, cudaMemcpyAsync(dC, h_centers, (size_t)m * ld * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
    if (h_radii)
        MEB_CUDA_OK(ctx, cudaMemcpyAsync(dR, h_radii, (size_t)m * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
    return meb_solve(ctx, m, d, dC, ld, dR, tol, precision_mode, h_params, h_center_out, h_radius_out, h_stats);
}
