// C-ABI entry points of libmeb_b200.so: context management and the per-primitive calls of
// include/meb.h.  Argument checking and launch sequencing only; all arithmetic is in the kernels.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>

#include "meb_internal.cuh"
#include "meb_ctrl.cuh"

// layout of ctx->small (doubles)
#define SM_EV 0          // [16] evaluation scalars scratch
#define SM_AUX 16        // [16] argmax / sums scratch
#define SM_X 32          // [d_max+1] assembled x = (r, c)

static size_t round_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

static void ctx_free_all(meb_ctx* c) {
    if (!c) return;
    cudaFree(c->vmask); cudaFree(c->vlist); cudaFree(c->part_multi); cudaFree(c->dyn_api); cudaFree(c->smask);
    cudaFree(c->mask); cudaFree(c->rec_lam); cudaFree(c->rec_rho); cudaFree(c->rec_t);
    cudaFree(c->list); cudaFree(c->blocksum); cudaFree(c->part_scalar); cudaFree(c->part_vec);
    cudaFree(c->part_mat); cudaFree(c->part_red); cudaFree(c->count_dev); cudaFree(c->part_sc); cudaFree(c->small);
    if (c->h_pinned) cudaFreeHost(c->h_pinned);
    for (int i = 0; i < 40; ++i) if (c->own[i]) cudaFree(c->own[i]);
    if (c->ev0) cudaEventDestroy(c->ev0);
    if (c->ev1) cudaEventDestroy(c->ev1);
    meb_free_graph_cache(c);
    if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
    if (c->sdev) cudaFree(c->sdev);
    if (c->h_sdev) cudaFreeHost(c->h_sdev);
    if (c->evpool) {
        for (int i = 0; i < 2 * MEB_EVPOOL; ++i) if (c->evpool[i]) cudaEventDestroy(c->evpool[i]);
        free(c->evpool);
    }
    for (int i = 0; i < 4; ++i) if (c->ev_solve[i]) cudaEventDestroy(c->ev_solve[i]);
    for (int i = 0; i < 8; ++i) if (c->ev_stage[i]) cudaEventDestroy(c->ev_stage[i]);
}

void meb_debug_cuda(const meb_ctx* ctx, const char* file, int line, int err) {
    if (ctx && ctx->debug) fprintf(stderr, "[meb] %s:%d: CUDA error %d (%s)\n", file, line, err, cudaGetErrorString((cudaError_t)err));
}

extern "C" int meb_version(void) { return 100; }

extern "C" const char* meb_strerror(int code) {
    switch (code) {
        case MEB_OK: return "ok";
        case MEB_W_NOT_CONVERGED: return "iteration cap reached; outputs hold the best iterate";
        case MEB_E_ARG: return "invalid argument";
        case MEB_E_INPUT: return "non-finite data or negative radius";
        case MEB_E_ALLOC: return "allocation failed";
        case MEB_E_CUDA: return "CUDA error (see meb_last_cuda_error)";
        case MEB_E_CAPACITY: return "capacity exceeded";
        default: return "unknown code";
    }
}

extern "C" void meb_default_params(meb_params* p) {
    if (!p) return;
    memset(p, 0, sizeof(*p));
    p->rho = 0.5; p->sigma0 = 1.0; p->kappa = 3.0; p->sigma_max = 1e8; p->tau = 1.0;
    p->armijo_shrink_min = 0.5;
    p->armijo_mu = 1e-4; p->tol_lo = 1e-2; p->tol_red_factor = 0.02;
    p->armijo_max_halvings = 30; p->cg_max = 500; p->dense_d_max = 128; p->inner_max = 50;
    p->outer_max = 200; p->max_rounds = 10; p->sample_rows = 1024; p->outer_max_lo = 30;
    p->armijo_multi = -1; p->ag_outer = 0; p->sigma_carry = 0.0;
}

extern "C" int meb_create(meb_ctx** out, int device, void* cuda_stream, int64_t m_max, int32_t d_max) {
    if (!out || m_max < 1 || d_max < 1 || m_max >= 2147483647LL - 64) return MEB_E_ARG;
    *out = nullptr;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return MEB_E_CUDA;
    meb_ctx* c = new (std::nothrow) meb_ctx();
    if (!c) return MEB_E_ALLOC;
    memset(c, 0, sizeof(*c));
    c->device = device;
    c->stream = (cudaStream_t)cuda_stream;
    c->m_max = m_max;
    c->d_max = d_max;
    cudaError_t e = cudaSetDevice(device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, device);
    const size_t nwords = (size_t)(m_max + 31) / 32 + 8;
    const size_t nseg = nwords / 2048 + 8;
    const size_t dpad = round_up((size_t)d_max + 1, 8);
    c->vec_rows = 2 * (int64_t)(c->sm_count > 0 ? c->sm_count : 148);
    c->small_len = SM_X + (int64_t)dpad + 64;
    c->h_pinned_len = 12 * (int64_t)dpad + 256;     // [0, 4 dpad + 256): read-backs; then 8 upload slots of dpad
#define TRY_ALLOC(ptr, bytes) if (e == cudaSuccess) e = cudaMalloc((void**)&(ptr), (bytes))
    TRY_ALLOC(c->mask, nwords * sizeof(uint32_t));
    TRY_ALLOC(c->smask, nwords * sizeof(uint32_t));
    if ((size_t)d_max * 8 > 1024) {                  // long rows (meb_long.cu): list of the balls with a multiplier row
        TRY_ALLOC(c->vmask, nwords * sizeof(uint32_t));
        TRY_ALLOC(c->vlist, ((size_t)m_max + 32) * sizeof(int32_t));
    }
    TRY_ALLOC(c->part_multi, (size_t)MEB_MAX_GRID * MEB_MULTI_MAX * sizeof(double));
    TRY_ALLOC(c->dyn_api, sizeof(MebDyn));
    TRY_ALLOC(c->rec_lam, (size_t)m_max * sizeof(double));
    TRY_ALLOC(c->rec_rho, (size_t)m_max * sizeof(double));
    TRY_ALLOC(c->rec_t, (size_t)m_max * sizeof(double));
    TRY_ALLOC(c->list, ((size_t)m_max + 32) * sizeof(int32_t));
    TRY_ALLOC(c->blocksum, nseg * sizeof(int32_t));
    TRY_ALLOC(c->part_scalar, (size_t)MEB_MAX_GRID * MEB_NPART * sizeof(double));
    TRY_ALLOC(c->part_vec, (size_t)c->vec_rows * dpad * sizeof(double));
    TRY_ALLOC(c->part_red, dpad * sizeof(double));
    {
        const size_t dpm = (size_t)((d_max < 128 ? d_max : 128) + 15) / 16 * 16;
        c->part_mat_len = (size_t)(c->vec_rows * 3 / 2) * (dpm * dpm + dpm);      // up to three SYRK CTAs per SM
    }
    TRY_ALLOC(c->part_mat, c->part_mat_len * sizeof(double));
    TRY_ALLOC(c->count_dev, 8 * sizeof(int32_t));
    TRY_ALLOC(c->part_sc, 1024 * sizeof(double));
    TRY_ALLOC(c->small, (size_t)c->small_len * sizeof(double));
#undef TRY_ALLOC
    if (e == cudaSuccess) e = cudaMallocHost((void**)&c->h_pinned, (size_t)c->h_pinned_len * sizeof(double));
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaMalloc(&c->sdev, meb_solver_dev_size());
    if (e == cudaSuccess) e = cudaMallocHost(&c->h_sdev, meb_solver_dev_size());
    if (e == cudaSuccess) e = cudaEventCreate(&c->ev0);
    if (e == cudaSuccess) e = cudaEventCreate(&c->ev1);
    if (e == cudaSuccess) {
        c->evpool = (cudaEvent_t*)calloc(2 * MEB_EVPOOL, sizeof(cudaEvent_t));
        if (!c->evpool) e = cudaErrorMemoryAllocation;
        for (int i = 0; e == cudaSuccess && i < 2 * MEB_EVPOOL; ++i) e = cudaEventCreate(&c->evpool[i]);
    }
    for (int i = 0; e == cudaSuccess && i < 4; ++i) e = cudaEventCreate(&c->ev_solve[i]);
    for (int i = 0; e == cudaSuccess && i < 8; ++i) e = cudaEventCreateWithFlags(&c->ev_stage[i], cudaEventDisableTiming);
    c->opt[MEB_OPT_STEPPED] = getenv("MEB_NO_GRAPH") ? 1 : 0;
    c->opt[MEB_OPT_NO_SMALL] = getenv("MEB_NO_SMALL") ? 1 : 0;
    c->opt[MEB_OPT_NO_ABORT] = getenv("MEB_NO_ABORT") ? 1 : 0;
    c->opt[MEB_OPT_NO_FUSED_SCREEN] = 0;
    c->debug = getenv("MEB_DEBUG") != nullptr;
    c->cur_class = MEB_PASS_NCLASS - 1;
    if (e == cudaSuccess) e = cudaMemsetAsync(c->count_dev, 0, 8 * sizeof(int32_t), c->stream);
    if (e != cudaSuccess) {
        const bool oom = (e == cudaErrorMemoryAllocation);
        ctx_free_all(c);
        delete c;
        cudaGetLastError();
        return oom ? MEB_E_ALLOC : MEB_E_CUDA;
    }
    *out = c;
    return MEB_OK;
}

extern "C" int meb_destroy(meb_ctx* ctx) {
    if (!ctx) return MEB_E_ARG;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    ctx_free_all(ctx);
    delete ctx;
    return MEB_OK;
}

extern "C" int meb_last_cuda_error(const meb_ctx* ctx) { return ctx ? ctx->last_cuda_error : 0; }

extern "C" int meb_set_option(meb_ctx* ctx, int option, int value) {
    if (!ctx || option < 0 || option >= MEB_OPT_NCOUNT) return MEB_E_ARG;
    ctx->opt[option] = value != 0;
    return MEB_OK;
}

extern "C" int meb_set_pass_timing(meb_ctx* ctx, int on) {
    if (!ctx) return MEB_E_ARG;
    ctx->time_passes = on != 0;
    return MEB_OK;
}

extern "C" int meb_last_pass_info(const meb_ctx* ctx, double* h_ms, double* h_bytes) {
    if (!ctx) return MEB_E_ARG;
    if (h_ms) *h_ms = ctx->last_pass_ms;
    if (h_bytes) *h_bytes = ctx->last_pass_bytes;
    return MEB_OK;
}

static int check_problem(const meb_ctx* ctx, int64_t m, int32_t d, const void* C, int64_t ld) {
    if (!ctx || !C || m < 1 || d < 1 || ld < d) return MEB_E_ARG;
    if (m > ctx->m_max || d > ctx->d_max) return MEB_E_CAPACITY;
    return MEB_OK;
}

// one streaming launch, optionally timed with CUDA events on the context's stream.  Short aligned rows
// go to the TMA-staged tile kernels (meb_tile.cu), everything else to the register-mapped kernels.
// which kernel family an evaluation of this problem uses (the dispatch of timed_stream)
int meb_eval_path(const meb_ctx* ctx, int prec, const void* C, int64_t ld, int64_t m, int32_t d) {
    StreamArgs a;
    memset(&a, 0, sizeof(a));
    a.C = C; a.ld = ld; a.m = m; a.d = d; a.part_vec = ctx->part_vec;
    if (meb_tile_applicable(OP_EVAL, prec, a)) return PATH_TILE;
    if (ctx->vlist != nullptr && meb_long_applicable(OP_EVAL, prec, a)) return PATH_LONG;
    return PATH_STREAM;
}
// the ascending list of the set bits of `mask` into idx_out[cap]; *h_count (host) = how many (MEB_E_CAPACITY if > cap)
int meb_compact_mask(meb_ctx* ctx, const uint32_t* mask, int64_t m, int32_t* idx_out, int64_t cap, int64_t* h_count) {
    int rc = meb_launch_compact_cap(ctx, mask, m, idx_out, cap, ctx->count_dev);
    if (rc != MEB_OK) return rc;
    MEB_CUDA_OK(ctx, cudaMemcpyAsync(ctx->h_pinned, ctx->count_dev, sizeof(int32_t), cudaMemcpyDeviceToHost, ctx->stream));
    MEB_CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
    const int64_t n = *(int32_t*)ctx->h_pinned;
    if (h_count) *h_count = n;
    return n > cap ? MEB_E_CAPACITY : MEB_OK;
}
static int timed_stream(meb_ctx* ctx, int op, int prec, const StreamArgs& a, double bytes, int* grid, int* path_out) {
    const bool tile = meb_tile_applicable(op, prec, a);
    const bool longk = !tile && ctx->vlist != nullptr && meb_long_applicable(op, prec, a);
    const int32_t* vlist = nullptr; const int32_t* vcount = nullptr;
    if (longk && op == OP_EVAL && a.dyn == nullptr && a.v_slot != nullptr) {
        // per-primitive call: the list of the balls with a multiplier row is built here (a solve keeps it up to date)
        int rcl = meb_build_vlist(ctx, a.v_slot, a.m, ctx->vlist, ctx->count_dev + 1);
        if (rcl != MEB_OK) return rcl;
        vlist = ctx->vlist; vcount = ctx->count_dev + 1;
    }
    if (longk) { int rc0 = meb_launch_long(ctx, 0, op, prec, a, vlist, vcount, grid); if (rc0 != MEB_OK) return rc0; }
    if (ctx->time_passes) MEB_CUDA_OK(ctx, cudaEventRecord(ctx->ev0, ctx->stream));
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    cudaStreamIsCapturing(ctx->stream, &cap);
    const bool pool = ctx->ev_record && !ctx->time_passes && ctx->evn < MEB_EVPOOL && cap == cudaStreamCaptureStatusNone;
    if (pool) MEB_CUDA_OK(ctx, cudaEventRecord(ctx->evpool[2 * ctx->evn], ctx->stream));
    int rc = tile ? meb_launch_tile(ctx, op, prec, a, grid)
                  : (longk ? meb_launch_long(ctx, 1, op, prec, a, vlist, vcount, grid) : meb_launch_stream(ctx, op, prec, a, grid));
    if (rc != MEB_OK) return rc;
    ctx->last_path = tile ? PATH_TILE : (longk ? PATH_LONG : PATH_STREAM);
    if (path_out) *path_out = ctx->last_path;
    if (pool) {
        MEB_CUDA_OK(ctx, cudaEventRecord(ctx->evpool[2 * ctx->evn + 1], ctx->stream));
        ctx->evclass[ctx->evn] = ctx->cur_class;
        // (long rows: the multiplier rows are read by vrow_kernel, outside the bracket)
        ctx->evbytes[ctx->evn] = bytes + ((op == OP_EVAL && !longk) ? ctx->ev_extra_bytes : 0.0);
        ctx->evcut[ctx->evn] = false;
        ctx->evn++;
    }
    ctx->last_pass_bytes = bytes;
    ctx->list_valid = false;
    if (ctx->time_passes && cap == cudaStreamCaptureStatusNone) {
        MEB_CUDA_OK(ctx, cudaEventRecord(ctx->ev1, ctx->stream));
        MEB_CUDA_OK(ctx, cudaEventSynchronize(ctx->ev1));
        float ms = 0.f;
        MEB_CUDA_OK(ctx, cudaEventElapsedTime(&ms, ctx->ev0, ctx->ev1));
        ctx->last_pass_ms = ms;
    }
    if (longk) {                    // balls with a multiplier row: after the bracket, so that the events time the
        rc = meb_launch_long(ctx, 2, op, prec, a, vlist, vcount, grid);      // streaming kernel alone
        if (rc != MEB_OK) return rc;
    }
    ctx->last_grid = *grid;
    return MEB_OK;
}

static void graph_side(ActiveArgs& a, const GraphSide* gs) {
    if (!gs) return;
    a.dyn = gs->dyn;
    for (int b = 0; b < 2; ++b) { a.U2[b] = gs->U2[b]; a.slot2[b] = gs->slot2[b]; a.V2[b] = gs->V2[b]; a.vcap2[b] = gs->vcap2[b]; }
}

static ActiveArgs active_args(meb_ctx* ctx, const EvalCall& c) {
    ActiveArgs a;
    memset(&a, 0, sizeof(a));
    a.C = c.C; a.ld = c.ld; a.U = c.U; a.v_slot = c.v_slot; a.V = c.V; a.ldv = c.ldv;
    a.x = c.x; a.d = c.d; a.dpad = (int32_t)round_up((size_t)c.d, 8); a.sigma = c.sigma;
    a.list = ctx->list; a.count = ctx->count_dev;
    a.rec_lam = ctx->rec_lam; a.rec_rho = ctx->rec_rho; a.rec_t = ctx->rec_t;
    a.part_vec = ctx->part_vec; a.part_sc = ctx->part_sc;
    graph_side(a, c.gs);
    return a;
}

// ascending list of the rows flagged by the last streaming pass (the active set of an evaluation)
int meb_ensure_list(meb_ctx* ctx, int64_t m) {
    if (ctx->list_valid) return MEB_OK;
    int rc = meb_launch_compact(ctx, ctx->mask, m, ctx->list, ctx->count_dev);
    if (rc == MEB_OK) ctx->list_valid = true;
    return rc;
}

int meb_eval_internal(meb_ctx* ctx, const EvalCall& c, double* out_scalars, double* grad,
                      double* t_out, double* lam_out) {
    StreamArgs s;
    memset(&s, 0, sizeof(s));
    s.C = c.C; s.ld = c.ld; s.R = c.R; s.U = c.U; s.v_slot = c.v_slot; s.V = c.V; s.ldv = c.ldv;
    s.x = c.x; s.m = c.m; s.d = c.d; s.sigma = c.sigma;
    s.mask = ctx->mask; s.rec_lam = ctx->rec_lam; s.rec_rho = ctx->rec_rho; s.rec_t = ctx->rec_t;
    s.t_out = t_out; s.lam_out = lam_out; s.part = ctx->part_scalar;
    s.part_vec = ctx->part_vec; s.dpad = (int32_t)round_up((size_t)c.d, 8);
    bool any_mult = c.U != nullptr;
    if (c.gs) {
        s.dyn = c.gs->dyn;
        for (int b = 0; b < 2; ++b) {
            s.U2[b] = c.gs->U2[b]; s.slot2[b] = c.gs->slot2[b]; s.V2[b] = c.gs->V2[b];
            s.vlist2[b] = c.gs->vlist2[b]; s.vcount2[b] = c.gs->vcount2[b];
        }
        any_mult = true;
        s.smask = ctx->smask;                    // written only while MebDyn::screen_on (low-precision run of a mixed solve)
        if (c.gs->multi > 0 && (c.gs->v || c.gs->dir)) {
            s.multi = c.gs->multi; s.dir = c.gs->dir ? c.gs->dir : c.gs->v->dir_raw; s.multi_part = ctx->part_multi;
        }
    }
    const double sz = c.prec == MEB_FP64 ? 8.0 : 4.0;
    const double bytes = (double)c.m * (c.d * sz + (c.R ? sz : 0) + (any_mult ? sz + 4 : 0));
    int grid = 0, path = PATH_STREAM;
    int rc = timed_stream(ctx, OP_EVAL, c.prec, s, bytes, &grid, &path);
    if (rc != MEB_OK) return rc;
    const bool fused = path == PATH_TILE;
    FinalizeArgs f;
    memset(&f, 0, sizeof(f));
    f.part = ctx->part_scalar; f.grid = grid; f.part_vec = ctx->part_vec; f.dpad = s.dpad;
    f.count = ctx->count_dev; f.x = c.x; f.xbar = c.xbar; f.sigma = c.sigma; f.tau = c.tau; f.d = c.d;
    f.out = out_scalars; f.grad = grad;
    if (c.gs) { f.dyn = c.gs->dyn; f.S = c.gs->S; if (c.gs->v) f.v = *c.gs->v; }
    if (s.multi > 0 && path != PATH_STREAM) f.multi_part = ctx->part_multi;  // kernels that carry the multi-trial code
    if (fused) {
        f.nvec = grid; f.tpb = 0;
    } else {                          // long rows: the vector part comes from the active-list kernel
        rc = meb_ensure_list(ctx, c.m);
        if (rc != MEB_OK) return rc;
        ActiveArgs a = active_args(ctx, c);
        if (c.gs) { a.cut_part = ctx->part_scalar; a.cut_grid = grid; }      // only a solve arms the early stop
        int nvec = 0;
        rc = meb_launch_active(ctx, MODE_ROWSUM, c.prec, a, &nvec);
        if (rc != MEB_OK) return rc;
        f.nvec = nvec; f.tpb = c.d > 2048 ? 1 : MEB_WARPS;
    }
    return meb_eval_finalize(ctx, f);
}

int meb_hvp_from_records(meb_ctx* ctx, const EvalCall& c, const double* ev_scalars, const double* q,
                         double* Hq) {
    int rc = meb_ensure_list(ctx, c.m);
    if (rc != MEB_OK) return rc;
    ActiveArgs a = active_args(ctx, c);
    a.q = q;
    int nvec = 0;
    rc = meb_launch_active(ctx, MODE_HVP, c.prec, a, &nvec);
    if (rc != MEB_OK) return rc;
    return meb_hvp_finalize(ctx, nvec, a.dpad, ctx->part_sc, ev_scalars, q, c.sigma, c.tau, c.d, Hq,
                            c.gs ? c.gs->dyn : nullptr);
}

static int check_eval_args(const meb_ctx* ctx, int prec, int64_t m, int32_t d, const void* C, int64_t ld,
                           const int32_t* v_slot, const void* V, int64_t ldv, const double* x, double sigma) {
    int rc = check_problem(ctx, m, d, C, ld);
    if (rc != MEB_OK) return rc;
    if ((prec != MEB_FP64 && prec != MEB_FP32) || !x || !(sigma > 0.0)) return MEB_E_ARG;
    if (v_slot && (!V || ldv < d)) return MEB_E_ARG;
    return MEB_OK;
}

extern "C" int meb_eval_alm(meb_ctx* ctx, int prec, int64_t m, int32_t d, const void* C, int64_t ld,
                            const void* R, const void* U, const int32_t* v_slot, const void* Vrows,
                            int64_t ldv, const double* x, const double* xbar, double sigma, double tau,
                            double* out_scalars, double* grad, double* t_out, double* lam_out,
                            int32_t* active_idx, double* active_rho, double* active_lam) {
    int rc = check_eval_args(ctx, prec, m, d, C, ld, v_slot, Vrows, ldv, x, sigma);
    if (rc != MEB_OK) return rc;
    if (!out_scalars || !grad || !(tau >= 0.0)) return MEB_E_ARG;
    EvalCall c{prec, m, d, C, ld, R, U, v_slot, Vrows, ldv, x, xbar, sigma, tau, nullptr};
    rc = meb_eval_internal(ctx, c, out_scalars, grad, t_out, lam_out);
    if (rc != MEB_OK) return rc;
    if (active_idx) {
        rc = meb_ensure_list(ctx, m);
        if (rc != MEB_OK) return rc;
        MEB_CUDA_OK(ctx, cudaMemcpyAsync(ctx->h_pinned, ctx->count_dev, sizeof(int32_t),
                                         cudaMemcpyDeviceToHost, ctx->stream));
        MEB_CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
        const int64_t n = *(int32_t*)ctx->h_pinned;
        if (n > 0) {
            MEB_CUDA_OK(ctx, cudaMemcpyAsync(active_idx, ctx->list, n * sizeof(int32_t),
                                             cudaMemcpyDeviceToDevice, ctx->stream));
            if (active_rho) { rc = meb_gather_vec_f64(ctx, ctx->rec_rho, ctx->list, n, active_rho); if (rc) return rc; }
            if (active_lam) { rc = meb_gather_vec_f64(ctx, ctx->rec_lam, ctx->list, n, active_lam); if (rc) return rc; }
        }
    }
    return MEB_OK;
}

// ---- multi-trial evaluation: Psi at several points of one line in ONE pass ------------------
namespace {
__global__ void multi_setup_kernel(MebDyn* dyn, const double* __restrict__ dir, int d, int n, double g0, double g1,
                                   double g2, double g3, double sigma, double tau, int has_mult) {
    __shared__ double red[8];
    double s = 0.0;
    for (int j = 1 + threadIdx.x; j <= d; j += blockDim.x) s = fma(dir[j], dir[j], s);
    s = warp_sum(s);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t += red[w];
        dyn->sigma_raw = sigma; dyn->tau_eff = tau; dyn->cur = 0; dyn->has_mult = has_mult; dyn->s0_abort = 1e300;
        dyn->multi_n = n;
        dyn->multi_gamma[0] = g0; dyn->multi_gamma[1] = g1; dyn->multi_gamma[2] = g2; dyn->multi_gamma[3] = g3;
        dyn->dir_r = dir[0]; dyn->dir_c2 = t; dyn->dir_c = sqrt(t);
    }
}
// psi_out[k] = r_k + (sigma/2) S_k + (tau/2sigma) ||x_k - xbar||^2 at x_k = x - gamma_k dir (reading 13)
__global__ void multi_psi_kernel(const double* __restrict__ part_multi, int grid, const MebDyn* dyn,
                                 const double* __restrict__ x, const double* __restrict__ xbar,
                                 const double* __restrict__ dir, int d, double* __restrict__ psi_out) {
    const int k = blockIdx.x, lane = threadIdx.x;
    if (k >= dyn->multi_n) return;
    const double g = dyn->multi_gamma[k];
    double s = 0.0, dx2 = 0.0;
    for (int b = lane; b < grid; b += 32) s += part_multi[(size_t)b * MEB_MULTI_MAX + k];
    for (int j = lane; j <= d; j += 32) { const double w = x[j] - g * dir[j] - (xbar ? xbar[j] : x[j] - g * dir[j]); dx2 = fma(w, w, dx2); }
    s = warp_sum(s); dx2 = warp_sum(dx2);
    if (lane == 0) psi_out[k] = (x[0] - g * dir[0]) + 0.5 * dyn->sigma_raw * s + 0.5 * (dyn->tau_eff / dyn->sigma_raw) * dx2;
}
}  // namespace

extern "C" int meb_eval_alm_multi(meb_ctx* ctx, int prec, int64_t m, int32_t d, const void* C, int64_t ld,
                                  const void* R, const void* U, const int32_t* v_slot, const void* Vrows, int64_t ldv,
                                  const double* x, const double* xbar, double sigma, double tau, const double* dir,
                                  int32_t n_steps, const double* h_gammas, double* out_scalars, double* grad,
                                  double* psi_out) {
    int rc = check_eval_args(ctx, prec, m, d, C, ld, v_slot, Vrows, ldv, x, sigma);
    if (rc != MEB_OK) return rc;
    if (!out_scalars || !grad || !(tau >= 0.0) || !dir || !h_gammas || !psi_out || n_steps < 1 || n_steps > MEB_MULTI_MAX)
        return MEB_E_ARG;
    double g[MEB_MULTI_MAX] = {0, 0, 0, 0};
    for (int k = 0; k < n_steps; ++k) { if (!(h_gammas[k] == h_gammas[k])) return MEB_E_ARG; g[k] = h_gammas[k]; }
    for (int k = 0; k < n_steps; ++k) if (g[k] < 0.0 || (k > 0 && g[k] < g[k - 1])) return MEB_E_ARG;   // farthest point last
    ctx->launches++;
    multi_setup_kernel<<<1, 256, 0, ctx->stream>>>(ctx->dyn_api, dir, d, n_steps, g[0], g[1], g[2], g[3], sigma, tau,
                                                   (U != nullptr || v_slot != nullptr) ? 1 : 0);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    GraphSide gs;
    memset(&gs, 0, sizeof(gs));
    gs.dyn = ctx->dyn_api;
    gs.U2[0] = const_cast<void*>(U); gs.slot2[0] = const_cast<int32_t*>(v_slot); gs.V2[0] = const_cast<void*>(Vrows);
    gs.multi = n_steps; gs.dir = dir;
    if (v_slot && ctx->vlist) {
        rc = meb_build_vlist(ctx, v_slot, m, ctx->vlist, ctx->count_dev + 1);
        if (rc != MEB_OK) return rc;
        gs.vlist2[0] = ctx->vlist; gs.vcount2[0] = ctx->count_dev + 1;
    }
    EvalCall c{prec, m, d, C, ld, R, U, v_slot, Vrows, ldv, x, xbar, sigma, tau, &gs};
    rc = meb_eval_internal(ctx, c, out_scalars, grad, nullptr, nullptr);
    if (rc != MEB_OK) return rc;
    if (ctx->last_path == PATH_STREAM) return MEB_E_CAPACITY;     // rows that are not 16-byte aligned: no multi-trial kernel
    ctx->launches++;
    multi_psi_kernel<<<n_steps, 32, 0, ctx->stream>>>(ctx->part_multi, ctx->last_grid, ctx->dyn_api, x, xbar, dir, d, psi_out);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}

extern "C" int meb_hvp(meb_ctx* ctx, int prec, int64_t m, int32_t d, const void* C, int64_t ld,
                       const void* R, const void* U, const int32_t* v_slot, const void* Vrows, int64_t ldv,
                       const double* x, double sigma, double tau, const double* q, double* Hq) {
    int rc = check_eval_args(ctx, prec, m, d, C, ld, v_slot, Vrows, ldv, x, sigma);
    if (rc != MEB_OK) return rc;
    if (!q || !Hq || !(tau >= 0.0)) return MEB_E_ARG;
    EvalCall c{prec, m, d, C, ld, R, U, v_slot, Vrows, ldv, x, nullptr, sigma, tau, nullptr};
    double* ev = ctx->small + SM_EV;
    rc = meb_eval_internal(ctx, c, ev, ctx->small + SM_X, nullptr, nullptr);
    if (rc != MEB_OK) return rc;
    return meb_hvp_from_records(ctx, c, ev, q, Hq);
}

extern "C" int meb_dense_hessian(meb_ctx* ctx, int prec, int64_t m, int32_t d, const void* C, int64_t ld,
                                 const void* R, const void* U, const int32_t* v_slot, const void* Vrows,
                                 int64_t ldv, const double* x, double sigma, double tau, double* H) {
    int rc = check_eval_args(ctx, prec, m, d, C, ld, v_slot, Vrows, ldv, x, sigma);
    if (rc != MEB_OK) return rc;
    if (!H || !(tau >= 0.0)) return MEB_E_ARG;
    if (d > 128) return MEB_E_CAPACITY;
    EvalCall c{prec, m, d, C, ld, R, U, v_slot, Vrows, ldv, x, nullptr, sigma, tau, nullptr};
    double* ev = ctx->small + SM_EV;
    rc = meb_eval_internal(ctx, c, ev, ctx->small + SM_X, nullptr, nullptr);
    if (rc != MEB_OK) return rc;
    return meb_dense_from_records(ctx, c, ev, H);
}

extern "C" int meb_update_multipliers(meb_ctx* ctx, int prec, int64_t m, int32_t d, const void* C,
                                      int64_t ld, const void* R, const void* U, const int32_t* v_slot,
                                      const void* Vrows, int64_t ldv, const double* x, double sigma,
                                      void* U_out, int32_t* v_slot_out, void* Vrows_out, int64_t ldv_out,
                                      int64_t cap_rows, int64_t* h_n_slots, double* h_sum_mult2) {
    int rc = check_eval_args(ctx, prec, m, d, C, ld, v_slot, Vrows, ldv, x, sigma);
    if (rc != MEB_OK) return rc;
    if (!U_out || !v_slot_out || !Vrows_out || ldv_out < d || cap_rows < 0) return MEB_E_ARG;
    EvalCall c{prec, m, d, C, ld, R, U, v_slot, Vrows, ldv, x, nullptr, sigma, 0.0, nullptr};
    rc = meb_eval_internal(ctx, c, ctx->small + SM_EV, ctx->small + SM_X, nullptr, nullptr);
    if (rc != MEB_OK) return rc;
    rc = meb_ensure_list(ctx, m);
    if (rc != MEB_OK) return rc;
    if (prec == MEB_FP64) rc = meb_fill_f64(ctx, (double*)U_out, m, 0.0);
    else rc = meb_fill_f32(ctx, (float*)U_out, m, 0.f);
    if (rc != MEB_OK) return rc;
    rc = meb_fill_i32(ctx, v_slot_out, m, -1);
    if (rc != MEB_OK) return rc;
    ActiveArgs a = active_args(ctx, c);
    a.U_out = U_out; a.slot_out = v_slot_out; a.V_out = Vrows_out; a.ldv_out = ldv_out; a.cap_rows = cap_rows;
    int nvec = 0;
    rc = meb_launch_active(ctx, MODE_WRITEV, prec, a, &nvec);
    if (rc != MEB_OK) return rc;
    rc = meb_scalar_sum(ctx, ctx->part_sc, nvec, ctx->small + SM_AUX);
    if (rc != MEB_OK) return rc;
    MEB_CUDA_OK(ctx, cudaMemcpyAsync(ctx->h_pinned, ctx->small + SM_AUX, sizeof(double), cudaMemcpyDeviceToHost,
                                     ctx->stream));
    MEB_CUDA_OK(ctx, cudaMemcpyAsync(ctx->h_pinned + 1, ctx->count_dev, sizeof(int32_t), cudaMemcpyDeviceToHost,
                                     ctx->stream));
    MEB_CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
    const int64_t n = *(int32_t*)(ctx->h_pinned + 1);
    if (h_n_slots) *h_n_slots = n;
    if (h_sum_mult2) *h_sum_mult2 = ctx->h_pinned[0];
    return n > cap_rows ? MEB_E_CAPACITY : MEB_OK;
}

// x = (r, c) assembled on the device from a host scalar and a device vector
static int assemble_x(meb_ctx* ctx, double r, const double* c, int32_t d) {
    ctx->h_pinned[8] = r;
    MEB_CUDA_OK(ctx, cudaMemcpyAsync(ctx->small + SM_X, ctx->h_pinned + 8, sizeof(double), cudaMemcpyHostToDevice,
                                     ctx->stream));
    MEB_CUDA_OK(ctx, cudaMemcpyAsync(ctx->small + SM_X + 1, c, (size_t)d * sizeof(double),
                                     cudaMemcpyDeviceToDevice, ctx->stream));
    return MEB_OK;
}

extern "C" int meb_screen_compact(meb_ctx* ctx, int64_t m, int32_t d, const float* C32, int64_t ld32,
                                  const float* R32, float r_hat, const double* c_hat, float tol_red,
                                  int32_t* idx_out, int64_t cap, int64_t* h_count, uint8_t* flags,
                                  int flags_are_input) {
    if (!ctx || !idx_out || cap < 0 || m < 1) return MEB_E_ARG;
    if (m > ctx->m_max) return MEB_E_CAPACITY;
    int rc;
    if (flags_are_input) {
        if (!flags) return MEB_E_ARG;
        rc = meb_launch_flags_to_mask(ctx, flags, m, ctx->mask);
        if (rc != MEB_OK) return rc;
    } else {
        rc = check_problem(ctx, m, d, C32, ld32);
        if (rc != MEB_OK) return rc;
        if (!c_hat) return MEB_E_ARG;
        rc = assemble_x(ctx, (double)r_hat, c_hat, d);
        if (rc != MEB_OK) return rc;
        StreamArgs s;
        memset(&s, 0, sizeof(s));
        s.C = C32; s.ld = ld32; s.R = R32; s.x = ctx->small + SM_X; s.m = m; s.d = d; s.sigma = 1.0;
        s.mask = ctx->mask; s.part = ctx->part_scalar; s.eps = (double)tol_red; s.flags_out = flags;
        int grid = 0;
        ctx->cur_class = MEB_PASS_SCREEN;
        rc = timed_stream(ctx, OP_SCREEN, MEB_FP32, s, (double)m * (d * 4.0 + (R32 ? 4 : 0)), &grid, nullptr);
        if (rc != MEB_OK) return rc;
    }
    rc = meb_launch_compact_cap(ctx, ctx->mask, m, idx_out, cap, ctx->count_dev);
    if (rc != MEB_OK) return rc;
    MEB_CUDA_OK(ctx, cudaMemcpyAsync(ctx->h_pinned, ctx->count_dev, sizeof(int32_t), cudaMemcpyDeviceToHost,
                                     ctx->stream));
    MEB_CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
    const int64_t n = *(int32_t*)ctx->h_pinned;
    if (h_count) *h_count = n;
    return n > cap ? MEB_E_CAPACITY : MEB_OK;
}

extern "C" int meb_feasibility_check(meb_ctx* ctx, int64_t m, int32_t d, const double* C, int64_t ld,
                                     const double* R, double r, const double* c, double eps_feas,
                                     const uint8_t* kept_mask, double* h_delta_max, int32_t* h_argmax,
                                     int32_t* viol_idx, int64_t cap, int64_t* h_n_viol) {
    int rc = check_problem(ctx, m, d, C, ld);
    if (rc != MEB_OK) return rc;
    if (!c || cap < 0 || (cap > 0 && !viol_idx)) return MEB_E_ARG;
    rc = assemble_x(ctx, r, c, d);
    if (rc != MEB_OK) return rc;
    StreamArgs s;
    memset(&s, 0, sizeof(s));
    s.C = C; s.ld = ld; s.R = R; s.x = ctx->small + SM_X; s.m = m; s.d = d; s.sigma = 1.0;
    s.mask = ctx->mask; s.part = ctx->part_scalar; s.eps = eps_feas; s.kept = kept_mask;
    int grid = 0;
    ctx->cur_class = MEB_PASS_FEAS;
    rc = timed_stream(ctx, OP_FEAS, MEB_FP64, s, (double)m * (d * 8.0 + (R ? 8 : 0) + (kept_mask ? 1 : 0)), &grid, nullptr);
    if (rc != MEB_OK) return rc;
    rc = meb_argmax_finalize(ctx, grid, ctx->small + SM_AUX);
    if (rc != MEB_OK) return rc;
    rc = meb_launch_compact_cap(ctx, ctx->mask, m, viol_idx ? viol_idx : ctx->list, viol_idx ? cap : 0,
                                ctx->count_dev);
    if (rc != MEB_OK) return rc;
    MEB_CUDA_OK(ctx, cudaMemcpyAsync(ctx->h_pinned, ctx->small + SM_AUX, 2 * sizeof(double),
                                     cudaMemcpyDeviceToHost, ctx->stream));
    MEB_CUDA_OK(ctx, cudaMemcpyAsync(ctx->h_pinned + 2, ctx->count_dev, sizeof(int32_t), cudaMemcpyDeviceToHost,
                                     ctx->stream));
    MEB_CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
    if (h_delta_max) *h_delta_max = ctx->h_pinned[0];
    if (h_argmax) *h_argmax = (int32_t)ctx->h_pinned[1];
    const int64_t n = *(int32_t*)(ctx->h_pinned + 2);
    if (h_n_viol) *h_n_viol = n;
    return (viol_idx && n > cap) ? MEB_E_CAPACITY : MEB_OK;
}

extern "C" int meb_ingest(meb_ctx* ctx, int64_t m, int32_t d, const double* C, int64_t ld, const double* R,
                          int32_t sample_rows, double* c0_out, double* scalars_out, float* C32, int64_t ld32,
                          float* R32) {
    int rc = check_problem(ctx, m, d, C, ld);
    if (rc != MEB_OK) return rc;
    if (!c0_out || !scalars_out || sample_rows < 1) return MEB_E_ARG;
    if (C32 && (ld32 < d || ld32 % 4 != 0)) return MEB_E_ARG;
    const int S = (int)(m < sample_rows ? m : sample_rows);
    rc = meb_sample_mean(ctx, C, ld, m, d, S, c0_out);
    if (rc != MEB_OK) return rc;
    if (ctx->shard) {               // sharded solve: c0 = mean of the ranks' sample means weighted by their rows (reading 3)
        rc = meb_shard_mean(ctx, c0_out, d, m);
        if (rc != MEB_OK) return rc;
    }
    StreamArgs s;
    memset(&s, 0, sizeof(s));
    s.C = C; s.ld = ld; s.R = R; s.x = nullptr; s.c0 = c0_out; s.m = m; s.d = d; s.sigma = 1.0;
    s.part = ctx->part_scalar; s.C32 = C32; s.ld32 = ld32; s.R32 = (C32 && R) ? R32 : nullptr;
    int grid = 0;
    const double bytes = (double)m * (d * 8.0 + (R ? 8 : 0)) + (C32 ? (double)m * (d * 4.0 + (R ? 4 : 0)) : 0.0);
    ctx->cur_class = MEB_PASS_INGEST;
    rc = timed_stream(ctx, OP_INGEST, MEB_FP64, s, bytes, &grid, nullptr);
    if (rc != MEB_OK) return rc;
    rc = meb_argmax_finalize(ctx, grid, scalars_out);
    if (rc == MEB_OK && ctx->shard) rc = meb_shard_argmax(ctx, scalars_out);     // L = max over the ranks, global index
    return rc;
}
