// Single-CTA controller kernels of the device-resident ripALM loop (see meb_ctrl.cuh).
#include "meb_ctrl.cuh"

namespace {

constexpr int CBLK = 1024;

__global__ void __launch_bounds__(CBLK) ctrl_init_kernel(SolverDev* S, const SolverVecs v, double sigma0,
                                                         int cur, int has_mult) {
    meb_ctrl_init_dev(S, v, sigma0, cur, has_mult);
}

// After a relaunch that only had to grow the V pools: keep everything, clear the stop flag.
__global__ void ctrl_resume_kernel(SolverDev* S) {
    S->done = 0;
    S->status = ST_RUNNING;
    S->dyn.s0_abort = 1e300;
}

// After the Newton direction Delta is in v.delta (Alg. 2 line 8): first Armijo trial x + Delta.
__global__ void __launch_bounds__(CBLK) ctrl_after_newton_kernel(SolverDev* S, const SolverVecs v) {
    __shared__ double sm[32];
    const int n = S->n;
    const double Ls = S->L;
    double sl = 0.0, dx2t = 0.0, dc2 = 0.0;
    for (int j = threadIdx.x; j < n; j += blockDim.x) {
        const double dj = v.delta[j];
        sl = fma(v.g[j], dj, sl);
        const double xj = v.xn[j] + dj;
        v.xt[j] = xj;
        v.dir_raw[j] = Ls * dj;
        const double dxb = xj - v.xbar[j];
        dx2t = fma(dxb, dxb, dx2t);
        if (j > 0) dc2 = fma(dj, dj, dc2);
    }
    sl = ctrl_block_sum(sl, sm);
    dx2t = ctrl_block_sum(dx2t, sm);
    dc2 = ctrl_block_sum(dc2, sm);
    __syncthreads();
    ctrl_to_raw(S, v, v.xt, v.x_raw);
    if (threadIdx.x == 0) {
        ctrl_arm_abort(S, true, v.xn[0] + v.delta[0], dx2t);
        S->slope = sl;
        S->tiny = (-sl <= S->slope_floor * fabs(S->psi_cur)) ? 1 : 0;
        S->eta = 1.0;
        S->ls = 0;
        S->phase = PH_ARMIJO;
        S->action = ACT_TRIAL;
        ctrl_arm_multi(S, 1.0, 0, Ls * v.delta[0], Ls * Ls * dc2);
    }
}

// One conjugate-gradient step on H Delta = -g after Hp = H_raw p is in v.Hp (reading 5).
// H~ = L H_raw in normalised units.
__global__ void __launch_bounds__(CBLK) ctrl_cg_step_kernel(SolverDev* S, const SolverVecs v) {
    __shared__ double sm[32];
    const int n = S->n;
    const double Ls = S->L;
    double pHp = 0.0;
    for (int j = threadIdx.x; j < n; j += blockDim.x) pHp = fma(v.p[j], Ls * v.Hp[j], pHp);
    pHp = ctrl_block_sum(pHp, sm);
    const double rr = S->cg_rr;
    const double alpha = rr / pHp;
    double rr_new = 0.0;
    for (int j = threadIdx.x; j < n; j += blockDim.x) {
        v.delta[j] = fma(alpha, v.p[j], v.delta[j]);
        const double rj = fma(-alpha, Ls * v.Hp[j], v.res[j]);
        v.res[j] = rj;
        rr_new = fma(rj, rj, rr_new);
    }
    rr_new = ctrl_block_sum(rr_new, sm);
    const double beta = rr_new / rr;
    for (int j = threadIdx.x; j < n; j += blockDim.x) v.p[j] = fma(beta, v.p[j], v.res[j]);
    __syncthreads();
    if (threadIdx.x == 0) {
        S->cg_rr = rr_new;
        S->cg_it++;
        S->cg_total++;
        S->cg_go = (sqrt(rr_new) > S->cg_tol && S->cg_it < S->cg_max) ? 1 : 0;
        if (S->in_graph) cudaGraphSetConditional(S->h_cg, S->cg_go ? 1u : 0u);
    }
}

// After the multiplier-update kernels wrote (U+, V+) into the other buffer (eq. (6)):
// capacity check, buffer flip, (alpha, beta) update, KKT test, sigma update,
// start of the next outer iteration.
__global__ void __launch_bounds__(CBLK) ctrl_after_update_kernel(SolverDev* S, const SolverVecs v,
                                                                 const int32_t* count) {
    meb_ctrl_after_update_dev(S, v, (long long)*count);
}

// U_next <- 0, slot_next <- -1 before the scatter of the multiplier update
template <typename T>
__global__ void reset_next_kernel(const MebDyn* dyn, T* U0, T* U1, int32_t* s0, int32_t* s1, int64_t m) {
    const int nxt = dyn->has_mult ? 1 - dyn->cur : 0;
    T* U = nxt ? U1 : U0;
    int32_t* sl = nxt ? s1 : s0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < m; i += (int64_t)gridDim.x * blockDim.x) {
        U[i] = T(0);
        sl[i] = -1;
    }
}

}  // namespace

int meb_ctrl_init(meb_ctx* ctx, SolverDev* S, const SolverVecs& v, double sigma0, int cur, int has_mult) {
    ctx->launches++; ctrl_init_kernel<<<1, CBLK, 0, ctx->stream>>>(S, v, sigma0, cur, has_mult);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}
int meb_ctrl_resume(meb_ctx* ctx, SolverDev* S) {
    ctx->launches++; ctrl_resume_kernel<<<1, 1, 0, ctx->stream>>>(S);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}
int meb_ctrl_after_newton(meb_ctx* ctx, SolverDev* S, const SolverVecs& v) {
    ctx->launches++; ctrl_after_newton_kernel<<<1, CBLK, 0, ctx->stream>>>(S, v);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}
int meb_ctrl_cg_step(meb_ctx* ctx, SolverDev* S, const SolverVecs& v) {
    ctx->launches++; ctrl_cg_step_kernel<<<1, CBLK, 0, ctx->stream>>>(S, v);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}
int meb_ctrl_after_update(meb_ctx* ctx, SolverDev* S, const SolverVecs& v, const int32_t* count) {
    ctx->launches++; ctrl_after_update_kernel<<<1, CBLK, 0, ctx->stream>>>(S, v, count);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}
int meb_reset_next(meb_ctx* ctx, int prec, const MebDyn* dyn, void* U0, void* U1, int32_t* s0, int32_t* s1,
                   int64_t m) {
    int64_t g = (m + 1023) / 1024;
    if (g > 148 * 8) g = 148 * 8;
    if (g < 1) g = 1;
    ctx->launches++;
    if (prec == MEB_FP64) reset_next_kernel<double><<<(int)g, 256, 0, ctx->stream>>>(dyn, (double*)U0, (double*)U1, s0, s1, m);
    else reset_next_kernel<float><<<(int)g, 256, 0, ctx->stream>>>(dyn, (float*)U0, (float*)U1, s0, s1, m);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}
