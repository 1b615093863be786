// Second level of the fixed-order reduction trees and the (d+1)-sized state updates.
// Single-CTA kernels: their inputs are the per-CTA partials written by the streaming / active-list
// kernels (a few thousand doubles), so they are latency-, not bandwidth-bound.
#include "meb_internal.cuh"
#include "meb_ctrl.cuh"

namespace {

constexpr int FBLOCK = 1024;

// scalar k of the CTA partials: lanes stride over the CTAs, xor tree (warp k handles scalar k)
__device__ __forceinline__ double partial_sum(const double* part, int grid, int k, int lane, int stride = MEB_NPART) {
    double s = 0.0;
    for (int b = lane; b < grid; b += 32) s += part[(size_t)b * stride + k];
    return warp_sum(s);
}
__device__ __forceinline__ double partial_max(const double* part, int grid, int k, int lane, int stride = MEB_NPART) {
    double s = 0.0;
    for (int b = lane; b < grid; b += 32) s = fmax(s, part[(size_t)b * stride + k]);
    return warp_max(s);
}

// out_scalars / grad of one ALM evaluation (reading 13 for psi_var).  Second level of the
// fixed-order reduction: CTA partials are added in index order (in S interleaved segments that are
// then added in order, so the order does not depend on timing).  With f.S != nullptr the same CTA then
// runs the controller step of the device-resident solver (meb_ctrl.cuh).
__global__ void __launch_bounds__(FBLOCK) eval_finalize_kernel(const FinalizeArgs f) {
    __shared__ double sm[104];
    __shared__ double ev_s[MEB_EVAL_NSCALARS];
    __shared__ double sc[MEB_NPART];
    __shared__ double seg[FBLOCK];
    __shared__ double multi_s[MEB_MULTI_MAX];
    __shared__ __align__(16) SolverDev sS;             // working copy of the solver state (controller step)
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (f.S) {
        const unsigned long long* src = reinterpret_cast<const unsigned long long*>(f.S);
        unsigned long long* dst = reinterpret_cast<unsigned long long*>(&sS);
        for (int q = threadIdx.x; q < (int)(sizeof(SolverDev) / 8); q += FBLOCK) dst[q] = src[q];
    }                                                   // (visible after the first __syncthreads below)
    const double* __restrict__ part = f.part;
    const double* __restrict__ part_vec = f.part_vec;
    const int grid = f.grid, d = f.d;
    const int dpad = f.vec_stride > 0 ? f.vec_stride : f.dpad;           // stride between the vector partials
    const int pstr = f.part_stride > 0 ? f.part_stride : MEB_NPART;
    const int mstr = f.multi_stride > 0 ? f.multi_stride : MEB_MULTI_MAX;
    double sigma = f.sigma, tau = f.tau;
    if (f.dyn) { sigma = f.dyn->sigma_raw; tau = f.dyn->tau_eff; }
    const double* x = f.x; const double* xbar = f.xbar;
    if (warp < 9) {
        double v;
        if (warp >= 5 && warp <= 7) v = partial_max(part, grid, warp, lane, pstr);
        else v = partial_sum(part, grid, warp, lane, pstr);
        if (lane == 0) sc[warp] = v;
    } else if (warp == 10) {
        const double v = partial_max(part, grid, MEB_PART_CUT, lane, pstr);
        if (lane == 0) sc[MEB_PART_CUT] = v;
    } else if (warp >= 11 && warp < 11 + MEB_MULTI_MAX && f.S && f.multi_part) {
        // predicted step sizes of a trial pass (multi-trial Armijo): CTA partials in index order
        const int k = warp - 11;
        double t = 0.0;
        for (int b = lane; b < grid; b += 32) t += f.multi_part[(size_t)b * mstr + k];
        t = warp_sum(t);
        if (lane == 0) multi_s[k] = t;
    } else if (warp == 9 && f.S) {
        // device time of the pass: last CTA end - first CTA start (globaltimer stamps of the tile kernel)
        long long t0 = 0x7fffffffffffffffLL, t1 = 0;
        for (int b = lane; b < grid; b += 32) {
            const long long s0 = __double_as_longlong(part[(size_t)b * pstr + 10]);
            const long long s1 = __double_as_longlong(part[(size_t)b * pstr + 11]);
            if (s1 > 0) { t0 = min(t0, s0); t1 = max(t1, s1); }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            t0 = min(t0, __shfl_xor_sync(MEB_FULL_MASK, t0, o));
            t1 = max(t1, __shfl_xor_sync(MEB_FULL_MASK, t1, o));
        }
        if (lane == 0) { sm[100] = __longlong_as_double(t0); sm[101] = __longlong_as_double(t1); }
    }
    // vector part: sum_i v+_i = sigma * sum_k lam_k b_k
    int nvec = f.nvec;
    if (nvec > 0 && f.tpb > 0) {           // active-list kernel: only CTAs b < ceil(count/tpb) had entries
        const int used = (*f.count + f.tpb - 1) / f.tpb;
        if (nvec > used) nvec = used;
    }
    double nv2 = 0.0, dx2 = 0.0;
    const double tos = tau / sigma;
    if (d <= FBLOCK) {
        const int dr = (d + 31) & ~31;
        int S = FBLOCK / dr;
        if (S > 32) S = 32;
        const int j = threadIdx.x % dr, sg = threadIdx.x / dr;
        double s = 0.0;
        if (sg < S && j < d)
            for (int b = sg; b < nvec; b += S) s += part_vec[(size_t)b * dpad + j];
        seg[threadIdx.x] = s;
        __syncthreads();
        if (threadIdx.x < d) {
            double t = 0.0;
            for (int q = 0; q < S; ++q) t += seg[q * dr + threadIdx.x];
            const double sv = sigma * t;
            const double dx = x[1 + threadIdx.x] - (xbar ? xbar[1 + threadIdx.x] : x[1 + threadIdx.x]);
            f.grad[1 + threadIdx.x] = -sv + tos * dx;
            nv2 = sv * sv;
            dx2 = dx * dx;
        }
    } else {
        const double* __restrict__ xr = x; const double* __restrict__ xbr = xbar ? xbar : x;
        double* __restrict__ gr = f.grad;
#pragma unroll 4
        for (int j = threadIdx.x; j < d; j += FBLOCK) {
            double s = 0.0;
            for (int b = 0; b < nvec; ++b) s += part_vec[(size_t)b * dpad + j];
            const double sv = sigma * s;
            const double dx = xr[1 + j] - xbr[1 + j];
            gr[1 + j] = -sv + tos * dx;
            nv2 = fma(sv, sv, nv2);
            dx2 = fma(dx, dx, dx2);
        }
    }
    { double dummy = 0.0; ctrl_block_sum3(nv2, dx2, dummy, sm); }
    __syncthreads();
    if (threadIdx.x == 0) {
        const bool cut = f.S && sc[MEB_PART_CUT] != 0.0;       // a CTA stopped early: certainly rejected (MebDyn::s0_abort)
        if (cut) sS.aborted++;
        if (f.S) {
            int np = f.multi_part ? sS.dyn.multi_n : 0;
            if (np > MEB_MULTI_MAX) np = MEB_MULTI_MAX;
            sS.pred_n = np;
            for (int k = 0; k < np; ++k) sS.pred_s[k] = multi_s[k];
        }
        if (f.S) {
            const long long t0 = __double_as_longlong(sm[100]), t1 = __double_as_longlong(sm[101]);
            if (t1 > t0) {
                const int q = sS.evals < 48 ? sS.evals : 47;          // MEB_TRACE history, indexed by evaluation
                sS.pass_hist[q] = (uint32_t)(t1 - t0);
                sS.act_hist[q] = cut ? 0xffffffffu : (uint32_t)(sc[3] + sc[4]);
                if (!cut) {
                    sS.pass_ns += (unsigned long long)(t1 - t0); sS.pass_count++;
                    sS.vrow_reads += (unsigned long long)(sS.dyn.has_mult ? sS.n_support : 0);
                }
            }
        }
        double* out = ev_s;
        const double dx0 = x[0] - (xbar ? xbar[0] : x[0]);
        dx2 += dx0 * dx0;
        f.grad[0] = 1.0 - sc[1] + tos * dx0;
        out[MEB_EV_PSI] = cut ? 1e290 : x[0] + 0.5 * sigma * sc[0] + 0.5 * tos * dx2;
        out[MEB_EV_SUM_UPLUS] = sc[1];
        out[MEB_EV_SUM_PROJ2] = sc[0];
        out[MEB_EV_SUM_DMULT2] = sc[2];
        out[MEB_EV_N_B1] = sc[3];
        out[MEB_EV_N_B3] = sc[4];
        out[MEB_EV_MAX_PFEAS] = sc[5];
        out[MEB_EV_MAX_COMPL] = sc[6];
        out[MEB_EV_MAX_DFEAS] = sc[7];
        out[MEB_EV_SUM_RHO] = sc[8];
        out[MEB_EV_NORM_SUM_VPLUS] = sqrt(nv2);
        out[MEB_EV_N_ACTIVE] = sc[3] + sc[4];          // active <=> branch B1 or B3
        out[12] = dx2;
        out[13] = 0.0; out[14] = 0.0; out[15] = 0.0;
    }
    __syncthreads();
    if (threadIdx.x < MEB_EVAL_NSCALARS) f.out[threadIdx.x] = ev_s[threadIdx.x];
    if (f.S) ctrl_after_eval(f.S, &sS, f.v, ev_s, sm);
}

// H q from the active-list partials (reading 1):
//  (Hq)_0 = (tau/sigma) q0 + sigma [ n1 q0 + 1/2 (n3 q0 + sum_{B3} w^T q1) ]
//  (Hq)_1 = (tau/sigma) q1 + sigma [ n1 q1 + 1/2 (sum_{B3} coef b + (n3 + sum rho) q1) ]
__global__ void __launch_bounds__(FBLOCK) hvp_finalize_kernel(
    const double* __restrict__ part_vec, int nvec, int tpb, const int32_t* __restrict__ count, int dpad,
    const double* __restrict__ part_sc, const double* __restrict__ ev, const double* __restrict__ q,
    double sigma, double tau, int d, double* __restrict__ Hq, const MebDyn* __restrict__ dyn, int nsc, int sc_stride) {
    if (dyn) { sigma = dyn->sigma_raw; tau = dyn->tau_eff; }
    const double n1 = ev[MEB_EV_N_B1], n3 = ev[MEB_EV_N_B3], srho = ev[MEB_EV_SUM_RHO];
    const double tos = tau / sigma;
    if (tpb > 0) { const int used = (*count + tpb - 1) / tpb; if (nvec > used) nvec = used; }
    for (int j = threadIdx.x; j < d; j += FBLOCK) {
        double s = 0.0;
        for (int b = 0; b < nvec; ++b) s += part_vec[(size_t)b * dpad + j];
        const double qj = q[1 + j];
        Hq[1 + j] = tos * qj + sigma * (n1 * qj + 0.5 * (s + (n3 + srho) * qj));
    }
    if (threadIdx.x < 32) {
        double s = 0.0;
        for (int b = threadIdx.x; b < nsc; b += 32) s += part_sc[(size_t)b * sc_stride];   // CTAs without list entries wrote 0
        s = warp_sum(s);
        if (threadIdx.x == 0) Hq[0] = tos * q[0] + sigma * (n1 * q[0] + 0.5 * (n3 * q[0] + s));
    }
}

// Long vectors (d > 1024): the per-CTA vector partials are first added by MANY CTAs (32 columns each, the 8
// warps of a CTA take interleaved partials and are then added in warp order: fixed order), so that the
// single-CTA finalize kernels read one vector instead of nvec of them.
__global__ void __launch_bounds__(256) reduce_partials_kernel(const double* __restrict__ part_vec, int nvec, int tpb,
                                                              const int32_t* __restrict__ count, int dpad, int d,
                                                              double* __restrict__ out) {
    __shared__ double sm[8][32];
    if (tpb > 0) { const int used = (*count + tpb - 1) / tpb; if (nvec > used) nvec = used; }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int j = blockIdx.x * 32 + lane;
    double s = 0.0;
    if (j < d)
        for (int b = warp; b < nvec; b += 8) s += part_vec[(size_t)b * dpad + j];
    sm[warp][lane] = s;
    __syncthreads();
    if (warp == 0 && j < d) {
        double t = 0.0;
#pragma unroll
        for (int w = 0; w < 8; ++w) t += sm[w][lane];
        out[j] = t;
    }
}

// arg-max style partials (feasibility / ingest): out[0] = max value, out[1] = index, out[2] = count sum
__global__ void __launch_bounds__(32) argmax_finalize_kernel(const double* __restrict__ part, int grid,
                                                             double* __restrict__ out) {
    const int lane = threadIdx.x;
    double bv = 0.0, bi = -1.0, cnt = 0.0;
    for (int b = lane; b < grid; b += 32) {
        const double v = part[(size_t)b * MEB_NPART], i = part[(size_t)b * MEB_NPART + 1];
        cnt += part[(size_t)b * MEB_NPART + 2];
        if (i >= 0.0 && (bi < 0.0 || v > bv || (v == bv && i < bi))) { bv = v; bi = i; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const double ov = __shfl_xor_sync(MEB_FULL_MASK, bv, o);
        const double oi = __shfl_xor_sync(MEB_FULL_MASK, bi, o);
        if (oi >= 0.0 && (bi < 0.0 || ov > bv || (ov == bv && oi < bi))) { bv = ov; bi = oi; }
    }
    cnt = warp_sum(cnt);
    if (lane == 0) { out[0] = bv; out[1] = bi; out[2] = cnt; }
}

__global__ void __launch_bounds__(32) scalar_sum_kernel(const double* __restrict__ v, int n,
                                                        double* __restrict__ out) {
    double s = 0.0;
    for (int b = threadIdx.x; b < n; b += 32) s += v[b];
    s = warp_sum(s);
    if (threadIdx.x == 0) out[0] = s;
}

// c0 = mean of the S rows floor(k m / S) (reading 3).  Stage 1: CTA (x, g) adds the rows of sample
// chunk g (S/32 rows, in order) for 256 columns -> part[g][j]; stage 2 adds the 32 chunks in order.
constexpr int SM_CHUNKS = 32;
__global__ void __launch_bounds__(256) sample_mean_kernel(const double* __restrict__ C, int64_t ld,
                                                          int64_t m, int d, int S,
                                                          double* __restrict__ part) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    const int g = blockIdx.y;
    if (j >= d) return;
    const int per = (S + SM_CHUNKS - 1) / SM_CHUNKS;
    const int k0 = g * per, k1 = min(S, k0 + per);
    double s = 0.0;
#pragma unroll 4
    for (int k = k0; k < k1; ++k) s += C[(((int64_t)k * m) / S) * ld + j];
    part[(size_t)g * d + j] = s;
}
__global__ void __launch_bounds__(256) sample_mean_final_kernel(const double* __restrict__ part, int d, int S,
                                                                double* __restrict__ c0) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= d) return;
    double s = 0.0;
#pragma unroll
    for (int g = 0; g < SM_CHUNKS; ++g) s += part[(size_t)g * d + j];
    c0[j] = s / (double)S;
}

template <typename T>
__global__ void fill_kernel(T* p, int64_t n, T v) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (int64_t)gridDim.x * blockDim.x)
        p[i] = v;
}

// gather rows idx[k] of a row-major matrix (and convert): reduced problem of P:L265-269
template <typename TI, typename TO>
__global__ void __launch_bounds__(256) gather_rows_kernel(const TI* __restrict__ src, int64_t ld_src,
                                                          const int32_t* __restrict__ idx, int64_t n, int d,
                                                          TO* __restrict__ dst, int64_t ld_dst,
                                                          const double* __restrict__ add) {
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    const int nw = (gridDim.x * blockDim.x) >> 5;
    for (int64_t k = warp; k < n; k += nw) {
        const TI* s = src + (int64_t)idx[k] * ld_src;
        TO* o = dst + k * ld_dst;
        for (int j = lane; j < d; j += 32) o[j] = (TO)s[j] + (add ? (TO)add[j] : (TO)0);
    }
}

template <typename TI, typename TO>
__global__ void __launch_bounds__(256) gather_vec_kernel(const TI* __restrict__ src,
                                                         const int32_t* __restrict__ idx, int64_t n,
                                                         TO* __restrict__ dst) {
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n;
         k += (int64_t)gridDim.x * blockDim.x)
        dst[k] = src ? (TO)src[idx[k]] : (TO)0;
}

// reduced-problem multipliers from the FP32 run: for list entry k (ball i = idx[k]):
// U_red[k] = U32[i]; if slot32[i] >= 0: V_red row k = V32 row slot32[i], slot_red[k] = k else -1
__global__ void __launch_bounds__(256) gather_mult_kernel(const float* __restrict__ U32,
                                                          const int32_t* __restrict__ slot32,
                                                          const float* __restrict__ V32, int64_t ldv32,
                                                          const int32_t* __restrict__ idx, int64_t n, int d,
                                                          double* __restrict__ U, int32_t* __restrict__ slot,
                                                          double* __restrict__ V, int64_t ldv) {
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    const int nw = (gridDim.x * blockDim.x) >> 5;
    for (int64_t k = warp; k < n; k += nw) {
        const int i = idx[k];
        const int s = slot32 ? slot32[i] : -1;
        if (lane == 0) { U[k] = (double)U32[i]; slot[k] = s >= 0 ? (int32_t)k : -1; }
        if (s >= 0)
            for (int j = lane; j < d; j += 32) V[k * ldv + j] = (double)V32[(int64_t)s * ldv32 + j];
    }
}

__global__ void set_kept_kernel(const int32_t* __restrict__ idx, int64_t n, uint8_t* __restrict__ kept) {
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n;
         k += (int64_t)gridDim.x * blockDim.x)
        kept[idx[k]] = 1;
}

}  // namespace

// ---- host wrappers ---------------------------------------------------------------------------------
int meb_eval_finalize(meb_ctx* ctx, const FinalizeArgs& f_in) {
    FinalizeArgs f = f_in;
    if (ctx->shard) {
        // sharded solve: first level of the reduction here, the ranks' records are added in rank order below
        int rc = meb_shard_pack_eval(ctx, f.part, f.grid, f.part_vec, f.nvec, f.tpb, f.count, f.dpad, f.d, f.multi_part);
        if (rc != MEB_OK) return rc;
        const int64_t rs = 16 + ((int64_t)f.d + 7) / 8 * 8;
        rc = meb_shard_exchange(ctx, rs);
        if (rc != MEB_OK) return rc;
        const double* rv = ctx->shard->recv;
        f.part = rv; f.grid = ctx->shard->nranks; f.part_stride = (int)rs;
        f.part_vec = rv + 16; f.nvec = ctx->shard->nranks; f.tpb = 0; f.dpad = (int)rs; f.vec_stride = 0;
        if (f.multi_part) { f.multi_part = rv + MEB_NPART; f.multi_stride = (int)rs; }
    }
    if (f.d > 256 && f.nvec > 8) {                 // long vectors: add the partials with many CTAs first
        ctx->launches++;
        reduce_partials_kernel<<<(f.d + 31) / 32, 256, 0, ctx->stream>>>(f.part_vec, f.nvec, f.tpb, f.count, f.dpad, f.d,
                                                                        ctx->part_red);
        f.part_vec = ctx->part_red; f.nvec = 1; f.tpb = 0;
    }
    ctx->launches++; eval_finalize_kernel<<<1, FBLOCK, 0, ctx->stream>>>(f);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}

int meb_hvp_finalize(meb_ctx* ctx, int nvec, int dpad, const double* part_sc, const double* ev,
                     const double* q, double sigma, double tau, int d, double* Hq, const MebDyn* dyn) {
    int tpb = d > 2048 ? 1 : MEB_WARPS;
    if (ctx->shard) {
        // sharded solve: this rank's partial goes into its record, the records of all ranks come back in rank order
        int rc = meb_shard_pack_hvp(ctx, part_sc, nvec, ctx->part_vec, nvec, tpb, ctx->count_dev, dpad, d);
        if (rc != MEB_OK) return rc;
        const int64_t rs = 8 + dpad;
        rc = meb_shard_exchange(ctx, rs);
        if (rc != MEB_OK) return rc;
        const double* rv = ctx->shard->recv;
        ctx->launches++;
        hvp_finalize_kernel<<<1, FBLOCK, 0, ctx->stream>>>(rv + 8, ctx->shard->nranks, 0, ctx->count_dev, (int)rs, rv, ev, q, sigma, tau, d,
                                                          Hq, dyn, ctx->shard->nranks, (int)rs);
        MEB_CUDA_OK(ctx, cudaGetLastError());
        return MEB_OK;
    }
    const double* pv = ctx->part_vec;
    int nv = nvec;
    if (d > 128 && nvec > 8) {                     // long vectors: add the partials with many CTAs first
        ctx->launches++;
        reduce_partials_kernel<<<(d + 31) / 32, 256, 0, ctx->stream>>>(ctx->part_vec, nvec, tpb, ctx->count_dev, dpad, d,
                                                                      ctx->part_red);
        pv = ctx->part_red; nv = 1;
    }
    ctx->launches++; hvp_finalize_kernel<<<1, FBLOCK, 0, ctx->stream>>>(pv, nv, nv == 1 && pv == ctx->part_red ? 0 : tpb, ctx->count_dev, dpad,
                                                       part_sc, ev, q, sigma, tau, d, Hq, dyn, nvec, 1);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}

int meb_argmax_finalize(meb_ctx* ctx, int grid, double* out) {
    ctx->launches++; argmax_finalize_kernel<<<1, 32, 0, ctx->stream>>>(ctx->part_scalar, grid, out);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}

int meb_scalar_sum(meb_ctx* ctx, const double* v, int n, double* out) {
    ctx->launches++; scalar_sum_kernel<<<1, 32, 0, ctx->stream>>>(v, n, out);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}

int meb_sample_mean(meb_ctx* ctx, const double* C, int64_t ld, int64_t m, int d, int S, double* c0) {
    const int gx = (d + 255) / 256;
    double* part = ctx->part_vec;                  // [32][d] scratch: vec_rows >= 32 rows of >= d doubles
    ctx->launches++; sample_mean_kernel<<<dim3(gx, SM_CHUNKS), 256, 0, ctx->stream>>>(C, ld, m, d, S, part);
    ctx->launches++; sample_mean_final_kernel<<<gx, 256, 0, ctx->stream>>>(part, d, S, c0);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}

static int grid_for(int64_t n, int per) {
    int64_t g = (n + per - 1) / per;
    if (g < 1) g = 1;
    if (g > 148 * 8) g = 148 * 8;
    return (int)g;
}

int meb_fill_f64(meb_ctx* ctx, double* p, int64_t n, double v) {
    ctx->launches++; fill_kernel<double><<<grid_for(n, 1024), 256, 0, ctx->stream>>>(p, n, v);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}
int meb_fill_f32(meb_ctx* ctx, float* p, int64_t n, float v) {
    ctx->launches++; fill_kernel<float><<<grid_for(n, 1024), 256, 0, ctx->stream>>>(p, n, v);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}
int meb_fill_i32(meb_ctx* ctx, int32_t* p, int64_t n, int32_t v) {
    ctx->launches++; fill_kernel<int32_t><<<grid_for(n, 1024), 256, 0, ctx->stream>>>(p, n, v);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}
int meb_fill_u8(meb_ctx* ctx, uint8_t* p, int64_t n, uint8_t v) {
    ctx->launches++; fill_kernel<uint8_t><<<grid_for(n, 1024), 256, 0, ctx->stream>>>(p, n, v);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}

int meb_gather_rows_f64(meb_ctx* ctx, const double* src, int64_t ld_src, const int32_t* idx, int64_t n, int d,
                        double* dst, int64_t ld_dst) {
    if (n <= 0) return MEB_OK;
    ctx->launches++; gather_rows_kernel<double, double><<<grid_for(n, 8), 256, 0, ctx->stream>>>(src, ld_src, idx, n, d, dst,
                                                                                 ld_dst, nullptr);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}
int meb_gather_vec_f64(meb_ctx* ctx, const double* src, const int32_t* idx, int64_t n, double* dst) {
    if (n <= 0) return MEB_OK;
    ctx->launches++; gather_vec_kernel<double, double><<<grid_for(n, 256), 256, 0, ctx->stream>>>(src, idx, n, dst);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}
int meb_gather_mult(meb_ctx* ctx, const float* U32, const int32_t* slot32, const float* V32, int64_t ldv32,
                    const int32_t* idx, int64_t n, int d, double* U, int32_t* slot, double* V, int64_t ldv) {
    if (n <= 0) return MEB_OK;
    ctx->launches++; gather_mult_kernel<<<grid_for(n, 8), 256, 0, ctx->stream>>>(U32, slot32, V32, ldv32, idx, n, d, U, slot, V,
                                                                ldv);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}
int meb_set_kept(meb_ctx* ctx, const int32_t* idx, int64_t n, uint8_t* kept) {
    if (n <= 0) return MEB_OK;
    ctx->launches++; set_kept_kernel<<<grid_for(n, 256), 256, 0, ctx->stream>>>(idx, n, kept);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}
