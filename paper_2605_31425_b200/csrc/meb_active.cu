// Passes over the ACTIVE balls only (lam_i != 0), driven by the compacted ascending index list
// (SURVEY 8(a) rows a1 vector part, a2, a6).  Only active rows contribute to sum_i v+_i and to
// sum_i P_i q, so these kernels touch |A| rows, not m.
//
//   MODE_ROWSUM   sum_k lam_k b_k                      -> gradient, P:L111 / L232
//   MODE_HVP      sum_{B3} coef_k b_k, sum_{B3} w_k^T q1   -> H q, P:L214-216 (P_i: reading 1)
//   MODE_WRITEV   v_k <- sigma lam_k b_k, u_i <- sigma t_i, slot_i <- k   -> eq. (6)
//
// A TEAM of threads (one warp, or the whole CTA for long rows) owns a list entry; thread t of the
// team owns columns t, t+TEAM, ... and accumulates them in its own slice of shared memory, so there
// are no atomics and the summation order is fixed: entries k = team, team + nteams, ... in order,
// then teams of a CTA in order, then CTAs in order (finalize kernels in meb_small.cu).
#include "meb_internal.cuh"

namespace {

template <int TEAM>
__device__ __forceinline__ double team_sum(double v, double* scratch) {
    v = warp_sum(v);
    if (TEAM == 32) return v;
    // whole CTA: combine the warps in index order
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) scratch[warp] = v;
    __syncthreads();
    double t = 0.0;
#pragma unroll
    for (int w = 0; w < MEB_WARPS; ++w) t += scratch[w];
    return t;
}

template <typename T, int TEAM, int MODE>
__global__ void __launch_bounds__(MEB_BLOCK, (MODE == MODE_WRITEV && TEAM == 32) ? 3 : 1) active_kernel(const ActiveArgs a_in) {
    ActiveArgs a = a_in;
    meb_resolve_dyn(a);
    extern __shared__ __align__(16) double acc_s[];          // [teams_per_block][dpad]
    __shared__ double scratch[MEB_WARPS];
    __shared__ double sc_red[MEB_WARPS];
    constexpr int TPB = MEB_BLOCK / TEAM;
    const int team = threadIdx.x / TEAM, tt = threadIdx.x % TEAM;
    const int d = a.d;
    double* acc = acc_s + (size_t)team * a.dpad;
    if (MODE == MODE_ROWSUM && a.cut_part != nullptr) {
        int cut = 0;
        for (int b = threadIdx.x; b < a.cut_grid; b += MEB_BLOCK)
            cut |= a.cut_part[(size_t)b * MEB_NPART + MEB_PART_CUT] != 0.0;
        if (__syncthreads_or(cut)) {                         // rejected trial: zero partials, nothing to read
            double* pv = a.part_vec + (size_t)blockIdx.x * a.dpad;
            for (int j = threadIdx.x; j < a.dpad; j += MEB_BLOCK) pv[j] = 0.0;
            if (threadIdx.x == 0) a.part_sc[blockIdx.x] = 0.0;
            return;
        }
    }
    if (blockIdx.x * TPB >= *a.count) {                      // no list entry for this CTA: the finalize
        if (threadIdx.x == 0) a.part_sc[blockIdx.x] = 0.0;   // kernels skip its vector partial
        return;
    }
    if (MODE != MODE_WRITEV)
        for (int j = tt; j < a.dpad; j += TEAM) acc[j] = 0.0;
    const T* __restrict__ C = static_cast<const T*>(a.C);
    const T* __restrict__ V = static_cast<const T*>(a.V);
    const double* __restrict__ cx = a.x + 1;
    const T inv_sig = T(1) / (T)a.sigma;
    const int n = *a.count;
    const int nteams = gridDim.x * TPB;
    double sc = 0.0;                                         // scalar partial (one per team, in thread 0)
    int kstart = blockIdx.x * TPB + team;
    if (MODE == MODE_WRITEV && TEAM == 32 && d <= 64) {
        // Short rows: the gather list[k] -> (slot, lam, t) -> rows of C and V is three dependent global loads per
        // entry, and one entry per warp at a time leaves the pass latency-bound (config 4: 5e6 entries, 3.8 ms).
        // Four entries of the team's sequence are loaded level by level, then written; same entries, same order
        // and same arithmetic as the loop below (fma(0, 1/sigma, b) = b for a row without v_i).
        constexpr int UB = 4, EP = 2;
        for (int kb = kstart; kb < n; kb += nteams * UB) {
            int ii[UB], sl[UB];
            double lam[UB], tv[UB];
            T cv[UB][EP], vv[UB][EP];
#pragma unroll
            for (int u = 0; u < UB; ++u) {
                const long long k = (long long)kb + (long long)u * nteams;
                ii[u] = k < n ? a.list[k] : -1;
            }
#pragma unroll
            for (int u = 0; u < UB; ++u) {
                const int i = ii[u];
                sl[u] = (i >= 0 && a.v_slot) ? a.v_slot[i] : -1;
                lam[u] = i >= 0 ? a.rec_lam[i] : 0.0;
                tv[u] = i >= 0 ? a.rec_t[i] : 0.0;
            }
#pragma unroll
            for (int u = 0; u < UB; ++u) {
                const T* rowp = C + (int64_t)(ii[u] >= 0 ? ii[u] : 0) * a.ld;
                const T* vrow = V + (int64_t)(sl[u] >= 0 ? sl[u] : 0) * a.ldv;
#pragma unroll
                for (int e = 0; e < EP; ++e) {
                    const int j = tt + 32 * e;
                    cv[u][e] = (ii[u] >= 0 && j < d) ? rowp[j] : T(0);
                    vv[u][e] = (sl[u] >= 0 && j < d) ? vrow[j] : T(0);
                }
            }
#pragma unroll
            for (int u = 0; u < UB; ++u) {
                if (ii[u] < 0) continue;                             // team-uniform
                const int k = kb + u * nteams;
                const T sl_ = (T)(a.sigma * lam[u]);
                T* vout = static_cast<T*>(a.V_out) + (int64_t)k * a.ldv_out;
                const bool store = k < a.cap_rows;
                double nb2 = 0.0;
#pragma unroll
                for (int e = 0; e < EP; ++e) {
                    const int j = tt + 32 * e;
                    if (j < d) {
                        T b = cv[u][e] - (T)cx[j];
                        b = fma(vv[u][e], inv_sig, b);
                        const T vp = sl_ * b;
                        if (store) vout[j] = vp;
                        nb2 = fma((double)vp, (double)vp, nb2);
                    }
                }
                nb2 = team_sum<TEAM>(nb2, scratch);
                if (tt == 0) {
                    const T up = (T)a.sigma * (T)tv[u];
                    static_cast<T*>(a.U_out)[ii[u]] = up;
                    a.slot_out[ii[u]] = store ? k : -1;
                    sc += (double)up * (double)up + nb2;
                }
            }
        }
        kstart = n;
    }
    if (MODE == MODE_ROWSUM && TEAM == MEB_BLOCK) {
        // Long rows, whole CTA per entry: FOUR entries of the CTA's sequence per sweep over the columns, so that a
        // thread has eight independent loads in flight per column instead of a load -> shared-memory update chain
        // per entry (the entries are still added in list order: a fixed chain of four FMAs per column).
        for (int kb = kstart; kb < n; kb += nteams * 4) {
            const T* rp[4]; const T* vp[4]; double lam[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const long long k = (long long)kb + (long long)u * nteams;
                const int i = k < n ? a.list[k] : -1;
                lam[u] = i >= 0 ? a.rec_lam[i] : 0.0;
                rp[u] = C + (int64_t)(i >= 0 ? i : 0) * a.ld;
                const int slot = (i >= 0 && a.v_slot) ? a.v_slot[i] : -1;
                vp[u] = slot >= 0 ? V + (int64_t)slot * a.ldv : nullptr;
            }
#pragma unroll 2
            for (int j = tt; j < d; j += TEAM) {
                const T cj = (T)cx[j];
                T b4[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    b4[u] = rp[u][j] - cj;
                    if (vp[u]) b4[u] = fma(vp[u][j], inv_sig, b4[u]);
                }
                double s = acc[j];
#pragma unroll
                for (int u = 0; u < 4; ++u) s = fma(lam[u], (double)b4[u], s);
                acc[j] = s;
            }
        }
        kstart = n;
    }
    for (int k = kstart; k < n; k += nteams) {
        const int i = a.list[k];
        const T* rowp = C + (int64_t)i * a.ld;
        const int slot = a.v_slot ? a.v_slot[i] : -1;
        const T* vrow = slot >= 0 ? V + (int64_t)slot * a.ldv : nullptr;
        if (MODE == MODE_ROWSUM) {
            const double lam = a.rec_lam[i];
            for (int j = tt; j < d; j += TEAM) {
                T b = rowp[j] - (T)cx[j];
                if (vrow) b = fma(vrow[j], inv_sig, b);
                acc[j] = fma(lam, (double)b, acc[j]);
            }
        } else if (MODE == MODE_HVP) {
            const double rho = a.rec_rho[i];
            if (rho > 1.5) continue;                          // B1: P_i = I, handled in the finalize
            double dot = 0.0, nb2 = 0.0;
            for (int j = tt; j < d; j += TEAM) {
                T b = rowp[j] - (T)cx[j];
                if (vrow) b = fma(vrow[j], inv_sig, b);
                const double bd = (double)b;
                dot = fma(bd, a.q[1 + j], dot);
                nb2 = fma(bd, bd, nb2);
            }
            dot = team_sum<TEAM>(dot, scratch);
            nb2 = team_sum<TEAM>(nb2, scratch);
            const double nb = sqrt(nb2);
            const double wq = dot / nb;                       // w_i^T q1
            const double coef = (a.q[0] - rho * wq) / nb;     // (P_i q)_1 = 1/2 (coef b + (1+rho) q1)
            for (int j = tt; j < d; j += TEAM) {
                T b = rowp[j] - (T)cx[j];
                if (vrow) b = fma(vrow[j], inv_sig, b);
                acc[j] = fma(coef, (double)b, acc[j]);
            }
            if (tt == 0) sc += wq;
        } else {  // MODE_WRITEV
            const double lam = a.rec_lam[i], t = a.rec_t[i];
            const T sl = (T)(a.sigma * lam);
            T* vout = static_cast<T*>(a.V_out) + (int64_t)k * a.ldv_out;
            const bool store = k < a.cap_rows;
            double nb2 = 0.0;
            for (int j = tt; j < d; j += TEAM) {
                T b = rowp[j] - (T)cx[j];
                if (vrow) b = fma(vrow[j], inv_sig, b);
                const T vp = sl * b;
                if (store) vout[j] = vp;
                nb2 = fma((double)vp, (double)vp, nb2);
            }
            nb2 = team_sum<TEAM>(nb2, scratch);
            if (tt == 0) {
                const T up = (T)a.sigma * (T)t;
                static_cast<T*>(a.U_out)[i] = up;
                a.slot_out[i] = store ? k : -1;
                sc += (double)up * (double)up + nb2;
            }
        }
    }
    // ---- CTA partials, fixed order ----
    __syncthreads();
    if (MODE != MODE_WRITEV) {
        double* pv = a.part_vec + (size_t)blockIdx.x * a.dpad;
        for (int j = threadIdx.x; j < d; j += MEB_BLOCK) {
            double s = 0.0;
#pragma unroll
            for (int tm = 0; tm < TPB; ++tm) s += acc_s[(size_t)tm * a.dpad + j];
            pv[j] = s;
        }
    }
    // scalar partial: teams in order
    if (TEAM == 32) {
        if (tt == 0) sc_red[team] = sc;
        __syncthreads();
        if (threadIdx.x == 0) {
            double s = 0.0;
            for (int tm = 0; tm < TPB; ++tm) s += sc_red[tm];
            a.part_sc[blockIdx.x] = s;
        }
    } else if (threadIdx.x == 0) {
        a.part_sc[blockIdx.x] = sc;
    }
}

// MODE_WRITEV for SHORT rows (d <= 32): eight lanes per list entry, four consecutive entries per warp and step, lane l8 of
// an entry owning the columns l8, l8 + 8, ...  A warp per entry spent 130 instructions on a row of 32 numbers and kept
// one row per warp in flight; here the instructions are shared by four rows and UB steps (16 rows per warp) are loaded
// level by level (list -> slot, lam, t -> rows of C and V) before any is used.  Consecutive entries are neighbouring
// balls and consecutive rows of the new pool, so the four rows of a step are read and written as one run.
// Same arithmetic per entry as the generic loop (fma(0, 1/sigma, b) = b for a row without v_i); ||v+||^2 is added over
// the eight lanes by an xor tree, entries in the fixed order of the static partition.
template <typename T>
__global__ void __launch_bounds__(MEB_BLOCK, 2) writev_short_kernel(const ActiveArgs a_in) {
    ActiveArgs a = a_in;
    meb_resolve_dyn(a);
    __shared__ double sc_red[MEB_WARPS];
    constexpr int UB = 4, EL = 4;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int sub = lane >> 3, l8 = lane & 7;
    const int d = a.d;
    const int n = *a.count;
    const T* __restrict__ C = static_cast<const T*>(a.C);
    const T* __restrict__ V = static_cast<const T*>(a.V);
    const T inv_sig = T(1) / (T)a.sigma;
    T cxe[EL];
#pragma unroll
    for (int e = 0; e < EL; ++e) cxe[e] = (l8 + 8 * e) < d ? (T)a.x[1 + l8 + 8 * e] : T(0);
    const long long NW = (long long)gridDim.x * MEB_WARPS;
    double sc = 0.0;
    for (long long q0 = (long long)blockIdx.x * MEB_WARPS + warp; q0 * 4 < n; q0 += NW * UB) {
        int ii[UB], sl[UB];
        long long kk[UB];
        double lam[UB], tv[UB];
        T cv[UB][EL], vv[UB][EL];
#pragma unroll
        for (int u = 0; u < UB; ++u) {
            kk[u] = (q0 + (long long)u * NW) * 4 + sub;
            ii[u] = kk[u] < n ? a.list[kk[u]] : -1;
        }
#pragma unroll
        for (int u = 0; u < UB; ++u) {
            const int i = ii[u];
            sl[u] = (i >= 0 && a.v_slot) ? a.v_slot[i] : -1;
            lam[u] = i >= 0 ? a.rec_lam[i] : 0.0;
            tv[u] = i >= 0 ? a.rec_t[i] : 0.0;
        }
#pragma unroll
        for (int u = 0; u < UB; ++u) {
            const T* rowp = C + (int64_t)(ii[u] >= 0 ? ii[u] : 0) * a.ld;
            const T* vrow = V + (int64_t)(sl[u] >= 0 ? sl[u] : 0) * a.ldv;
#pragma unroll
            for (int e = 0; e < EL; ++e) {
                const int j = l8 + 8 * e;
                cv[u][e] = (ii[u] >= 0 && j < d) ? rowp[j] : T(0);
                vv[u][e] = (sl[u] >= 0 && j < d) ? vrow[j] : T(0);
            }
        }
#pragma unroll
        for (int u = 0; u < UB; ++u) {
            const bool on = ii[u] >= 0;
            const T sl_ = (T)(a.sigma * lam[u]);
            T* vout = static_cast<T*>(a.V_out) + (int64_t)kk[u] * a.ldv_out;
            const bool store = on && kk[u] < a.cap_rows;
            double nb2 = 0.0;
#pragma unroll
            for (int e = 0; e < EL; ++e) {
                const int j = l8 + 8 * e;
                if (j < d) {
                    T b = cv[u][e] - cxe[e];
                    b = fma(vv[u][e], inv_sig, b);
                    const T vp = sl_ * b;
                    if (store) vout[j] = vp;
                    nb2 = fma((double)vp, (double)vp, nb2);
                }
            }
            nb2 += __shfl_xor_sync(MEB_FULL_MASK, nb2, 1);
            nb2 += __shfl_xor_sync(MEB_FULL_MASK, nb2, 2);
            nb2 += __shfl_xor_sync(MEB_FULL_MASK, nb2, 4);
            if (on && l8 == 0) {
                const T up = (T)a.sigma * (T)tv[u];
                static_cast<T*>(a.U_out)[ii[u]] = up;
                a.slot_out[ii[u]] = store ? (int32_t)kk[u] : -1;
                sc += (double)up * (double)up + nb2;
            }
        }
    }
    // scalar partial: the four entries of a warp, then the warps, in index order
    sc += __shfl_xor_sync(MEB_FULL_MASK, sc, 8);
    sc += __shfl_xor_sync(MEB_FULL_MASK, sc, 16);
    if (lane == 0) sc_red[warp] = sc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < MEB_WARPS; ++w) t += sc_red[w];
        a.part_sc[blockIdx.x] = t;
    }
}

template <typename T, int MODE>
int launch_active_t(meb_ctx* ctx, const ActiveArgs& a, int* grid_out) {
    const bool wide = a.d > 2048;
    const int tpb = wide ? 1 : MEB_WARPS;
    const size_t smem = (MODE == MODE_WRITEV) ? 0 : (size_t)tpb * a.dpad * sizeof(double);
    if (smem > 220 * 1024) return MEB_E_CAPACITY;
    int grid = ctx->sm_count * (smem > 100 * 1024 ? 1 : 2);
    if ((int64_t)grid > ctx->vec_rows) grid = (int)ctx->vec_rows;
    if (MODE == MODE_WRITEV && !wide) {          // no vector partials: as many CTAs as fit (part_sc holds 1024)
        grid = ctx->sm_count * 4;
        if (grid > 1024) grid = 1024;
    }
    cudaError_t e;
    if (MODE == MODE_WRITEV && a.d <= 32) {
        grid = ctx->sm_count * 2;
        ctx->launches++;
        writev_short_kernel<T><<<grid, MEB_BLOCK, 0, ctx->stream>>>(a);
        e = cudaSuccess;
    } else if (wide) {
        auto kern = active_kernel<T, MEB_BLOCK, MODE>;
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) { ctx->launches++; kern<<<grid, MEB_BLOCK, smem, ctx->stream>>>(a); }
    } else {
        auto kern = active_kernel<T, 32, MODE>;
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) { ctx->launches++; kern<<<grid, MEB_BLOCK, smem, ctx->stream>>>(a); }
    }
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e != cudaSuccess) { ctx->last_cuda_error = (int)e; return MEB_E_CUDA; }
    *grid_out = grid;
    return MEB_OK;
}

}  // namespace

int meb_launch_active(meb_ctx* ctx, int mode, int prec, const ActiveArgs& a, int* grid_out) {
    if (prec == MEB_FP64) {
        if (mode == MODE_ROWSUM) return launch_active_t<double, MODE_ROWSUM>(ctx, a, grid_out);
        if (mode == MODE_HVP) return launch_active_t<double, MODE_HVP>(ctx, a, grid_out);
        return launch_active_t<double, MODE_WRITEV>(ctx, a, grid_out);
    }
    if (mode == MODE_ROWSUM) return launch_active_t<float, MODE_ROWSUM>(ctx, a, grid_out);
    if (mode == MODE_HVP) return launch_active_t<float, MODE_HVP>(ctx, a, grid_out);
    return launch_active_t<float, MODE_WRITEV>(ctx, a, grid_out);
}
