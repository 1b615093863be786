// Dense generalized Hessian for moderate d (SURVEY 8(a) rows a2', a3) and its Cholesky solve.
//
//   H = (tau/sigma) I + sigma [ n1 I + 1/2 [[n3, s^T],[s, (n3 + sum rho) I - sum_{B3} rho_i w_i w_i^T]] ]
//   with w_i = b_i/||b_i||, s = sum_{B3} w_i        (P:L187 with P_i of reading 1).
//
// The data-dependent part is a weighted SYRK over the ACTIVE B3 rows with SIGNED weights rho_i in
// (-1, 1).  It is FP64 and d <= 128, so it runs on the FP64 pipes: 16 x 16 threads, each owning a
// BS x BS register block of the d x d accumulator (interleaved ownership: conflict-free shared
// loads), fed from a shared tile of RB normalised rows.  Static list partition + fixed-order
// combination of the per-CTA partial matrices: deterministic.
#include <string.h>

#include "meb_internal.cuh"
#include "meb_ctrl.cuh"
#include "meb_ldlt.cuh"

namespace {

// Threads of a CTA: KS row groups of TD x TD threads; thread (ty, tx) of a group owns the B x B block
// {ty + TD i} x {tx + TD j} of the DP x DP accumulator (DP = TD * B) and group kg takes rows kg, kg + KS, ... of a
// tile.  TD = 8, KS = 4 for DP <= 48 (a 16 x 16 grid would leave 1-4 FMAs per thread and row), TD = 16, KS = 1 above.
template <int TD> struct SyrkShape {
    static constexpr int KS = MEB_BLOCK / (TD * TD);
    static constexpr int RB = TD == 8 ? 32 : 16;            // rows per shared tile
};

// The list is a gather (list[k] -> rho_i, slot_i -> rows of C and V): three dependent levels of global loads.  They
// are software-pipelined over three tiles -- while the FMAs of tile t run, the rows of tile t+1, the (rho, slot) of
// tile t+2 and the list entries of tile t+3 are in flight in registers -- because with two CTAs per SM nothing else
// hides that latency (config 4, 5e6-1e7 active rows: 3.5 ms per Hessian before the pipeline).
template <typename T, int TD, int B>
__global__ void __launch_bounds__(MEB_BLOCK) syrk_kernel(const ActiveArgs a_in, double* __restrict__ part_mat) {
    constexpr int DP = TD * B;
    constexpr int KS = SyrkShape<TD>::KS;
    constexpr int RB = SyrkShape<TD>::RB;
    constexpr int RPW = RB / MEB_WARPS;                      // rows per warp in the fill phase
    constexpr int EPL = (DP + 31) / 32;                      // elements per lane and row
    ActiveArgs a = a_in;
    meb_resolve_dyn(a);
    extern __shared__ __align__(16) double sm[];             // W[RB][DP], rho[RB], then (KS > 1) red[DP*DP + DP]
    double* W = sm;
    double* rho_s = sm + (size_t)RB * DP;
    const int tx = threadIdx.x % TD, ty = (threadIdx.x / TD) % TD, kg = threadIdx.x / (TD * TD);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int d = a.d;
    const T* __restrict__ C = static_cast<const T*>(a.C);
    const T* __restrict__ V = static_cast<const T*>(a.V);
    const T inv_sig = T(1) / (T)a.sigma;
    const int n = *a.count;
    if (blockIdx.x * RB >= n) return;                        // no tile for this CTA: the finalize skips it
    double acc[B][B];
    double accs[B];
#pragma unroll
    for (int i = 0; i < B; ++i) {
        accs[i] = 0.0;
#pragma unroll
        for (int j = 0; j < B; ++j) acc[i][j] = 0.0;
    }
    T cxr[EPL];
#pragma unroll
    for (int e = 0; e < EPL; ++e) cxr[e] = (lane + 32 * e) < d ? (T)a.x[1 + lane + 32 * e] : T(0);

    // pipeline registers of the RPW rows this warp fills
    int i_a[RPW];                                            // level 1: list entries (tile t+3)
    int i_b[RPW], slot_b[RPW]; double rho_b[RPW];            // level 2: (rho, slot) of tile t+2
    T cq[RPW][EPL], vq[RPW][EPL]; double rho_c[RPW];         // level 3: raw rows of tile t+1
    auto level1 = [&](int k0) {
#pragma unroll
        for (int r = 0; r < RPW; ++r) {
            const int k = k0 + warp * RPW + r;
            i_a[r] = (k0 >= 0 && k < n) ? a.list[k] : -1;
        }
    };
    auto level2 = [&]() {
#pragma unroll
        for (int r = 0; r < RPW; ++r) {
            const int i = i_a[r];
            i_b[r] = i;
            rho_b[r] = i >= 0 ? a.rec_rho[i] : 2.0;          // B1 rows (rho = 2): P_i = I, no SYRK term
            slot_b[r] = (i >= 0 && a.v_slot) ? a.v_slot[i] : -1;
        }
    };
    auto level3 = [&]() {
#pragma unroll
        for (int r = 0; r < RPW; ++r) {
            const int i = i_b[r];
            const double rho = rho_b[r];
            const bool use = i >= 0 && rho < 1.5;
            const int slot = slot_b[r];
            rho_c[r] = use ? rho : 2.0;
            const T* rowp = C + (int64_t)(use ? i : 0) * a.ld;
            const T* vrow = V + (int64_t)(slot >= 0 ? slot : 0) * a.ldv;
#pragma unroll
            for (int e = 0; e < EPL; ++e) {
                const int j = lane + 32 * e;
                cq[r][e] = (use && j < d) ? rowp[j] : T(0);
                vq[r][e] = (use && slot >= 0 && j < d) ? vrow[j] : T(0);
            }
        }
    };
    const int kstep = gridDim.x * RB;
    int k0 = blockIdx.x * RB;
    auto tile_at = [&](int q) {                              // first list entry of the q-th tile after k0, or -1
        const long long k = (long long)k0 + (long long)q * kstep;
        return k < n ? (int)k : -1;
    };
    level1(k0); level2(); level3();                          // tile 0 -> level 3
    level1(tile_at(1)); level2();                            // tile 1 -> level 2
    level1(tile_at(2));                                      // tile 2 -> level 1
    for (; k0 < n; k0 += kstep) {
        __syncthreads();
        // normalise the rows of this tile (level 3 registers) into shared memory
#pragma unroll
        for (int r = 0; r < RPW; ++r) {
            const int rr = warp * RPW + r;
            const bool use = rho_c[r] < 1.5;
            double bd[EPL];
            double nb2 = 0.0;
#pragma unroll
            for (int e = 0; e < EPL; ++e) {
                T b = cq[r][e] - cxr[e];
                b = fma(vq[r][e], inv_sig, b);
                bd[e] = (use && lane + 32 * e < d) ? (double)b : 0.0;
                nb2 = fma(bd[e], bd[e], nb2);
            }
            nb2 = warp_sum(nb2);
            const double inv = use ? rsqrt(nb2) : 0.0;
#pragma unroll
            for (int e = 0; e < EPL; ++e)
                if (lane + 32 * e < DP) W[(size_t)rr * DP + lane + 32 * e] = bd[e] * inv;
            if (lane == 0) rho_s[rr] = use ? rho_c[r] : 0.0;
        }
        __syncthreads();
        level3();                                            // rows of the next tile
        level2();                                            // (rho, slot) of the tile after it
        level1(tile_at(3));                                  // list entries three tiles ahead
#pragma unroll 4
        for (int rr = kg; rr < RB; rr += KS) {
            const double rho = rho_s[rr];
            const double* w = W + (size_t)rr * DP;
            double wq[B], wp[B];
#pragma unroll
            for (int j = 0; j < B; ++j) wq[j] = w[tx + TD * j];
#pragma unroll
            for (int i = 0; i < B; ++i) wp[i] = rho * w[ty + TD * i];
#pragma unroll
            for (int i = 0; i < B; ++i)
#pragma unroll
                for (int j = 0; j < B; ++j) acc[i][j] = fma(wp[i], wq[j], acc[i][j]);
            if (ty == 0) {
#pragma unroll
                for (int j = 0; j < B; ++j) accs[j] += wq[j];
            }
        }
    }
    // per-CTA partial: [DP*DP] matrix then [DP] vector; the row groups are added in index order
    double* pm = part_mat + (size_t)blockIdx.x * ((size_t)DP * DP + DP);
    if (KS > 1) {
        double* red = sm + (size_t)RB * DP + RB;
        for (int gk = 0; gk < KS; ++gk) {
            __syncthreads();
            if (kg == gk) {
#pragma unroll
                for (int i = 0; i < B; ++i)
#pragma unroll
                    for (int j = 0; j < B; ++j) {
                        const int e = (ty + TD * i) * DP + tx + TD * j;
                        red[e] = (gk == 0 ? 0.0 : red[e]) + acc[i][j];
                    }
                if (ty == 0) {
#pragma unroll
                    for (int j = 0; j < B; ++j) {
                        const int e = DP * DP + tx + TD * j;
                        red[e] = (gk == 0 ? 0.0 : red[e]) + accs[j];
                    }
                }
            }
        }
        __syncthreads();
        for (int e = threadIdx.x; e < DP * DP + DP; e += MEB_BLOCK) pm[e] = red[e];
    } else {
#pragma unroll
        for (int i = 0; i < B; ++i)
#pragma unroll
            for (int j = 0; j < B; ++j) pm[(size_t)(ty + TD * i) * DP + tx + TD * j] = acc[i][j];
        if (ty == 0) {
#pragma unroll
            for (int j = 0; j < B; ++j) pm[(size_t)DP * DP + tx + TD * j] = accs[j];
        }
    }
}

// Rows of at most 48 columns (DP = 8 B): the variant the large active sets of short-row instances run (config 4: 5e6
// rows of 32 numbers per Hessian).  Differences to syrk_kernel, which spent 180 warp instructions per row there:
//  * fill: EIGHT lanes per row (lane l8 owns the columns l8, l8 + 8, ...), so a warp normalises its four rows of the
//    tile at once -- a quarter of the loads, shuffles and rsqrt sequences per row;
//  * the fill also stores rho_i w_i next to w_i and accumulates s = sum w_i, which takes 4 multiplications and the
//    additions of s out of the inner loop of every thread;
//  * only the blocks on and below the diagonal are accumulated (B (B + 1) / 2 of B^2 FMAs per thread and row; the
//    finalize kernel reads H from the lower triangle).
// Same three-level software pipeline of the gather, same static partition and fixed-order combination.
template <typename T, int B>
__global__ void __launch_bounds__(MEB_BLOCK, B <= 4 ? 3 : 2) syrk8_kernel(const ActiveArgs a_in, double* __restrict__ part_mat) {
    constexpr int TD = 8, DP = TD * B, KS = SyrkShape<TD>::KS, RB = SyrkShape<TD>::RB;
    static_assert(RB == 4 * MEB_WARPS, "four rows per warp and tile");
    ActiveArgs a = a_in;
    meb_resolve_dyn(a);
    extern __shared__ __align__(16) double sm[];             // W[RB][DP], Wr[RB][DP], then red[DP*DP + DP]
    double* W = sm;
    double* Wr = sm + (size_t)RB * DP;
    double* red = sm + 2 * (size_t)RB * DP;
    const int tx = threadIdx.x % TD, ty = (threadIdx.x / TD) % TD, kg = threadIdx.x / (TD * TD);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int sub = lane >> 3, l8 = lane & 7;
    const int rr = warp * 4 + sub;                           // my row of a tile in the fill phase
    const int d = a.d;
    const T* __restrict__ C = static_cast<const T*>(a.C);
    const T* __restrict__ V = static_cast<const T*>(a.V);
    const T inv_sig = T(1) / (T)a.sigma;
    const int n = *a.count;
    if (blockIdx.x * RB >= n) return;                        // no tile for this CTA: the finalize skips it
    double acc[B][B];
    double accs[B];                                          // fill lanes: my columns of s = sum of the w rows I normalised
#pragma unroll
    for (int i = 0; i < B; ++i) {
        accs[i] = 0.0;
#pragma unroll
        for (int j = 0; j < B; ++j) acc[i][j] = 0.0;
    }
    T cxr[B];
#pragma unroll
    for (int e = 0; e < B; ++e) cxr[e] = (l8 + 8 * e) < d ? (T)a.x[1 + l8 + 8 * e] : T(0);
    int i_a;                                                 // level 1: list entry (tile t+3)
    int i_b, slot_b; double rho_b;                           // level 2: (rho, slot) of tile t+2
    T cq[B], vq[B]; double rho_c;                            // level 3: raw row of tile t+1
    auto level1 = [&](int k0) {
        const int k = k0 + rr;
        i_a = (k0 >= 0 && k < n) ? a.list[k] : -1;
    };
    auto level2 = [&]() {
        const int i = i_a;
        i_b = i;
        rho_b = i >= 0 ? a.rec_rho[i] : 2.0;                 // B1 rows (rho = 2): P_i = I, no SYRK term
        slot_b = (i >= 0 && a.v_slot) ? a.v_slot[i] : -1;
    };
    auto level3 = [&]() {
        const int i = i_b;
        const bool use = i >= 0 && rho_b < 1.5;
        rho_c = use ? rho_b : 2.0;
        const T* rowp = C + (int64_t)(use ? i : 0) * a.ld;
        const T* vrow = V + (int64_t)(slot_b >= 0 ? slot_b : 0) * a.ldv;
#pragma unroll
        for (int e = 0; e < B; ++e) {
            const int j = l8 + 8 * e;
            cq[e] = (use && j < d) ? rowp[j] : T(0);
            vq[e] = (use && slot_b >= 0 && j < d) ? vrow[j] : T(0);
        }
    };
    const int kstep = gridDim.x * RB;
    int k0 = blockIdx.x * RB;
    auto tile_at = [&](int q) {                              // first list entry of the q-th tile after k0, or -1
        const long long k = (long long)k0 + (long long)q * kstep;
        return k < n ? (int)k : -1;
    };
    level1(k0); level2(); level3();
    level1(tile_at(1)); level2();
    level1(tile_at(2));
    for (; k0 < n; k0 += kstep) {
        __syncthreads();
        {   // normalise my row of this tile (level 3 registers) into shared memory
            const bool use = rho_c < 1.5;
            double bd[B];
            double nb2 = 0.0;
#pragma unroll
            for (int e = 0; e < B; ++e) {
                T b = cq[e] - cxr[e];
                b = fma(vq[e], inv_sig, b);
                bd[e] = (use && l8 + 8 * e < d) ? (double)b : 0.0;
                nb2 = fma(bd[e], bd[e], nb2);
            }
            nb2 += __shfl_xor_sync(MEB_FULL_MASK, nb2, 1);
            nb2 += __shfl_xor_sync(MEB_FULL_MASK, nb2, 2);
            nb2 += __shfl_xor_sync(MEB_FULL_MASK, nb2, 4);
            const double inv = use ? rsqrt(nb2) : 0.0;
            const double rho = use ? rho_c : 0.0;
#pragma unroll
            for (int e = 0; e < B; ++e) {
                const double w = bd[e] * inv;
                W[(size_t)rr * DP + l8 + 8 * e] = w;
                Wr[(size_t)rr * DP + l8 + 8 * e] = rho * w;
                accs[e] += w;
            }
        }
        __syncthreads();
        level3();                                            // row of the next tile
        level2();                                            // (rho, slot) of the tile after it
        level1(tile_at(3));                                  // list entry three tiles ahead
#pragma unroll 4
        for (int r2 = kg; r2 < RB; r2 += KS) {
            const double* w = W + (size_t)r2 * DP;
            const double* wr = Wr + (size_t)r2 * DP;
            double wq[B], wp[B];
#pragma unroll
            for (int j = 0; j < B; ++j) wq[j] = w[tx + TD * j];
#pragma unroll
            for (int i = 0; i < B; ++i) wp[i] = wr[ty + TD * i];
#pragma unroll
            for (int i = 0; i < B; ++i)
#pragma unroll
                for (int j = 0; j <= i; ++j) acc[i][j] = fma(wp[i], wq[j], acc[i][j]);
        }
    }
    // per-CTA partial: [DP*DP] matrix (lower blocks; the others stay zero) then [DP] vector.  Row groups are added
    // in index order; s: the 32 fill rows (warp, sub) in index order.
    double* pm = part_mat + (size_t)blockIdx.x * ((size_t)DP * DP + DP);
    __syncthreads();
#pragma unroll
    for (int e = 0; e < B; ++e) W[(size_t)rr * DP + l8 + 8 * e] = accs[e];
    for (int gk = 0; gk < KS; ++gk) {
        __syncthreads();
        if (kg == gk) {
#pragma unroll
            for (int i = 0; i < B; ++i)
#pragma unroll
                for (int j = 0; j < B; ++j) {
                    const int e = (ty + TD * i) * DP + tx + TD * j;
                    red[e] = (gk == 0 ? 0.0 : red[e]) + acc[i][j];
                }
        }
    }
    if (threadIdx.x < DP) {
        double s = 0.0;
#pragma unroll 4
        for (int q = 0; q < RB; ++q) s += W[(size_t)q * DP + threadIdx.x];
        red[DP * DP + threadIdx.x] = s;
    }
    __syncthreads();
    for (int e = threadIdx.x; e < DP * DP + DP; e += MEB_BLOCK) pm[e] = red[e];
}

__global__ void __launch_bounds__(256) dense_finalize_kernel(const double* __restrict__ part_mat, int nparts,
                                                             const int32_t* __restrict__ count,
                                                             int dp, int d, const double* __restrict__ ev,
                                                             double sigma, double tau, double* __restrict__ H,
                                                             const MebDyn* __restrict__ dyn, int rb, long long pstride) {
    if (dyn) { sigma = dyn->sigma_raw; tau = dyn->tau_eff; }
    if (rb > 0) {
        const int ntiles = (*count + rb - 1) / rb;        // CTAs b < ntiles wrote a partial
        if (nparts > ntiles) nparts = ntiles;
    }
    const double n1 = ev[MEB_EV_N_B1], n3 = ev[MEB_EV_N_B3], srho = ev[MEB_EV_SUM_RHO];
    const double tos = tau / sigma;
    const int n = d + 1;
    const size_t stride = pstride > 0 ? (size_t)pstride : (size_t)dp * dp + dp;
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < n * n; e += gridDim.x * blockDim.x) {
        const int p = e / n, q = e % n;
        double v;
        if (p == 0 && q == 0) {
            v = tos + sigma * (n1 + 0.5 * n3);
        } else if (p == 0 || q == 0) {
            const int j = (p == 0 ? q : p) - 1;
            double s = 0.0;
            for (int b = 0; b < nparts; ++b) s += part_mat[b * stride + (size_t)dp * dp + j];
            v = 0.5 * sigma * s;
        } else {
            double s = 0.0;
            const int hi = (p > q ? p : q) - 1, lo = (p > q ? q : p) - 1;       // lower triangle (syrk8 fills no other)
            for (int b = 0; b < nparts; ++b) s += part_mat[b * stride + (size_t)hi * dp + lo];
            v = -0.5 * sigma * s;
            if (p == q) v += tos + sigma * (n1 + 0.5 * (n3 + srho));
        }
        H[(size_t)p * n + q] = v;
    }
}

// Solve (scale * H) delta = -g for one SPD matrix of order n <= 16*BS - 1, one CTA of 16 x 16 threads.
// Square-root-free Cholesky (H = L D L^T, no pivoting: H is SPD) on the AUGMENTED matrix
// M = [H; -g^T]: eliminating column k also updates the right-hand-side row n, so after the n column
// steps row n holds D L^{-1}(-g) and only the backward substitution with L^T is left.
// The matrix lives in REGISTERS: thread (ty, tx) owns M[ty + 16 ii][tx + 16 jj], jj <= ii < BS.
// Column steps are grouped in phases of 16 (KB = k / 16) that are unrolled at compile time, so inside
// a phase the code is straight-line: every thread updates its (BS-KB)(BS-KB+1)/2 live entries with
// multipliers masked to zero outside the trailing block (no branches), the owners of column k+1
// publish it to shared memory (where it stays as row k+1 of L D for the backward substitution)
// together with 1/d_{k+1}, computed by the diagonal's owner while the others are still updating.
// One __syncthreads per column.
template <int BS>
__global__ void __launch_bounds__(256) ldlt_solve_kernel(const double* __restrict__ H, const double* __restrict__ g,
                                                         int n, double scale, double* __restrict__ delta,
                                                         int* __restrict__ info, SolverDev* S, const SolverVecs v) {
    extern __shared__ __align__(16) double Lm[];          // LdltShape<BS>::smem_doubles(n)
    __shared__ int bad;
    const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
    double a[BS][BS];
#pragma unroll
    for (int ii = 0; ii < BS; ++ii)
#pragma unroll
        for (int jj = 0; jj < BS; ++jj) {
            // unconditional loads from clamped addresses (all in flight at once), selected afterwards
            const int i = ty + 16 * ii, j = tx + 16 * jj;
            double v0 = 0.0;
            if (jj <= ii) {
                const int ic = i < n ? i : n - 1, jc = j < n ? j : n - 1;
                const double hv = H[(size_t)ic * n + jc];
                const double gv = g[jc];
                const bool live = j < n && j <= i;
                v0 = (live && i < n) ? scale * hv : ((live && i == n) ? -gv : 0.0);
            }
            a[ii][jj] = v0;
        }
    const double* z = meb_ldlt_solve_regs<BS>(a, n, Lm, &bad);
    for (int e = tid; e < n; e += 256) delta[e] = z[e];
    if (tid == 0 && info) *info = bad;
    if (S) meb_ctrl_after_newton_dev(S, v, z, n);
}

template <typename T>
int launch_syrk(meb_ctx* ctx, const ActiveArgs& a, int dp, double* part_mat, int grid, int* rb_out) {
    const int bs = dp / 16;
    const int td = bs <= 3 ? 8 : 16;
    const int rb = td == 8 ? SyrkShape<8>::RB : SyrkShape<16>::RB;
    const size_t smem = td == 8 ? (2 * (size_t)rb * dp + (size_t)dp * dp + dp) * sizeof(double)
                                : ((size_t)rb * dp + rb) * sizeof(double);
    *rb_out = rb;
#define MEB_SYRK_CASE(BSV, TD, B) case BSV: ctx->launches++; syrk_kernel<T, TD, B><<<grid, MEB_BLOCK, smem, ctx->stream>>>(a, part_mat); break;
#define MEB_SYRK8_CASE(BSV, B) case BSV: ctx->launches++; syrk8_kernel<T, B><<<grid, MEB_BLOCK, smem, ctx->stream>>>(a, part_mat); break;
    switch (bs) {
        MEB_SYRK8_CASE(1, 2) MEB_SYRK8_CASE(2, 4) MEB_SYRK8_CASE(3, 6) MEB_SYRK_CASE(4, 16, 4)
        MEB_SYRK_CASE(5, 16, 5) MEB_SYRK_CASE(6, 16, 6) MEB_SYRK_CASE(7, 16, 7) MEB_SYRK_CASE(8, 16, 8)
        default: return MEB_E_CAPACITY;
    }
#undef MEB_SYRK_CASE
#undef MEB_SYRK8_CASE
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}

}  // namespace

// H (device, (d+1)^2) from the records of the last streaming pass.  d <= 128.
int meb_dense_from_records(meb_ctx* ctx, const EvalCall& c, const double* ev_scalars, double* H) {
    if (c.d > 128) return MEB_E_CAPACITY;
    { const int rcl = meb_ensure_list(ctx, c.m); if (rcl != MEB_OK) return rcl; }
    const int dp = (c.d + 15) / 16 * 16;
    const size_t per = (size_t)dp * dp + dp;
    const size_t avail = ctx->part_mat_len;
    int grid = ctx->sm_count * (dp <= 32 ? 3 : 2);      // (d <= 32: the 80-register instance of syrk8, three CTAs per SM)
    if ((size_t)grid * per > avail) grid = (int)(avail / per);
    if (grid < 1) return MEB_E_CAPACITY;
    ActiveArgs a;
    memset(&a, 0, sizeof(a));
    a.C = c.C; a.ld = c.ld; a.U = c.U; a.v_slot = c.v_slot; a.V = c.V; a.ldv = c.ldv; a.x = c.x; a.d = c.d;
    a.sigma = c.sigma; a.list = ctx->list; a.count = ctx->count_dev;
    a.rec_lam = ctx->rec_lam; a.rec_rho = ctx->rec_rho; a.rec_t = ctx->rec_t;
    if (c.gs) {
        a.dyn = c.gs->dyn;
        for (int b = 0; b < 2; ++b) { a.U2[b] = c.gs->U2[b]; a.slot2[b] = c.gs->slot2[b]; a.V2[b] = c.gs->V2[b]; a.vcap2[b] = c.gs->vcap2[b]; }
    }
    int rb = 0;
    int rc = c.prec == MEB_FP64 ? launch_syrk<double>(ctx, a, dp, ctx->part_mat, grid, &rb)
                                : launch_syrk<float>(ctx, a, dp, ctx->part_mat, grid, &rb);
    if (rc != MEB_OK) return rc;
    const int n = c.d + 1;
    int fgrid = (n * n + 255) / 256;
    if (fgrid > 64) fgrid = 64;
    if (ctx->shard) {                     // sharded solve: records of the ranks' partial matrices, added in rank order
        rc = meb_shard_pack_mat(ctx, ctx->part_mat, grid, ctx->count_dev, rb, (int64_t)per);
        if (rc != MEB_OK) return rc;
        rc = meb_shard_exchange(ctx, (int64_t)per);
        if (rc != MEB_OK) return rc;
        ctx->launches++;
        dense_finalize_kernel<<<fgrid, 256, 0, ctx->stream>>>(ctx->shard->recv, ctx->shard->nranks, ctx->count_dev, dp, c.d, ev_scalars,
                                                             c.sigma, c.tau, H, c.gs ? c.gs->dyn : nullptr, 0, (long long)per);
        MEB_CUDA_OK(ctx, cudaGetLastError());
        return MEB_OK;
    }
    ctx->launches++; dense_finalize_kernel<<<fgrid, 256, 0, ctx->stream>>>(ctx->part_mat, grid, ctx->count_dev, dp, c.d, ev_scalars, c.sigma,
                                                          c.tau, H, c.gs ? c.gs->dyn : nullptr, rb, 0);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}

// delta <- -(scale*H)^{-1} g on the device; info_dev (nullable) receives 0 or the failing pivot + 1
int meb_chol_solve(meb_ctx* ctx, const double* H, const double* g, int n, double scale, double* delta,
                   int* info_dev, SolverDev* S, const SolverVecs* v) {
    SolverVecs vv;
    memset(&vv, 0, sizeof(vv));
    if (S && v) vv = *v;
    const int bs = (n + 1 + 15) / 16;                       // augmented order n + 1 <= 16 bs
    if (bs > 9) return MEB_E_CAPACITY;
    const int np = 16 * bs;
    const size_t smem = ((size_t)n * (np | 1) + 2 * (size_t)np) * sizeof(double);      // = LdltShape<bs>::smem_doubles(n)
#define MEB_LDLT_CASE(B)                                                                                        \
    case B:                                                                                                     \
        MEB_CUDA_OK(ctx, cudaFuncSetAttribute(ldlt_solve_kernel<B>, cudaFuncAttributeMaxDynamicSharedMemorySize, \
                                              (int)smem));                                                      \
        ctx->launches++;                                                                                        \
        ldlt_solve_kernel<B><<<1, 256, smem, ctx->stream>>>(H, g, n, scale, delta, info_dev, S, vv);                   \
        break;
    switch (bs) {
        MEB_LDLT_CASE(1) MEB_LDLT_CASE(2) MEB_LDLT_CASE(3) MEB_LDLT_CASE(4) MEB_LDLT_CASE(5)
        MEB_LDLT_CASE(6) MEB_LDLT_CASE(7) MEB_LDLT_CASE(8) MEB_LDLT_CASE(9)
        default: return MEB_E_CAPACITY;
    }
#undef MEB_LDLT_CASE
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}
