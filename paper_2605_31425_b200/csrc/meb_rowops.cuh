// Per-row arithmetic shared by the streaming kernels (meb_stream.cu: register/LDG mapping for long or
// unaligned rows; meb_tile.cu: TMA-staged lane-per-row mapping for short rows): the accumulators of a
// pass, the scalar epilogue of one ball and the fixed-order
// block reduction.  Nothing here is used by, or shared with, the CPU oracle.
#pragma once
#include "meb_internal.cuh"

namespace {

// ---- per-lane accumulators of one pass -----------------------------------------------------------
struct Acc {
    double s0 = 0, s1 = 0, s2 = 0, s3 = 0;  // sums   (eval: proj2, uplus, dmult2, rho)
    double m0 = 0, m1 = 0, m2 = 0;          // maxima (eval: pfeas, compl, dfeas; feas/ingest: m0 = value)
    long long i0 = -1;                      // argmax index for m0 (feas/ingest)
    int n0 = 0, n1 = 0;                     // counts (eval: n_b1, n_b3; ingest: bad entries)
};

template <typename T> __device__ __forceinline__ T t_sqrt(T v);
template <> __device__ __forceinline__ double t_sqrt<double>(double v) { return sqrt(v); }
template <> __device__ __forceinline__ float t_sqrt<float>(float v) { return sqrtf(v); }

// Epilogue for one row, executed by the lane that owns it (lane L <-> row tile*32+L).
// ri, ui: radius and multiplier u_i of the row (already loaded); lam_out receives lam_i (EVAL).
template <typename T, int OP>
__device__ __forceinline__ bool row_epilogue_core(const StreamArgs& a, int64_t row, bool valid, bool hasv,
                                                  T nb2, T ne2, T ev, T vv, T r, T sig, T ri, T ui, Acc& acc,
                                                  double& lam_out) {
    lam_out = 0.0;
    if (!valid) return false;
    if (OP == OP_EVAL) {
        if (!hasv && ui == T(0)) {
            // Fast path: a ball without multipliers that lies clearly inside the current ball is in
            // branch B2 (nb <= -a = r - r_i) and every one of its terms is exactly zero.  The margin
            // keeps balls near the branch boundary on the exact path below.
            const T apf = r - ri;
            if (apf > T(0) && nb2 <= apf * apf * T(0.998)) {
                if (a.t_out) a.t_out[row] = 0.0;
                if (a.lam_out) a.lam_out[row] = 0.0;
                return false;
            }
        }
        const T av = ri - r + ui / sig;                    // a_i
        const T nb = t_sqrt<T>(nb2);
        T t, lam;
        int br;
        if (nb <= av)       { t = av;   lam = T(1); br = 1; }      // P:L115, printed order
        else if (nb <= -av) { t = T(0); lam = T(0); br = 2; }
        else { const T s = (av + nb) / T(2); t = s; lam = s / nb; br = 3; }
        const T lnb = lam * nb;
        const T uplus = sig * t;
        const T sl = sig * lam;
        T dv2;
        T eb;                                               // <c_i - c, b_i>
        T ne;
        if (hasv) {
            const T bv = ev + vv / sig;                     // <b_i, v_i>
            dv2 = sl * sl * nb2 - T(2) * sl * bv + vv;      // ||sigma lam b - v||^2
            if (dv2 < T(0)) dv2 = T(0);
            eb = ne2 + ev / sig;
            ne = t_sqrt<T>(ne2);
        } else {
            dv2 = sl * sl * nb2;
            eb = nb2;
            ne = nb;
        }
        const T du = uplus - ui;
        const T ap = r - ri;                                // (r - r_i, c - c_i)
        T pf;
        if (ne <= ap)       pf = T(0);
        else if (ne <= -ap) pf = t_sqrt<T>(ap * ap + ne * ne);
        else                pf = (ne - ap) * T(0.70710678118654752440);
        T cp = ap * uplus - sl * eb;
        cp = cp < T(0) ? -cp : cp;
        T df = (sl * nb - uplus) * T(0.70710678118654752440);
        if (df < T(0)) df = T(0);
        acc.s0 += (double)(t * t + lnb * lnb);
        acc.s1 += (double)uplus;
        acc.s2 += (double)(du * du + dv2);
        acc.m0 = fmax(acc.m0, (double)pf);
        acc.m1 = fmax(acc.m1, (double)cp);
        acc.m2 = fmax(acc.m2, (double)df);
        if (br == 1) acc.n0++;
        if (br == 3) { acc.n1++; acc.s3 += (double)(av / nb); }
        if (a.t_out) a.t_out[row] = (double)t;
        if (a.lam_out) a.lam_out[row] = (double)lam;
        lam_out = (double)lam;
        if (br != 2) {
            a.rec_lam[row] = (double)lam;
            a.rec_rho[row] = br == 1 ? 2.0 : (double)(av / nb);
            a.rec_t[row] = (double)t;
            return true;
        }
        return false;
    } else if (OP == OP_FEAS) {
        const double viol = (double)ri + (double)t_sqrt<T>(nb2) - (double)r;
        if (acc.i0 < 0 || viol > acc.m0) { acc.m0 = viol; acc.i0 = row; }
        bool flag = viol > a.eps;
        if (flag && a.kept && a.kept[row]) flag = false;
        return flag;
    } else if (OP == OP_SCREEN) {
        const T s = (r - ri) - t_sqrt<T>(nb2);              // s_i
        const bool flag = s <= (T)a.eps;
        if (a.flags_out) a.flags_out[row] = flag ? 1 : 0;
        return flag;
    } else {  // OP_INGEST
        const double val = (double)t_sqrt<T>(nb2) + (double)ri;
        // rows with a non-finite entry (0 * e accumulated in ne2 is then NaN) or a bad radius
        if (!(ne2 == T(0)) || !(ri >= T(0)) || !((double)ri < 1.79e308)) acc.n0++;
        if (acc.i0 < 0 || val > acc.m0) { acc.m0 = val; acc.i0 = row; }
        if (a.R32) a.R32[row] = (float)ri;
        return false;
    }
}

// ---- early stop of a doomed Armijo trial (MebDyn::s0_abort) -------------------------------------------
// Every warp keeps its running part of sum_i ||Pi(z_i)||^2 (Acc::s0) in a shared-memory slot; a warp that finds
// the sum over the slots of its CTA above the threshold raises the CTA's flag, and the warps of the CTA stop.
// Everything stays inside the CTA (no global flag, no atomics: same-address traffic between the two dies costs
// ~30 ns per access).  One CTA's part exceeding the threshold is sufficient (not necessary) for
// Psi(trial) > Psi(x); a pass that is cut short is rejected exactly as it would have been when run to the end.
struct AbortCtl {
    volatile double* slots = nullptr;       // [32] running sums of the warps, [32] = the CTA's flag
    double thr = 0.0;
    bool on = false;
};
// call before the first __syncthreads of the kernel; slots: 33 doubles of shared memory
__device__ __forceinline__ void abort_init(AbortCtl& c, const MebDyn* dyn, double* slots) {
    c.slots = slots;
    if (threadIdx.x < 33) slots[threadIdx.x] = 0.0;
    if (dyn == nullptr) return;
    const double thr = dyn->s0_abort;
    if (!(thr < 1e299)) return;
    c.thr = thr; c.on = true;
}
__device__ __forceinline__ bool abort_seen(const AbortCtl& c) { return c.on && c.slots[32] != 0.0; }
// warp-collective; returns true when the CTA's part crossed the threshold
__device__ __forceinline__ bool abort_publish(AbortCtl& c, const Acc& acc, int nwarps) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const double w = warp_sum(acc.s0);
    if (lane == 0) c.slots[warp] = w;
    __syncwarp();
    const double t = warp_sum(lane < nwarps ? c.slots[lane] : 0.0);
    const bool crossed = t > c.thr;
    if (crossed && lane == 0) c.slots[32] = 1.0;
    return crossed;
}
// thread 0, after the CTA's partials were stored
__device__ __forceinline__ void abort_store(const AbortCtl& c, double* part) {
    part[(size_t)blockIdx.x * MEB_NPART + MEB_PART_CUT] = (c.on && c.slots[32] != 0.0) ? 1.0 : 0.0;
}

// ---- multi-trial Armijo (MebDyn::multi_n) -----------------------------------------------------------------------
// Per-lane sums of ||Pi(z_i)||^2 at the predicted points x_t - gamma_k Delta, k < multi_n.
template <bool ON> struct MultiAcc { double s[ON ? MEB_MULTI_MAX : 1]; __device__ MultiAcc() { for (int k = 0; k < (ON ? MEB_MULTI_MAX : 1); ++k) s[k] = 0.0; } };

// One row at the trial point: nb2 = ||b_i||^2, p = <b_i, Delta c>.  At x_t - gamma Delta the shifted point is
// (a_i + gamma Delta r, b_i + gamma Delta c), so ||b||^2 = nb2 + 2 gamma p + gamma^2 ||Delta c||^2.
template <typename T>
__device__ __forceinline__ void multi_row(MultiAcc<true>& ma, const StreamArgs& a, int cap, T nb2, T p, T r, T sig, T ri, T ui) {
    const int nm = a.dyn ? (a.dyn->multi_n < cap ? a.dyn->multi_n : cap) : 0;
    if (nm <= 0) return;
    const T av = ri - r + ui / sig;
    const T dr = (T)a.dyn->dir_r, dc2 = (T)a.dyn->dir_c2;
    {   // balls that stay strictly inside at every predicted point add exactly zero: ||b + g dc|| <= ||b|| + g ||dc||
        const T gmax = (T)a.dyn->multi_gamma[nm - 1];
        const T reach = t_sqrt<T>(nb2) + gmax * (T)a.dyn->dir_c;
        const T amax = av + (dr > T(0) ? gmax * dr : T(0));
        if (reach <= -amax) return;
    }
#pragma unroll
    for (int k = 0; k < MEB_MULTI_MAX; ++k) {
        if (k < nm) {
            const T g = (T)a.dyn->multi_gamma[k];
            T nk2 = fma(g, fma(g, dc2, T(2) * p), nb2);
            if (nk2 < T(0)) nk2 = T(0);
            const T nk = t_sqrt<T>(nk2);
            const T ak = fma(g, dr, av);
            T pr2;
            if (nk <= ak) pr2 = ak * ak + nk2;                      // P:L115, printed order
            else if (nk <= -ak) pr2 = T(0);
            else { const T s2 = ak + nk; pr2 = T(0.5) * s2 * s2; }    // 2 ((a + nb)/2)^2
            ma.s[k] += (double)pr2;
        }
    }
}
template <typename T>
__device__ __forceinline__ void multi_row(MultiAcc<false>&, const StreamArgs&, int, T, T, T, T, T, T) {}

// per-CTA partials of the predictions: lanes (xor tree), then warps in index order
__device__ __forceinline__ void multi_store(MultiAcc<true>& ma, const StreamArgs& a, int nwarps) {
    __shared__ double mred[16][MEB_MULTI_MAX];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < MEB_MULTI_MAX; ++k) {
        const double v = warp_sum(ma.s[k]);
        if (lane == 0 && warp < 16) mred[warp][k] = v;
    }
    __syncthreads();
    if (threadIdx.x < MEB_MULTI_MAX && a.multi_part) {
        double t = 0.0;
        for (int w = 0; w < nwarps; ++w) t += mred[w][threadIdx.x];
        a.multi_part[(size_t)blockIdx.x * MEB_MULTI_MAX + threadIdx.x] = t;
    }
}
__device__ __forceinline__ void multi_store(MultiAcc<false>&, const StreamArgs&, int) {}

// Same, loading r_i and u_i of the row from global memory.
template <typename T, int OP>
__device__ __forceinline__ bool row_epilogue(const StreamArgs& a, int64_t row, bool valid, bool hasv,
                                             T nb2, T ne2, T ev, T vv, T r, T sig, Acc& acc) {
    T ri = T(0), ui = T(0);
    if (valid) {
        const T* R = static_cast<const T*>(a.R);
        if (R) ri = R[row];
        if (OP == OP_EVAL) {
            const T* U = static_cast<const T*>(a.U);
            if (U) ui = U[row];
        }
    }
    double lam;
    return row_epilogue_core<T, OP>(a, row, valid, hasv, nb2, ne2, ev, vv, r, sig, ri, ui, acc, lam);
}

// Fixed-order reduction of the per-lane accumulators to one partial per CTA.
template <int OP>
__device__ __forceinline__ void block_reduce_store(Acc& acc, double* part, int nwarps = MEB_WARPS) {
    __shared__ double red[16][MEB_NPART];          // up to 16 warps per CTA (meb_tile.cu)
    __shared__ long long redi[16];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double v[MEB_NPART];
#pragma unroll
    for (int k = 0; k < MEB_NPART; ++k) v[k] = 0.0;
    long long bi = acc.i0;
    if (OP == OP_EVAL) {
        v[0] = warp_sum(acc.s0); v[1] = warp_sum(acc.s1); v[2] = warp_sum(acc.s2);
        v[3] = warp_sum((double)acc.n0); v[4] = warp_sum((double)acc.n1);
        v[5] = warp_max(acc.m0); v[6] = warp_max(acc.m1); v[7] = warp_max(acc.m2);
        v[8] = warp_sum(acc.s3);
    } else {
        // (value, index) arg-max, smaller index wins ties; lanes without rows carry i0 = -1
        double bv = acc.m0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const double ov = __shfl_xor_sync(MEB_FULL_MASK, bv, o);
            const long long oi = __shfl_xor_sync(MEB_FULL_MASK, bi, o);
            if (oi >= 0 && (bi < 0 || ov > bv || (ov == bv && oi < bi))) { bv = ov; bi = oi; }
        }
        v[0] = bv;
        v[2] = warp_sum((double)acc.n0);
    }
    if (lane == 0) {
#pragma unroll
        for (int k = 0; k < MEB_NPART; ++k) red[warp][k] = v[k];
        redi[warp] = bi;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double o[MEB_NPART];
#pragma unroll
        for (int k = 0; k < MEB_NPART; ++k) o[k] = red[0][k];
        long long oi = redi[0];
        for (int w = 1; w < nwarps; ++w) {
            if (OP == OP_EVAL) {
                o[0] += red[w][0]; o[1] += red[w][1]; o[2] += red[w][2]; o[3] += red[w][3];
                o[4] += red[w][4]; o[8] += red[w][8];
                o[5] = fmax(o[5], red[w][5]); o[6] = fmax(o[6], red[w][6]); o[7] = fmax(o[7], red[w][7]);
            } else {
                const long long wi = redi[w];
                if (wi >= 0 && (oi < 0 || red[w][0] > o[0] || (red[w][0] == o[0] && wi < oi))) {
                    o[0] = red[w][0]; oi = wi;
                }
                o[2] += red[w][2];
            }
        }
        if (OP != OP_EVAL) o[1] = (double)oi;
#pragma unroll
        for (int k = 0; k < MEB_NPART; ++k) part[(size_t)blockIdx.x * MEB_NPART + k] = o[k];
    }
}

// Load one chunk of VEC elements starting at column `col` of a row; zero beyond d / invalid rows.
template <typename T, int VEC>
__device__ __forceinline__ void load_chunk(const T* rowp, int col, int d, bool valid, T (&out)[VEC]) {
#pragma unroll
    for (int j = 0; j < VEC; ++j) out[j] = T(0);
    if (!valid || col >= d) return;
    if (VEC > 1 && col + VEC <= d) {
        typedef typename VecOf<T>::type V;
        const V v = ldg_stream(reinterpret_cast<const V*>(rowp + col));
        const T* pv = reinterpret_cast<const T*>(&v);
#pragma unroll
        for (int j = 0; j < VEC; ++j) out[j] = pv[j];
    } else {
#pragma unroll
        for (int j = 0; j < VEC; ++j)
            if (col + j < d) out[j] = __ldg(rowp + col + j);
    }
}

}  // namespace
