// Streaming map-reduce passes over the balls.
//
// One kernel template serves the four passes that read every centre row exactly once:
//   OP_EVAL    proximal augmented Lagrangian evaluation
//   OP_FEAS    full FP64 feasibility check
//   OP_SCREEN  FP32 boundary screening
//   OP_INGEST  initial radius / validation / FP32 shadow  (reading 3)
//
// Mapping (B200): a warp owns tiles of 32 consecutive rows.  G lanes cooperate on one row
// (G in {1,2,4,8,16,32}), each lane loading CPT 16-byte chunks (ld.global.nc, L1 no-allocate), so a
// warp-wide load instruction covers 32/G rows x 16*G contiguous bytes (full 32 B sectors).  Partial
// sums are combined inside the G-lane group with xor shuffles, then TRANSPOSED so that lane L holds
// the row sums of row L of the tile: the scalar epilogue (sqrt, divide, branch of P:L115, ~100
// FP64 instructions) runs once per 32 rows instead of once per row.  That keeps the pass
// HBM-bound at d = 10..32 where a row is only 80..256 bytes.
// Rows longer than 512 chunks use the loop kernel (a whole warp per row, 8 loads in flight).
//
// Determinism: tiles are assigned statically (tile -> warp round-robin), every lane accumulates its
// own rows in a fixed order, then xor-shuffle tree -> shared memory -> per-CTA partial in global
// memory; a second kernel adds the CTA partials in index order.  No floating-point atomics.
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
template <typename T, int OP>
__device__ __forceinline__ bool row_epilogue(const StreamArgs& a, int64_t row, bool valid, bool hasv,
                                             T nb2, T ne2, T ev, T vv, T r, T sig, Acc& acc) {
    if (!valid) return false;
    const T* R = static_cast<const T*>(a.R);
    const T ri = R ? R[row] : T(0);
    if (OP == OP_EVAL) {
        const T* U = static_cast<const T*>(a.U);
        const T ui = U ? U[row] : T(0);
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

// Fixed-order reduction of the per-lane accumulators to one partial per CTA.
template <int OP>
__device__ __forceinline__ void block_reduce_store(Acc& acc, double* part) {
    __shared__ double red[MEB_WARPS][MEB_NPART];
    __shared__ long long redi[MEB_WARPS];
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
        for (int w = 1; w < MEB_WARPS; ++w) {
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

namespace {

// ---- tiled kernel: G lanes per row, CPT chunks per lane (G * CPT * VEC >= d) ---------------------
template <typename T, int G, int CPT, int VEC, int OP, bool SHADOW>
__global__ void __launch_bounds__(MEB_BLOCK) stream_tile_kernel(const StreamArgs a) {
    constexpr int RPW = 32 / G;                     // rows per warp-wide load instruction
    constexpr int NPAD = G * CPT * VEC;             // padded row length held in shared memory
    __shared__ __align__(16) T cs[NPAD];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int gl = lane % G, gw = lane / G;
    const int d = a.d;
    const int64_t m = a.m;
    const T* __restrict__ C = static_cast<const T*>(a.C);
    const T* __restrict__ V = static_cast<const T*>(a.V);
    const bool HASV = (OP == OP_EVAL) && a.v_slot != nullptr;

    const double* cptr = (OP == OP_INGEST) ? a.c0 : a.x + 1;
    for (int j = threadIdx.x; j < NPAD; j += MEB_BLOCK) cs[j] = j < d ? (T)cptr[j] : T(0);
    __syncthreads();
    T creg[CPT][VEC];
#pragma unroll
    for (int k = 0; k < CPT; ++k)
#pragma unroll
        for (int j = 0; j < VEC; ++j) creg[k][j] = cs[(gl + k * G) * VEC + j];

    const T r = (OP == OP_INGEST) ? T(0) : (T)a.x[0];
    const T sig = (T)a.sigma;
    const T inv_sig = T(1) / sig;
    Acc acc;

    const int64_t ntiles = (m + 31) >> 5;
    const int64_t stride = (int64_t)gridDim.x * MEB_WARPS;
    for (int64_t tile = (int64_t)blockIdx.x * MEB_WARPS + warp; tile < ntiles; tile += stride) {
        const int64_t row0 = tile << 5;
        const int64_t myrow = row0 + lane;
        const bool myvalid = myrow < m;
        int myslot = -1;
        if (HASV && myvalid) myslot = a.v_slot[myrow];
        T my_nb2 = T(0), my_ne2 = T(0), my_ev = T(0), my_vv = T(0);
#pragma unroll(G <= 8 ? G : 4)
        for (int it = 0; it < G; ++it) {
            const int rsub = it * RPW + gw;
            const int64_t row = row0 + rsub;
            const bool valid = row < m;
            const T* rowp = C + row * a.ld;
            T e[CPT][VEC];
#pragma unroll
            for (int k = 0; k < CPT; ++k) load_chunk<T, VEC>(rowp, (gl + k * G) * VEC, d, valid, e[k]);
            int slot = -1;
            if (HASV) slot = __shfl_sync(MEB_FULL_MASK, myslot, rsub);
            const bool anyv = HASV && __any_sync(MEB_FULL_MASK, slot >= 0);
            T s_nb2 = T(0), s_ne2 = T(0), s_ev = T(0), s_vv = T(0);
            if (!anyv) {
#pragma unroll
                for (int k = 0; k < CPT; ++k)
#pragma unroll
                    for (int j = 0; j < VEC; ++j) {
                        const T ee = e[k][j] - creg[k][j];
                        s_nb2 = fma(ee, ee, s_nb2);
                        if (OP == OP_INGEST) s_ne2 = fma(e[k][j], T(0), s_ne2);   // NaN iff a non-finite entry
                        if (SHADOW) e[k][j] = ee;
                    }
            } else {
                const T* vrow = V + (int64_t)(slot < 0 ? 0 : slot) * a.ldv;
#pragma unroll
                for (int k = 0; k < CPT; ++k) {
                    T v[VEC];
                    load_chunk<T, VEC>(vrow, (gl + k * G) * VEC, d, valid && slot >= 0, v);
#pragma unroll
                    for (int j = 0; j < VEC; ++j) {
                        const T ee = e[k][j] - creg[k][j];
                        const T b = fma(v[j], inv_sig, ee);
                        s_nb2 = fma(b, b, s_nb2);
                        s_ne2 = fma(ee, ee, s_ne2);
                        s_ev = fma(ee, v[j], s_ev);
                        s_vv = fma(v[j], v[j], s_vv);
                    }
                }
            }
            if (SHADOW && valid) {       // FP32 shadow of the centred rows (reading 8)
                float* srow = a.C32 + row * a.ld32;
#pragma unroll
                for (int k = 0; k < CPT; ++k) {
                    const int col = (gl + k * G) * VEC;
#pragma unroll
                    for (int j = 0; j < VEC; ++j)
                        if (col + j < d) srow[col + j] = (float)e[k][j];
                }
            }
#pragma unroll
            for (int o = G / 2; o > 0; o >>= 1) {
                s_nb2 += __shfl_xor_sync(MEB_FULL_MASK, s_nb2, o);
                if (OP == OP_INGEST) s_ne2 += __shfl_xor_sync(MEB_FULL_MASK, s_ne2, o);
                if (anyv) {
                    s_ne2 += __shfl_xor_sync(MEB_FULL_MASK, s_ne2, o);
                    s_ev += __shfl_xor_sync(MEB_FULL_MASK, s_ev, o);
                    s_vv += __shfl_xor_sync(MEB_FULL_MASK, s_vv, o);
                }
            }
            // transpose: lane L owns row L of the tile = iteration L / RPW, group L % RPW
            const int src = (lane % RPW) * G;
            const bool take = (it == lane / RPW);
            const T g0 = __shfl_sync(MEB_FULL_MASK, s_nb2, src);
            if (take) my_nb2 = g0;
            if (OP == OP_INGEST) {
                const T g1 = __shfl_sync(MEB_FULL_MASK, s_ne2, src);
                if (take) my_ne2 = g1;
            }
            if (anyv) {
                const T g1 = __shfl_sync(MEB_FULL_MASK, s_ne2, src);
                const T g2 = __shfl_sync(MEB_FULL_MASK, s_ev, src);
                const T g3 = __shfl_sync(MEB_FULL_MASK, s_vv, src);
                if (take) { my_ne2 = g1; my_ev = g2; my_vv = g3; }
            }
        }
        const bool flag = row_epilogue<T, OP>(a, myrow, myvalid, myslot >= 0, my_nb2, my_ne2, my_ev,
                                              my_vv, r, sig, acc);
        if (OP != OP_INGEST) {
            const uint32_t bits = __ballot_sync(MEB_FULL_MASK, flag);
            if (lane == 0) a.mask[tile] = bits;
        }
    }
    block_reduce_store<OP>(acc, a.part);
}

// ---- loop kernel: one warp per row, any d -----------------------------------------------------------
template <typename T, int VEC, int OP, bool SHADOW>
__global__ void __launch_bounds__(MEB_BLOCK) stream_loop_kernel(const StreamArgs a) {
    constexpr int UNR = 8;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int d = a.d;
    const int64_t m = a.m;
    const T* __restrict__ C = static_cast<const T*>(a.C);
    const T* __restrict__ V = static_cast<const T*>(a.V);
    const bool HASV = (OP == OP_EVAL) && a.v_slot != nullptr;
    const double* __restrict__ cptr = (OP == OP_INGEST) ? a.c0 : a.x + 1;
    const T r = (OP == OP_INGEST) ? T(0) : (T)a.x[0];
    const T sig = (T)a.sigma;
    const T inv_sig = T(1) / sig;
    const int nchunks = (d + VEC - 1) / VEC;
    Acc acc;

    const int64_t ntiles = (m + 31) >> 5;
    const int64_t stride = (int64_t)gridDim.x * MEB_WARPS;
    for (int64_t tile = (int64_t)blockIdx.x * MEB_WARPS + warp; tile < ntiles; tile += stride) {
        const int64_t row0 = tile << 5;
        const int64_t myrow = row0 + lane;
        const bool myvalid = myrow < m;
        int myslot = -1;
        if (HASV && myvalid) myslot = a.v_slot[myrow];
        T my_nb2 = T(0), my_ne2 = T(0), my_ev = T(0), my_vv = T(0);
        for (int it = 0; it < 32; ++it) {
            const int64_t row = row0 + it;
            if (row >= m) break;                       // warp-uniform
            const T* rowp = C + row * a.ld;
            int slot = -1;
            if (HASV) slot = __shfl_sync(MEB_FULL_MASK, myslot, it);
            T s_nb2 = T(0), s_ne2 = T(0), s_ev = T(0), s_vv = T(0);
            if (slot < 0) {
                for (int c0 = lane; c0 < nchunks; c0 += 32 * UNR) {
                    T e[UNR][VEC];
#pragma unroll
                    for (int u = 0; u < UNR; ++u)
                        load_chunk<T, VEC>(rowp, (c0 + 32 * u) * VEC, d, true, e[u]);
#pragma unroll
                    for (int u = 0; u < UNR; ++u) {
                        const int col = (c0 + 32 * u) * VEC;
#pragma unroll
                        for (int j = 0; j < VEC; ++j) {
                            if (col + j < d) {
                                const T ee = e[u][j] - (T)__ldg(cptr + col + j);
                                s_nb2 = fma(ee, ee, s_nb2);
                                if (OP == OP_INGEST) s_ne2 = fma(e[u][j], T(0), s_ne2);
                                if (SHADOW) a.C32[row * a.ld32 + col + j] = (float)ee;
                            }
                        }
                    }
                }
            } else {
                const T* vrow = V + (int64_t)slot * a.ldv;
                for (int c0 = lane; c0 < nchunks; c0 += 32 * 4) {
                    T e[4][VEC], v[4][VEC];
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        load_chunk<T, VEC>(rowp, (c0 + 32 * u) * VEC, d, true, e[u]);
                        load_chunk<T, VEC>(vrow, (c0 + 32 * u) * VEC, d, true, v[u]);
                    }
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int col = (c0 + 32 * u) * VEC;
#pragma unroll
                        for (int j = 0; j < VEC; ++j) {
                            if (col + j < d) {
                                const T ee = e[u][j] - (T)__ldg(cptr + col + j);
                                const T b = fma(v[u][j], inv_sig, ee);
                                s_nb2 = fma(b, b, s_nb2);
                                s_ne2 = fma(ee, ee, s_ne2);
                                s_ev = fma(ee, v[u][j], s_ev);
                                s_vv = fma(v[u][j], v[u][j], s_vv);
                            }
                        }
                    }
                }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                s_nb2 += __shfl_xor_sync(MEB_FULL_MASK, s_nb2, o);
                if (OP == OP_INGEST) s_ne2 += __shfl_xor_sync(MEB_FULL_MASK, s_ne2, o);
                if (slot >= 0) {
                    s_ne2 += __shfl_xor_sync(MEB_FULL_MASK, s_ne2, o);
                    s_ev += __shfl_xor_sync(MEB_FULL_MASK, s_ev, o);
                    s_vv += __shfl_xor_sync(MEB_FULL_MASK, s_vv, o);
                }
            }
            if (it == lane) { my_nb2 = s_nb2; my_ne2 = s_ne2; my_ev = s_ev; my_vv = s_vv; }
        }
        const bool flag = row_epilogue<T, OP>(a, myrow, myvalid, myslot >= 0, my_nb2, my_ne2, my_ev,
                                              my_vv, r, sig, acc);
        if (OP != OP_INGEST) {
            const uint32_t bits = __ballot_sync(MEB_FULL_MASK, flag);
            if (lane == 0) a.mask[tile] = bits;
        }
    }
    block_reduce_store<OP>(acc, a.part);
}

}  // namespace

// ---- host-side dispatch ---------------------------------------------------------------------------
namespace {

template <typename KernelT>
int launch_sized(meb_ctx* ctx, KernelT kernel, const StreamArgs& a, int* grid_out) {
    int occ = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, MEB_BLOCK, 0);
    if (e != cudaSuccess) { ctx->last_cuda_error = (int)e; return MEB_E_CUDA; }
    if (occ < 1) occ = 1;
    const int64_t ntiles = (a.m + 31) / 32;
    int64_t want = (ntiles + MEB_WARPS - 1) / MEB_WARPS;
    int64_t cap = (int64_t)ctx->sm_count * occ;          // one resident wave, grid-stride inside
    if (cap > MEB_MAX_GRID) cap = MEB_MAX_GRID;
    int grid = (int)(want < cap ? want : cap);
    if (grid < 1) grid = 1;
    StreamArgs b = a;
    ctx->launches++; kernel<<<grid, MEB_BLOCK, 0, ctx->stream>>>(b);
    e = cudaGetLastError();
    if (e != cudaSuccess) { ctx->last_cuda_error = (int)e; return MEB_E_CUDA; }
    *grid_out = grid;
    return MEB_OK;
}

template <typename T, int OP, bool SHADOW>
int dispatch_shape(meb_ctx* ctx, const StreamArgs& a, bool aligned, int* grid_out) {
    constexpr int VEC = VecOf<T>::N;
    if (!aligned) return launch_sized(ctx, stream_loop_kernel<T, 1, OP, SHADOW>, a, grid_out);
    const int nchunks = (a.d + VEC - 1) / VEC;
    if (nchunks <= 4)   return launch_sized(ctx, stream_tile_kernel<T, 4, 1, VEC, OP, SHADOW>, a, grid_out);
    if (nchunks <= 8)   return launch_sized(ctx, stream_tile_kernel<T, 4, 2, VEC, OP, SHADOW>, a, grid_out);
    if (nchunks <= 16)  return launch_sized(ctx, stream_tile_kernel<T, 4, 4, VEC, OP, SHADOW>, a, grid_out);
    if (nchunks <= 32)  return launch_sized(ctx, stream_tile_kernel<T, 8, 4, VEC, OP, SHADOW>, a, grid_out);
    if (nchunks <= 64)  return launch_sized(ctx, stream_tile_kernel<T, 8, 8, VEC, OP, SHADOW>, a, grid_out);
    if (nchunks <= 128) return launch_sized(ctx, stream_tile_kernel<T, 16, 8, VEC, OP, SHADOW>, a, grid_out);
    if (nchunks <= 256) return launch_sized(ctx, stream_tile_kernel<T, 32, 8, VEC, OP, SHADOW>, a, grid_out);
    if (nchunks <= 512) return launch_sized(ctx, stream_tile_kernel<T, 32, 16, VEC, OP, SHADOW>, a, grid_out);
    return launch_sized(ctx, stream_loop_kernel<T, VEC, OP, SHADOW>, a, grid_out);
}

template <typename T>
bool rows_aligned(const void* p, int64_t ld) {
    return ((uintptr_t)p % 16 == 0) && ((ld * (int64_t)sizeof(T)) % 16 == 0);
}

}  // namespace

// Launches one streaming pass.  Per-CTA partials land in a.part[grid * MEB_NPART].
int meb_launch_stream(meb_ctx* ctx, int op, int prec, const StreamArgs& a, int* grid_out) {
    if (prec == MEB_FP64) {
        bool al = rows_aligned<double>(a.C, a.ld);
        if (a.v_slot) al = al && rows_aligned<double>(a.V, a.ldv);
        switch (op) {
            case OP_EVAL: return dispatch_shape<double, OP_EVAL, false>(ctx, a, al, grid_out);
            case OP_FEAS: return dispatch_shape<double, OP_FEAS, false>(ctx, a, al, grid_out);
            case OP_INGEST:
                if (a.C32) return dispatch_shape<double, OP_INGEST, true>(ctx, a, al, grid_out);
                return dispatch_shape<double, OP_INGEST, false>(ctx, a, al, grid_out);
            default: return MEB_E_ARG;
        }
    } else {
        bool al = rows_aligned<float>(a.C, a.ld);
        if (a.v_slot) al = al && rows_aligned<float>(a.V, a.ldv);
        switch (op) {
            case OP_EVAL: return dispatch_shape<float, OP_EVAL, false>(ctx, a, al, grid_out);
            case OP_SCREEN: return dispatch_shape<float, OP_SCREEN, false>(ctx, a, al, grid_out);
            default: return MEB_E_ARG;
        }
    }
}
