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
#include "meb_rowops.cuh"

namespace {

// ---- tiled kernel: G lanes per row, CPT chunks per lane (G * CPT * VEC >= d) ---------------------
template <typename T, int G, int CPT, int VEC, int OP, bool SHADOW>
__global__ void __launch_bounds__(MEB_BLOCK) stream_tile_kernel(const StreamArgs a_in) {
    StreamArgs a = a_in;
    meb_resolve_dyn(a);
    long long t_start = 0;
    if (threadIdx.x == 0) asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_start));
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
    __shared__ double abort_slots[33];
    AbortCtl ab;
    if (OP == OP_EVAL) abort_init(ab, a.dyn, abort_slots);
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
        if (OP == OP_EVAL && abort_seen(ab)) break;
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
        if (OP == OP_EVAL && ab.on && abort_publish(ab, acc, MEB_WARPS)) break;
    }
    block_reduce_store<OP>(acc, a.part);
    if (threadIdx.x == 0) {                 // device time stamps of this CTA (ns), read by the finalize kernel
        long long t_end;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_end));
        a.part[(size_t)blockIdx.x * MEB_NPART + 10] = __longlong_as_double(t_start);
        a.part[(size_t)blockIdx.x * MEB_NPART + 11] = __longlong_as_double(t_end);
        if (OP == OP_EVAL) abort_store(ab, a.part);
    }
}

// ---- loop kernel: one warp per row, any d -----------------------------------------------------------
template <typename T, int VEC, int OP, bool SHADOW>
__global__ void __launch_bounds__(MEB_BLOCK) stream_loop_kernel(const StreamArgs a_in) {
    StreamArgs a = a_in;
    meb_resolve_dyn(a);
    long long t_start = 0;
    if (threadIdx.x == 0) asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_start));
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
    // the centre, converted to T once, in dynamic shared memory (padded with zeros to whole chunks)
    extern __shared__ __align__(16) unsigned char loop_dyn_smem[];
    T* cs = reinterpret_cast<T*>(loop_dyn_smem);
    for (int j = threadIdx.x; j < nchunks * VEC; j += MEB_BLOCK) cs[j] = j < d ? (T)cptr[j] : T(0);
    __shared__ double abort_slots[33];
    AbortCtl ab;
    if (OP == OP_EVAL) abort_init(ab, a.dyn, abort_slots);
    __syncthreads();

    // rows per warp tile: 32, or 16 / 8 when there are too few rows to occupy the GPU with 32-row tiles
    const int rts = a.rt_shift ? a.rt_shift : 5;
    const int RT = 1 << rts;
    const int64_t ntiles = (m + RT - 1) >> rts;
    const int64_t stride = (int64_t)gridDim.x * MEB_WARPS;
    for (int64_t tile = (int64_t)blockIdx.x * MEB_WARPS + warp; tile < ntiles; tile += stride) {
        if (OP == OP_EVAL && abort_seen(ab)) break;
        const int64_t row0 = tile << rts;
        const int64_t myrow = row0 + lane;
        const bool myvalid = lane < RT && myrow < m;
        int myslot = -1;
        if (HASV && myvalid) myslot = a.v_slot[myrow];
        T my_nb2 = T(0), my_ne2 = T(0), my_ev = T(0), my_vv = T(0);
        for (int it = 0; it < RT; ++it) {
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
                                const T ee = e[u][j] - cs[col + j];
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
                                const T ee = e[u][j] - cs[col + j];
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
            if (lane == 0) {
                if (rts == 5) a.mask[tile] = bits;
                else if (rts == 4) reinterpret_cast<uint16_t*>(a.mask)[tile] = (uint16_t)bits;
                else reinterpret_cast<uint8_t*>(a.mask)[tile] = (uint8_t)bits;
            }
        }
        if (OP == OP_EVAL && ab.on && abort_publish(ab, acc, MEB_WARPS)) break;
    }
    block_reduce_store<OP>(acc, a.part);
    if (threadIdx.x == 0) {                 // device time stamps of this CTA (ns), read by the finalize kernel
        long long t_end;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_end));
        a.part[(size_t)blockIdx.x * MEB_NPART + 10] = __longlong_as_double(t_start);
        a.part[(size_t)blockIdx.x * MEB_NPART + 11] = __longlong_as_double(t_end);
        if (OP == OP_EVAL) abort_store(ab, a.part);
    }
}

}  // namespace

// ---- host-side dispatch ---------------------------------------------------------------------------
namespace {

template <typename KernelT>
int launch_sized(meb_ctx* ctx, KernelT kernel, const StreamArgs& a, int* grid_out, size_t smem = 0, bool loop_kernel = false) {
    if (smem > 220 * 1024) return MEB_E_CAPACITY;            // centre does not fit in shared memory (d > ~28,000)
    int occ = 0;
    cudaError_t e = cudaSuccess;
    if (smem > 48 * 1024) e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, MEB_BLOCK, smem);
    if (e != cudaSuccess) { ctx->last_cuda_error = (int)e; return MEB_E_CUDA; }
    if (occ < 1) occ = 1;
    StreamArgs b = a;
    int64_t ntiles = (a.m + 31) / 32;
    if (loop_kernel) {               // few long rows: smaller warp tiles so that every SM gets rows
        const int64_t full = (int64_t)ctx->sm_count * occ * MEB_WARPS;
        b.rt_shift = 5;
        if (ntiles < 2 * full) b.rt_shift = 4;
        if ((a.m + 15) / 16 < 2 * full) b.rt_shift = 3;
        ntiles = (a.m + (1 << b.rt_shift) - 1) >> b.rt_shift;
    }
    int64_t want = (ntiles + MEB_WARPS - 1) / MEB_WARPS;
    int64_t cap = (int64_t)ctx->sm_count * occ;          // one resident wave, grid-stride inside
    if (cap > MEB_MAX_GRID) cap = MEB_MAX_GRID;
    int grid = (int)(want < cap ? want : cap);
    if (grid < 1) grid = 1;
    ctx->launches++; kernel<<<grid, MEB_BLOCK, smem, ctx->stream>>>(b);
    e = cudaGetLastError();
    if (e != cudaSuccess) { ctx->last_cuda_error = (int)e; return MEB_E_CUDA; }
    *grid_out = grid;
    return MEB_OK;
}

template <typename T, int OP, bool SHADOW>
int dispatch_shape(meb_ctx* ctx, const StreamArgs& a, bool aligned, int* grid_out) {
    constexpr int VEC = VecOf<T>::N;
    if (!aligned) return launch_sized(ctx, stream_loop_kernel<T, 1, OP, SHADOW>, a, grid_out, ((size_t)a.d * sizeof(T) + 15) / 16 * 16, true);
    const int nchunks = (a.d + VEC - 1) / VEC;
    if (nchunks <= 4)   return launch_sized(ctx, stream_tile_kernel<T, 4, 1, VEC, OP, SHADOW>, a, grid_out);
    if (nchunks <= 8)   return launch_sized(ctx, stream_tile_kernel<T, 4, 2, VEC, OP, SHADOW>, a, grid_out);
    if (nchunks <= 16)  return launch_sized(ctx, stream_tile_kernel<T, 4, 4, VEC, OP, SHADOW>, a, grid_out);
    if (nchunks <= 32)  return launch_sized(ctx, stream_tile_kernel<T, 8, 4, VEC, OP, SHADOW>, a, grid_out);
    if (nchunks <= 64)  return launch_sized(ctx, stream_tile_kernel<T, 8, 8, VEC, OP, SHADOW>, a, grid_out);
    if (nchunks <= 128) return launch_sized(ctx, stream_tile_kernel<T, 16, 8, VEC, OP, SHADOW>, a, grid_out);
    if (nchunks <= 256) return launch_sized(ctx, stream_tile_kernel<T, 32, 8, VEC, OP, SHADOW>, a, grid_out);
    // rows longer than 256 chunks (4 KB): the warp-per-row loop kernel (centre in shared memory, 8 loads in
    // flight per lane) beats a 16-chunks-per-lane register tile, which needs ~250 registers (one CTA per SM)
    return launch_sized(ctx, stream_loop_kernel<T, VEC, OP, SHADOW>, a, grid_out, (size_t)nchunks * 16, true);
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
        if (a.dyn) al = al && rows_aligned<double>(a.V2[0], a.ldv) && rows_aligned<double>(a.V2[1], a.ldv);
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
        if (a.dyn) al = al && rows_aligned<float>(a.V2[0], a.ldv) && rows_aligned<float>(a.V2[1], a.ldv);
        switch (op) {
            case OP_EVAL: return dispatch_shape<float, OP_EVAL, false>(ctx, a, al, grid_out);
            case OP_SCREEN: return dispatch_shape<float, OP_SCREEN, false>(ctx, a, al, grid_out);
            default: return MEB_E_ARG;
        }
    }
}
