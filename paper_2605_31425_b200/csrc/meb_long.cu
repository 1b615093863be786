// TMA-staged streaming map-reduce for LONG rows (row > 1024 bytes): SURVEY 8(a) rows a0, a1, a7, a8 at
// d = 1e3 .. 1e4 (BASELINE configs 3 and 5: rows of 4 KB .. 80 KB).
//
// B200 mapping.  One persistent CTA per SM, W warps (16 for rows up to 16 KB, 8 above), WARP PER ROW.  Every warp runs its own ring of NS
// shared-memory stages; a stage is one contiguous SEGMENT of a row (up to 4 KB), fetched by one bulk asynchronous
// copy (cp.async.bulk global -> shared, completion on an mbarrier: the TMA engine moves the bytes), so each SM keeps
// W * (NS - 1) segments (~100 KB) of HBM reads in flight no matter what the lanes are doing.  Lane L reads the
// 16-byte chunks L, L + 32, ... of a segment (conflict-free LDS.128) against the centre held in shared memory and
// accumulates ||c_i - c||^2 on two chains; one xor-shuffle tree per ROW parks the row's sums in one lane, and the
// scalar epilogue (branch of P:L115, multiplier, KKT terms) runs for a BATCH of up to 32 rows at once, lane per
// row.  Rows are assigned row -> warp statically and round-robin over all warps of the grid (row = gw + k GW),
// which balances the warps to within one row.
//
// Flags go into a PRE-ZEROED bit mask with atomicOr (integer: order-independent).  Rows that carry a multiplier
// row v_i (slot >= 0; a few hundred at most away from degenerate supports) are left to vrow_kernel, which walks
// the list of such rows with one warp per row and plain 128-bit loads of both rows; its per-CTA partials are
// appended to those of the streaming kernel.  The gradient's vector part comes from the active-list kernel
// (meb_active.cu), as for every long-row evaluation.
//
// Determinism: static row -> warp assignment, per-lane accumulation in a fixed order, xor-shuffle trees, warps added
// in index order, CTA partials added in index order by the finalize kernel.  No floating-point atomics.
#include <string.h>

#include <type_traits>

#include "meb_internal.cuh"
#include "meb_rowops.cuh"

namespace {

__device__ __forceinline__ uint32_t lsmem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void lbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(lsmem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void lbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(lsmem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void lbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "LWAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra LWAIT_DONE;\n"
        "bra LWAIT_LOOP;\n"
        "LWAIT_DONE:\n"
        "}\n" ::"r"(lsmem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void lbulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     lsmem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(lsmem_u32(bar))
                 : "memory");
}

struct LongCfg {
    int W, NS;                 // warps per CTA, ring stages per warp
    uint32_t seg_bytes;        // bytes of a full segment, a multiple of 512 (32 lanes x 16 bytes)
    uint32_t data_bytes;       // bytes of a row that are fetched: its d columns rounded up to whole 16-byte chunks
    int nseg;                  // segments per row
    int nch;                   // 16-byte chunks per row
    int multi;                 // OP_EVAL: number of extra step sizes predicted per row (0: none)
    uint32_t off_dir;          // byte offset of the direction Delta c (multi > 0) in the dynamic shared memory
    uint32_t off_ring, off_bars, smem_total;
};

template <typename T> struct LChunk;
template <> struct LChunk<double> { typedef double2 type; static constexpr int N = 2; };
template <> struct LChunk<float>  { typedef float4 type;  static constexpr int N = 4; };

constexpr int LONG_MAXW = 16;
constexpr int LONG_THREADS = LONG_MAXW * 32;

template <typename T, int OP, bool SHADOW, bool MULTI>
__global__ void __launch_bounds__(LONG_THREADS, 1) long_kernel(const StreamArgs a, const LongCfg cfg) {
    typedef typename LChunk<T>::type V4;
    constexpr int VEC = LChunk<T>::N;
    extern __shared__ __align__(128) unsigned char smem[];
    double sigma_d = a.sigma;
    const void* Up = a.U; const int32_t* slotp = a.v_slot;
    if (a.dyn) {
        const int cur = a.dyn->cur;
        const bool hm = a.dyn->has_mult != 0;
        sigma_d = a.dyn->sigma_raw;
        Up = hm ? a.U2[cur] : nullptr; slotp = hm ? a.slot2[cur] : nullptr;
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int d = a.d;
    const int64_t m = a.m;
    const int W = cfg.W, NS = cfg.NS, nch = cfg.nch, nseg = cfg.nseg;
    const uint32_t seg_bytes = cfg.seg_bytes;
    T* cs = reinterpret_cast<T*>(smem);
    T* ds = reinterpret_cast<T*>(smem + cfg.off_dir);
    unsigned char* ring = smem + cfg.off_ring + (size_t)warp * NS * seg_bytes;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + cfg.off_bars) + warp * NS;
    const unsigned char* __restrict__ Cb = static_cast<const unsigned char*>(a.C);
    const T* __restrict__ Ug = static_cast<const T*>(Up);
    const T* __restrict__ Rg = static_cast<const T*>(a.R);
    const size_t row_bytes = (size_t)a.ld * sizeof(T);

    long long t_start = 0;
    if (threadIdx.x == 0) asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_start));
    const double* cptr = (OP == OP_INGEST) ? a.c0 : a.x + 1;
    const bool domulti = MULTI && a.dyn != nullptr && a.dyn->multi_n > 0;
#pragma unroll 8
    for (int j = threadIdx.x; j < nch * VEC; j += LONG_THREADS) cs[j] = j < d ? (T)cptr[j] : T(0);
    if (MULTI && domulti) {
#pragma unroll 8
        for (int j = threadIdx.x; j < nch * VEC; j += LONG_THREADS) ds[j] = j < d ? (T)a.dir[1 + j] : T(0);
    }
    if (lane == 0) {
        for (int s = 0; s < NS; ++s) lbar_init(&bars[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __shared__ double abort_slots[33];
    AbortCtl ab;
    if (OP == OP_EVAL) abort_init(ab, a.dyn, abort_slots);
    __syncthreads();

    const T r = (OP == OP_INGEST) ? T(0) : (T)a.x[0];
    const T sig = (T)sigma_d;
    Acc acc;
    MultiAcc<MULTI> macc;
    const V4* cs4 = reinterpret_cast<const V4*>(cs);
    const V4* ds4 = reinterpret_cast<const V4*>(ds);
    const int cps = (int)(seg_bytes / 16);                      // chunks of a full segment
    const bool haspad = nch * VEC != d;

    // rows of this warp: gw, gw + GW, ...
    const int64_t gw = (int64_t)warp * gridDim.x + blockIdx.x;
    const int64_t GW = (int64_t)gridDim.x * W;
    // ---- producer cursor (all lanes keep it; lane 0 issues) ----
    int64_t p_row = gw;
    int p_seg = 0, p_slot = 0;
    uint32_t issued = 0, consumed = 0;
    auto issue_one = [&]() {
        const uint32_t off = (uint32_t)p_seg * seg_bytes;
        const uint32_t bytes = (cfg.data_bytes - off) < seg_bytes ? (cfg.data_bytes - off) : seg_bytes;
        if (lane == 0) {
            lbar_expect_tx(&bars[p_slot], bytes);
            lbulk_g2s(ring + (size_t)p_slot * seg_bytes, Cb + (size_t)p_row * row_bytes + off, bytes, &bars[p_slot]);
        }
        if (++p_seg == nseg) { p_seg = 0; p_row += GW; }
        p_slot = (p_slot + 1 == NS) ? 0 : p_slot + 1;
        ++issued;
    };
    if (warp < W)
        for (int k = 0; k < NS && p_row < m; ++k) issue_one();

    int c_slot = 0;
    uint32_t parity = 0;
    bool aborted = false;
    // Epilogues are BATCHED: the sums of the q-th row of a batch are parked in lane q (its radius, multiplier and slot
    // are requested by that lane when the row starts to stream), and after 32 rows -- or the warp's last row -- every
    // lane runs the scalar epilogue of its own row: 32 times fewer epilogue instructions issued than with one
    // epilogue per row, which matters for rows of a few KB.
    int q = 0;
    // rows per batch: 32 for rows of a few KB, fewer for very long rows (the early stop of a doomed trial is
    // tested once per batch)
    int qmax = cfg.data_bytes >= 131072u ? 1 : (131072u / cfg.data_bytes > 32u ? 32 : (int)(131072u / cfg.data_bytes));
    {   // at least four batches per warp, so that a doomed trial of a small problem can still be cut
        const int64_t per_warp = (m + (int64_t)gridDim.x * W - 1) / ((int64_t)gridDim.x * W);
        if (per_warp < 4 * (int64_t)qmax) qmax = per_warp >= 4 ? (int)(per_warp / 4) : 1;
    }
    int64_t my_row = -1;
    T my_nb2 = T(0), my_f0 = T(0), my_p0 = T(0), ri = T(0), ui = T(0);
    int myslot = -1;
    auto flush = [&]() {
        if (lane < q && myslot < 0) {                                   // rows with a multiplier row: vrow_kernel
            double mylam;
            const bool flag = row_epilogue_core<T, OP>(a, my_row, true, false, my_nb2, my_f0, T(0), T(0), r, sig, ri, ui, acc, mylam);
            if (OP != OP_INGEST && flag) atomicOr(&a.mask[my_row >> 5], 1u << (my_row & 31));
            if (OP == OP_EVAL && a.smask != nullptr && a.dyn != nullptr && a.dyn->screen_on != 0) {
                // fused screening, the arithmetic of OP_SCREEN (the switch and the threshold are re-read
                // here, once per batch of rows, rather than kept in registers across the streaming loop)
                const T sslack = (r - ri) - t_sqrt<T>(my_nb2);
                if (sslack <= (T)(a.dyn->screen_factor * a.x[0])) atomicOr(&a.smask[my_row >> 5], 1u << (my_row & 31));
            }
            if (MULTI) multi_row<T>(macc, a, cfg.multi, my_nb2, my_p0, r, sig, ri, ui);
        }
        q = 0;
    };
    if (warp < W)
    for (int64_t row = gw; row < m; row += GW) {
        if (lane == q) {                                                // per-row scalars: requested now, used at the flush
            my_row = row; ri = T(0); ui = T(0); myslot = -1;
            if (Rg) ri = Rg[row];
            if (OP == OP_EVAL && Ug) ui = Ug[row];
            if (OP == OP_EVAL && slotp) myslot = slotp[row];
        }
        T s0 = T(0), s1 = T(0), f0 = T(0), p0 = T(0);
        for (int sg = 0; sg < nseg; ++sg) {
            lbar_wait(&bars[c_slot], parity);
            const V4* st4 = reinterpret_cast<const V4*>(ring + (size_t)c_slot * seg_bytes);
            const int ch0 = sg * cps;
            const int nchs = (nch - ch0) < cps ? (nch - ch0) : cps;
            const V4* c4 = cs4 + ch0;
            const V4* d4 = ds4 + ch0;
            float* srow = SHADOW ? a.C32 + row * a.ld32 : nullptr;
            auto chunk = [&](auto pm, int qc, bool last) {
                constexpr bool PM = decltype(pm)::value;
                const V4 ev4 = st4[qc];
                const V4 cv4 = c4[qc];
                const T* e = reinterpret_cast<const T*>(&ev4);
                const T* cc = reinterpret_cast<const T*>(&cv4);
                T ee[VEC];
#pragma unroll
                for (int j = 0; j < VEC; ++j) {
                    ee[j] = e[j] - cc[j];
                    if (last && (ch0 + qc) * VEC + j >= d) ee[j] = T(0);     // padding of the last chunk of the row
                    if (j & 1) s1 = fma(ee[j], ee[j], s1); else s0 = fma(ee[j], ee[j], s0);
                    if (OP == OP_INGEST) f0 = fma((last && (ch0 + qc) * VEC + j >= d) ? T(0) : e[j], T(0), f0);
                }
                if constexpr (PM) {
                    const V4 dv4 = d4[qc];
                    const T* dd = reinterpret_cast<const T*>(&dv4);
#pragma unroll
                    for (int j = 0; j < VEC; ++j) p0 = fma(ee[j], dd[j], p0);
                }
                if (SHADOW) {
                    const int col = (ch0 + qc) * VEC;
                    if (VEC == 2 && col + 1 < d) {
                        float2 o; o.x = (float)ee[0]; o.y = (float)ee[1];
                        *reinterpret_cast<float2*>(srow + col) = o;          // ld32 is a multiple of 4
                    } else {
#pragma unroll
                        for (int j = 0; j < VEC; ++j) if (col + j < d) srow[col + j] = (float)ee[j];
                    }
                }
            };
            const bool tail_seg = haspad && (ch0 + nchs == nch);
            auto walk = [&](auto pm) {
                if (nchs == cps && !tail_seg && (cps & 255) == 0) {
                    for (int q0 = lane; q0 < cps; q0 += 256) {
#pragma unroll
                        for (int u = 0; u < 8; ++u) chunk(pm, q0 + 32 * u, false);
                    }
                } else {
                    int qc = lane;
                    for (; qc + 96 < nchs; qc += 128) { chunk(pm, qc, false); chunk(pm, qc + 32, false); chunk(pm, qc + 64, false); chunk(pm, qc + 96, tail_seg && qc + 96 == nchs - 1); }
                    for (; qc < nchs; qc += 32) chunk(pm, qc, tail_seg && qc == nchs - 1);
                }
            };
            if (MULTI && domulti) walk(std::true_type{}); else walk(std::false_type{});
            __syncwarp();
            if (p_row < m && !aborted) {
                if (lane == 0) asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                issue_one();
            }
            ++consumed;
            if (++c_slot == NS) { c_slot = 0; parity ^= 1u; }
        }
        T nb2 = s0 + s1;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            nb2 += __shfl_xor_sync(MEB_FULL_MASK, nb2, o);
            if (OP == OP_INGEST) f0 += __shfl_xor_sync(MEB_FULL_MASK, f0, o);
            if (MULTI && domulti) p0 += __shfl_xor_sync(MEB_FULL_MASK, p0, o);
        }
        if (lane == q) { my_nb2 = nb2; my_f0 = f0; my_p0 = p0; }
        if (++q == qmax) {
            flush();
            if (OP == OP_EVAL && ab.on) {
                if (abort_seen(ab) || abort_publish(ab, acc, W)) { aborted = true; break; }
            }
        }
    }
    if (warp < W && !aborted) flush();
    // copies still in flight must land before the CTA may exit
    while (consumed < issued) {
        lbar_wait(&bars[c_slot], parity);
        ++consumed;
        if (++c_slot == NS) { c_slot = 0; parity ^= 1u; }
    }
    if (MULTI) multi_store(macc, a, W);
    block_reduce_store<OP>(acc, a.part, W);
    if (threadIdx.x == 0) {                 // device time stamps of this CTA (ns), read by the finalize kernel
        long long t_end;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_end));
        a.part[(size_t)blockIdx.x * MEB_NPART + 10] = __longlong_as_double(t_start);
        a.part[(size_t)blockIdx.x * MEB_NPART + 11] = __longlong_as_double(t_end);
        if (OP == OP_EVAL) abort_store(ab, a.part);
    }
}

// ---- rows that carry a multiplier row v_i: one warp per list entry, plain loads of both rows -------------------
// vlist[0 .. *vcount): ascending indices of the balls with slot >= 0.  CTA b writes its partial to
// part[(part_base + b) * MEB_NPART ...] (zeros when it has no entry): the finalize kernel adds them after the
// partials of the streaming kernel.
// TEAM = 32: warp per entry; TEAM = MEB_BLOCK: the whole CTA per entry (rows of 16 KB and more: one warp would need
// dozens of dependent-latency rounds per row).
template <typename T, bool MULTI, int TEAM>
__global__ void __launch_bounds__(MEB_BLOCK) vrow_kernel(const StreamArgs a_in, const int32_t* __restrict__ vlist,
                                                         const int32_t* __restrict__ vcount, int part_base, int multi) {
    typedef typename VecOf<T>::type V4;
    constexpr int VEC = VecOf<T>::N;
    StreamArgs a = a_in;
    const int32_t* vl = vlist; const int32_t* vc = vcount;
    if (a.dyn) {                                   // the list of the current multiplier buffer
        const int cur = a.dyn->cur;
        vl = a.vlist2[cur]; vc = a.vcount2[cur];
    }
    meb_resolve_dyn(a);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int d = a.d;
    const T* __restrict__ C = static_cast<const T*>(a.C);
    const T* __restrict__ V = static_cast<const T*>(a.V);
    const T* __restrict__ Ug = static_cast<const T*>(a.U);
    const T* __restrict__ Rg = static_cast<const T*>(a.R);
    const double* __restrict__ cx = a.x + 1;
    const T r = (T)a.x[0];
    const T sig = (T)a.sigma;
    const T inv_sig = T(1) / sig;
    const int n = (a.v_slot != nullptr && vc != nullptr) ? *vc : 0;
    const bool vec_ok = ((a.ld * (int64_t)sizeof(T)) % 16 == 0) && ((a.ldv * (int64_t)sizeof(T)) % 16 == 0) &&
                        ((uintptr_t)C % 16 == 0) && ((uintptr_t)V % 16 == 0);
    Acc acc;
    MultiAcc<MULTI> macc;
    __shared__ double vred[MEB_WARPS][5];
    constexpr int TPB = MEB_BLOCK / TEAM;
    const int tt = TEAM == 32 ? lane : (int)threadIdx.x;
    const int nteams = gridDim.x * TPB;
    for (int k = blockIdx.x * TPB + (TEAM == 32 ? warp : 0); k < n; k += nteams) {
        const int64_t row = vl[k];
        const int slot = a.v_slot[row];
        if (slot < 0) continue;                    // (a stale list entry cannot happen; defensive)
        const T* rowp = C + row * a.ld;
        const T* vrow = V + (int64_t)slot * a.ldv;
        T nb2 = T(0), ne2 = T(0), evd = T(0), vv = T(0), p0 = T(0);
        auto elem = [&](T cj, T vj, int col) {
            const T ee = cj - (T)cx[col];
            const T b = fma(vj, inv_sig, ee);
            nb2 = fma(b, b, nb2); ne2 = fma(ee, ee, ne2); evd = fma(ee, vj, evd); vv = fma(vj, vj, vv);
            if (MULTI) p0 = fma(b, (T)a.dir[1 + col], p0);
        };
        if (vec_ok) {
            const int nchunks = d / VEC;
            for (int c0 = tt; c0 < nchunks; c0 += TEAM * 4) {
                V4 e[4], v[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int c = c0 + TEAM * u;
                    if (c < nchunks) {
                        e[u] = ldg_stream(reinterpret_cast<const V4*>(rowp) + c);
                        v[u] = ldg_stream(reinterpret_cast<const V4*>(vrow) + c);
                    }
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int c = c0 + TEAM * u;
                    if (c < nchunks) {
                        const T* ep = reinterpret_cast<const T*>(&e[u]);
                        const T* vp = reinterpret_cast<const T*>(&v[u]);
#pragma unroll
                        for (int j = 0; j < VEC; ++j) elem(ep[j], vp[j], c * VEC + j);
                    }
                }
            }
            for (int col = nchunks * VEC + tt; col < d; col += TEAM) elem(__ldg(rowp + col), __ldg(vrow + col), col);
        } else {
            for (int col = tt; col < d; col += TEAM) elem(__ldg(rowp + col), __ldg(vrow + col), col);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            nb2 += __shfl_xor_sync(MEB_FULL_MASK, nb2, o);
            ne2 += __shfl_xor_sync(MEB_FULL_MASK, ne2, o);
            evd += __shfl_xor_sync(MEB_FULL_MASK, evd, o);
            vv += __shfl_xor_sync(MEB_FULL_MASK, vv, o);
            if (MULTI) p0 += __shfl_xor_sync(MEB_FULL_MASK, p0, o);
        }
        if (TEAM != 32) {                                   // warps of the CTA in index order
            __syncthreads();
            if (lane == 0) { vred[warp][0] = (double)nb2; vred[warp][1] = (double)ne2; vred[warp][2] = (double)evd; vred[warp][3] = (double)vv; vred[warp][4] = (double)p0; }
            __syncthreads();
            double t5[5] = {0, 0, 0, 0, 0};
            for (int w = 0; w < MEB_WARPS; ++w)
#pragma unroll
                for (int q5 = 0; q5 < 5; ++q5) t5[q5] += vred[w][q5];
            nb2 = (T)t5[0]; ne2 = (T)t5[1]; evd = (T)t5[2]; vv = (T)t5[3]; p0 = (T)t5[4];
        }
        if (tt == 0) {
            const T ri = Rg ? Rg[row] : T(0);
            const T ui = Ug ? Ug[row] : T(0);
            double mylam;
            const bool flag = row_epilogue_core<T, OP_EVAL>(a, row, true, true, nb2, ne2, evd, vv, r, sig, ri, ui, acc, mylam);
            if (flag) atomicOr(&a.mask[row >> 5], 1u << (row & 31));
            if (a.smask != nullptr && a.dyn != nullptr && a.dyn->screen_on != 0) {      // fused screening: ||c_i - c||^2 = ne2
                const T sslack = (r - ri) - t_sqrt<T>(ne2);
                if (sslack <= (T)(a.dyn->screen_factor * a.x[0])) atomicOr(&a.smask[row >> 5], 1u << (row & 31));
            }
            if (MULTI) multi_row<T>(macc, a, multi, nb2, p0, r, sig, ri, ui);
        }
    }
    StreamArgs b = a;
    b.part = a.part + (size_t)part_base * MEB_NPART;
    b.multi_part = a.multi_part ? a.multi_part + (size_t)part_base * MEB_MULTI_MAX : nullptr;
    if (MULTI) multi_store(macc, b, MEB_WARPS);
    block_reduce_store<OP_EVAL>(acc, b.part, MEB_WARPS);
    if (threadIdx.x == 0) {
        b.part[(size_t)blockIdx.x * MEB_NPART + MEB_PART_CUT] = 0.0;
        b.part[(size_t)blockIdx.x * MEB_NPART + 10] = 0.0;       // no time stamps: the finalize kernel skips t1 <= 0
        b.part[(size_t)blockIdx.x * MEB_NPART + 11] = 0.0;
    }
}

// list of the balls with slot >= 0 as a bit mask (input of the compaction that builds vlist)
__global__ void __launch_bounds__(256) slot_mask_kernel(const int32_t* __restrict__ slot, int64_t m,
                                                        uint32_t* __restrict__ mask) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t n32 = (m + 31) / 32 * 32;
    if (i >= n32) return;
    const bool f = i < m && slot[i] >= 0;
    const uint32_t bits = __ballot_sync(MEB_FULL_MASK, f);
    if ((threadIdx.x & 31) == 0) mask[i >> 5] = bits;
}

// vlist[nxt] <- the active list of the accepted pass (the rows the multiplier update just gave a slot)
__global__ void __launch_bounds__(256) copy_vlist_kernel(const int32_t* __restrict__ list, const int32_t* __restrict__ count,
                                                         const MebDyn* dyn, int32_t* v0, int32_t* v1, int32_t* c0, int32_t* c1,
                                                         int64_t cap) {
    const int nxt = dyn->has_mult ? 1 - dyn->cur : 0;
    int32_t* dst = nxt ? v1 : v0;
    const int n = *count;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n && k < cap; k += (int64_t)gridDim.x * blockDim.x)
        dst[k] = list[k];
    if (blockIdx.x == 0 && threadIdx.x == 0) *(nxt ? c1 : c0) = n < cap ? n : (int32_t)cap;
}

constexpr size_t LONG_SMEM_BUDGET = 212 * 1024;

bool make_long_cfg(const StreamArgs& a, size_t esize, int multi, LongCfg* out) {
    LongCfg c;
    memset(&c, 0, sizeof(c));
    c.nch = (int)(((size_t)a.d * esize + 15) / 16);
    c.data_bytes = (uint32_t)c.nch * 16u;
    c.multi = multi;
    const size_t cs_bytes = ((size_t)c.nch * 16 + 127) / 128 * 128;
    const size_t fixed = cs_bytes * (multi > 0 ? 2 : 1) + LONG_MAXW * 8 * sizeof(uint64_t) + 256;
    if (fixed + (size_t)2 * 2 * 2048 > LONG_SMEM_BUDGET) return false;
    // one stage per row up to 8 KB, else 4 KB segments
    uint32_t seg = c.data_bytes <= 8192 ? (c.data_bytes + 511u) / 512u * 512u : 4096u;
    // rows of a few KB: 16 warps (the per-row wait / reduce / issue chain of a warp is long compared with the
    // time its row takes to stream, so 8 warps do not keep the ring busy); very long rows: 8 warps, deeper rings
    int W = c.data_bytes <= 16384u ? LONG_MAXW : 8, NS = 0;
    for (;;) {
        NS = (int)((LONG_SMEM_BUDGET - fixed) / ((size_t)W * seg));
        if (NS >= 3 || (NS >= 2 && seg <= 2048 && W <= 4)) break;
        if (seg > 2048) seg = (seg / 2 + 511u) / 512u * 512u;       // smaller segments before fewer warps
        else if (W > 4) W -= 2;
        else return false;
    }
    if (NS > 6) NS = 6;
    // the direction of the multi-trial code must not starve the ring (FP64 rows of 80 KB: centre + direction = 160 KB)
    if (multi > 0 && (size_t)W * NS * seg < (size_t)96 * 1024 && (size_t)W * NS * seg < (size_t)c.data_bytes * 8) return false;
    c.W = W; c.NS = NS; c.seg_bytes = seg;
    c.nseg = (int)((c.data_bytes + seg - 1) / seg);
    c.off_dir = (uint32_t)cs_bytes;
    c.off_ring = (uint32_t)(cs_bytes * (multi > 0 ? 2 : 1));
    c.off_bars = (uint32_t)(c.off_ring + (size_t)W * NS * seg);
    c.smem_total = (uint32_t)((c.off_bars + (size_t)LONG_MAXW * 8 * sizeof(uint64_t) + 127) / 128 * 128);
    *out = c;
    return true;
}

template <typename KernelT>
int launch_long(meb_ctx* ctx, KernelT kernel, const StreamArgs& a, const LongCfg& c, int* grid_out) {
    int grid = ctx->sm_count > 0 ? ctx->sm_count : 148;
    const int64_t want = (a.m + c.W - 1) / c.W;                 // one row per warp at least
    if (want < grid) grid = (int)want;
    if (grid < 1) grid = 1;
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem_total);
    if (e != cudaSuccess) { ctx->last_cuda_error = (int)e; return MEB_E_CUDA; }
    ctx->launches++;
    kernel<<<grid, LONG_THREADS, c.smem_total, ctx->stream>>>(a, c);
    e = cudaGetLastError();
    if (e != cudaSuccess) { ctx->last_cuda_error = (int)e; return MEB_E_CUDA; }
    *grid_out = grid;
    return MEB_OK;
}

}  // namespace

bool meb_long_applicable(int op, int prec, const StreamArgs& a) {
    const size_t esize = prec == MEB_FP64 ? 8 : 4;
    const size_t row_bytes = (size_t)a.ld * esize;
    if (row_bytes <= 1024 && a.d <= 256) return false;          // short rows: meb_tile.cu
    if (row_bytes % 16 != 0 || ((uintptr_t)a.C % 16) != 0) return false;
    LongCfg c;
    return make_long_cfg(a, esize, 0, &c);
}

// Three steps, so that the caller can bracket the streaming kernel ALONE with its CUDA events:
//   phase 0: zero the mask (flags are OR-ed in);  phase 1: the streaming kernel, *grid_out = its CTAs;
//   phase 2: for an evaluation with multipliers, vrow_kernel over `vlist`; *grid_out += its CTAs (in: the grid of phase 1).
int meb_launch_long(meb_ctx* ctx, int phase, int op, int prec, const StreamArgs& a, const int32_t* vlist, const int32_t* vcount,
                    int* grid_out) {
    const size_t esize = prec == MEB_FP64 ? 8 : 4;
    int multi = (op == OP_EVAL) ? a.multi : 0;
    LongCfg c;
    if (multi > 0 && !make_long_cfg(a, esize, multi, &c)) multi = 0;      // no room for the direction: no predictions
    if (multi == 0 && !make_long_cfg(a, esize, 0, &c)) return MEB_E_CAPACITY;
    StreamArgs b = a;
    b.multi = multi;
    if (phase == 0) {
        if (op != OP_INGEST) {
            const size_t nwords = (size_t)(a.m + 31) / 32;
            cudaError_t e = cudaMemsetAsync(a.mask, 0, nwords * sizeof(uint32_t), ctx->stream);
            if (e == cudaSuccess && op == OP_EVAL && a.smask != nullptr)
                e = cudaMemsetAsync(a.smask, 0, nwords * sizeof(uint32_t), ctx->stream);    // (screening flags are OR-ed in too)
            if (e != cudaSuccess) { ctx->last_cuda_error = (int)e; return MEB_E_CUDA; }
        }
        return MEB_OK;
    }
    if (phase == 1) {
        int grid = 0, rc = MEB_E_ARG;
        if (prec == MEB_FP64) {
            switch (op) {
                case OP_EVAL:
                    rc = multi > 0 ? launch_long(ctx, long_kernel<double, OP_EVAL, false, true>, b, c, &grid)
                                   : launch_long(ctx, long_kernel<double, OP_EVAL, false, false>, b, c, &grid);
                    break;
                case OP_FEAS: rc = launch_long(ctx, long_kernel<double, OP_FEAS, false, false>, b, c, &grid); break;
                case OP_INGEST:
                    rc = a.C32 ? launch_long(ctx, long_kernel<double, OP_INGEST, true, false>, b, c, &grid)
                               : launch_long(ctx, long_kernel<double, OP_INGEST, false, false>, b, c, &grid);
                    break;
                default: return MEB_E_ARG;
            }
        } else {
            switch (op) {
                case OP_EVAL:
                    rc = multi > 0 ? launch_long(ctx, long_kernel<float, OP_EVAL, false, true>, b, c, &grid)
                                   : launch_long(ctx, long_kernel<float, OP_EVAL, false, false>, b, c, &grid);
                    break;
                case OP_SCREEN: rc = launch_long(ctx, long_kernel<float, OP_SCREEN, false, false>, b, c, &grid); break;
                default: return MEB_E_ARG;
            }
        }
        if (rc == MEB_OK) *grid_out = grid;
        return rc;
    }
    int grid = *grid_out;
    if (op == OP_EVAL && (a.v_slot != nullptr || a.dyn != nullptr)) {
        const int gv = 32;                                        // 256 warps: supports of a few thousand rows at most
        const bool wide = c.data_bytes >= 16384u;                 // CTA per entry
        ctx->launches++;
#define MEB_VROW(T, M) do { if (wide) vrow_kernel<T, M, MEB_BLOCK><<<gv, MEB_BLOCK, 0, ctx->stream>>>(b, vlist, vcount, grid, multi); \
                            else vrow_kernel<T, M, 32><<<gv, MEB_BLOCK, 0, ctx->stream>>>(b, vlist, vcount, grid, multi); } while (0)
        if (prec == MEB_FP64) { if (multi > 0) MEB_VROW(double, true); else MEB_VROW(double, false); }
        else { if (multi > 0) MEB_VROW(float, true); else MEB_VROW(float, false); }
#undef MEB_VROW
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) { ctx->last_cuda_error = (int)e; return MEB_E_CUDA; }
        grid += gv;
    }
    *grid_out = grid;
    return MEB_OK;
}

// vlist <- ascending indices of the balls with slot[i] >= 0, *vcount <- how many (uses ctx->vmask as scratch)
int meb_build_vlist(meb_ctx* ctx, const int32_t* slot, int64_t m, int32_t* vlist, int32_t* vcount) {
    const int64_t n32 = (m + 31) / 32 * 32;
    ctx->launches++;
    slot_mask_kernel<<<(unsigned)((n32 + 255) / 256), 256, 0, ctx->stream>>>(slot, m, ctx->vmask);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return meb_launch_compact_cap(ctx, ctx->vmask, m, vlist, m, vcount);
}

int meb_copy_vlist(meb_ctx* ctx, const int32_t* list, const int32_t* count, const MebDyn* dyn, int32_t* v0, int32_t* v1,
                   int32_t* c0, int32_t* c1, int64_t cap) {
    ctx->launches++;
    copy_vlist_kernel<<<64, 256, 0, ctx->stream>>>(list, count, dyn, v0, v1, c0, c1, cap);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}
