// TMA-staged streaming map-reduce for SHORT rows (row <= 1024 bytes): SURVEY 8(a) rows a0, a1, a7, a8.
//
// B200 mapping.  One persistent CTA per SM.  Every warp runs its own producer/consumer ring of NS
// shared-memory stages; a stage is one contiguous block of 32*R rows of C, fetched by ONE bulk
// asynchronous copy (cp.async.bulk global -> shared, completion on an mbarrier: the TMA engine moves
// the bytes, no registers, no per-thread address arithmetic), so each SM keeps W*(NS-1) stages
// (~100 KB) of HBM reads in flight regardless of how long the per-row epilogue is.  Inside a stage
// the mapping is LANE PER ROW: lane L reads its row from shared memory in 16-byte chunks (chunk
// order rotated by the lane index when the row stride is an even number of 16-byte slots, which
// makes the quarter-warp LDS.128 conflict-free), accumulates ||c_i - c||^2 with no shuffles, and runs
// the scalar epilogue (branch of P:L115, multiplier, KKT terms) for its own row.
//
// Fused evaluation (OP_EVAL): for every ACTIVE row of the stage (lam_i != 0, found by ballot) the
// warp adds lam_i b_i into per-lane register accumulators straight from the shared-memory copy of
// the row -- the gradient's vector part sum_i v+_i costs no second pass over C.
//
// Determinism: static stage -> warp assignment, per-lane / per-warp accumulation in a fixed order,
// warps combined in index order, CTA partials combined in index order by the finalize kernel.
#include <stdlib.h>
#include <string.h>

#include <type_traits>

#include "meb_internal.cuh"
#include "meb_rowops.cuh"

namespace {

// ---- mbarrier / bulk-copy PTX -------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
// one contiguous block global -> shared through the TMA engine; bytes is a multiple of 16
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// a row of zeros stands in for the multiplier row of a ball that has none (rows of at most 1024 bytes)
__device__ __align__(32) const double tile_zero_row[128] = {};

template <typename T> struct Chunk;
template <> struct Chunk<double> { typedef double2 type; static constexpr int N = 2; };
template <> struct Chunk<float>  { typedef float4 type;  static constexpr int N = 4; };

struct TileCfg {
    int G, logG;           // lanes per row (1, 2 or 4); a sub-tile is 32/G rows
    int R;                 // sub-tiles per stage
    int NS;                // stages per warp
    int W;                 // warps per CTA
    uint32_t row_bytes;    // ld * sizeof(T), a multiple of 16
    uint32_t stage_rows;   // R * 32 / G
    uint32_t stage_bytes;  // whole stage: rows, then per-row scalars u_i, r_i, slot_i (each 16-byte aligned)
    uint32_t off_u, off_r, off_slot;   // byte offsets of the per-row scalars inside a stage
    int nch;               // 16-byte chunks that cover the d columns of a row
    int rot;               // 1: rotate the chunk order by the row index (bank conflicts)
    int rowfast;           // 1: lane -> (row = lane % RPT, g = lane / RPT) instead of (row = lane / G, g = lane % G)
    int sc_tma;            // 1: per-row scalars come with the stage (their arrays are 16-byte aligned)
    int lognchp;           // gradient part: 2^lognchp = lanes that cover one row (>= nch, at most 32); the warp
                           // walks 32 >> lognchp active rows at a time
    uint32_t off_dir;      // byte offset of the direction Delta c (multi-trial Armijo), same layout as the centre
    int multi;             // predictions the kernel may be asked for (0: instance without the multi-trial code)
    uint32_t off_tiles;    // byte offsets inside the dynamic shared memory
    uint32_t off_bars;
    uint32_t off_vec;
    uint32_t smem_total;
};

// ---- the kernel ------------------------------------------------------------------------------------
// G  = lanes per row (compile time: chunk offsets become immediates);
// CH = 16-byte chunks per lane when a whole warp walks ONE row (active rows, shadow): ceil(nch / 32).
// MAXT = threads per CTA the instance may be launched with: stages of 8 KB and more leave room for at most 12
// warps, and those launches use the 384-thread instance, which may keep 168 registers per thread (the 512-thread
// one is held to 128 and rematerialises addresses inside the per-row loops).
template <typename T, int OP, int G, int CH, bool SHADOW, int MAXT, bool MULTI>
__global__ void __launch_bounds__(MAXT, 1) tile_kernel(const StreamArgs a, const TileCfg cfg) {
    typedef typename Chunk<T>::type V4;
    constexpr int VEC = Chunk<T>::N;
    constexpr int LG = G == 1 ? 0 : (G == 2 ? 1 : 2);
    constexpr int RPT = 32 / G;                                          // rows per sub-tile
    extern __shared__ __align__(128) unsigned char smem[];
    // device-resident parameters of a solve graph override the launch-time ones (no copy of `a`)
    double sigma_d = a.sigma;
    const void* Up = a.U; const int32_t* slotp = a.v_slot; const void* Vp = a.V;
    if (a.dyn) {
        const int cur = a.dyn->cur;
        const bool hm = a.dyn->has_mult != 0;
        sigma_d = a.dyn->sigma_raw;
        Up = hm ? a.U2[cur] : nullptr; slotp = hm ? a.slot2[cur] : nullptr; Vp = hm ? a.V2[cur] : nullptr;
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int d = a.d;
    const int m = (int)a.m;                                              // m < 2^31 - 64 (meb.h)
    const int W = cfg.W, NS = cfg.NS, R = cfg.R, nch = cfg.nch;
    // lane -> (row of the sub-tile, which of the G interleaved chunk sets): the host picks the mapping whose
    // quarter-warp LDS.128 wavefronts collide less for this row stride
    const int xsh = cfg.rowfast ? 5 - LG : 0;                            // partner lanes of a row differ in bits xsh..
    const int g = cfg.rowfast ? lane >> (5 - LG) : lane & (G - 1);
    const int rl = cfg.rowfast ? lane & (RPT - 1) : lane >> LG;
    T* cs = reinterpret_cast<T*>(smem);                                  // centre, padded to whole chunks
    unsigned char* tiles = smem + cfg.off_tiles + (size_t)warp * NS * cfg.stage_bytes;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + cfg.off_bars) + warp * NS;
    const unsigned char* __restrict__ Cb = static_cast<const unsigned char*>(a.C);
    const T* __restrict__ Vg = static_cast<const T*>(Vp);
    const T* __restrict__ Ug = static_cast<const T*>(Up);
    const T* __restrict__ Rg = static_cast<const T*>(a.R);
    const bool HASU = (OP == OP_EVAL) && Ug != nullptr;
    const bool HASV = (OP == OP_EVAL) && slotp != nullptr;
    const bool HASR = Rg != nullptr;

    long long t_start = 0;
    if (threadIdx.x == 0) asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_start));
    const double* cptr = (OP == OP_INGEST) ? a.c0 : a.x + 1;
    for (int j = threadIdx.x; j < nch * VEC; j += blockDim.x) cs[j] = j < d ? (T)cptr[j] : T(0);
    // multi-trial Armijo: this pass also predicts Psi at further points along Delta (MebDyn::multi_n), which
    // needs <b_i, Delta c> per row: Delta c sits in shared memory next to the centre
    const bool domulti = MULTI && a.dyn != nullptr && a.dyn->multi_n > 0;
    const int doff4 = (int)(cfg.off_dir / 16);                          // Delta c chunk = centre chunk + doff4
    if (MULTI) {
        T* dsm = reinterpret_cast<T*>(smem + cfg.off_dir);
        for (int j = threadIdx.x; j < nch * VEC; j += blockDim.x) dsm[j] = (domulti && j < d) ? (T)a.dir[1 + j] : T(0);
    }
    MultiAcc<MULTI> macc;
    if (lane == 0) {
        for (int s = 0; s < NS; ++s) mbar_init(&bars[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __shared__ double abort_slots[33];
    AbortCtl ab;
    if (OP == OP_EVAL) abort_init(ab, a.dyn, abort_slots);
    __syncthreads();

    const T r = (OP == OP_INGEST) ? T(0) : (T)a.x[0];
    const T sig = (T)sigma_d;
    const T inv_sig = T(1) / sig;
    Acc acc;
    // whole-warp-per-row view: lane owns chunks cl, cl + 32 (columns (cl + 32 q) * VEC + e).  Rows of at most
    // 16 chunks (OP_EVAL only) leave lanes over: the warp is split into RP = 32 / nchp groups of nchp lanes and
    // walks RP rows at a time, group `grp` taking rows grp, grp + RP, ... of a sub-tile.
    const int lognchp = (OP == OP_EVAL) ? cfg.lognchp : 5;
    const int cl = lane & ((1 << lognchp) - 1);
    const int grp = lane >> lognchp;
    const int RP = 32 >> lognchp;
    double vacc[CH][VEC], vaccB[CH][VEC];                              // two accumulation chains (rows rs, rs + RP)
    T creg[CH][VEC];
    const V4* cs4 = reinterpret_cast<const V4*>(cs);
#pragma unroll
    for (int q = 0; q < CH; ++q) {
        const int ch = cl + 32 * q;
        V4 cv;
        if (ch < nch) cv = cs4[ch];
        const T* cc = reinterpret_cast<const T*>(&cv);
#pragma unroll
        for (int e = 0; e < VEC; ++e) { vacc[q][e] = 0.0; vaccB[q][e] = 0.0; creg[q][e] = ch < nch ? cc[e] : T(0); }
    }

    // stages: st = gw, gw + GW, ...  (consecutive stages go to different SMs)
    const int rows_per_stage = (int)cfg.stage_rows;
    const int nstages = (m + rows_per_stage - 1) / rows_per_stage;
    const int gw = warp * (int)gridDim.x + (int)blockIdx.x;
    const int GW = (int)gridDim.x * W;
    const int mine = gw < nstages ? (nstages - gw + GW - 1) / GW : 0;
    const uint32_t sc_row_bytes = cfg.sc_tma ? ((HASU ? (uint32_t)sizeof(T) : 0u) + (HASR ? (uint32_t)sizeof(T) : 0u) + (HASV ? 4u : 0u)) : 0u;

    auto issue = [&](int k, int s) {                    // k-th stage of this warp -> ring slot s
        const int row0 = (gw + k * GW) * rows_per_stage;
        const int nrows = (m - row0) < rows_per_stage ? (m - row0) : rows_per_stage;
        const uint32_t nb = (uint32_t)(nrows & ~3);                      // rows whose scalars come in 16-byte units
        unsigned char* dst = tiles + (size_t)s * cfg.stage_bytes;
        const uint32_t rbytes = (uint32_t)nrows * cfg.row_bytes;
        mbar_expect_tx(&bars[s], rbytes + nb * sc_row_bytes);
        bulk_g2s(dst, Cb + (size_t)row0 * cfg.row_bytes, rbytes, &bars[s]);
        if (sc_row_bytes != 0u && nb > 0u) {
            if (HASU) bulk_g2s(dst + cfg.off_u, Ug + row0, nb * (uint32_t)sizeof(T), &bars[s]);
            if (HASR) bulk_g2s(dst + cfg.off_r, Rg + row0, nb * (uint32_t)sizeof(T), &bars[s]);
            if (HASV) bulk_g2s(dst + cfg.off_slot, slotp + row0, nb * 4u, &bars[s]);
        }
    };
    if (lane == 0)
        for (int k = 0; k < NS && k < mine; ++k) issue(k, k);

    const int ldT = (int)(cfg.row_bytes / sizeof(T));
    const int n_g = (nch - g + G - 1) >> LG;                             // my chunks: g, g + G, ...
    const int start = cfg.rot ? (rl % n_g) : 0;                          // rotated start (bank conflicts)
    const bool haspad = nch * VEC != d;

    int s = 0;
    uint32_t parity = 0;
    int srow0 = gw * rows_per_stage;
    const int srow_step = GW * rows_per_stage;
    bool aborted = false;
    int kend = mine;
    for (int k = 0; k < kend; ++k, srow0 += srow_step) {
        mbar_wait(&bars[s], parity);
        if (OP == OP_EVAL && !aborted && abort_seen(ab)) {
            aborted = true;                                              // stages in flight are still waited for,
            kend = (k + NS < mine) ? k + NS : mine;                      // nothing new is issued
        }
        if (aborted) { if (++s == NS) { s = 0; parity ^= 1u; } continue; }
        unsigned char* sbase = tiles + (size_t)s * cfg.stage_bytes;
        T* stage = reinterpret_cast<T*>(sbase);
        const T* Us = reinterpret_cast<const T*>(sbase + cfg.off_u);
        const T* Rs = reinterpret_cast<const T*>(sbase + cfg.off_r);
        const int32_t* Ss = reinterpret_cast<const int32_t*>(sbase + cfg.off_slot);
        const int snrows = (m - srow0) < rows_per_stage ? (m - srow0) : rows_per_stage;
        const int nbulk = cfg.sc_tma ? (snrows & ~3) : 0;
        for (int rr = 0; rr < R; ++rr) {
            const int rs0 = rr * RPT;                                    // first row of the sub-tile in the stage
            const int row0 = srow0 + rs0;
            if (row0 >= m) break;                                        // warp-uniform
            const int myrs = rs0 + rl;
            const int myrow = row0 + rl;
            const bool myvalid = myrow < m;
            T* rowp = stage + (size_t)myrs * ldT;
            // per-row scalars: staged with the rows, or (tail rows / unaligned arrays) read from global memory
            int myslot = -1;
            T ri = T(0), ui = T(0);
            if (myvalid) {
                if (myrs < nbulk) {
                    if (HASV) myslot = Ss[myrs];
                    if (HASR) ri = Rs[myrs];
                    if (HASU) ui = Us[myrs];
                } else {
                    if (HASV) myslot = slotp[myrow];
                    if (HASR) ri = Rg[myrow];
                    if (HASU) ui = Ug[myrow];
                }
            }
            T nb2 = T(0), ne2 = T(0), evd = T(0), vv = T(0), pdot = T(0);
            if (haspad) {                                                // zero the padding of the last chunk
                if (myvalid && g == 0)
                    for (int j = d; j < nch * VEC; ++j) rowp[j] = T(0);
                __syncwarp();
            }
            // a sub-tile with multiplier rows runs ONE loop for all its lanes (v = 0 where a row has none): two
            // divergent loops, one per kind of row, cost more than the few extra multiplications
            const bool wv = HASV && __any_sync(MEB_FULL_MASK, myvalid && myslot >= 0);
            if (myvalid) {
                if (!wv) {
                    T s0 = T(0), s1 = T(0), f0 = T(0);
                    const V4* rp = reinterpret_cast<const V4*>(rowp) + g;
                    const V4* cp = cs4 + g;
                    uint64_t s01 = 0ull, p01 = 0ull;                     // FP32: (s0, s1) and the two halves of pdot, packed pairs
                    T pp = T(0);
                    auto chunk = [&](auto pm, const V4* rq, const V4* cq) {
                        constexpr bool PM = decltype(pm)::value;
                        const V4 ev4 = *rq;
                        const V4 cv4 = *cq;
                        if constexpr (sizeof(T) == 4 && OP != OP_INGEST) {
                            // packed FP32 pairs (FADD2 / FFMA2 of sm_100): the same operations in the same order
                            // as the scalar form below (s0 takes columns 0 and 2 of the chunk, s1 columns 1 and 3)
                            const uint64_t* e2 = reinterpret_cast<const uint64_t*>(&ev4);
                            const uint64_t* c2 = reinterpret_cast<const uint64_t*>(&cv4);
                            uint64_t d0, d1;
                            asm("sub.f32x2 %0, %1, %2;" : "=l"(d0) : "l"(e2[0]), "l"(c2[0]));
                            asm("sub.f32x2 %0, %1, %2;" : "=l"(d1) : "l"(e2[1]), "l"(c2[1]));
                            asm("fma.rn.f32x2 %0, %1, %1, %0;" : "+l"(s01) : "l"(d0));
                            asm("fma.rn.f32x2 %0, %1, %1, %0;" : "+l"(s01) : "l"(d1));
                            if constexpr (PM) {
                                const V4 dv4 = *(cq + doff4);
                                const uint64_t* q2 = reinterpret_cast<const uint64_t*>(&dv4);
                                asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(p01) : "l"(d0), "l"(q2[0]));
                                asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(p01) : "l"(d1), "l"(q2[1]));
                            }
                            return;
                        }
                        const T* e = reinterpret_cast<const T*>(&ev4);
                        const T* cc = reinterpret_cast<const T*>(&cv4);
                        V4 dv4 = V4();
                        if constexpr (PM) dv4 = *(cq + doff4);
                        const T* dd = reinterpret_cast<const T*>(&dv4);
#pragma unroll
                        for (int j = 0; j < VEC; ++j) {
                            const T ee = e[j] - cc[j];
                            if (j & 1) s1 = fma(ee, ee, s1); else s0 = fma(ee, ee, s0);
                            if (OP == OP_INGEST) f0 = fma(e[j], T(0), f0);   // NaN iff a non-finite entry
                            if constexpr (PM) pp = fma(ee, dd[j], pp);
                        }
                    };
                    auto walk = [&](auto pm) {
                        if (!cfg.rot) {                                  // my chunks g, g + G, ... in order
                            const V4* rq = rp;
                            const V4* cq = cp;
                            int c = 0;
                            for (; c + 4 <= n_g; c += 4, rq += 4 * G, cq += 4 * G) {
                                chunk(pm, rq, cq); chunk(pm, rq + G, cq + G); chunk(pm, rq + 2 * G, cq + 2 * G); chunk(pm, rq + 3 * G, cq + 3 * G);
                            }
                            for (; c < n_g; ++c, rq += G, cq += G) chunk(pm, rq, cq);
                        } else {                                         // same trip count, start rotated by the row index
                            int ci = start;
                            for (int c = 0; c < n_g; ++c) {
                                chunk(pm, rp + ci * G, cp + ci * G);
                                ci = (ci + 1 == n_g) ? 0 : ci + 1;
                            }
                        }
                    };
                    if (MULTI && domulti) walk(std::true_type{}); else walk(std::false_type{});
                    if constexpr (sizeof(T) == 4 && OP != OP_INGEST) {
                        float p0, p1;
                        asm("mov.b64 {%0, %1}, %2;" : "=f"(p0), "=f"(p1) : "l"(s01));
                        s0 = (T)p0; s1 = (T)p1;
                        if (MULTI) {
                            asm("mov.b64 {%0, %1}, %2;" : "=f"(p0), "=f"(p1) : "l"(p01));
                            pp = (T)p0 + (T)p1;
                        }
                    }
                    pdot = pp;
                    nb2 = s0 + s1;
                    if (OP == OP_INGEST) ne2 = f0;
                } else {                                                 // sub-tile with multiplier rows v_i
                    // 16-byte chunks of the V row straight from global memory (rows of the pool are in ascending
                    // ball order, so neighbouring lanes read neighbouring pool rows); a lane whose row has no v_i
                    // reads a row of zeros instead (one broadcast sector), which keeps the loop free of predicates.
                    // The V loads of a batch of 8 chunks are issued together (one exposed latency per batch), then
                    // the arithmetic runs on registers.  Chunk order rotated by the row index like the rows
                    // without multipliers (lanes of a quarter warp would otherwise read the same banks).
                    const V4* rp = reinterpret_cast<const V4*>(rowp);
                    const bool v16 = (a.ldv * (int64_t)sizeof(T)) % 16 == 0 && (reinterpret_cast<uintptr_t>(Vg) % 16) == 0;
                    const bool hasrow = myslot >= 0;
                    const T* vrowT = hasrow ? Vg + (int64_t)myslot * a.ldv : reinterpret_cast<const T*>(tile_zero_row);
                    const V4* vrow4 = reinterpret_cast<const V4*>(vrowT);
                    // FAST: whole batches, no column padding, aligned pool rows, power-of-two chunk count
                    auto vwalk = [&](auto fast) {
                        constexpr bool FAST = decltype(fast)::value;
                        for (int k0 = 0; k0 < n_g; k0 += 8) {
                            V4 vb[8];
                            int cidx[8];
#pragma unroll
                            for (int u = 0; u < 8; ++u) {
                                int ci = start + k0 + u;
                                if (FAST) ci &= n_g - 1; else if (ci >= n_g) ci -= n_g;
                                cidx[u] = g + (ci << LG);
                            }
#pragma unroll
                            for (int u = 0; u < 8; ++u) {
                                const int c = cidx[u];
                                if (FAST) {
                                    vb[u] = __ldg(vrow4 + c);
                                } else {
                                    vb[u] = V4();
                                    if (k0 + u < n_g) {
                                        if (v16) {
                                            vb[u] = __ldg(vrow4 + c);
                                        } else {
                                            T* vq = reinterpret_cast<T*>(&vb[u]);
#pragma unroll
                                            for (int j = 0; j < VEC; ++j) vq[j] = (c * VEC + j < d) ? __ldg(vrowT + c * VEC + j) : T(0);
                                        }
                                    }
                                }
                            }
#pragma unroll
                            for (int u = 0; u < 8; ++u) {
                                const int c = cidx[u];
                                if (FAST || k0 + u < n_g) {
                                    const V4 ev4 = rp[c];
                                    const V4 cv4 = cs4[c];
                                    const T* e = reinterpret_cast<const T*>(&ev4);
                                    const T* cc = reinterpret_cast<const T*>(&cv4);
                                    const T* vq = reinterpret_cast<const T*>(&vb[u]);
                                    const int col = c * VEC;
#pragma unroll
                                    for (int j = 0; j < VEC; ++j) {
                                        const T ee = e[j] - cc[j];               // padding of the row was zeroed above
                                        const T v = (FAST || col + j < d) ? vq[j] : T(0);   // padding of the pool row is not
                                        const T bq = fma(v, inv_sig, ee);
                                        if (MULTI && domulti) pdot = fma(bq, reinterpret_cast<const T*>(cs4 + doff4)[col + j], pdot);
                                        nb2 = fma(bq, bq, nb2);
                                        ne2 = fma(ee, ee, ne2);
                                        evd = fma(ee, v, evd);
                                        vv = fma(v, v, vv);
                                    }
                                }
                            }
                        }
                    };
                    if (!haspad && v16 && (n_g & 7) == 0 && (n_g & (n_g - 1)) == 0) vwalk(std::true_type{});
                    else vwalk(std::false_type{});
                }
            }
#pragma unroll
            for (int o = G >> 1; o > 0; o >>= 1) {                       // combine the G lanes of a row
                const int ox = o << xsh;
                nb2 += __shfl_xor_sync(MEB_FULL_MASK, nb2, ox);
                if (MULTI && domulti) pdot += __shfl_xor_sync(MEB_FULL_MASK, pdot, ox);
                if (HASV || OP == OP_INGEST) ne2 += __shfl_xor_sync(MEB_FULL_MASK, ne2, ox);
                if (HASV) {
                    evd += __shfl_xor_sync(MEB_FULL_MASK, evd, ox);
                    vv += __shfl_xor_sync(MEB_FULL_MASK, vv, ox);
                }
            }
            double mylam;
            const bool flag = row_epilogue_core<T, OP>(a, myrow, myvalid && g == 0, myslot >= 0, nb2, ne2, evd, vv,
                                                       r, sig, ri, ui, acc, mylam);
            if (MULTI && domulti && myvalid && g == 0) multi_row<T>(macc, a, cfg.multi, nb2, pdot, r, sig, ri, ui);
            if (OP != OP_INGEST) {
                uint32_t bits = __ballot_sync(MEB_FULL_MASK, flag);      // bit of the g = 0 lane of row rl
                if (G == 1) {
                    if (lane == 0) a.mask[row0 >> 5] = bits;
                } else {   // RPT-bit piece of the 32-row mask word: lane q < RPT takes the flag of row q
                    uint32_t piece = bits;                               // rowfast: lane q < RPT is row q, g = 0
                    if (!cfg.rowfast) {
                        const bool f2 = __shfl_sync(MEB_FULL_MASK, (int)flag, (lane << LG) & 31) != 0 && lane < RPT;
                        piece = __ballot_sync(MEB_FULL_MASK, f2);
                    }
                    if (lane == 0) {
                        if (G == 2) reinterpret_cast<uint16_t*>(a.mask)[row0 >> 4] = (uint16_t)piece;
                        else reinterpret_cast<uint8_t*>(a.mask)[row0 >> 3] = (uint8_t)piece;
                    }
                }
                if (OP == OP_EVAL && bits != 0u) {
                    // gradient vector part: sum over the ACTIVE rows of lam_i b_i, from shared memory.  The active
                    // rows of the sub-tile are first compacted (ascending) into a warp-private list of (row, lam_i,
                    // slot of v_i); group `grp` of the warp then walks the entries grp, grp + RP, ..., lane `cl` of
                    // the group owning the 16-byte chunks cl, cl + 32 of every row.  Work is proportional to the
                    // number of active rows (a loop over all 32 rows that skipped the inactive ones cost a third of
                    // the pass's instructions on config 4, where every second row is active).
                    __shared__ double lam_w[16][32];
                    __shared__ int32_t slot_w[16][32];
                    __shared__ uint8_t row_w[16][32];
                    if (flag) {                                          // flag only on the g = 0 lane of a row
                        const int o = __popc(bits & ((1u << lane) - 1u));
                        lam_w[warp][o] = mylam; slot_w[warp][o] = myslot; row_w[warp][o] = (uint8_t)rl;
                    }
                    __syncwarp();
                    const int nact = __popc(bits);
                    const bool v16a = (a.ldv * (int64_t)sizeof(T)) % 16 == 0 && (reinterpret_cast<uintptr_t>(Vg) % 16) == 0;
                    auto load_v = [&](int slot, int ch) -> V4 {          // chunk ch of pool row `slot` (zero if none)
                        V4 vb = V4();
                        if (slot >= 0) {
                            const T* vrow = Vg + (int64_t)slot * a.ldv + ch * VEC;
                            if (v16a) {
                                vb = __ldg(reinterpret_cast<const V4*>(vrow));
                            } else {
                                T* vq = reinterpret_cast<T*>(&vb);
#pragma unroll
                                for (int j = 0; j < VEC; ++j) vq[j] = (ch * VEC + j < d) ? __ldg(vrow + j) : T(0);
                            }
                        }
                        return vb;
                    };
                    const bool anyv = HASV && __any_sync(MEB_FULL_MASK, flag && myslot >= 0);
                    if (anyv && MAXT == 384) {
                        // rows with a multiplier row v_i: b_i = c_i - c + v_i / sigma.  The pool rows come from
                        // global memory (L1 / L2: the norm part has just read them); the loads of FOUR entries of
                        // my group are issued before any of them is used.  Entries alternate between the two
                        // accumulation chains.  (384-thread instance only: the batch spills in the 512-thread one.)
                        // FAST: every lane of a group owns a chunk, no column padding, aligned pool rows; an entry
                        // without v_i (or past the end of the list) reads the row of zeros.
                        auto gwalk = [&](auto fast) {
                            constexpr bool FAST = decltype(fast)::value;
                            for (int k0 = grp; k0 < nact; k0 += 4 * RP) {
                                double lam4[4];
                                int sl4[4], r4[4];
                                V4 vb[4][CH];
#pragma unroll
                                for (int u = 0; u < 4; ++u) {
                                    const int kq = k0 + u * RP;
                                    const bool on = kq < nact;
                                    lam4[u] = on ? lam_w[warp][kq] : 0.0;
                                    sl4[u] = on ? slot_w[warp][kq] : -1;
                                    r4[u] = on ? (int)row_w[warp][kq] : (FAST ? (int)row_w[warp][k0] : -1);
                                }
#pragma unroll
                                for (int u = 0; u < 4; ++u)
#pragma unroll
                                    for (int q = 0; q < CH; ++q) {
                                        const int ch = cl + 32 * q;
                                        if (FAST) {
                                            const T* vrow = sl4[u] >= 0 ? Vg + (int64_t)sl4[u] * a.ldv : reinterpret_cast<const T*>(tile_zero_row);
                                            vb[u][q] = __ldg(reinterpret_cast<const V4*>(vrow) + ch);
                                        } else {
                                            vb[u][q] = load_v(ch < nch ? sl4[u] : -1, ch);
                                        }
                                    }
#pragma unroll
                                for (int u = 0; u < 4; ++u) {
                                    if (!FAST && r4[u] < 0) continue;    // (FAST: lam = 0 on a valid row adds exactly zero)
                                    const V4* rp4 = reinterpret_cast<const V4*>(stage + (size_t)(rs0 + r4[u]) * ldT);
#pragma unroll
                                    for (int q = 0; q < CH; ++q) {
                                        const int ch = cl + 32 * q;
                                        if (FAST || ch < nch) {
                                            const V4 ev4 = rp4[ch];
                                            const T* e = reinterpret_cast<const T*>(&ev4);
                                            const T* vq = reinterpret_cast<const T*>(&vb[u][q]);
#pragma unroll
                                            for (int j = 0; j < VEC; ++j) {
                                                T bj = e[j] - creg[q][j];
                                                if (FAST) bj = fma(vq[j], inv_sig, bj);
                                                else if (sl4[u] >= 0 && ch * VEC + j < d) bj = fma(vq[j], inv_sig, bj);
                                                if (u & 1) vaccB[q][j] = fma(lam4[u], (double)bj, vaccB[q][j]);
                                                else vacc[q][j] = fma(lam4[u], (double)bj, vacc[q][j]);
                                            }
                                        }
                                    }
                                }
                            }
                        };
                        if (CH == 1 && !haspad && v16a && nch == (1 << lognchp)) gwalk(std::true_type{});
                        else gwalk(std::false_type{});
                    } else {
                        // two entries of my group per step (chains A and B); a missing second entry repeats the
                        // first row with lam = 0 and adds exactly zero.  FAST as above (then an entry without v_i
                        // reads the row of zeros and the loop has no predicates).
                        auto gwalk2 = [&](auto fast, auto withv) {
                            constexpr bool FAST = decltype(fast)::value;
                            constexpr bool WV = decltype(withv)::value;
                            for (int k0 = grp; k0 < nact; k0 += 2 * RP) {
                                const int kB = k0 + RP;
                                const bool hasB = kB < nact;
                                const double lamA = lam_w[warp][k0];
                                const double lamB = hasB ? lam_w[warp][kB] : 0.0;
                                const int rA = row_w[warp][k0];
                                const int rB = hasB ? (int)row_w[warp][kB] : rA;
                                const int slotA = WV ? slot_w[warp][k0] : -1;
                                const int slotB = (WV && hasB) ? slot_w[warp][kB] : -1;
                                const V4* rpA = reinterpret_cast<const V4*>(stage + (size_t)(rs0 + rA) * ldT);
                                const V4* rpB = reinterpret_cast<const V4*>(stage + (size_t)(rs0 + rB) * ldT);
#pragma unroll
                                for (int q = 0; q < CH; ++q) {
                                    const int ch = cl + 32 * q;
                                    if (FAST || ch < nch) {
                                        V4 vA = V4(), vB = V4();
                                        if (WV && FAST) {
                                            const T* pa = slotA >= 0 ? Vg + (int64_t)slotA * a.ldv : reinterpret_cast<const T*>(tile_zero_row);
                                            const T* pb = slotB >= 0 ? Vg + (int64_t)slotB * a.ldv : reinterpret_cast<const T*>(tile_zero_row);
                                            vA = __ldg(reinterpret_cast<const V4*>(pa) + ch);
                                            vB = __ldg(reinterpret_cast<const V4*>(pb) + ch);
                                        } else if (WV) {
                                            vA = load_v(slotA, ch); vB = load_v(slotB, ch);
                                        }
                                        const V4 eA = rpA[ch];
                                        const V4 eB = rpB[ch];
                                        const T* ea = reinterpret_cast<const T*>(&eA);
                                        const T* eb = reinterpret_cast<const T*>(&eB);
                                        const T* va = reinterpret_cast<const T*>(&vA);
                                        const T* vbq = reinterpret_cast<const T*>(&vB);
#pragma unroll
                                        for (int j = 0; j < VEC; ++j) {
                                            T bA = ea[j] - creg[q][j], bB = eb[j] - creg[q][j];
                                            if (WV && FAST) { bA = fma(va[j], inv_sig, bA); bB = fma(vbq[j], inv_sig, bB); }
                                            else if (WV) {
                                                if (slotA >= 0 && ch * VEC + j < d) bA = fma(va[j], inv_sig, bA);
                                                if (slotB >= 0 && ch * VEC + j < d) bB = fma(vbq[j], inv_sig, bB);
                                            }
                                            vacc[q][j] = fma(lamA, (double)bA, vacc[q][j]);
                                            vaccB[q][j] = fma(lamB, (double)bB, vaccB[q][j]);
                                        }
                                    }
                                }
                            }
                        };
                        const bool fastg = CH == 1 && !haspad && v16a && nch == (1 << lognchp);
                        if (anyv) { if (fastg) gwalk2(std::true_type{}, std::true_type{}); else gwalk2(std::false_type{}, std::true_type{}); }
                        else { if (fastg) gwalk2(std::true_type{}, std::false_type{}); else gwalk2(std::false_type{}, std::false_type{}); }
                    }
                    __syncwarp();                                        // the lists are rewritten by the next sub-tile
                }
            }
            if (SHADOW) {                       // FP32 shadow of the centred rows (reading 8)
                const int nr = (m - row0) < RPT ? (m - row0) : RPT;
#pragma unroll 4
                for (int rs = 0; rs < nr; ++rs) {
                    const V4* rp4 = reinterpret_cast<const V4*>(stage + (size_t)(rs0 + rs) * ldT);
                    float* srow = a.C32 + (int64_t)(row0 + rs) * a.ld32;
#pragma unroll
                    for (int q = 0; q < CH; ++q) {
                        const int ch = lane + 32 * q;
                        if (ch < nch) {
                            const V4 ev4 = rp4[ch];
                            const T* e = reinterpret_cast<const T*>(&ev4);
                            const int col = ch * VEC;
                            if (VEC == 2 && col + 1 < d) {
                                float2 o;
                                o.x = (float)(e[0] - creg[q][0]);
                                o.y = (float)(e[1] - creg[q][1]);
                                *reinterpret_cast<float2*>(srow + col) = o;       // ld32 is a multiple of 4
                            } else {
#pragma unroll
                                for (int j = 0; j < VEC; ++j)
                                    if (col + j < d) srow[col + j] = (float)(e[j] - creg[q][j]);
                            }
                        }
                    }
                }
            }
        }
        if (OP == OP_EVAL && ab.on && (k & 3) == 0 && abort_publish(ab, acc, W)) {
            aborted = true;
            kend = (k + NS < mine) ? k + NS : mine;
        }
        __syncwarp();
        if (lane == 0 && k + NS < mine && !aborted) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // accesses above before the refill
            issue(k + NS, s);
        }
        if (++s == NS) { s = 0; parity ^= 1u; }
    }
    // ---- CTA partials, fixed order ----
    if (OP == OP_EVAL) {
        double* vs = reinterpret_cast<double*>(smem + cfg.off_vec);      // [W][CH * 32 * VEC]
        constexpr int VW = CH * 32 * VEC;
        __syncthreads();
#pragma unroll
        for (int q = 0; q < CH; ++q)
#pragma unroll
            for (int j = 0; j < VEC; ++j) vacc[q][j] += vaccB[q][j];
        for (int o = 1 << lognchp; o < 32; o <<= 1)                     // row groups of the warp, fixed order
#pragma unroll
            for (int q = 0; q < CH; ++q)
#pragma unroll
                for (int j = 0; j < VEC; ++j) vacc[q][j] += __shfl_xor_sync(MEB_FULL_MASK, vacc[q][j], o);
        if (grp == 0) {
#pragma unroll
            for (int q = 0; q < CH; ++q)
#pragma unroll
                for (int j = 0; j < VEC; ++j) vs[(size_t)warp * VW + (cl + 32 * q) * VEC + j] = vacc[q][j];
        }
        __syncthreads();
        double* pv = a.part_vec + (size_t)blockIdx.x * a.dpad;
        for (int j = threadIdx.x; j < d; j += blockDim.x) {
            double sacc = 0.0;
            for (int w = 0; w < W; ++w) sacc += vs[(size_t)w * VW + j];
            pv[j] = sacc;
        }
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

}  // namespace

// ---- host-side configuration and dispatch --------------------------------------------------------
namespace {

constexpr size_t TILE_SMEM_BUDGET = 212 * 1024;     // of the 227 KB a CTA may use on sm_100

bool aligned16(const void* p) { return ((uintptr_t)p % 16) == 0; }

int lanes_per_row(const StreamArgs& a, size_t esize);

bool make_cfg(const StreamArgs& a, size_t esize, int cpl, int grid, TileCfg* out) {
    TileCfg c;
    memset(&c, 0, sizeof(c));
    c.row_bytes = (uint32_t)(a.ld * (int64_t)esize);
    c.nch = (int)(((size_t)a.d * esize + 15) / 16);
    c.G = lanes_per_row(a, esize);
    c.lognchp = 0;
    while (c.lognchp < 5 && (1 << c.lognchp) < c.nch) ++c.lognchp;
    c.logG = c.G == 1 ? 0 : (c.G == 2 ? 1 : 2);
    const int rpt = 32 / c.G;
    const int slots = (int)(c.row_bytes / 16);
    {   // bank conflicts of the quarter-warp LDS.128 (8 lanes, 8 slots of 16 bytes per wavefront): lane
        // (rl, g) reads slot S rl + g + G ((c + rot rl) mod n_g); pick the rotation with fewer collisions
        auto collisions = [&](int rowfast, int rot) {
            int coll = 0;
            for (int q = 0; q < 4; ++q) {                     // the four quarter-warps
                int cnt[8] = {0, 0, 0, 0, 0, 0, 0, 0};
                for (int l = 8 * q; l < 8 * q + 8; ++l) {
                    const int g = rowfast ? l / rpt : l % c.G, rl = rowfast ? l % rpt : l / c.G;
                    const int n_g = (c.nch - g + c.G - 1) / c.G;
                    const int ci = rot && n_g > 0 ? rl % n_g : 0;
                    cnt[(slots * rl + g + c.G * ci) & 7]++;
                }
                for (int b = 0; b < 8; ++b) if (cnt[b] > 1) coll += cnt[b] - 1;
            }
            return coll;
        };
        int best = collisions(0, 0);
        c.rot = 0; c.rowfast = 0;
        bool try_rowfast = c.G > 1;
#ifdef MEB_TUNING
        if (getenv("MEB_TILE_NO_ROWFAST")) try_rowfast = false;
#endif
        if (try_rowfast) {
            const int cr = collisions(1, 0);
            if (cr < best) { best = cr; c.rowfast = 1; }
        }
        // rotation costs instructions: use it only against severe (>= 4-way on average) conflicts
        if (best >= 24) {
            const int c0 = collisions(c.rowfast, 1);
            if (c0 < best) { best = c0; c.rot = 1; }
        }
    }
    // stage of about 12 KB of rows, but never so large that a small problem lands on a handful of warps
    int R = (int)(6656 / ((size_t)rpt * c.row_bytes));
    if (R < 1) R = 1;
    if (R > 8) R = 8;
    while (R > 1 && (a.m + (int64_t)rpt * R - 1) / ((int64_t)rpt * R) < (int64_t)grid * 16 * 4) --R;
    c.R = R;
    c.stage_rows = (uint32_t)(R * rpt);
    c.off_u = c.stage_rows * c.row_bytes;
    c.off_r = c.off_u + c.stage_rows * (uint32_t)esize;
    c.off_slot = c.off_r + c.stage_rows * (uint32_t)esize;
    c.stage_bytes = (c.off_slot + c.stage_rows * 4u + 127u) / 128u * 128u;
    c.sc_tma = 1;
    const void* ptrs[] = {a.U, a.R, a.v_slot, a.U2[0], a.U2[1], a.slot2[0], a.slot2[1]};
    for (const void* q : ptrs) if (q && !aligned16(q)) c.sc_tma = 0;
    const size_t cs1 = ((size_t)c.nch * 16 + 127) / 128 * 128;
    c.multi = a.multi > 0 ? a.multi : 0;
    c.off_dir = (uint32_t)cs1;
    const size_t cs_bytes = cs1 * (c.multi > 0 ? 2 : 1);               // centre, then Delta c for the multi-trial instances
    int W = 16, NS = 0;
    int want_ns = 2;
#ifdef MEB_TUNING                     // tuning knobs of experimental builds (build.sh -DMEB_TUNING); clamped
    if (getenv("MEB_TILE_NS")) want_ns = atoi(getenv("MEB_TILE_NS")) < 3 ? 2 : (atoi(getenv("MEB_TILE_NS")) > 3 ? 4 : 3);
    if (getenv("MEB_TILE_W")) { W = atoi(getenv("MEB_TILE_W")); W = W < 2 ? 2 : (W > 16 ? 16 : W); }
    if (getenv("MEB_TILE_R")) {
        c.R = atoi(getenv("MEB_TILE_R"));
        c.R = c.R < 1 ? 1 : (c.R > 8 ? 8 : c.R);
        c.stage_rows = (uint32_t)(c.R * rpt);
        c.off_u = c.stage_rows * c.row_bytes;
        c.off_r = c.off_u + c.stage_rows * (uint32_t)esize;
        c.off_slot = c.off_r + c.stage_rows * (uint32_t)esize;
        c.stage_bytes = (c.off_slot + c.stage_rows * 4u + 127u) / 128u * 128u;
    }
#endif
    for (; W >= 2; --W) {
        const size_t fixed = cs_bytes + 16 * 4 * sizeof(uint64_t) + 256;
        if (fixed + (size_t)W * want_ns * c.stage_bytes > TILE_SMEM_BUDGET) continue;
        NS = (int)((TILE_SMEM_BUDGET - fixed) / ((size_t)W * c.stage_bytes));
        if (NS > 4) NS = 4;
        break;
    }
    if (NS < 2) return false;
    c.W = W; c.NS = NS;
    c.off_tiles = (uint32_t)cs_bytes;
    c.off_bars = (uint32_t)(cs_bytes + (size_t)W * NS * c.stage_bytes);
    c.off_vec = c.off_tiles;          // the per-warp vector partials reuse the stage ring (all stages consumed by then)
    c.smem_total = (uint32_t)((c.off_bars + (size_t)W * NS * sizeof(uint64_t) + 127) / 128 * 128);
    *out = c;
    return true;
}

size_t cfg_smem(const TileCfg& c, int cpl) {
    const size_t vec_end = (size_t)c.off_vec + (size_t)c.W * 32 * cpl * sizeof(double);
    return vec_end > c.smem_total ? vec_end : c.smem_total;
}

template <typename KernelT>
int launch_cfg(meb_ctx* ctx, KernelT kernel512, KernelT kernel384, const StreamArgs& a, size_t esize, int cpl, int* grid_out) {
    int grid = ctx->sm_count > 0 ? ctx->sm_count : 148;            // one persistent CTA per SM
    TileCfg c;
    if (!make_cfg(a, esize, cpl, grid, &c)) return MEB_E_CAPACITY;
    KernelT kernel = c.W <= 12 ? kernel384 : kernel512;
    const int64_t nstages = (a.m + c.stage_rows - 1) / c.stage_rows;
    if (nstages < grid) grid = (int)nstages;                       // stage k -> CTA k % grid, warp k / grid
    if (grid < 1) grid = 1;
    const size_t smem = cfg_smem(c, cpl);
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) { ctx->last_cuda_error = (int)e; return MEB_E_CUDA; }
    ctx->launches++;
    kernel<<<grid, 32 * c.W, smem, ctx->stream>>>(a, c);
    e = cudaGetLastError();
    if (e != cudaSuccess) { ctx->last_cuda_error = (int)e; return MEB_E_CUDA; }
    *grid_out = grid;
    return MEB_OK;
}

int lanes_per_row(const StreamArgs& a, size_t esize) {
    const size_t rb = (size_t)a.ld * esize;
    // sub-tile of at most ~8 KB.  (Two lanes per row for 256-byte rows, i.e. stages of 4 KB, were measured on config 4:
    // the pass slows from 0.60 to 0.90 ms -- the kernel is bound by per-stage instruction overhead.)
    return rb <= 256 ? 1 : (rb <= 416 ? 2 : 4);
}

// G is fixed by the row length; CH = 2 only occurs with G = 4 (rows longer than 512 bytes)
template <typename T, int OP, bool SHADOW, bool MULTI>
int launch_g(meb_ctx* ctx, const StreamArgs& a, bool want_ch, int* grid_out) {
    const int nch = (int)(((size_t)a.d * sizeof(T) + 15) / 16);        // <= 64 (rows of at most 1024 bytes)
    constexpr int VEC = 16 / sizeof(T);
    const int G = lanes_per_row(a, sizeof(T));
    if (G == 1) return launch_cfg(ctx, tile_kernel<T, OP, 1, 1, SHADOW, 512, MULTI>, tile_kernel<T, OP, 1, 1, SHADOW, 384, MULTI>, a, sizeof(T), VEC, grid_out);
    if (G == 2) return launch_cfg(ctx, tile_kernel<T, OP, 2, 1, SHADOW, 512, MULTI>, tile_kernel<T, OP, 2, 1, SHADOW, 384, MULTI>, a, sizeof(T), VEC, grid_out);
    if (!want_ch || nch <= 32)
        return launch_cfg(ctx, tile_kernel<T, OP, 4, 1, SHADOW, 512, MULTI>, tile_kernel<T, OP, 4, 1, SHADOW, 384, MULTI>, a, sizeof(T), VEC, grid_out);
    return launch_cfg(ctx, tile_kernel<T, OP, 4, 2, SHADOW, 512, MULTI>, tile_kernel<T, OP, 4, 2, SHADOW, 384, MULTI>, a, sizeof(T), 2 * VEC, grid_out);
}

}  // namespace

bool meb_tile_applicable(int op, int prec, const StreamArgs& a) {
    const size_t esize = prec == MEB_FP64 ? 8 : 4;
    const size_t row_bytes = (size_t)a.ld * esize;
    if (row_bytes > 1024 || row_bytes % 16 != 0 || ((uintptr_t)a.C % 16) != 0) return false;
    if (a.d > 256) return false;
    if (op == OP_EVAL && a.part_vec == nullptr) return false;
    return true;
}

int meb_launch_tile(meb_ctx* ctx, int op, int prec, const StreamArgs& a, int* grid_out) {
    if (prec == MEB_FP64) {
        switch (op) {
            case OP_EVAL:
                if (a.multi > 0) return launch_g<double, OP_EVAL, false, true>(ctx, a, true, grid_out);
                return launch_g<double, OP_EVAL, false, false>(ctx, a, true, grid_out);
            case OP_FEAS: return launch_g<double, OP_FEAS, false, false>(ctx, a, false, grid_out);
            case OP_INGEST:
                if (a.C32) return launch_g<double, OP_INGEST, true, false>(ctx, a, true, grid_out);
                return launch_g<double, OP_INGEST, false, false>(ctx, a, false, grid_out);
            default: return MEB_E_ARG;
        }
    }
    switch (op) {
        case OP_EVAL:
            if (a.multi > 0) return launch_g<float, OP_EVAL, false, true>(ctx, a, true, grid_out);
            return launch_g<float, OP_EVAL, false, false>(ctx, a, true, grid_out);
        case OP_SCREEN: return launch_g<float, OP_SCREEN, false, false>(ctx, a, false, grid_out);
        default: return MEB_E_ARG;
    }
}
