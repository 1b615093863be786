// Stable stream compaction of a bit mask into an ascending int32 index list
// (screening set I_red; violated set V; active set of an evaluation).
//
// Bit b of mask[w] is ball 32*w + b (written by the streaming kernels with __ballot_sync).
// Two launches, integer work only, so the result is bit-exact and order-stable by construction:
//   1. each CTA counts the bits of its segment of SEG_WORDS words            -> segsum[s]
//   2. each CTA adds segsum[0..s) (parallel reduce), rescans its own segment with warp ballots /
//      shuffles and writes the indices at their final position; CTA 0 also writes the total.
#include "meb_internal.cuh"

namespace {

constexpr int SEG_WORDS = 2048;          // 65536 balls per segment
constexpr int CBLOCK = 256;

__global__ void __launch_bounds__(CBLOCK) compact_count_kernel(const uint32_t* __restrict__ mask,
                                                               int64_t nwords, int64_t m,
                                                               int32_t* __restrict__ segsum) {
    __shared__ int wsum[CBLOCK / 32];
    const int64_t w0 = (int64_t)blockIdx.x * SEG_WORDS;
    int cnt = 0;
    for (int k = threadIdx.x; k < SEG_WORDS; k += CBLOCK) {
        const int64_t w = w0 + k;
        if (w < nwords) {
            uint32_t bits = mask[w];
            if ((w + 1) * 32 > m) bits &= (m - w * 32 >= 32) ? 0xffffffffu : ((1u << (m - w * 32)) - 1u);
            cnt += __popc(bits);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(MEB_FULL_MASK, cnt, o);
    if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = cnt;
    __syncthreads();
    if (threadIdx.x == 0) {
        int t = 0;
        for (int w = 0; w < CBLOCK / 32; ++w) t += wsum[w];
        segsum[blockIdx.x] = t;
    }
}

__global__ void __launch_bounds__(CBLOCK) compact_write_kernel(const uint32_t* __restrict__ mask,
                                                               int64_t nwords, int64_t m,
                                                               const int32_t* __restrict__ segsum,
                                                               int nseg, int32_t* __restrict__ list,
                                                               int64_t cap, int32_t* __restrict__ count) {
    __shared__ long long sred[CBLOCK / 32];
    __shared__ int wtot[CBLOCK / 32];
    __shared__ long long base_s;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // exclusive prefix of the segment sums up to this CTA (and the grand total in CTA 0)
    long long pre = 0, tot = 0;
    for (int s = threadIdx.x; s < nseg; s += CBLOCK) {
        const int v = segsum[s];
        if (s < (int)blockIdx.x) pre += v;
        tot += v;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        pre += __shfl_xor_sync(MEB_FULL_MASK, pre, o);
        tot += __shfl_xor_sync(MEB_FULL_MASK, tot, o);
    }
    if (lane == 0) sred[warp] = pre;
    __syncthreads();
    if (threadIdx.x == 0) {
        long long p = 0;
        for (int w = 0; w < CBLOCK / 32; ++w) p += sred[w];
        base_s = p;
    }
    __syncthreads();
    if (blockIdx.x == 0) {
        if (lane == 0) sred[warp] = tot;
        __syncthreads();
        if (threadIdx.x == 0) {
            long long p = 0;
            for (int w = 0; w < CBLOCK / 32; ++w) p += sred[w];
            *count = (int32_t)p;
        }
    }
    long long base = base_s;
    const int64_t w0 = (int64_t)blockIdx.x * SEG_WORDS;
    // the segment is scanned in rounds of CBLOCK words: thread k handles word w0 + round*CBLOCK + k
    for (int round = 0; round < SEG_WORDS / CBLOCK; ++round) {
        const int64_t w = w0 + (int64_t)round * CBLOCK + threadIdx.x;
        uint32_t bits = 0;
        if (w < nwords) {
            bits = mask[w];
            if ((w + 1) * 32 > m) bits &= (m - w * 32 >= 32) ? 0xffffffffu : ((1u << (m - w * 32)) - 1u);
        }
        const int c = __popc(bits);
        int incl = c;                                   // inclusive scan inside the warp
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(MEB_FULL_MASK, incl, o);
            if (lane >= o) incl += v;
        }
        if (lane == 31) wtot[warp] = incl;
        __syncthreads();
        int wpre = 0, rtot = 0;
        for (int k = 0; k < CBLOCK / 32; ++k) {
            const int v = wtot[k];
            if (k < warp) wpre += v;
            rtot += v;
        }
        long long pos = base + wpre + (incl - c);
        while (bits) {
            const int b = __ffs(bits) - 1;
            bits &= bits - 1;
            if (pos < cap) list[pos] = (int32_t)(w * 32 + b);
            ++pos;
        }
        base += rtot;
        __syncthreads();
    }
}

// Small problems (up to 2M balls): ONE CTA of 1024 threads.  Thread t owns the contiguous run of W words
// [t W, (t+1) W): it counts its bits, one block-wide exclusive scan (warp shuffles + warp totals in
// shared memory, two barriers in all) gives its output offset, and it writes its indices in order.
__global__ void __launch_bounds__(1024) compact_single_kernel(const uint32_t* __restrict__ mask, int64_t nwords,
                                                              int64_t m, int32_t* __restrict__ list, int64_t cap,
                                                              int32_t* __restrict__ count) {
    __shared__ int wtot[32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int W = (int)((nwords + 1023) / 1024);
    const int64_t w0 = (int64_t)threadIdx.x * W;
    auto word = [&](int64_t w) -> uint32_t {
        if (w >= nwords) return 0u;
        uint32_t bits = mask[w];
        if ((w + 1) * 32 > m) bits &= (m - w * 32 >= 32) ? 0xffffffffu : ((1u << (m - w * 32)) - 1u);
        return bits;
    };
    int c = 0;
#pragma unroll 4
    for (int k = 0; k < W; ++k) c += __popc(word(w0 + k));
    int incl = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(MEB_FULL_MASK, incl, o);
        if (lane >= o) incl += v;
    }
    if (lane == 31) wtot[warp] = incl;
    __syncthreads();
    int wpre = 0, tot = 0;
#pragma unroll
    for (int k = 0; k < 32; ++k) {
        const int v = wtot[k];
        if (k < warp) wpre += v;
        tot += v;
    }
    if (threadIdx.x == 0) *count = tot;
    if (c == 0) return;
    long long pos = (long long)wpre + (incl - c);
    for (int k = 0; k < W; ++k) {
        uint32_t bits = word(w0 + k);
        while (bits) {
            const int b = __ffs(bits) - 1;
            bits &= bits - 1;
            if (pos < cap) list[pos] = (int32_t)((w0 + k) * 32 + b);
            ++pos;
        }
    }
}

// uint8 flags -> bit mask (the "flags given" input mode of meb_screen_compact)
__global__ void __launch_bounds__(256) flags_to_mask_kernel(const uint8_t* __restrict__ flags, int64_t m,
                                                           uint32_t* __restrict__ mask) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t n32 = (m + 31) / 32 * 32;
    if (i >= n32) return;
    const bool f = i < m && flags[i] != 0;
    const uint32_t bits = __ballot_sync(MEB_FULL_MASK, f);
    if ((threadIdx.x & 31) == 0) mask[i >> 5] = bits;
}

}  // namespace

// list[cap] <- ascending indices of the set bits of mask (first m bits); *count_dev <- how many.
int meb_launch_compact_cap(meb_ctx* ctx, const uint32_t* mask, int64_t m, int32_t* list, int64_t cap,
                           int32_t* count_dev) {
    const int64_t nwords = (m + 31) / 32;
    if (nwords <= 64 * 1024) {                     // up to 2M balls: one CTA, one launch
        ctx->launches++; compact_single_kernel<<<1, 1024, 0, ctx->stream>>>(mask, nwords, m, list, cap, count_dev);
        MEB_CUDA_OK(ctx, cudaGetLastError());
        return MEB_OK;
    }
    const int nseg = (int)((nwords + SEG_WORDS - 1) / SEG_WORDS);
    ctx->launches++; compact_count_kernel<<<nseg, CBLOCK, 0, ctx->stream>>>(mask, nwords, m, ctx->blocksum);
    ctx->launches++; compact_write_kernel<<<nseg, CBLOCK, 0, ctx->stream>>>(mask, nwords, m, ctx->blocksum, nseg, list, cap,
                                                           count_dev);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}

int meb_launch_compact(meb_ctx* ctx, const uint32_t* mask, int64_t m, int32_t* list, int32_t* count_dev) {
    return meb_launch_compact_cap(ctx, mask, m, list, m, count_dev);
}

int meb_launch_flags_to_mask(meb_ctx* ctx, const uint8_t* flags, int64_t m, uint32_t* mask) {
    const int64_t n32 = (m + 31) / 32 * 32;
    const int64_t grid = (n32 + 255) / 256;
    ctx->launches++; flags_to_mask_kernel<<<(unsigned)grid, 256, 0, ctx->stream>>>(flags, m, mask);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}
