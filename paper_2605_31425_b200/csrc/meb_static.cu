// Allocation-free feasibility maximum (the a-posteriori check of the mixed-precision method):
//
//     viol_i = r_i + ||c - c_i|| - r,      Delta_max = max_i viol_i,      argmax = its smallest index.
//
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
// it): no context, no workspace argument.  The scratch of the two-level reduction -- one (value, index) pair per tile
// of 256 rows -- lives in a file-scope __device__ array of MEB_STATIC_MAX_TILES pairs (1 MiB; every GPU that loads the
// library holds it until the process exits).  Nothing here calls cudaMalloc, cudaFree or an allocating library routine.
//
// The array is SHARED by all calls and keeps the last call's contents.  Nothing in it has to start at zero: the first
// kernel overwrites every pair the second kernel reads (tiles 0 .. ntiles-1) on every call.  Two calls that overlap
// on the GPU (different streams, or concurrent host threads) RACE on it; calls on one stream are ordered and safe.
//
// Deterministic: static row -> warp -> tile mapping, lanes combined by an xor tree, tiles by index.
#include <stdint.h>

#include <cuda_runtime.h>

#include "../../include/meb.h"

namespace {

constexpr int ST_THREADS = 256;
constexpr int ST_WARPS = ST_THREADS / 32;
constexpr int ST_TILE_ROWS = 256;                           // rows of one tile = one pair of the scratch
constexpr int ST_ROWS_PER_WARP = ST_TILE_ROWS / ST_WARPS;   // 32
constexpr int ST_MAX_TILES = MEB_STATIC_MAX_TILES;
constexpr int ST_MAX_DEVICES = 64;

struct __align__(16) StPair { double value; long long index; };

// Host code must never hand `st_scratch` to a kernel: on the host this name is a stand-in, not a device address.
// The launcher below resolves it with cudaGetSymbolAddress once per device; device code may name it directly.
static __device__ __align__(256) StPair st_scratch[ST_MAX_TILES];

StPair* st_scratch_addr[ST_MAX_DEVICES];                    // per device, resolved at the first call on it
bool st_scratch_known[ST_MAX_DEVICES];

__device__ __forceinline__ double st_warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// larger value wins; equal values: the smaller index (a tile without rows carries index -1 and never wins)
__device__ __forceinline__ void st_take(double& bv, long long& bi, double v, long long i) {
    if (i >= 0 && (bi < 0 || v > bv || (v == bv && i < bi))) { bv = v; bi = i; }
}

// Tile t = rows 256 t .. 256 t + 255; warp w of the CTA walks rows 32 w .. 32 w + 31 of the tile, lanes over the
// columns.  A CTA handles tiles blockIdx.x, blockIdx.x + gridDim.x, ...
__global__ void __launch_bounds__(ST_THREADS) st_tile_kernel(const double* __restrict__ C, long long ld,
                                                             const double* __restrict__ R, long long m, int d, double r,
                                                             const double* __restrict__ c, long long ntiles,
                                                             StPair* __restrict__ scratch) {
    __shared__ double wv[ST_WARPS];
    __shared__ long long wi[ST_WARPS];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (long long t = blockIdx.x; t < ntiles; t += gridDim.x) {
        double bv = 0.0;
        long long bi = -1;
        const long long row0 = t * ST_TILE_ROWS + (long long)warp * ST_ROWS_PER_WARP;
        for (int q = 0; q < ST_ROWS_PER_WARP; ++q) {
            const long long i = row0 + q;
            if (i >= m) break;
            const double* __restrict__ rowp = C + i * ld;
            double s0 = 0.0, s1 = 0.0;
            int j = lane;
            for (; j + 32 < d; j += 64) {
                const double e0 = c[j] - rowp[j], e1 = c[j + 32] - rowp[j + 32];
                s0 = fma(e0, e0, s0);
                s1 = fma(e1, e1, s1);
            }
            if (j < d) { const double e = c[j] - rowp[j]; s0 = fma(e, e, s0); }
            const double n2 = st_warp_sum(s0 + s1);
            const double viol = (R ? R[i] : 0.0) + sqrt(n2) - r;
            st_take(bv, bi, viol, i);
        }
        if (lane == 0) { wv[warp] = bv; wi[warp] = bi; }
        __syncthreads();
        if (threadIdx.x == 0) {
            double tv = 0.0;
            long long ti = -1;
            for (int w = 0; w < ST_WARPS; ++w) st_take(tv, ti, wv[w], wi[w]);
            scratch[t].value = tv;
            scratch[t].index = ti;
        }
        __syncthreads();
    }
}

// one CTA: thread k takes tiles k, k + 256, ...; threads are then combined in index order
__global__ void __launch_bounds__(ST_THREADS) st_final_kernel(const StPair* __restrict__ scratch, long long ntiles,
                                                              double* __restrict__ out) {
    __shared__ double tv[ST_THREADS];
    __shared__ long long ti[ST_THREADS];
    double bv = 0.0;
    long long bi = -1;
    for (long long t = threadIdx.x; t < ntiles; t += ST_THREADS) st_take(bv, bi, scratch[t].value, scratch[t].index);
    tv[threadIdx.x] = bv;
    ti[threadIdx.x] = bi;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 1; k < ST_THREADS; ++k) st_take(bv, bi, tv[k], ti[k]);
        out[0] = bv;
        out[1] = (double)bi;
    }
}

}  // namespace

extern "C" MEB_API int meb_feasibility_max_static(void* cuda_stream, int64_t m, int32_t d, const double* C, int64_t ld,
                                                  const double* R, double r, const double* c, double* out2) {
    if (!C || !c || !out2 || m < 1 || d < 1 || ld < d) return MEB_E_ARG;
    const int64_t ntiles = (m + ST_TILE_ROWS - 1) / ST_TILE_ROWS;
    if (ntiles > ST_MAX_TILES) return MEB_E_CAPACITY;       // m > MEB_STATIC_MAX_ROWS: the static scratch is too small
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= ST_MAX_DEVICES) return MEB_E_CUDA;
    if (!st_scratch_known[dev]) {                           // set-up, once per device, with that device current
        StPair* p = nullptr;
        if (cudaGetSymbolAddress((void**)&p, st_scratch) != cudaSuccess || !p) return MEB_E_CUDA;
        st_scratch_addr[dev] = p;
        st_scratch_known[dev] = true;
    }
    StPair* scratch = st_scratch_addr[dev];
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    const int64_t cap = 148 * 8;                            // one wave of 256-thread CTAs on a B200
    const int grid = (int)(ntiles < cap ? ntiles : cap);
    st_tile_kernel<<<grid, ST_THREADS, 0, stream>>>(C, (long long)ld, R, (long long)m, (int)d, r, c, (long long)ntiles, scratch);
    if (cudaGetLastError() != cudaSuccess) return MEB_E_CUDA;
    st_final_kernel<<<1, ST_THREADS, 0, stream>>>(scratch, (long long)ntiles, out2);
    if (cudaGetLastError() != cudaSuccess) return MEB_E_CUDA;
    return MEB_OK;
}
