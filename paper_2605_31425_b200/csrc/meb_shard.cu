// Sharded solves: the balls of ONE instance partitioned over several GPUs (P:L351 names
// multi-GPU as future work, P:L179 / L218 give the separable structure that makes it natural).
//
// Every rank streams its own rows with the unchanged kernels.  What crosses the GPUs is the FIRST level of each
// reduction tree: the rank adds its per-CTA partials in index order into one record (d + O(10) doubles; (d+1)^2 for
// the dense Hessian), the records of all ranks are all-gathered in rank order (the caller's collective: NCCL over
// NVLink / NVSwitch, 80 KB at d = 1e4: latency-bound), and the unchanged second-level kernels add the nranks
// records in rank order.  Sums are therefore bit-identical on every rank, the replicated controllers take identical
// decisions, and no floating-point atomics or order-dependent collectives (all-reduce) are involved.
#include <string.h>

#include "meb_internal.cuh"
#include "meb_ctrl.cuh"

namespace {

constexpr int PK = 256;

// column j of the record's vector part: partials b < used added in index order (coalesced across the threads)
__global__ void __launch_bounds__(PK) pack_eval_kernel(const double* __restrict__ part, int grid,
                                                       const double* __restrict__ part_vec, int nvec, int tpb,
                                                       const int32_t* __restrict__ count, int dpad, int d,
                                                       const double* __restrict__ multi_part, double* __restrict__ rec) {
    if (nvec > 0 && tpb > 0) { const int used = (*count + tpb - 1) / tpb; if (nvec > used) nvec = used; }
    const int j = (blockIdx.x - 1) * PK + threadIdx.x;
    if (blockIdx.x == 0) {
        const int k = threadIdx.x;
        if (k < MEB_NPART) {
            double v = 0.0;
            if (k < 10) {
                const bool is_max = (k >= 5 && k <= 7) || k == MEB_PART_CUT;
                for (int b = 0; b < grid; ++b) {
                    const double p = part[(size_t)b * MEB_NPART + k];
                    v = is_max ? fmax(v, p) : v + p;
                }
            }
            rec[k] = v;                                  // slots 10, 11 (time stamps): 0 = none
        } else if (k < MEB_NPART + MEB_MULTI_MAX) {
            double v = 0.0;
            if (multi_part)
                for (int b = 0; b < grid; ++b) v += multi_part[(size_t)b * MEB_MULTI_MAX + (k - MEB_NPART)];
            rec[k] = v;
        }
        return;
    }
    if (j < d) {
        double s = 0.0;
        for (int b = 0; b < nvec; ++b) s += part_vec[(size_t)b * dpad + j];
        rec[16 + j] = s;
    }
}

__global__ void __launch_bounds__(PK) pack_hvp_kernel(const double* __restrict__ part_sc, int nsc,
                                                      const double* __restrict__ part_vec, int nvec, int tpb,
                                                      const int32_t* __restrict__ count, int dpad, int d,
                                                      double* __restrict__ rec) {
    if (tpb > 0) { const int used = (*count + tpb - 1) / tpb; if (nvec > used) nvec = used; }
    if (blockIdx.x == 0) {
        if (threadIdx.x == 0) {
            double s = 0.0;
            for (int b = 0; b < nsc; ++b) s += part_sc[b];       // CTAs without list entries wrote 0
            rec[0] = s;
        }
        return;
    }
    const int j = (blockIdx.x - 1) * PK + threadIdx.x;
    if (j < d) {
        double s = 0.0;
        for (int b = 0; b < nvec; ++b) s += part_vec[(size_t)b * dpad + j];
        rec[8 + j] = s;
    }
}

__global__ void __launch_bounds__(PK) pack_mat_kernel(const double* __restrict__ part_mat, int nparts,
                                                      const int32_t* __restrict__ count, int rb, long long per,
                                                      double* __restrict__ rec) {
    const int ntiles = (*count + rb - 1) / rb;
    if (nparts > ntiles) nparts = ntiles;
    const long long e = (long long)blockIdx.x * PK + threadIdx.x;
    if (e >= per) return;
    double s = 0.0;
    for (int b = 0; b < nparts; ++b) s += part_mat[(size_t)b * per + e];
    rec[e] = s;
}

__global__ void pack_small_kernel(const double* __restrict__ src, int n, double* __restrict__ rec, double tail, int has_tail) {
    for (int k = threadIdx.x; k < n; k += blockDim.x) rec[k] = src[k];
    if (has_tail && threadIdx.x == 0) rec[n] = tail;
}
// (value, local index, count) -> (value, global index, count)
__global__ void pack_argmax_kernel(const double* __restrict__ src, double row_offset, double* __restrict__ rec) {
    rec[0] = src[0]; rec[1] = src[1] >= 0.0 ? src[1] + row_offset : -1.0; rec[2] = src[2]; rec[3] = 0.0;
}

__global__ void __launch_bounds__(PK) combine_kernel(const double* __restrict__ recv, int nranks, long long stride,
                                                     int mode, int d, double* __restrict__ out) {
    if (mode == 0) {                                     // (value, index, count): arg-max, smallest index on ties
        if (threadIdx.x == 0 && blockIdx.x == 0) {
            double bv = 0.0, bi = -1.0, cnt = 0.0;
            for (int r = 0; r < nranks; ++r) {
                const double v = recv[(size_t)r * stride], i = recv[(size_t)r * stride + 1];
                cnt += recv[(size_t)r * stride + 2];
                if (i >= 0.0 && (bi < 0.0 || v > bv || (v == bv && i < bi))) { bv = v; bi = i; }
            }
            out[0] = bv; out[1] = bi; out[2] = cnt;
        }
        return;
    }
    double wsum = 0.0;                                   // weighted mean of the ranks' vectors, rank order
    for (int r = 0; r < nranks; ++r) wsum += recv[(size_t)r * stride + d];
    for (int j = blockIdx.x * PK + threadIdx.x; j < d; j += gridDim.x * PK) {
        double s = 0.0;
        for (int r = 0; r < nranks; ++r) s += (recv[(size_t)r * stride + d] / wsum) * recv[(size_t)r * stride + j];
        out[j] = s;
    }
}

}  // namespace

extern "C" int64_t meb_shard_record_doubles(int32_t d) {
    const int64_t dpad = ((int64_t)d + 7) / 8 * 8;
    int64_t n = 16 + dpad + 8;
    if (d <= 128) {
        const int64_t dp = ((int64_t)d + 15) / 16 * 16;
        if (dp * dp + dp + 8 > n) n = dp * dp + dp + 8;
    }
    return n;
}

// all-gather of the first n doubles of every rank's send record; afterwards record r starts at recv + r * n
int meb_shard_exchange(meb_ctx* ctx, int64_t n) {
    MebShard* sh = ctx->shard;
    if (!sh || n > sh->rec_doubles) return MEB_E_CAPACITY;
    if (sh->nranks == 1) {                               // degenerate: a device copy stands in for the collective
        MEB_CUDA_OK(ctx, cudaMemcpyAsync(sh->recv, sh->send, (size_t)n * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));
        return MEB_OK;
    }
    return sh->allgather(sh->user, n) == 0 ? MEB_OK : MEB_E_CUDA;
}

int meb_shard_pack_eval(meb_ctx* ctx, const double* part, int grid, const double* part_vec, int nvec, int tpb,
                        const int32_t* count, int dpad, int d, const double* multi_part) {
    ctx->launches++;
    pack_eval_kernel<<<1 + (d + PK - 1) / PK, PK, 0, ctx->stream>>>(part, grid, part_vec, nvec, tpb, count, dpad, d, multi_part,
                                                                   ctx->shard->send);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}
int meb_shard_pack_hvp(meb_ctx* ctx, const double* part_sc, int nsc, const double* part_vec, int nvec, int tpb,
                       const int32_t* count, int dpad, int d) {
    ctx->launches++;
    pack_hvp_kernel<<<1 + (d + PK - 1) / PK, PK, 0, ctx->stream>>>(part_sc, nsc, part_vec, nvec, tpb, count, dpad, d, ctx->shard->send);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}
int meb_shard_pack_mat(meb_ctx* ctx, const double* part_mat, int nparts, const int32_t* count, int rb, int64_t per) {
    ctx->launches++;
    pack_mat_kernel<<<(unsigned)((per + PK - 1) / PK), PK, 0, ctx->stream>>>(part_mat, nparts, count, rb, (long long)per, ctx->shard->send);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}
int meb_shard_pack_small(meb_ctx* ctx, const double* src, int n) {
    ctx->launches++;
    pack_small_kernel<<<1, 128, 0, ctx->stream>>>(src, n, ctx->shard->send, 0.0, 0);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}
// c0 of this rank's rows and its weight (the number of rows) -> the weighted mean over the ranks, in c0
int meb_shard_mean(meb_ctx* ctx, double* c0, int d, int64_t m_local) {
    ctx->launches++;
    pack_small_kernel<<<1, 256, 0, ctx->stream>>>(c0, d, ctx->shard->send, (double)m_local, 1);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    int rc = meb_shard_exchange(ctx, (int64_t)d + 8);
    if (rc != MEB_OK) return rc;
    return meb_shard_combine(ctx, 1, d, c0);
}
// (value, index, count) arg-max of this rank (device, 3 doubles, local index) -> the global one, in place
int meb_shard_argmax(meb_ctx* ctx, double* scal3) {
    ctx->launches++;
    pack_argmax_kernel<<<1, 1, 0, ctx->stream>>>(scal3, (double)ctx->shard->row_offset, ctx->shard->send);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    int rc = meb_shard_exchange(ctx, 4);
    if (rc != MEB_OK) return rc;
    return meb_shard_combine(ctx, 0, 0, scal3);
}
int meb_shard_combine(meb_ctx* ctx, int mode, int d, double* out) {
    // stride = the n of the exchange that preceded: 4 for the arg-max records, d + 8 for the weighted vectors
    const long long stride = mode == 0 ? 4 : (long long)d + 8;
    ctx->launches++;
    combine_kernel<<<mode == 0 ? 1 : (d + PK - 1) / PK, PK, 0, ctx->stream>>>(ctx->shard->recv, ctx->shard->nranks, stride, mode, d, out);
    MEB_CUDA_OK(ctx, cudaGetLastError());
    return MEB_OK;
}
