// Register-tiled LDL^T solve of one SPD system of order n <= 16*BS - 1 by one group of 16 x 16 threads
// (threads 0..255 of the CTA), shared by the stand-alone Newton-solve kernel (meb_dense.cu) and the
// single-CTA solver of small problems (meb_smallsolve.cu).
//
// Square-root-free Cholesky (H = L D L^T, no pivoting: H is SPD) on the AUGMENTED matrix
// M = [H; -g^T]: eliminating column k also updates the right-hand-side row n, so after the n column
// steps row n holds D L^{-1}(-g) and only the backward substitution with L^T is left.
// The matrix lives in REGISTERS: thread (ty, tx) owns M[ty + 16 ii][tx + 16 jj], jj <= ii < BS.
// Column steps are grouped in phases of 16 (KB = k / 16) that are unrolled at compile time, so inside
// a phase the code is straight-line: every thread updates its (BS-KB)(BS-KB+1)/2 live entries with
// multipliers that are masked to zero only in the pivot block, the owners of column k+1 publish it to
// shared memory (where it stays as row k+1 of L D for the backward substitution), and every thread
// forms 1/d_k itself with a fast reciprocal.  One __syncthreads per column.
#pragma once
#include "meb_internal.cuh"

// 1/d for d > 0 in full precision: hardware seed (about 20 bits) + two Newton steps, 4 dependent FMAs
// (the IEEE division subroutine is several times longer and sits on the critical path of every column)
__device__ __forceinline__ double meb_fast_rcp(double d) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d));
    double e = fma(-d, r, 1.0);
    r = fma(r, e, r);
    e = fma(-d, r, 1.0);
    return fma(r, e, r);
}

template <int BS> struct LdltShape {
    static constexpr int NP = 16 * BS;
    static constexpr int LDL = NP | 1;
    // doubles of shared memory: n rows of L D, 1/d, the solution
    __host__ __device__ static size_t smem_doubles(int n) { return (size_t)n * LDL + 2 * (size_t)NP; }
};

// a: augmented lower triangle in registers (entries outside it are ignored).  Lm: shared memory of
// LdltShape<BS>::smem_doubles(n) doubles.  All 256 threads of the group call it (tid = 0..255; the CTA may
// hold more threads only if they do not touch Lm meanwhile and all of them reach the __syncthreads inside:
// callers use CTAs of exactly 256 threads).  On return z = Lm + n*LDL + NP holds the solution (n doubles)
// and *bad (shared) is 0 or the index + 1 of the first non-positive pivot.
template <int BS>
__device__ __forceinline__ double* meb_ldlt_solve_regs(double (&a)[BS][BS], int n, double* Lm, int* bad) {
    constexpr int NP = LdltShape<BS>::NP;
    constexpr int ldl = LdltShape<BS>::LDL;
    double* invd = Lm + (size_t)n * ldl;
    double* z = invd + NP;
    const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
    if (tid == 0) *bad = 0;
    if (tx == 0) {                                        // publish column 0
#pragma unroll
        for (int ii = 0; ii < BS; ++ii) Lm[ty + 16 * ii] = a[ii][0];
    }
    __syncthreads();
#pragma unroll
    for (int KB = 0; KB < BS; ++KB) {
        if (16 * KB < n) {
#pragma unroll 1
            for (int kk = 0; kk < 16; ++kk) {
                const int k = 16 * KB + kk;
                if (k >= n) break;                        // uniform
                const double* col = Lm + (size_t)k * ldl;
                double dk = col[k];
                if (!(dk > 0.0)) { if (tid == 0) *bad = k + 1; dk = 1.0; }
                const double ninv = -meb_fast_rcp(dk);    // every thread forms 1/d_k itself (no serial owner)
                if (tid == 0) invd[k] = -ninv;
                // multipliers; only block KB holds rows / columns <= k, which are masked to zero
                double lik[BS], cj[BS];
#pragma unroll
                for (int q = KB; q < BS; ++q) {
                    double c1 = col[ty + 16 * q], c2 = col[tx + 16 * q];
                    if (q == KB) {
                        c1 = (ty + 16 * KB > k) ? c1 : 0.0;
                        c2 = (tx + 16 * KB > k) ? c2 : 0.0;
                    }
                    lik[q] = c1 * ninv;
                    cj[q] = c2;
                }
#pragma unroll
                for (int ii = KB; ii < BS; ++ii)
#pragma unroll
                    for (int jj = KB; jj <= ii; ++jj) a[ii][jj] = fma(lik[ii], cj[jj], a[ii][jj]);
                const int k1 = k + 1;
                if (k1 < n && tx == (k1 & 15)) {          // owners of column k+1 publish it
                    double* cn = Lm + (size_t)k1 * ldl;
                    if (kk < 15) {
#pragma unroll
                        for (int ii = KB; ii < BS; ++ii) cn[ty + 16 * ii] = a[ii][KB];
                    } else if (KB + 1 < BS) {
#pragma unroll
                        for (int ii = KB + 1; ii < BS; ++ii) cn[ty + 16 * ii] = a[ii][KB + 1 < BS ? KB + 1 : KB];
                    }
                }
                __syncthreads();
            }
        }
    }
    // row n of L D is spread over the columns' shared rows: z_k = Lm[k][n] / d_k; then L^T x = z,
    // column-oriented by one warp with z in REGISTERS (lane L holds z[L + 32 q]): per step one shuffle
    // broadcasts x_k and every lane updates its entries j < k with L_kj = Lm[j][k] * invd[j].
    if (tid < 32) {
        constexpr int ZQ = (NP + 31) / 32;
        double zr[ZQ], dj[ZQ];
#pragma unroll
        for (int q = 0; q < ZQ; ++q) {
            const int j = tid + 32 * q;
            dj[q] = j < n ? invd[j] : 0.0;
            zr[q] = j < n ? Lm[(size_t)j * ldl + n] * dj[q] : 0.0;
        }
        for (int k = n - 1; k > 0; --k) {
            double lv[ZQ];
#pragma unroll
            for (int q = 0; q < ZQ; ++q) {
                const int j = tid + 32 * q;
                lv[q] = j < k ? Lm[(size_t)j * ldl + k] * dj[q] : 0.0;     // independent of the x chain
            }
            double xk = 0.0;
#pragma unroll
            for (int q = 0; q < ZQ; ++q) {
                const double t = __shfl_sync(MEB_FULL_MASK, zr[q], k & 31);
                if (q == (k >> 5)) xk = t;
            }
#pragma unroll
            for (int q = 0; q < ZQ; ++q) zr[q] = fma(-lv[q], xk, zr[q]);
        }
#pragma unroll
        for (int q = 0; q < ZQ; ++q) {
            const int j = tid + 32 * q;
            if (j < n) z[j] = zr[q];
        }
    }
    __syncthreads();
    return z;
}
