/*
 * meb.h  --  C-ABI of the B200-native minimum-enclosing-ball library (libmeb_b200.so).
 *
 * Method: mixed-precision relative-type inexact proximal augmented Lagrangian method (ripALM)
 * for the minimum enclosing ball of m balls in R^d, "Mixed-Precision GPU Acceleration for
 * Large-Scale Minimum Enclosing Ball Problems" (Liang & Yang).  Citations P:L<n> are line
 * numbers of the paper text; "reading n" refers to DESIGN.md, "Readings of the paper".
 *
 * Problem:   min r   s.t.  ||c - c_i|| + r_i <= r,  i = 1..m,
 * as a second-order cone program (r - r_i, c - c_i) in Q_{d+1}  (eq. (1)).
 *
 * CONVENTIONS (all entry points)
 *  - Every function returns an int status: MEB_OK (0), a negative MEB_E_* error, or the positive
 *    warning MEB_W_NOT_CONVERGED (outputs then hold the best iterate).  No exceptions, no exit(),
 *    no global state.  Nothing is written to outputs on MEB_E_ARG.
 *  - Pointers are DEVICE pointers owned by the caller unless the argument name starts with h_
 *    (HOST pointer owned by the caller).  The library never frees or keeps a caller pointer
 *    beyond the call.  The context owns all workspace and the stream handle it was given.
 *  - Layout ("structure of arrays"): centres C row-major, row i at C + i*ld, ld >= d
 *    elements (all m*ld elements must be readable: rows are fetched in whole 16-byte units, the padding
 *    values are ignored); radii R[m] (NULL = points, all r_i = 0); multipliers U[m] and sparse V:
 *    v_slot[i] >= 0 is the row of ball i in Vrows (row stride ldv), v_slot[i] < 0 means v_i = 0;
 *    v_slot == NULL means all v_i = 0.  A dense V (the paper's layout) is v_slot[i] = i.
 *    (u_i = 0 implies v_i = 0 because multipliers are projections onto Q.)
 *  - prec: MEB_FP64 -> C, R, U, Vrows are double arrays; MEB_FP32 -> float arrays (the
 *    low-precision copy of P:L250; per-ball arithmetic in float, all sums over balls and the
 *    (d+1)-sized state in double, reading 8).  x, xbar, q, outputs are always double.
 *  - x = (r, c) is a (d+1)-vector, x[0] = r.  Notation for ball i:
 *        a_i = r_i - r + u_i/sigma,  b_i = c_i - c + v_i/sigma,  nb_i = ||b_i||,
 *        B1: nb <= a  -> Pi(z) = z      (t = a,        lam = 1)
 *        B2: nb <= -a -> Pi(z) = 0      (t = 0,        lam = 0)      [tested after B1]
 *        B3: else     -> t = (a+nb)/2,  lam = t/nb,   Pi(z_i) = (t_i, lam_i b_i).
 *    A ball is ACTIVE iff lam_i != 0.
 *  - Sizes: 1 <= m < 2^31 - 64, 1 <= d, ld >= d.  Indices are int32.
 *  - Determinism: every reduction uses a static row->thread assignment, warp shuffles and a
 *    fixed-order two-level tree; no floating-point atomics.  Same inputs, same bits.
 *  - Thread safety: one context per host thread.
 */
#ifndef MEB_H_
#define MEB_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define MEB_API __attribute__((visibility("default")))
#else
#define MEB_API
#endif

#define MEB_OK 0
#define MEB_W_NOT_CONVERGED 1   /* iteration cap hit; outputs hold the best iterate */
#define MEB_E_ARG (-1)          /* null pointer, bad size, bad tolerance or mode */
#define MEB_E_INPUT (-2)        /* NaN/Inf in the data or a negative radius */
#define MEB_E_ALLOC (-3)        /* device or host allocation failed */
#define MEB_E_CUDA (-4)         /* CUDA error; see meb_last_cuda_error */
#define MEB_E_CAPACITY (-5)     /* problem larger than the context (m_max, d_max) or an output list too small */

#define MEB_FP64 0
#define MEB_FP32 1

#define MEB_MODE_FP64 0         /* ripALM in FP64 on all m balls ("ripALM") */
#define MEB_MODE_MIXED 1        /* mp-ripALM of Section 4.2 */

typedef struct meb_ctx meb_ctx;

/* Free constants of Algorithms 1-2 and Section 4.2;
 * the paper names them without values: readings 3, 4, 5, 9, 10, 12. */
typedef struct meb_params {
    double rho;                 /* rho in [0,1) of the relative stopping condition (5)     0.5  */
    double sigma0;              /* sigma_0, normalised units                               1    */
    double kappa;               /* sigma_{k+1} = min(sigma_max, kappa sigma_k)             3    */
    double sigma_max;           /*                                                         1e8  */
    double tau;                 /* tau_k (constant)                                        1    */
    double armijo_mu;           /* sufficient-decrease constant                            1e-4 */
    double tol_lo;              /* stopping tolerance of the low-precision run    1e-2 */
    double tol_red_factor;      /* tol_red = factor * r_hat (reading 9, pinned by Table 1) 0.02 */
    int32_t armijo_max_halvings;/*                                                         30   */
    int32_t cg_max;             /* CG iteration cap                                        500  */
    int32_t dense_d_max;        /* d <= this: dense (d+1)x(d+1) H + Cholesky; else CG      128  */
    int32_t inner_max;          /* semismooth Newton iterations per outer iteration        50   */
    int32_t outer_max;          /*                                                         200  */
    int32_t max_rounds;         /* active-set refinement rounds               10   */
    int32_t sample_rows;        /* rows whose mean is the initial centre c^0               1024 */
    int32_t outer_max_lo;       /* outer iterations of the low-precision run (reading 17)     30   */
    double armijo_shrink_min;   /* a rejected Armijo trial halves eta, or multiplies it by this factor when the
                                 * parabola through Psi(x), Psi'(x; Delta), Psi(x + eta Delta) puts its minimiser
                                 * below it (trials bound to fail are skipped); 0.5 = plain halving (reading 4)  0.5  */
    int32_t armijo_multi;       /* every Armijo trial pass also evaluates Psi at the next armijo_multi halvings of its
                                 * step (same bytes, one more dot product per row), and halvings already known to fail
                                 * are skipped (DESIGN reading 19); 0 = off; -1 = automatic:
                                 * 4 for rows longer than 1 KB, off for shorter rows, where the per-row cost of the
                                 * predictions exceeds what the skipped (and anyway cut-short) trials cost         -1   */
    int32_t ag_outer;           /* the first ag_outer outer iterations solve subproblem (4) with the accelerated
                                 * gradient method instead of semismooth Newton (DESIGN reading 20)       0    */
    double sigma_carry;         /* mixed mode: the FP64 run on the reduced problem starts at
                                 * sigma = max(sigma0, sigma_carry * sigma reached by the low-precision run) when that
                                 * run converged (its multipliers are the warm start); 0 = reset to sigma0
                                 * (DESIGN reading 11)                                                             0    */
} meb_params;

/* Counters and residuals of one meb_solve (host struct). */
typedef struct meb_stats {
    int32_t converged;          /* 1 if KKT_max <= tol and the full feasibility check passed */
    int32_t outer_iters;        /* Algorithm 1 iterations, all phases */
    int32_t newton_iters;       /* Algorithm 2 iterations, all phases */
    int32_t cg_iters;
    int32_t passes_fp64_full;   /* streaming passes over all m rows in FP64 (eval, check, init) */
    int32_t passes_fp32_full;   /* streaming passes over all m rows of the FP32 shadow */
    int32_t passes_reduced;     /* streaming passes over the reduced problem */
    int32_t rounds;             /* refinement rounds of the mixed mode */
    int64_t n_reduced;          /* |I_red| entering the last FP64 phase */
    int64_t n_support;          /* balls with u_i > 0 at the end */
    double kkt;                 /* final relative KKT residual (reading 7) */
    double kkt_terms[5];        /* the five terms of KKT_max */
    double delta_max;           /* max_i(r_i + ||c - c_i||) - r_alg from the final full check */
    double radius_alg;          /* radius of the last iterate (before the feasible-radius step 7) */
    double length_scale;        /* L = r^0 (reading 3) */
    double ms_total, ms_phase_lo, ms_phase_hi, ms_check;   /* device times (CUDA events) */
    double bytes_streamed;      /* algorithmic bytes of all streaming passes */
    /* per pass class (MEB_PASS_*): device time of the streaming launches (CUDA events recorded on the
     * context's stream around each launch, read after the solve), their algorithmic bytes and count */
    double pass_ms[8];
    double pass_bytes[8];
    int32_t pass_count[8];
    int64_t kernel_launches;    /* kernels of this library launched by the solve */
    int32_t passes_cut;         /* Armijo trial passes (counted in passes_*) stopped early because the partial sum
                                 * of Psi already exceeded Psi(x): certain rejections */
    int32_t trials_skipped;     /* Armijo step sizes never evaluated because a trial pass had already shown that Psi at
                                 * that step exceeds Psi(x) (multi-trial line search) */
    /* the same per pass class, from CUDA-EVENT pairs recorded on the context's stream around every streaming
     * launch: filled for launches made outside CUDA graphs (ingest, screen, feasibility always; the evaluation
     * passes when the solve is host-stepped, MEB_OPT_STEPPED).  Passes that were cut short are left out. */
    double pass_ev_ms[8];
    double pass_ev_bytes[8];
    int32_t pass_ev_count[8];
    int32_t ag_iters;           /* accelerated-gradient inner iterations (meb_params.ag_outer) */
    int32_t reserved0;
} meb_stats;

/* classes of streaming passes in meb_stats.pass_* */
enum {
    MEB_PASS_INGEST = 0,       /* a0: FP64 read of all m rows (+ FP32 shadow write in mixed mode) */
    MEB_PASS_EVAL_FP64 = 1,    /* a1 over all m rows, FP64 */
    MEB_PASS_EVAL_FP32 = 2,    /* a1 over all m rows of the FP32 shadow */
    MEB_PASS_SCREEN = 3,       /* a7 over all m rows of the FP32 shadow */
    MEB_PASS_FEAS = 4,         /* a8 over all m rows, FP64 */
    MEB_PASS_EVAL_REDUCED = 5, /* a1 over the reduced problem (L2-resident, not an HBM claim) */
    MEB_PASS_NCLASS = 8
};

/* Scalars written by meb_eval_alm into out_scalars[MEB_EVAL_NSCALARS] (device, double). */
enum {
    MEB_EV_PSI = 0,        /* psi_var = r + (sigma/2) sum ||Pi(z_i)||^2 + (tau/2sigma)||x-xbar||^2 (reading 13) */
    MEB_EV_SUM_UPLUS = 1,  /* sum_i u+_i,  u+_i = sigma t_i   */
    MEB_EV_SUM_PROJ2 = 2,  /* sum_i ||Pi(z_i)||^2   */
    MEB_EV_SUM_DMULT2 = 3, /* sum_i ||(u+_i - u_i, v+_i - v_i)||^2, right side of (5)  */
    MEB_EV_N_B1 = 4,
    MEB_EV_N_B3 = 5,
    MEB_EV_MAX_PFEAS = 6,  /* max_i dist((r - r_i, c - c_i), Q)   */
    MEB_EV_MAX_COMPL = 7,  /* max_i |(r - r_i) u+_i + <c - c_i, v+_i>|   */
    MEB_EV_MAX_DFEAS = 8,  /* max_i dist((u+_i, v+_i), Q)   */
    MEB_EV_SUM_RHO = 9,    /* sum over B3 of rho_i = a_i/nb_i (for the generalized Hessian)      */
    MEB_EV_NORM_SUM_VPLUS = 10, /* || sum_i v+_i ||   */
    MEB_EV_N_ACTIVE = 11,
    MEB_EVAL_NSCALARS = 16
};

/* ---- context ------------------------------------------------------------------------------ */
/* Creates a context on CUDA device `device` that launches on `cuda_stream` (a cudaStream_t, may be
 * NULL = legacy default stream) and can hold problems up to m_max x d_max.  Workspace is
 * allocated here (about 40 bytes per ball plus O(grid * d)).  Errors: MEB_E_ARG, MEB_E_ALLOC, MEB_E_CUDA. */
MEB_API int meb_create(meb_ctx** out, int device, void* cuda_stream, int64_t m_max, int32_t d_max);
MEB_API int meb_destroy(meb_ctx* ctx);
MEB_API const char* meb_strerror(int code);
MEB_API int meb_last_cuda_error(const meb_ctx* ctx);           /* cudaError_t of the last MEB_E_CUDA */
MEB_API void meb_default_params(meb_params* h_params);          /* fills the defaults listed above */
MEB_API int meb_version(void);

/* Behaviour switches of a context (tests, profiling and measurement; none changes a result).  At meb_create the
 * environment variables MEB_NO_GRAPH, MEB_NO_SMALL, MEB_NO_ABORT (any value) preset the first three to 1. */
enum {
    MEB_OPT_STEPPED = 0,   /* 1: meb_solve sequences the SAME kernels and controller steps from the host instead of
                            *    launching its CUDA graph (profilers list every launch; every streaming launch gets a
                            *    CUDA-event pair, meb_stats.pass_ev_*) */
    MEB_OPT_NO_SMALL = 1,  /* 1: small (reduced) problems run through the general kernels, not the single-CTA solver */
    MEB_OPT_NO_ABORT = 2,  /* 1: doomed Armijo trials are not cut short (results are bit-identical either way) */
    MEB_OPT_NO_FUSED_SCREEN = 3,   /* 1: the screening of the mixed mode always runs as its own pass (long rows normally
                                    * take the retain rule from the last evaluation pass of the low-precision run; same
                                    * kept set either way) */
    MEB_OPT_NCOUNT = 4
};
MEB_API int meb_set_option(meb_ctx* ctx, int option, int value);    /* MEB_E_ARG for an unknown option */

/* ---- whole solve (Algorithm 1, Algorithm 2, Section 4.2) -------
 * centers, radii: DEVICE, FP64.  h_center_out[d], h_radius_out, h_stats: HOST.
 * Returns the unique optimum to relative KKT tolerance `tol` (reading 7); the returned
 * radius is max_i(||c - c_i|| + r_i) for the returned centre (step 7 of the algorithm statement).
 * Errors: MEB_E_ARG, MEB_E_INPUT, MEB_E_CAPACITY, MEB_E_ALLOC, MEB_E_CUDA; MEB_W_NOT_CONVERGED. */
MEB_API int meb_solve(meb_ctx* ctx, int64_t m, int32_t d, const double* centers, int64_t ld,
              const double* radii, double tol, int precision_mode, const meb_params* h_params,
              double* h_center_out, double* h_radius_out, meb_stats* h_stats);

/* ---- the same solve with the balls PARTITIONED over several GPUs (the paper's stated
 * future work; the constraint-wise separable structure that allows it: P:L179, L218) ----
 * One process per GPU.  This rank holds the contiguous rows [row_offset, row_offset + m_local) of an instance of
 * m_global balls: centers_local / radii_local are DEVICE arrays of m_local rows.  The (d+1)-sized state and the
 * controller are replicated; at every reduction point (evaluation, Hessian-vector product or dense Hessian,
 * initial point, feasibility check) the rank packs its partial into xchg_send (DEVICE, xchg_doubles doubles:
 * at least meb_shard_record_doubles(d)), calls allgather(user, n), which must place the first n doubles of every
 * rank's xchg_send at xchg_recv + r * n (DEVICE, nranks * xchg_doubles doubles) for r = 0..nranks-1, ORDERED ON THE
 * CONTEXT'S STREAM (e.g. ncclAllGather on that stream; return 0 on success), and the second-level kernels add the
 * nranks records in rank order.  All ranks therefore compute bit-identical iterates.  Records are d + O(10) doubles
 * ((d+1)^2 for the dense Hessian, d <= 128).  The solve is host-stepped (one decision read-back per evaluation).
 * Outputs as meb_solve; meb_stats counts this rank's passes and bytes.  Every rank must pass the same tol, mode
 * and parameters.  m_local >= 1. */
typedef int (*meb_allgather_fn)(void* user, int64_t n_doubles);
MEB_API int64_t meb_shard_record_doubles(int32_t d);
MEB_API int meb_solve_sharded(meb_ctx* ctx, int32_t rank, int32_t nranks, int64_t m_local, int64_t row_offset,
                      int64_t m_global, int32_t d, const double* centers_local, int64_t ld,
                      const double* radii_local, double tol, int precision_mode, const meb_params* h_params,
                      double* xchg_send, double* xchg_recv, int64_t xchg_doubles, meb_allgather_fn allgather,
                      void* user, double* h_center_out, double* h_radius_out, meb_stats* h_stats);

/* Same, with HOST input buffers: uploads centres (and radii) to device memory owned by the context
 * (host->device copies are part of the call), then solves.  This is the end-to-end entry point. */
MEB_API int meb_solve_host(meb_ctx* ctx, int64_t m, int32_t d, const double* h_centers, int64_t ld,
                   const double* h_radii, double tol, int precision_mode, const meb_params* h_params,
                   double* h_center_out, double* h_radius_out, meb_stats* h_stats);

/* ---- batched solves of small independent instances (the small-m end of the paper's
 * experiments) ----
 * nprob instances in R^d stored back to back: instance k owns rows h_row_offsets[k] .. h_row_offsets[k+1]-1 of
 * `centers` (DEVICE, FP64, row stride ld) and of `radii` (DEVICE, nullable = points).  Every instance needs
 * 1 <= m_k <= 4096 and d <= 126 (else MEB_E_CAPACITY).  One persistent CTA per instance runs the FP64 ripALM
 * of Algorithms 1-2 from its own initial point (reading 3), then the feasible-radius
 * step; three launches for the whole batch, one host synchronisation.
 * h_row_offsets[nprob+1]: HOST.  Outputs (HOST, owned by the caller): h_centers_out[nprob*d],
 * h_radii_out[nprob], h_status_out[nprob] (nullable; MEB_OK, MEB_W_NOT_CONVERGED or MEB_E_INPUT per instance),
 * h_kkt_out[nprob] (nullable; relative KKT residual reached, reading 7).  Workspace is owned by the context and
 * grows on demand (MEB_E_ALLOC).  Returns the worst per-instance status, or MEB_E_ARG / MEB_E_CUDA. */
MEB_API int meb_solve_batch(meb_ctx* ctx, int32_t nprob, const int64_t* h_row_offsets, int32_t d,
                            const double* centers, int64_t ld, const double* radii, double tol,
                            const meb_params* h_params, double* h_centers_out, double* h_radii_out,
                            int32_t* h_status_out, double* h_kkt_out);

/* ---- a0: ingest (reading 3; P:L250 low-precision copy) ---------------------------------------
 * c0_out[d] (device, double) = mean of the S = min(m, sample_rows) rows floor(k*m/S);
 * scalars_out[0] = L = max_i(||c_i - c0|| + r_i), scalars_out[1] = argmax (as double),
 * scalars_out[2] = number of rows with a non-finite entry, or a negative or non-finite radius (validation).
 * If C32 != NULL also writes the FP32 shadow C32[i,:] = fl32(c_i - c0) (row stride ld32, a multiple
 * of 4) and R32[i] = fl32(r_i) (R32 may be NULL when R is NULL). */
MEB_API int meb_ingest(meb_ctx* ctx, int64_t m, int32_t d, const double* C, int64_t ld, const double* R,
               int32_t sample_rows, double* c0_out, double* scalars_out,
               float* C32, int64_t ld32, float* R32);

/* ---- a1: one evaluation of the proximal augmented Lagrangian
 * One streaming pass over the m rows.  out_scalars[MEB_EVAL_NSCALARS] and grad[d+1] are device doubles:
 *   grad = (1;0) - (sum u+; sum v+) + (tau/sigma)(x - xbar).
 * Optional outputs (NULL to skip): t_out[m], lam_out[m] per-ball doubles (Pi(z_i) = (t_i, lam_i b_i));
 * active_idx[>= m] ascending int32 list of the active balls (its length is out_scalars[MEB_EV_N_ACTIVE]),
 * active_rho[k] = a/nb of list entry k (2.0 marks a B1 ball), active_lam[k]. */
MEB_API int meb_eval_alm(meb_ctx* ctx, int prec, int64_t m, int32_t d, const void* C, int64_t ld,
                 const void* R, const void* U, const int32_t* v_slot, const void* Vrows, int64_t ldv,
                 const double* x, const double* xbar, double sigma, double tau,
                 double* out_scalars, double* grad, double* t_out, double* lam_out,
                 int32_t* active_idx, double* active_rho, double* active_lam);

/* ---- a1 with several points of one line (multi-trial Armijo; DESIGN reading 19) ----------
 * Same pass as meb_eval_alm at x (out_scalars, grad as there), which ALSO returns
 *   psi_out[k] = psi_var(x - h_gammas[k] * dir),  k < n_steps <= 4      (device doubles; dir: device [d+1])
 * from ||b_i||^2, <b_i, dir_c> and ||dir_c||^2 of every ball: one read of the rows whatever n_steps is.
 * h_gammas must be non-negative and non-decreasing.  Inside meb_solve every Armijo trial pass uses this to
 * predict the next halvings of its step.  Rows must be 16-byte aligned (else MEB_E_CAPACITY). */
MEB_API int meb_eval_alm_multi(meb_ctx* ctx, int prec, int64_t m, int32_t d, const void* C, int64_t ld,
                       const void* R, const void* U, const int32_t* v_slot, const void* Vrows, int64_t ldv,
                       const double* x, const double* xbar, double sigma, double tau, const double* dir,
                       int32_t n_steps, const double* h_gammas, double* out_scalars, double* grad, double* psi_out);

/* ---- a2: generalized-Hessian-vector product (P_i: reading 1) ---------------
 *   Hq = (tau/sigma) q + sigma sum_i P_i q,  P_i = I (B1), 0 (B2),
 *   1/2 [[1, w^T],[w, (1+rho) I - rho w w^T]] (B3), w = b/nb, rho = a/nb.
 * One streaming pass to classify the balls, then a pass over the ACTIVE rows only.  q, Hq: device [d+1]. */
MEB_API int meb_hvp(meb_ctx* ctx, int prec, int64_t m, int32_t d, const void* C, int64_t ld,
            const void* R, const void* U, const int32_t* v_slot, const void* Vrows, int64_t ldv,
            const double* x, double sigma, double tau, const double* q, double* Hq);

/* ---- a2': dense generalized Hessian, for moderate d (SURVEY 8(a) row a2') ---------------
 *   H[(d+1) x (d+1)] (device, double, row-major, full symmetric matrix).  d <= 128 (else MEB_E_CAPACITY). */
MEB_API int meb_dense_hessian(meb_ctx* ctx, int prec, int64_t m, int32_t d, const void* C, int64_t ld,
                      const void* R, const void* U, const int32_t* v_slot, const void* Vrows,
                      int64_t ldv, const double* x, double sigma, double tau, double* H);

/* ---- a6: multiplier update (eq. (6); batched form P:L181-183) ----------------------
 *   u_i <- sigma t_i for all i;  v_i <- sigma lam_i b_i for the active balls, stored as the rows of
 *   Vrows_out in ascending ball order with v_slot_out[i] = its row or -1.  Output arrays must not
 *   alias the inputs.  cap_rows = rows available in Vrows_out (MEB_E_CAPACITY if too few;
 *   n_slots is still written).  h_n_slots (host) = number of rows written;
 *   h_sum_mult2 (host) = sum_i (u_i^2 + ||v_i||^2) of the NEW multipliers (last term of P:L107). */
MEB_API int meb_update_multipliers(meb_ctx* ctx, int prec, int64_t m, int32_t d, const void* C, int64_t ld,
                           const void* R, const void* U, const int32_t* v_slot, const void* Vrows,
                           int64_t ldv, const double* x, double sigma,
                           void* U_out, int32_t* v_slot_out, void* Vrows_out, int64_t ldv_out,
                           int64_t cap_rows, int64_t* h_n_slots, double* h_sum_mult2);

/* ---- a7: FP32 boundary screening + stream compaction ------------------------------
 *   s_i = r_hat - r_i - ||c_hat - c_i|| in float;  keep i iff s_i <= tol_red.
 *   idx_out[cap]: ascending int32 indices of the kept balls; h_count (host) = how many
 *   (MEB_E_CAPACITY if > cap, idx_out then holds the first cap).
 *   flags (device, uint8[m], nullable): flags_are_input = 0 -> written with the computed flags;
 *   flags_are_input = 1 -> C32/R32 are ignored and the compaction uses these flags verbatim
 *   (bit-exact compaction test, independent of floating point). */
MEB_API int meb_screen_compact(meb_ctx* ctx, int64_t m, int32_t d, const float* C32, int64_t ld32,
                       const float* R32, float r_hat, const double* c_hat, float tol_red,
                       int32_t* idx_out, int64_t cap, int64_t* h_count,
                       uint8_t* flags, int flags_are_input);

/* ---- a8: full FP64 a-posteriori feasibility check ---------------------------------
 *   viol_i = r_i + ||c - c_i|| - r;  h_delta_max = max_i viol_i, h_argmax = its smallest index;
 *   viol_idx[cap] = ascending indices with viol_i > eps_feas and kept_mask[i] == 0
 *   (kept_mask uint8[m] nullable = nothing kept); h_n_viol = their number.  c: device [d]. */
MEB_API int meb_feasibility_check(meb_ctx* ctx, int64_t m, int32_t d, const double* C, int64_t ld,
                          const double* R, double r, const double* c, double eps_feas,
                          const uint8_t* kept_mask, double* h_delta_max, int32_t* h_argmax,
                          int32_t* viol_idx, int64_t cap, int64_t* h_n_viol);

/* ---- a8': the feasibility maximum WITHOUT any allocation ---------------------------
 *   out2 (DEVICE, 2 doubles): out2[0] = max_i (r_i + ||c - c_i|| - r), out2[1] = its smallest index.
 * For callers that cannot call cudaMalloc (under CUDA graph capture, serving loops): no context, no
 * workspace; nothing is allocated or freed, nothing is synchronised.  The scratch of the two-level
 * reduction is a file-scope __device__ array of MEB_STATIC_MAX_TILES (value, index) pairs = 1 MiB that
 * every GPU holding the library keeps until exit, so m <= MEB_STATIC_MAX_ROWS (else MEB_E_CAPACITY).
 * C (m x d FP64, row stride ld), R (nullable = points), c: DEVICE pointers on the CURRENT device;
 * cuda_stream: a cudaStream_t (NULL = legacy default stream); the kernels are queued on it and the call
 * returns without waiting.  All calls share the scratch: calls ordered on one stream are safe, calls
 * that overlap on the GPU (other streams, other host threads) race.  Not thread-safe on first use per
 * device.  Errors: MEB_E_ARG (null pointer, m < 1, d < 1, ld < d), MEB_E_CAPACITY, MEB_E_CUDA. */
#define MEB_STATIC_MAX_TILES 65536
#define MEB_STATIC_MAX_ROWS (256LL * MEB_STATIC_MAX_TILES)      /* 16,777,216 balls */
MEB_API int meb_feasibility_max_static(void* cuda_stream, int64_t m, int32_t d, const double* C, int64_t ld,
                                       const double* R, double r, const double* c, double* out2);

/* ---- measurement helper ------------------------------------------------------------------------
 * Device time (ms, CUDA events on the context's stream) and algorithmic bytes of the most recent
 * streaming-pass launch made through this context (eval/hvp-classify/screen/feasibility/ingest). */
MEB_API int meb_last_pass_info(const meb_ctx* ctx, double* h_ms, double* h_bytes);
/* on != 0: every streaming launch is bracketed by CUDA events and synchronised (measurement only). */
MEB_API int meb_set_pass_timing(meb_ctx* ctx, int on);

#ifdef __cplusplus
}
#endif
#endif /* MEB_H_ */
