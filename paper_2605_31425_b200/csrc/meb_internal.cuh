// Internal declarations shared by the translation units of libmeb_b200.so (sm_100a only).
// Nothing here is used by, or shared with, the CPU oracle.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/meb.h"

#define MEB_FULL_MASK 0xffffffffu
#define MEB_BLOCK 256                 // threads per CTA of every streaming kernel
#define MEB_WARPS (MEB_BLOCK / 32)
#define MEB_MAX_GRID 2368             // 148 SMs x 16: upper bound on CTAs of a streaming launch

// number of per-CTA scalar partials written by the streaming kernels
#define MEB_NPART 12
#define MEB_PART_CUT 9     // per-CTA partial: 1 if the CTA cut its pass short (MebDyn::s0_abort)
#define MEB_EVPOOL 4096               // streaming launches of one solve that get an event pair
#define MEB_MULTI_MAX 4               // step sizes an Armijo trial pass can predict besides its own (meb_params.armijo_multi)

// A sharded solve: this rank holds rows [row_offset, row_offset + m_local) of an
// m_global-ball instance.  At every reduction point the rank packs its partial into `send` (one record of at most
// rec_doubles doubles), the caller's all-gather fills `recv` with the records of all ranks in RANK ORDER, and the
// unchanged second-level kernels add the nranks records in that order: every rank forms bit-identical sums and the
// replicated controllers take identical decisions.
struct MebShard {
    int32_t rank, nranks;
    int64_t row_offset, m_global;
    double* send; double* recv; int64_t rec_doubles;
    meb_allgather_fn allgather; void* user;
};

struct meb_ctx {
    int device;
    cudaStream_t stream;
    int64_t m_max;
    int32_t d_max;
    int sm_count;
    int last_cuda_error;
    // ---- workspace (device) ----
    uint32_t* mask;         // [ceil(m/32)] active / flag bit mask of the last streaming pass
    uint32_t* vmask;        // [ceil(m/32)] scratch: balls with a multiplier row (meb_build_vlist)
    int32_t* vlist;         // [m] ascending list of the balls with a multiplier row, per-primitive calls (long rows)
    double* part_multi;     // [MEB_MAX_GRID * MEB_MULTI_MAX] per-CTA partials of the predicted step sizes
    uint32_t* smask;        // bit mask of the fused screening (same size as mask)
    double* rec_lam;        // [m] lam_i of active balls (dense-indexed, sparse writes)
    double* rec_rho;        // [m] rho_i = a/nb (2.0 marks B1)
    double* rec_t;          // [m] t_i of active balls
    int32_t* list;          // [m] compacted ascending index list
    int32_t* blocksum;      // [nseg + 2] per-segment popcounts of the compaction; [nseg] = total
    double* part_scalar;    // [MEB_MAX_GRID * MEB_NPART] per-CTA scalar partials
    double* part_vec;       // [vec_rows * (d_max+8)] per-CTA vector partials of the list kernels
    double* part_red;       // [d_max+8] sum of the vector partials (long vectors, meb_small.cu)
    int64_t vec_rows;
    double* part_mat;       // per-CTA partial matrices of the dense-Hessian SYRK
    size_t part_mat_len;
    int32_t* count_dev;     // [8] device counters (compaction totals)
    double* part_sc;        // [1024] per-CTA scalar partials of the active-list kernels
    int last_grid;          // CTAs of the last streaming launch (its partials are still in part_scalar)
    bool list_valid;        // ctx->list / count_dev hold the compaction of the mask of the last streaming pass
    double* small;          // small device state: scalars, vectors of length d+1 (see meb_api.cu)
    int64_t small_len;
    double* h_pinned;       // pinned host mirror for small read-backs
    int64_t h_pinned_len;
    // ---- owned copies for meb_solve / meb_solve_host ----
    void* own[40];
    size_t own_bytes[40];
    // ---- measurement ----
    cudaEvent_t ev0, ev1;
    double last_pass_ms;
    double last_pass_bytes;
    bool time_passes;
    // event pool: one (start, stop) pair per streaming launch of a solve, read after the solve
    cudaEvent_t* evpool;    // [2 * MEB_EVPOOL]
    int evclass[MEB_EVPOOL];
    double evbytes[MEB_EVPOOL];
    int evn;
    bool ev_record;         // on inside meb_solve
    int cur_class;          // MEB_PASS_* of the next streaming launch
    int64_t launches;       // kernels launched through this context
    // ---- device-resident solver (meb_ctrl.cuh, meb_solver.cu) ----
    void* sdev;             // SolverDev on the device
    void* h_sdev;           // pinned host mirror
    void* graph_cache;      // instantiated solve graphs (meb_solver.cu)
    cudaStream_t cap_stream; // private stream used only to CAPTURE graphs (the legacy default stream cannot capture)
    // ---- behaviour switches (meb_set_option; preset from the environment in meb_create) ----
    int opt[MEB_OPT_NCOUNT];
    bool debug;             // MEB_DEBUG: print file:line of CUDA errors
    // ---- per-context events and pinned staging ring of meb_solve ----
    cudaEvent_t ev_solve[4];        // start, end of the low-precision phase, end of the FP64 phase, end
    cudaEvent_t ev_stage[8];        // one per slot of the pinned upload ring (the slot is free once its copy ran)
    int stage_next;
    bool evcut[MEB_EVPOOL];         // stepped solves: the launch was a trial pass that was cut short
    double ev_extra_bytes;          // stepped solves: bytes of the multiplier rows the next evaluation pass reads
    int last_path;                  // kernel family of the last streaming launch (PATH_* in meb_api.cu)
    struct MebDyn* dyn_api;         // device MebDyn of the per-primitive multi-trial call
    MebShard* shard;                // non-null inside meb_solve_sharded
};

// prints file:line and the CUDA error string to stderr when the context was created with MEB_DEBUG set
void meb_debug_cuda(const meb_ctx* ctx, const char* file, int line, int err);

#define MEB_CUDA_OK(ctx, expr)                                   \
    do {                                                         \
        cudaError_t e__ = (expr);                                \
        if (e__ != cudaSuccess) {                                \
            (ctx)->last_cuda_error = (int)e__;                   \
            meb_debug_cuda((ctx), __FILE__, __LINE__, (int)e__); \
            return MEB_E_CUDA;                                   \
        }                                                        \
    } while (0)

// ------------------------------------------------------------------------------------------------
// device helpers
// ------------------------------------------------------------------------------------------------
template <typename T> struct VecOf;
template <> struct VecOf<double> { typedef double2 type; static constexpr int N = 2; };
template <> struct VecOf<float>  { typedef float4 type;  static constexpr int N = 4; };

__device__ __forceinline__ double2 ldg_stream(const double2* p) {
    double2 r;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0,%1}, [%2];" : "=d"(r.x), "=d"(r.y) : "l"(p));
    return r;
}
__device__ __forceinline__ float4 ldg_stream(const float4* p) {
    float4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p));
    return r;
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(MEB_FULL_MASK, v, o);
    return v;
}
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(MEB_FULL_MASK, v, o));
    return v;
}

// Parameters that change while a solve graph runs live in device memory (no host round trip):
struct MebDyn {
    double sigma_raw;       // sigma / L   (reading 3: kernels run on the raw data)
    double tau_eff;         // tau / L^2
    int32_t cur;            // which of the two multiplier buffers holds (U, V) of the current outer iteration
    int32_t has_mult;       // 0: all multipliers are zero (first outer iteration)
    // Early stop of an Armijo trial that is certain to be rejected: Psi = r + (sigma/2) sum_i ||Pi(z_i)||^2 + prox
    // only grows as balls are added, so once the running sum exceeds s0_abort (the value at which
    // Psi(trial) = Psi(x)) the rest of the pass cannot change the decision.  1e300: never (not a trial).
    // A CTA whose own part of the sum crosses it stops and marks its partial (slot MEB_PART_CUT).
    double s0_abort;
    // Multi-trial Armijo (DESIGN reading 19): a trial pass at x_t = x + eta Delta also forms
    // sum_i ||Pi(z_i)||^2 at the multi_n further points x_t - gamma_k Delta (gamma_k = eta (1 - 2^-k): the next
    // halvings of eta) from ||b_i||^2, <b_i, Delta c> and ||Delta c||^2 -- no extra bytes.  0: not a trial pass.
    int32_t multi_n;
    // Screening fused into the evaluation passes of the low-precision run: with screen_on the pass also
    // sets, in StreamArgs::smask, the bit of every ball with r - r_i - ||c - c_i|| <= screen_factor * r -- the
    // retain rule at the point it evaluates; after the last accepted evaluation that is the rule at (r_hat, c_hat).
    int32_t screen_on;
    double multi_gamma[MEB_MULTI_MAX];
    double dir_r;           // Delta r (raw units)
    double dir_c2;          // ||Delta c||^2 (raw units)
    double dir_c;           // ||Delta c||
    double screen_factor;   // tol_red / r_hat (meb_params.tol_red_factor)
};

// host-side launch helpers implemented in the .cu files -------------------------------------------
struct StreamArgs {
    const void* C; int64_t ld;
    const void* R;               // nullable
    const void* U;               // nullable (all zero)
    const int32_t* v_slot;       // nullable
    const void* V; int64_t ldv;
    const double* x;             // device (d+1): (r, c)
    int64_t m; int32_t d;
    double sigma;
    // outputs
    uint32_t* mask;
    double* rec_lam; double* rec_rho; double* rec_t;
    double* t_out; double* lam_out;      // nullable dense per-ball outputs
    double* part;                        // [grid * MEB_NPART]
    // feasibility / screening
    double eps; const uint8_t* kept; uint8_t* flags_out;
    // ingest
    float* C32; int64_t ld32; float* R32; const double* c0;
    int32_t rt_shift;            // loop kernel: rows per warp tile = 1 << rt_shift (5, 4 or 3; set by the launcher)
    // fused evaluation (meb_tile.cu): per-CTA partial of sum_i lam_i b_i, [grid][dpad]
    double* part_vec; int32_t dpad;
    // device-resident parameters (solve graph): if dyn != nullptr it overrides sigma, U, v_slot, V
    const MebDyn* dyn;
    const void* U2[2]; const int32_t* slot2[2]; const void* V2[2];
    // long rows (meb_long.cu): list of the balls with a multiplier row, per multiplier buffer
    const int32_t* vlist2[2]; const int32_t* vcount2[2];
    // multi-trial Armijo: direction Delta (device, (d+1), raw units), host-side switch (0: kernel without it),
    // per-CTA partials [grid][MEB_MULTI_MAX]
    const double* dir; int32_t multi; double* multi_part;
    uint32_t* smask;             // nullable: bit mask of the fused screening (MebDyn::screen_on), [ceil(m / 32)]
};

// resolves the device-resident parameters of a solve graph into the plain fields
__device__ __forceinline__ void meb_resolve_dyn(StreamArgs& a) {
    if (a.dyn) {
        const int cur = a.dyn->cur;
        const bool hm = a.dyn->has_mult != 0;
        a.sigma = a.dyn->sigma_raw;
        a.U = hm ? a.U2[cur] : nullptr;
        a.v_slot = hm ? a.slot2[cur] : nullptr;
        a.V = hm ? a.V2[cur] : nullptr;
    }
}

enum StreamOp { OP_EVAL = 0, OP_FEAS = 1, OP_SCREEN = 2, OP_INGEST = 3 };

int meb_launch_stream(meb_ctx* ctx, int op, int prec, const StreamArgs& a, int* grid_out);
// TMA-staged lane-per-row kernels (meb_tile.cu).  meb_tile_applicable: rows of at most 1024 bytes whose
// start and stride are multiples of 16 bytes.  For OP_EVAL the kernel also accumulates sum_i lam_i b_i
// (a.part_vec), so no active-list pass is needed for the gradient.
bool meb_tile_applicable(int op, int prec, const StreamArgs& a);
int meb_launch_tile(meb_ctx* ctx, int op, int prec, const StreamArgs& a, int* grid_out);
// TMA-staged warp-per-row kernels for long rows (meb_long.cu): rows longer than 1024 bytes whose start and stride
// are multiples of 16 bytes.  The launcher zeroes a.mask, launches the streaming kernel and (evaluation with
// multipliers) the kernel that handles the balls on vlist; *grid_out counts the partials of both.
bool meb_long_applicable(int op, int prec, const StreamArgs& a);
int meb_launch_long(meb_ctx* ctx, int phase, int op, int prec, const StreamArgs& a, const int32_t* vlist,
                    const int32_t* vcount, int* grid_out);
int meb_build_vlist(meb_ctx* ctx, const int32_t* slot, int64_t m, int32_t* vlist, int32_t* vcount);
int meb_copy_vlist(meb_ctx* ctx, const int32_t* list, const int32_t* count, const MebDyn* dyn, int32_t* v0, int32_t* v1,
                   int32_t* c0, int32_t* c1, int64_t cap);
int meb_launch_compact(meb_ctx* ctx, const uint32_t* mask, int64_t m, int32_t* list, int32_t* count_dev);

// ---- active-list passes (meb_active.cu) ----
enum ActiveMode { MODE_ROWSUM = 0, MODE_HVP = 1, MODE_WRITEV = 2 };

struct ActiveArgs {
    const void* C; int64_t ld;
    const void* U;
    const int32_t* v_slot; const void* V; int64_t ldv;
    const double* x;                 // (r, c)
    int32_t d; int32_t dpad;
    double sigma;
    const int32_t* list; const int32_t* count;
    const double* rec_lam; const double* rec_rho; const double* rec_t;
    const double* q;                 // hvp: (q0, q1)
    double* part_vec;                // [grid][dpad]
    double* part_sc;                 // [grid][2]
    void* U_out; int32_t* slot_out; void* V_out; int64_t ldv_out; int64_t cap_rows;
    // device-resident parameters (solve graph): override sigma, U, v_slot, V and, for MODE_WRITEV,
    // the output buffers (the multiplier buffer that is NOT current)
    const MebDyn* dyn;
    void* U2[2]; int32_t* slot2[2]; void* V2[2]; int64_t vcap2[2];
    // MODE_ROWSUM after a streaming evaluation: per-CTA partials of that pass ([cut_grid][MEB_NPART]); if any of
    // its CTAs stopped early (MEB_PART_CUT: a doomed Armijo trial) the row sum is skipped, the trial is rejected anyway
    const double* cut_part; int32_t cut_grid;
};

__device__ __forceinline__ void meb_resolve_dyn(ActiveArgs& a) {
    if (a.dyn) {
        const int cur = a.dyn->cur;
        const bool hm = a.dyn->has_mult != 0;
        const int nxt = hm ? 1 - cur : 0;
        a.sigma = a.dyn->sigma_raw;
        a.U = hm ? a.U2[cur] : nullptr;
        a.v_slot = hm ? a.slot2[cur] : nullptr;
        a.V = hm ? a.V2[cur] : nullptr;
        a.U_out = a.U2[nxt]; a.slot_out = a.slot2[nxt]; a.V_out = a.V2[nxt]; a.cap_rows = a.vcap2[nxt];
    }
}


int meb_launch_active(meb_ctx* ctx, int mode, int prec, const ActiveArgs& a, int* grid_out);
int meb_launch_compact_cap(meb_ctx* ctx, const uint32_t* mask, int64_t m, int32_t* list, int64_t cap,
                           int32_t* count_dev);
int meb_launch_flags_to_mask(meb_ctx* ctx, const uint8_t* flags, int64_t m, uint32_t* mask);

// ---- second-level reductions and small kernels (meb_small.cu) ----
struct FinalizeArgs;
int meb_eval_finalize(meb_ctx* ctx, const FinalizeArgs& f);
int meb_hvp_finalize(meb_ctx* ctx, int nvec, int dpad, const double* part_sc, const double* ev,
                     const double* q, double sigma, double tau, int d, double* Hq, const MebDyn* dyn);
int meb_argmax_finalize(meb_ctx* ctx, int grid, double* out);
int meb_scalar_sum(meb_ctx* ctx, const double* v, int n, double* out);
int meb_sample_mean(meb_ctx* ctx, const double* C, int64_t ld, int64_t m, int d, int S, double* c0);
int meb_fill_f64(meb_ctx* ctx, double* p, int64_t n, double v);
int meb_fill_f32(meb_ctx* ctx, float* p, int64_t n, float v);
int meb_fill_i32(meb_ctx* ctx, int32_t* p, int64_t n, int32_t v);
int meb_fill_u8(meb_ctx* ctx, uint8_t* p, int64_t n, uint8_t v);
int meb_gather_rows_f64(meb_ctx* ctx, const double* src, int64_t ld_src, const int32_t* idx, int64_t n, int d,
                        double* dst, int64_t ld_dst);
int meb_gather_vec_f64(meb_ctx* ctx, const double* src, const int32_t* idx, int64_t n, double* dst);
int meb_gather_mult(meb_ctx* ctx, const float* U32, const int32_t* slot32, const float* V32, int64_t ldv32,
                    const int32_t* idx, int64_t n, int d, double* U, int32_t* slot, double* V, int64_t ldv);
int meb_set_kept(meb_ctx* ctx, const int32_t* idx, int64_t n, uint8_t* kept);

// ---- internal composite passes (meb_api.cu), used by the solver ----
// layout of ctx->small (doubles): see meb_api.cu
struct SolverDev;
struct SolverVecs;
// device-resident side of a call made while a solve graph is being captured: the multipliers are
// double-buffered and selected on the device by dyn->cur; sigma and tau come from dyn
struct GraphSide {
    const MebDyn* dyn;
    void* U2[2]; int32_t* slot2[2]; void* V2[2]; int64_t vcap2[2];
    int32_t* vlist2[2]; int32_t* vcount2[2];     // long rows: balls with a multiplier row, per multiplier buffer
    int32_t multi;                               // > 0: evaluation kernels with the multi-trial code
    const double* dir;                           // direction Delta (raw units) when there is no SolverVecs (meb_eval_alm_multi)
    SolverDev* S; const SolverVecs* v;
};
struct EvalCall {
    int prec; int64_t m; int32_t d;
    const void* C; int64_t ld; const void* R; const void* U;
    const int32_t* v_slot; const void* V; int64_t ldv;
    const double* x; const double* xbar; double sigma; double tau;
    const GraphSide* gs;         // nullable
};
// One evaluation: streaming pass (+ the vector part of the gradient: fused in the tile kernel, or by
// the active-list kernel after a compaction) + finalize.  The active list is built lazily
// (meb_ensure_list) because only the Newton solve and the multiplier update need it.
int meb_eval_internal(meb_ctx* ctx, const EvalCall& c, double* out_scalars, double* grad,
                      double* t_out, double* lam_out);
int meb_ensure_list(meb_ctx* ctx, int64_t m);
int meb_hvp_from_records(meb_ctx* ctx, const EvalCall& c, const double* ev_scalars, const double* q, double* Hq);

// ---- dense Hessian and Cholesky (meb_dense.cu) ----
int meb_dense_from_records(meb_ctx* ctx, const EvalCall& c, const double* ev_scalars, double* H);
// With S != nullptr the kernel also runs the controller step that follows a Newton solve (first Armijo trial).
int meb_chol_solve(meb_ctx* ctx, const double* H, const double* g, int n, double scale, double* delta,
                   int* info_dev, SolverDev* S, const SolverVecs* v);

// ---- sharded solves (meb_shard.cu): pack the local partial into the send record, all-gather, return the stride ----
int meb_shard_exchange(meb_ctx* ctx, int64_t n_doubles);
// evaluation: per-CTA scalars [grid][MEB_NPART], vector partials [nvec][dpad] (tpb / count: see FinalizeArgs),
// predictions [grid][MEB_MULTI_MAX] (nullable) -> record [0..11] scalars, [12..15] predictions, [16..16+d) vector
int meb_shard_pack_eval(meb_ctx* ctx, const double* part, int grid, const double* part_vec, int nvec, int tpb,
                        const int32_t* count, int dpad, int d, const double* multi_part);
// hvp: record [0] = sum of the scalar partials, [8 .. 8+d) = sum of the vector partials
int meb_shard_pack_hvp(meb_ctx* ctx, const double* part_sc, int nsc, const double* part_vec, int nvec, int tpb,
                       const int32_t* count, int dpad, int d);
// dense Hessian: record [0 .. per) = sum of the per-CTA partial matrices that were written (CTAs b < ceil(count / rb))
int meb_shard_pack_mat(meb_ctx* ctx, const double* part_mat, int nparts, const int32_t* count, int rb, int64_t per);
// small records: n doubles from `src` (device) -> send[0..n)
int meb_shard_pack_small(meb_ctx* ctx, const double* src, int n);
// combine the gathered small records (stride rec) on the device: mode 0: (value, index, count) arg-max records ->
// out[0] = max value, out[1] = its index (smallest on ties), out[2] = sum of counts; mode 1: weighted mean of the
// d-vectors rec[0..d) with weights rec[d] / sum of weights -> out[0..d)
int meb_shard_combine(meb_ctx* ctx, int mode, int d, double* out);
int meb_shard_mean(meb_ctx* ctx, double* c0, int d, int64_t m_local);
int meb_shard_argmax(meb_ctx* ctx, double* scal3);

// ---- matrix-free Newton direction in one persistent kernel (meb_cg.cu) ----
int meb_launch_cg(meb_ctx* ctx, const EvalCall& c, double* W, int64_t wc_cap, double* rho_c, unsigned int* bar);

// ---- controller kernels of the device-resident solver (meb_ctrl.cu) ----
int meb_ctrl_init(meb_ctx* ctx, SolverDev* S, const SolverVecs& v, double sigma0, int cur, int has_mult);
int meb_ctrl_resume(meb_ctx* ctx, SolverDev* S);
int meb_ctrl_after_newton(meb_ctx* ctx, SolverDev* S, const SolverVecs& v);
int meb_ctrl_cg_step(meb_ctx* ctx, SolverDev* S, const SolverVecs& v);
int meb_ctrl_after_update(meb_ctx* ctx, SolverDev* S, const SolverVecs& v, const int32_t* count);
int meb_reset_next(meb_ctx* ctx, int prec, const MebDyn* dyn, void* U0, void* U1, int32_t* s0, int32_t* s1,
                   int64_t m);
void meb_free_graph_cache(meb_ctx* ctx);
size_t meb_solver_dev_size();

// ---- single-CTA solver of small problems (meb_smallsolve.cu) ----
enum { PATH_TILE = 0, PATH_LONG = 1, PATH_STREAM = 2 };
int meb_eval_path(const meb_ctx* ctx, int prec, const void* C, int64_t ld, int64_t m, int32_t d);
int meb_compact_mask(meb_ctx* ctx, const uint32_t* mask, int64_t m, int32_t* idx_out, int64_t cap, int64_t* h_count);
bool meb_wide_applicable(int prec, int64_t m, int32_t d);
int meb_launch_wide_solve(meb_ctx* ctx, const void* C, int64_t ld, const void* R, int64_t m, int32_t d, int64_t ldv,
                          void* const U2[2], int32_t* const slot2[2], void* const V2[2], SolverDev* S,
                          const SolverVecs& v, double* W);
bool meb_small_applicable(int prec, int64_t m, int32_t d);
int meb_launch_small_solve(meb_ctx* ctx, const void* C, int64_t ld, const void* R, int64_t m, int32_t d, int64_t ldv,
                           void* const U2[2], int32_t* const slot2[2], void* const V2[2], SolverDev* S,
                           const SolverVecs& v);
