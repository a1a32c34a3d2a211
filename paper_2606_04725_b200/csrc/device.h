// device.h -- device-side data layout and kernel launch wrappers shared by factor.cu / ipm.cu / api.cu.
//
// HBM layout (all owned by the handle, allocated once in nmpc_analyze):
//   L   : one dense column-major panel per supernode s, r_s x w_s (leading dimension r_s rounded up to even), at panel_ptr[s]
//   U   : one dense column-major update (Schur complement) matrix per supernode, (r_s-w_s)^2, at upd_ptr[s];
//         only the lower triangle is written and read (multifrontal extend-add, parent pulls from children
//         in a fixed order -> bitwise reproducible)
//   ctr : per supernode r_s - w_s doubles at rel_ptr[s]: contribution vector of the forward solve
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "models.cuh"

namespace nmpc {

struct DevSym {                   // device copies of the symbolic arrays (symbolic.h)
    int32_t ns = 0;
    int64_t n = 0;
    int32_t aug_col = -1;         // pivot position (== original index n) of the right-hand-side row (symbolic.h), -1 = none: its
                                  // pivot is taken as 1 without a test, the solves treat its right-hand side / solution as 0
    const int32_t* sn_start = nullptr;
    const int64_t* rows_ptr = nullptr;
    const int32_t* rows = nullptr;
    const int32_t* child_ptr = nullptr;
    const int32_t* child_idx = nullptr;
    const int64_t* rel_ptr = nullptr;
    const int32_t* rel = nullptr;
    const int64_t* panel_ptr = nullptr;
    const int64_t* upd_ptr = nullptr;
    const int64_t* kent_ptr = nullptr;
    const int32_t* kent_src = nullptr;
    const int32_t* kent_dst = nullptr;
    const int32_t* perm = nullptr;
    double* L = nullptr;
    double* U = nullptr;
    double* ctr = nullptr;
    double* dinv = nullptr;       // n: 1 / L_jj at pivot position j (written by the factorization, used by the solves)
    int32_t* fail_col = nullptr;  // first failing pivot position (INT_MAX = none)
};

constexpr int BIG_NB = 64;        // block size used by the triangular-solve kernels for the diagonal blocks
constexpr int TILE = 64;          // tile size of the tiled (HBM-resident) fronts
constexpr int BWD_CH = 8;         // tiles of the ancestors' rows one chunk task of the backward solve takes (solve.cu)
constexpr int SMALL_ROWS_MAX = 240;  // upper bound on the rows (leading dimension) of a front handled by one CTA in shared memory

__host__ __device__ inline int ld_even(int r) { return (r + 1) & ~1; }   // = symbolic.h: panel_ld

// Block boundaries of a tiled front (rows == columns): nbp blocks of 64 over the pivot columns [0,w) (last one ragged),
// then blocks over the update rows [w,r); when w is odd the first update block has 63 rows so that every later
// boundary is even (16-byte aligned operand loads).
__host__ __device__ inline int tile_bound(int k, int w, int r, int nbp) {
    if (k < nbp) return k * TILE;
    if (k == nbp) return w;
    const int v = w + TILE - (w & 1) + TILE * (k - nbp - 1);
    return v < r ? v : r;
}
__host__ __device__ inline int tile_nbp(int w) { return (w + TILE - 1) / TILE; }
__host__ __device__ inline int tile_nbu(int w, int r) {
    if (r <= w) return 0;
    const int e1 = w + TILE - (w & 1);
    return r <= e1 ? 1 : 1 + (r - e1 + TILE - 1) / TILE;
}

// Task lists of the persistent task-DAG kernels, built once by nmpc_analyze.
//   factor task   (type, sn, I, J): type 0 = whole small front in shared memory, 1 = tile (I,J) of a tiled front (left-looking)
//   solve task    (type, sn, I, dir): type 0 = whole supernode, 1 = block row I (forward) / helper sums of block column I
//                 (backward) of a tiled supernode, 2 (backward) = chunk c of the ancestors' rows for block column J, I = J | c << 16,
//                 3 (backward) = the chain of the diagonal blocks of a tiled supernode;
//                 dir 0 = forward (L v = P b), 1 = backward (L^T x = v); forward tasks first, then the backward tasks top-down
// Completion flags are EPOCH-valued (no reset between calls): call number e stores e into a flag and adds 1 to a counter,
// so "done in this call" is flag >= e, counter >= e * target; the claim counter advances by ntasks + grid per call.
// The forward and the backward half of the solves have their own call numbers (a fused solve runs the backward half only).
struct DagPlan {
    const int4* ftasks = nullptr;        // factorization
    int32_t n_ftasks = 0;
    const int4* stasks = nullptr;        // solves: n_sfwd forward tasks, then the backward tasks
    int32_t n_stasks = 0, n_sfwd = 0;
    const int32_t* cls = nullptr;        // ns: 0 small, 1 tiled
    const int32_t* tbase = nullptr;      // ns: base of the front's (nbp x nbt + 1) slots in tile_done / tile_kptr
    const int32_t* bbase = nullptr;      // ns: base of the front's nbp slots in blk_f / blk_b
    const int32_t* target = nullptr;     // ns: factor completions that finish the front (1, or the number of tiles)
    const int32_t* target_f = nullptr;   // ns: forward-solve completions (1 or nbt);  backward: 1 or nbp
    const int32_t* target_b = nullptr;
    const int64_t* tile_kptr = nullptr;  // per tile slot: start of its K entries (kent arrays sorted by tile for tiled fronts)
    const int64_t* cb_ptr = nullptr;     // ns: offset into cbnd of the child's block boundaries in its (tiled) parent, else -1
    const int32_t* cbnd = nullptr;
    const int32_t* sn_parent = nullptr;  // ns
    uint32_t* sync = nullptr;            // [0] factor claim, [1] forward-solve claim, [2] backward-solve claim, then the arrays below
    uint32_t* fac_done = nullptr;        // ns
    uint32_t* sol_done_f = nullptr;      // ns
    uint32_t* sol_done_b = nullptr;      // ns
    uint32_t* tile_done = nullptr;       // tile slots
    uint32_t* blk_f = nullptr;           // block slots
    uint32_t* blk_b = nullptr;
    uint32_t* blk_u = nullptr;           // block slots: finished chunk tasks of the backward solve per block column
    uint32_t* blk_s = nullptr;           // block slots: helper sum S_J of the backward solve written
    double* bsum = nullptr;              // nt: the helper sums (pivot positions)
    const int32_t* cbase = nullptr;      // ns: first chunk of a tiled supernode in cdep_ptr
    const int64_t* cdep_ptr = nullptr;   // per chunk (supernode, c): the flags (word offsets into sync, all "done when >= call
    const uint32_t* cdep = nullptr;      // number") of the pieces of x its rows belong to
    const int64_t* pbase = nullptr;      // ns: offset into bpart of a tiled supernode's partial sums [chunk][w]
    double* bpart = nullptr;
    uint32_t* sub_done = nullptr;        // block slots: published 8-column blocks of the diagonal tile L_JJ, (epoch-1)*16 + count
#ifdef NMPC_TRACE_BUILD                     // measurement build only (libnmpc_b200_aids.so, include/nmpc_aids.h)
    unsigned long long* ftrace = nullptr;   // 8 timestamps per factor task / per solve task
    unsigned long long* strace = nullptr;
#endif
    int64_t sync_words = 0;
    int32_t small_max_r = 0;
    int32_t sbuf = 0;                    // doubles per staged column block of the small-supernode solves
    int32_t fgrid = 0, sgrid = 0;
    size_t fsmem = 0, ssmem = 0;
};

// ---- factor.cu ----
// one_cta_per_sm: latency mode (small problems whose largest fronts then fit one CTA's shared memory), else two CTAs per SM
cudaError_t configure_factor_kernels(int max_smem_bytes, bool one_cta_per_sm, int* ctas_per_sm, size_t* smem_bytes, int* small_max_r);
// epoch_dev (may be null): device words {factor call number, solve call number} that override `epoch` (CUDA-graph replay)
void launch_factor(const DevSym& D, const DagPlan& F, const double* Kval, double eta, uint32_t epoch, const uint32_t* epoch_dev,
                   cudaStream_t st);
void launch_reset_fail(const DevSym& D, cudaStream_t st);                                   // fail_col = INT_MAX
#ifdef NMPC_TRACE_BUILD
cudaError_t read_potrf_cycles(unsigned long long* out8, bool reset);   // measurement build: phase cycles of the diagonal-tile POTRFs
#endif
// ---- solve.cu ----
cudaError_t configure_solve_kernels(int max_smem_bytes, int small_max_r, int* ctas_per_sm, size_t* smem_bytes, int* sbuf_doubles);
// rhs_inout (original ordering, n doubles) is overwritten by K^-1 rhs; x is the handle's permuted work vector.
// epoch_f / epoch_b: call numbers of the forward / backward half (epoch_dev, may be null: two device words that override them).
// fused: backward half only, v = L^-1 P b is read from the right-hand-side row of the factor and rhs_inout is written only.
void launch_solve(const DevSym& D, const DagPlan& F, double* rhs_inout, double* x, uint32_t epoch_f, uint32_t epoch_b,
                  const uint32_t* epoch_dev, bool fused, cudaStream_t st);

// ---- ipm.cu ----
struct DevModel {                 // device copies of the model maps (symbolic.h: ModelMaps) + parameters
    ModelDesc desc;
    int64_t n = 0, m = 0, nnzJ = 0, nnzW = 0, nnzK = 0;
    int64_t m_dyn = 0;                                                  // rows [0, m_dyn): dynamics h_k; [m_dyn, m): general linear rows
    const double* g_val = nullptr;                                      // their values, in J order from J_ptr[m_dyn] on
    const double* cl = nullptr; const double* cu = nullptr;             // m: row intervals cl <= c(y) <= cu (gamma tube included), +-inf = no such side
    const int64_t* J_ptr = nullptr; const int32_t* J_idx = nullptr;
    const int64_t* jt_ptr = nullptr; const int32_t* jt_idx = nullptr; const int32_t* jt_row = nullptr;
    const int64_t* trip_ptr = nullptr; const int32_t* trip_a = nullptr; const int32_t* trip_b = nullptr; const int32_t* trip_r = nullptr;
    const int32_t* k_w = nullptr; const int32_t* k_diag = nullptr;
    const int64_t* wf_ptr = nullptr; const int32_t* wf_idx = nullptr; const int32_t* wf_src = nullptr;   // symmetric CSR of W (-> Wval index)
    const double* lb = nullptr; const double* ub = nullptr;             // n, +-inf allowed
    double* x0 = nullptr; double* ref = nullptr;                       // parameters p = (x0, ref)
};

struct IpmVectors {               // primal-dual iterate and work vectors (device)
    double *y, *sp, *sm, *wp, *wm, *zL, *zU;                 // z = (y, s+, s-, w+, w-, zL, zU)
    double *c, *gradf, *Jval, *Wval, *Kval;                  // model evaluation + assembled K values
    double *r_pp, *r_pm, *q, *t, *sigx, *b, *dy;             // residuals, Sigma, rhs, step
    double *rho;                                             // refinement: minus the un-condensed residual, then the correction
    double *yt, *ct;                                         // line search: trial point y + alpha dy and c(yt)
    double *dsp, *dsm, *dwp, *dwm, *dzL, *dzU;
    double *partial;                                         // block partials of the reductions
    double *scal;                                            // device scalars (see ipm.cu)
};

constexpr int RED_BLOCKS = 256;   // fixed number of reduction blocks -> fixed summation tree
constexpr int NSCAL = 16;

void launch_model_eval(const DevModel& M, const double* y, const double* wp, const double* wm, const double* lam,
                       double* c, double* gradf, double* Jval, double* Wval, cudaStream_t st);
void launch_assemble_K(const DevModel& M, const double* Jval, const double* Wval, const double* sigx, const double* q,
                       double eta, double* Kval, cudaStream_t st);
void launch_kkt_multiply(int64_t n, const int64_t* ptr, const int32_t* idx, const int32_t* src, const double* Kval, double eta,
                         const double* x, double* y, cudaStream_t st);
void launch_cold_init_y(const DevModel& M, const IpmVectors& V, const double* u_init, int use_y0, double kappa_push, double mu0,
                        cudaStream_t st);
void launch_cold_init_s(const DevModel& M, const IpmVectors& V, double gamma, double s_floor, double mu0, cudaStream_t st);
void launch_warm_push(const DevModel& M, const IpmVectors& V, double warm_push, cudaStream_t st);
void launch_residuals(const DevModel& M, const IpmVectors& V, double gamma, cudaStream_t st);
// par (may be null): device doubles {mu, tau} that override the scalar arguments (CUDA-graph replay)
void launch_sigma_rhs(const DevModel& M, const IpmVectors& V, double mu, const double* par, cudaStream_t st);
void launch_step(const DevModel& M, const IpmVectors& V, double mu, double tau, const double* par, cudaStream_t st);
// fail_col (may be null): device flag of the factorization; the update is skipped when it reports a failed pivot
void launch_update(const DevModel& M, const IpmVectors& V, const int32_t* fail_col, cudaStream_t st);
void launch_objective(const DevModel& M, const IpmVectors& V, cudaStream_t st);
// iterative refinement of dy on the un-condensed first block row of Eq. (10): rho <- -((W + eta I) dy + J^T(dw+ - dw-) - dzL + dzU
// + r_d) with the eliminated directions of the last launch_step; after K^-1 rho: dy += rho.  Both skip when *fail_col reports a
// failed pivot (fail_col may be null).
void launch_refine_residual(const DevModel& M, const IpmVectors& V, double eta, const int32_t* fail_col, cudaStream_t st);
void launch_add_correction(const DevModel& M, const IpmVectors& V, const int32_t* fail_col, cudaStream_t st);
// filter line search (options.globalization): trial point yt = y + alpha dy, then (after a model evaluation c(yt) -> ct)
// scal[0..4] <- theta (1-norm of the lifted equality residuals), sum of the logarithms of the barrier, f(yt), number of
// arguments outside the barrier's domain, and (with_grad) grad phi_mu^T d at alpha = 0
void launch_trial_point(const DevModel& M, const IpmVectors& V, double alpha, cudaStream_t st);
void launch_merit(const DevModel& M, const IpmVectors& V, double alpha, double mu, double gamma, int with_grad, cudaStream_t st);


// ---- hykkt.cu: vector kernels of the HyKKT variant (nmpc_hykkt_solve) ----
void launch_hk_residuals(const DevModel& M, const IpmVectors& V, cudaStream_t st);
void launch_hk_rhs(const DevModel& M, const IpmVectors& V, double mu, double gamma_h, cudaStream_t st);
// out_n = a_n + sign * J^T v_m (a_n may be null)
void launch_hk_jt(const DevModel& M, const IpmVectors& V, const double* v_m, const double* a_n, double sign, double* out_n, cudaStream_t st);
// out_m = J u_n + shift_m (shift may be null); scal[0] = p . out (p may be null), scal[1] = out . out
void launch_hk_j(const DevModel& M, const IpmVectors& V, const double* u_n, const double* shift_m, const double* p_m, double* out_m, cudaStream_t st);
// x += alpha p, r -= alpha Sp, scal[1] = r . r
void launch_hk_cg_update(const DevModel& M, const IpmVectors& V, double alpha, double* x, double* r, const double* p, const double* Sp, cudaStream_t st);
// p = r + beta p (init: p = r, x = 0)
void launch_hk_cg_dir(const DevModel& M, double beta, const double* r, double* p, double* x, int init, cudaStream_t st);
void launch_hk_step(const DevModel& M, const IpmVectors& V, double mu, double tau, cudaStream_t st);
void launch_hk_update(const DevModel& M, const IpmVectors& V, cudaStream_t st);
void launch_fill(int64_t n, double v, double* out, cudaStream_t st);

}  // namespace nmpc
