/* include/nmpc.h -- C-ABI of the B200-native KKT hot path of the parametric interior-point NMPC method of
 * arxiv/paper_2606_04725 ("GPU-Accelerated Direct Transcription-Based Nonlinear Model Predictive Control").
 *
 * The library implements, in hand-written CUDA for sm_100a (fp64), the per-IPM-iteration linear solve of the
 * paper's Algorithm 2 (LiftedIPM):
 *
 *   symbolic analysis, once per OCP structure   SymCholesky, Eq. (18)-(19); Alg. 2 lines 10-12
 *   numeric Cholesky on the fixed structure     NumCholesky, Eq. (20)-(21); Alg. 2 line 13
 *   triangular solves                            Eq. (22)-(25);             Alg. 2 line 14
 *   condensed lifted KKT assembly                Eq. (14), (16)-(17);        Alg. 2 lines 5-9
 *   IPM iteration + NMPC parameter update        Eq. (26)-(28), Alg. 1 lines 9-11
 *
 * Conventions (all entry points)
 *   - C99, no exceptions cross the boundary, no global state; every call returns an nmpc_status.
 *   - "HOST" pointers are ordinary host memory; "DEVICE" pointers are CUDA device memory of the device that
 *     was current when the handle was created (e.g. torch tensor.data_ptr()).  Every call selects that device
 *     for its own duration and restores the caller's current device before it returns.
 *   - Ownership: the caller owns every pointer it passes.  The library copies what it needs during the call and
 *     never frees or retains caller memory; DEVICE buffers must stay valid until the handle's stream has
 *     finished the work of the call (every call that returns a HOST result synchronises that stream itself).
 *   - The handle owns all internal host and device memory; nmpc_destroy releases it.
 *   - One handle <-> one CUDA stream <-> one host thread.  fp64 only.  There is no CPU fallback on the numeric
 *     path: without a CUDA device nmpc_analyze returns NMPC_E_CUDA.
 */
#ifndef NMPC_H
#define NMPC_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct nmpc_handle_s*   nmpc_handle;   /* opaque: symbolic data + device buffers + IPM state     */
typedef struct nmpc_symbolic_s* nmpc_symbolic; /* opaque: host-only symbolic analysis (no CUDA required)  */

typedef enum {
    NMPC_OK = 0,
    NMPC_E_ARG = 1,      /* NULL / out-of-range argument                                                  */
    NMPC_E_PATTERN = 2,  /* pattern not lower-triangular CSR, unsorted, duplicate or missing diagonal      */
    NMPC_E_ALLOC = 3,    /* host or device allocation failed                                              */
    NMPC_E_CUDA = 4,     /* CUDA runtime error (no device, launch failure); see nmpc_last_error           */
    NMPC_E_STATE = 5,    /* wrong call order (solve before a successful factor, ipm_solve without a model) */
    NMPC_E_NOT_SPD = 6,  /* a pivot was <= 0 or non-finite; *info = first failing column (original index)  */
    NMPC_E_INERTIA = 7,  /* the eta schedule exceeded eta_max (Eq. 13)                   */
    NMPC_E_MAXITER = 8,  /* max_iter IPM iterations without meeting Eq. (28)                               */
    NMPC_E_STEP = 9      /* non-finite iterate                                                             */
} nmpc_status;

enum { NMPC_MODEL_NONE = 0, NMPC_MODEL_VDP = 1, NMPC_MODEL_DISTILL = 2, NMPC_MODEL_PLATE = 3 };
enum { NMPC_ORDER_AUTO = 0, NMPC_ORDER_NATURAL = 1, NMPC_ORDER_AMD = 2, NMPC_ORDER_ND = 3, NMPC_ORDER_TIME_ND = 4 };

/* Sparsity pattern of the condensed KKT matrix K (Eq. 17): HOST, lower triangle in CSR (row i holds the
 * columns j <= i, strictly increasing, the diagonal present in every row).  nnz = rowptr[n].               */
typedef struct {
    int64_t n, nnz;
    const int64_t* rowptr;   /* n+1 */
    const int32_t* colind;   /* nnz */
} nmpc_pattern;

/* Stage-structured parametric OCP  P_k(p_k)  (Problems 4-6) with a built-in stage model.
 * Variables y = [x_1,u_1,...,x_N,u_N] (nv = nx+nu per stage); x_0 and the references are PARAMETERS.
 * Equalities h_k = x_k - x_{k-1} - dt F(x_k,u_k) (implicit Euler), bounds lb <= (x,u) <= ub.
 * model_params (HOST, copied), by model:
 *   VDP     [w_x, w_u]                      F = (x2, (1-x1^2) x2 - x1 + u);  l = w_x |x-r|^2 + w_u u^2
 *   DISTILL [alpha, D, F_feed, x_feed, A_c, A_t, A_r, feed_index, u_bar, w_u]   (Problem 29)
 *   PLATE   [g, a, kappa_r, T_amb, b, nseg, w_T, w_u]    5-point heat equation + radiative loss, edge heaters
 * lb/ub: HOST, length nx+nu (one stage, repeated over stages); +-INFINITY = no bound.
 * u_init: HOST, length nu, cold-start input guess.
 * General linear rows (Problem 5/6: inequality constraints g and the control-horizon constraints
 * y_c,u = y_c,u_c; reading G22 of DESIGN.md): n_g rows  g_lo <= G y <= g_hi  over the whole y, stacked below the N*nx dynamics
 * rows; G as HOST CSR (g_rowptr[n_g+1], g_colind strictly increasing per row, g_val), all copied.  g_lo == g_hi: an equality
 * row, lifted like every equality (Eq. 16: g_lo - gamma <= . <= g_hi + gamma); else an inequality row, either side may be
 * -+INFINITY (one-sided).  n_g = 0: none (the pointers are ignored).  m = N*nx + n_g rows in all (slacks, multipliers, J). */
typedef struct {
    int32_t model;
    int32_t N, nx, nu, nr;       /* nr = reference entries per stage                                        */
    double  dt;
    const double* model_params;
    int32_t n_model_params;
    const double* lb;
    const double* ub;
    const double* u_init;
    int64_t n_g;
    const int64_t* g_rowptr;
    const int32_t* g_colind;
    const double* g_val;
    const double* g_lo;
    const double* g_hi;
} nmpc_ocp;

/* Options; pass NULL for the defaults (nmpc_default_options).  IPM constants are the readings S0 of
 * DESIGN.md section 3 (the paper prints none).                                          */
typedef struct {
    int32_t ordering;            /* NMPC_ORDER_*                                                            */
    int32_t nd_leaf;             /* nested-dissection leaf size (variables)                                 */
    int32_t relax_small;         /* always merge a child supernode into its parent if the merged width <= this;
                                    -1 (default) = auto: nmpc_analyze uses 32 (small latency-bound problems) or 64,
                                    the host-only nmpc_symbolic_analyze 8 */
    double  relax_zeros;         /* else merge if the explicit zeros introduced stay below this fraction      */
    int32_t smem_front_max;      /* fronts with <= this many rows run in the one-CTA shared-memory kernel     */
    int32_t use_graph;           /* replay one IPM iteration (S6-S10 + the next S2) as a CUDA graph, 1 launch/iter  */
    /* IPM (Algorithm 2) */
    double gamma, eps_outer, mu0, mu_warm, kappa_eps, kappa_mu, theta_mu, tau_min, kappa_push, s_floor, s_max;
    int32_t max_iter;
    double eta_first, eta_grow_first, eta_grow, eta_shrink, eta_min, eta_max, warm_push;
    int32_t time_phases;         /* record CUDA-event phase times in nmpc_stats (adds event overhead)         */
    /* ---- SURVEY.md section 8(f) item 2, both off by default (reading G8): ---- */
    int32_t refine_steps;        /* iterative refinement steps of the Newton direction on the UN-condensed first block row of
                                    Eq. (10): rho = (W + eta I) dy + J^T(dw+ - dw-) - dzL + dzU + r_d, K ddy = -rho; 0..4.  One
                                    step makes the IPM path insensitive to the elimination order      */
    int32_t globalization;       /* 0 = fraction to the boundary only; 1 = filter line search on the primal step ("line search
                                    with step size alpha", Eq. 26, read as Algorithm A of ref. [17] without
                                    second-order correction / restoration, reading G20)                                      */
    double  gamma_theta, gamma_phi, delta_sw, s_theta, s_phi, eta_phi, theta_max_fact, theta_min_fact;   /* constants of [17] */
    int32_t ls_max_backtracks;
    int32_t grid_limit;          /* 0 = none.  Upper bound on the CTAs of the persistent factor / solve kernels of this handle, so
                                    that the kernels of several handles driven concurrently (nmpc_ipm_solve_batch) share the SMs */
    int32_t epoch_limit;         /* 0 = automatic.  Test hook: the completion flags of the persistent kernels are
                                    call-number valued and are zeroed before a counter could overflow (after ~1e4..1e6
                                    factorizations); a small value (>= 3) forces that restart every few calls           */
    /* ---- the HyKKT variant (nmpc_hykkt_solve, reading G21) ---- */
    double  gamma_h;             /* weight of the augmented-Lagrangian term in K_g = W + Sigma_x + eta I + gamma_h J^T J   */
    double  cg_tol;              /* CG on S = J K_g^-1 J^T stops at |r|_2 <= cg_tol |rhs|_2                                 */
    int32_t cg_max_iter;
    /* ---- right-hand-side row: Eq. (22), L v = P b, computed INSIDE the numeric factorization ---- */
    int32_t fuse_rhs;            /* 1: the analysed structure is [K b; b^T 0] (one extra variable ordered last), so that the
                                    factorization leaves v = L^-1 P b in the last row of the panels and the Newton system of an
                                    IPM iteration needs the backward solve (Eq. 24) only; nmpc_factor_rhs / nmpc_solve_fused
                                    expose the same for a bare handle.  0: off.  -1 (default): on when the handle has a model.
                                    nmpc_factor / nmpc_solve / nmpc_get_factor / nmpc_get_info behave the same either way (they
                                    report the factor of K alone)                                                           */
} nmpc_options;

typedef struct {                 /* filled by nmpc_get_info; arrays are HOST pointers owned by the handle     */
    int64_t n, nnz_K, nnz_L;     /* nnz_L = sum over supernodes of panel entries on or below the diagonal     */
    int64_t panel_doubles, update_doubles;
    double  flops;               /* sum_j cc_j^2 over the columns of L (cc_j = column count incl. diagonal)   */
    int32_t nsuper, nlevels, max_front, max_width, n_large_fronts;
    int32_t ordering_used;
    double  analyze_ms;
    const int32_t* perm;         /* n: perm[i] = original index of the variable at pivot position i (Eq. 19)  */
    const int32_t* super_start;  /* nsuper+1                                                                  */
    const int64_t* rows_ptr;     /* nsuper+1                                                                  */
    const int32_t* rows;         /* rows of each supernode in pivot order (first w are its own columns)       */
    const int32_t* super_parent; /* nsuper, -1 = root                                                         */
    const int32_t* super_level;  /* nsuper, 0 = leaf level                                                    */
    const int32_t* etree_parent; /* n, elimination tree on pivot positions, -1 = root; with fused_rhs
                                    the roots of K's forest point to n (the right-hand-side row)                        */
    int32_t fused_rhs;           /* 1 if the handle carries the right-hand-side row (options.fuse_rhs)                   */
} nmpc_sym_info;

typedef struct {                 /* filled by nmpc_ipm_solve (HOST)                                           */
    int32_t status, iters, factorizations, eta_retries;
    double  E0, mu, eta_last, objective;
    double  ms_total, ms_eval, ms_assemble, ms_factor, ms_solve, ms_vector;   /* CUDA-event phase sums        */
} nmpc_stats;

typedef struct {                 /* one row per IPM iteration, for parity traces and per-iteration timing (HOST,
                                    caller array)                                                              */
    double mu, E0, Emu, eta, alpha_pr, alpha_du;
    double backtracks;           /* halvings of the filter line search in this iteration (globalization = 1);
                                    nmpc_hykkt_solve: conjugate-gradient iterations of this IPM iteration               */
    double ms_iter;              /* device time of the whole iteration (CUDA events on the handle's stream, from the
                                    launch of S6 to the launch of the next iteration's S6 / the end of the solve)   */
    double ms_eval, ms_assemble, ms_factor, ms_solve, ms_vector;   /* phase split, only with options.time_phases  */
} nmpc_trace_row;

void nmpc_default_options(nmpc_options* out);

/* ---- host-only symbolic analysis (Eq. 18-19; no CUDA needed): ordering P, elimination tree, column counts,
 *      supernode partition, level sets, scatter maps.  `ocp` may be NULL (bare pattern).  If `pattern` is NULL
 *      and `ocp` names a model, the pattern of K = W + Sigma_x + J^T Q J is derived from the model.          */
nmpc_status nmpc_symbolic_analyze(const nmpc_pattern* pattern, const nmpc_ocp* ocp, const nmpc_options* opt,
                                  nmpc_symbolic* out);
nmpc_status nmpc_symbolic_info(nmpc_symbolic sym, nmpc_sym_info* out);
/* Pattern of K derived from the model (lower CSR).  Two-call protocol: with rowptr == NULL only *nnz is set. */
nmpc_status nmpc_symbolic_pattern(nmpc_symbolic sym, int64_t* nnz, int64_t* rowptr /*n+1*/, int32_t* colind);
/* scatter map: for K value index e (pattern order), supernode and offset into the concatenated panels (layout as
 * nmpc_get_factor: column-major, leading dimension r_s rounded up to even).                                 */
nmpc_status nmpc_symbolic_kmap(nmpc_symbolic sym, int32_t* super_of_entry /*nnz*/, int64_t* panel_offset /*nnz*/);
void        nmpc_symbolic_destroy(nmpc_symbolic sym);

/* ---- Alg. 2 lines 10-12: analysis once per structure; uploads all integer maps; allocates L.  cuda_stream is a
 *      cudaStream_t.  NULL = the library creates its own blocking stream (ordered with the legacy default stream,
 *      which itself cannot carry the CUDA-graph capture of the IPM iteration).                                 */
nmpc_status nmpc_analyze(const nmpc_pattern* pattern, const nmpc_ocp* ocp, const nmpc_options* opt,
                         void* cuda_stream, nmpc_handle* out);

/* ---- Alg. 1 line 11 / PAPER.md:362: parameter update p = (x0, ref); DEVICE pointers, x0[nx], ref[N*nr];
 *      asynchronous on the stream; no structural work.                                                       */
nmpc_status nmpc_update_params(nmpc_handle h, const double* x0_dev, const double* ref_dev);
/*      same from HOST buffers (copies through pinned staging inside the call)                                */
nmpc_status nmpc_update_params_host(nmpc_handle h, const double* x0_host, const double* ref_host);

/* ---- Eq. (20)-(21): numeric Cholesky of K + eta I.  values_dev: DEVICE, nnz doubles in pattern order.
 *      Synchronises the stream to read the pivot flag.  On NMPC_E_NOT_SPD *info_host = failing original column. */
nmpc_status nmpc_factor(nmpc_handle h, const double* values_dev, double eta, int64_t* info_host);

/* ---- Eq. (22)-(25): rhs_inout_dev DEVICE n*nrhs doubles (column-major), overwritten by K^-1 rhs.  Async.   */
nmpc_status nmpc_solve(nmpc_handle h, double* rhs_inout_dev, int32_t nrhs);

/* ---- Eq. (22)-(25) with NO allocation behind it: the same two-sided solve as nmpc_solve, for callers that cannot have
 *      cudaMalloc on their path (CUDA-graph capture, tight serving loops).  The permuted work vector of the solve kernel is a
 *      file-scope device array of the library, NMPC_STATIC_SOLVE_DOUBLES doubles = 2 MiB, which every GPU that loads the
 *      library holds until the process exits; the call makes no cudaMalloc / cudaFree and calls no allocating routine (the
 *      first call on a device looks the array's device address up once, cudaGetSymbolAddress).
 *      rhs_dev: DEVICE, n doubles, read only.  out_dev: DEVICE, n doubles, receives K^-1 rhs (may equal rhs_dev: in place).
 *      Asynchronous on the handle's stream.  Errors: NMPC_E_STATE before a successful nmpc_factor / nmpc_factor_rhs;
 *      NMPC_E_ARG when the structure needs more than NMPC_STATIC_SOLVE_DOUBLES work doubles (n + 1 with the right-hand-side
 *      row, else n) -- nmpc_last_error says so; use nmpc_solve then.
 *      ALL calls on one device share the array (any handle, any stream); it keeps the last call's contents and the part a
 *      call uses is cleared first.  Calls that OVERLAP on the GPU (different streams or handles) race on it: serialise them. */
#define NMPC_STATIC_SOLVE_DOUBLES 262144
nmpc_status nmpc_solve_static(nmpc_handle h, const double* rhs_dev, double* out_dev);

/* ---- Eq. (20)-(22) in one pass (handles with the right-hand-side row, options.fuse_rhs; else NMPC_E_STATE): numeric
 *      Cholesky of K + eta I with b = rhs_dev (DEVICE, n doubles, copied) carried as an extra row, which leaves v = L^-1 P b
 *      in the factor.  nmpc_solve_fused then runs the backward solve only: out_dev (DEVICE, n) <- P^T L^-T v = K^-1 b
 *      (Eq. 24-25; async).  nmpc_solve stays valid on the same factorization for any other right-hand side.            */
nmpc_status nmpc_factor_rhs(nmpc_handle h, const double* values_dev, const double* rhs_dev, double eta, int64_t* info_host);
nmpc_status nmpc_solve_fused(nmpc_handle h, double* out_dev);

/* ---- y = K x with the values last passed to nmpc_factor (+eta I), for residual checks.  Async.            */
nmpc_status nmpc_kkt_multiply(nmpc_handle h, const double* x_dev, double* y_dev);

/* ---- Algorithm 2 (LiftedIPM) on the current parameters.  warm = 0: cold start (y_inout_dev is ignored on input
 *      unless use_y0 != 0); warm = 1: z <- stored z* of the previous solve (Alg. 1 line 10).  y_inout_dev DEVICE n.
 *      trace (HOST, may be NULL) receives up to trace_cap rows.  z* is stored for the next warm start only when the
 *      solve converged (NMPC_OK) or stopped at max_iter with a finite iterate; after NMPC_E_STEP / NMPC_E_INERTIA the
 *      next call with warm = 1 starts cold.                                                                     */
nmpc_status nmpc_ipm_solve(nmpc_handle h, int32_t warm, int32_t use_y0, double* y_inout_dev, nmpc_stats* stats_host,
                           nmpc_trace_row* trace_host, int32_t trace_cap);
/*      end-to-end form with HOST buffers: parameters in, primal solution out (copies inside the call)        */
nmpc_status nmpc_ipm_solve_host(nmpc_handle h, int32_t warm, const double* x0_host, const double* ref_host,
                                double* y_out_host, nmpc_stats* stats_host);

/* ---- The HyKKT variant of Algorithm 2 ("the system can be reformulated using either Lifted-KKT or HyKKT
 *      ... a hybrid direct-iterative approach based on an augmented Lagrangian formulation ... the proposed framework and its
 *      implementation also support HyKKT"; reading G21 of DESIGN.md section 3).  The equalities h(y) = 0 are kept exact (no
 *      gamma tube, no slacks); primal-dual iterate (y, lam, zL, zU).  Per IPM iteration: K_g = W + Sigma_x + eta I + gamma_h J^T J
 *      is assembled, factored (Eq. 20-21, same pattern and kernels as Eq. 17's K) and used for 2 + #CG triangular-solve pairs
 *      (Eq. 22-25): conjugate gradients on S dlam = J K_g^-1 (r1 + gamma_h J^T r2) - r2, then dy = K_g^-1 (r1 + gamma_h J^T r2
 *      - J^T dlam).  Arguments, warm start, statuses, stats and trace as nmpc_ipm_solve (trace.backtracks = CG iterations of the
 *      iteration; stats.eta_retries counts inertia retries).  The iterate shares the handle's storage with nmpc_ipm_solve
 *      (lam lives in w+): do not alternate warm starts between the two variants on one handle.
 *      nmpc_get_iterate returns lam in wp_dev (wm_dev == 0, slacks unused).                                              */
nmpc_status nmpc_hykkt_solve(nmpc_handle h, int32_t warm, int32_t use_y0, double* y_inout_dev, nmpc_stats* stats_host,
                             nmpc_trace_row* trace_host, int32_t trace_cap);

/* ---- Independent OCP instances (the scenarios of the uncertainty domain D_xi):
 *      `count` handles, each created on its OWN CUDA stream (a handle's stream must not be shared), solved concurrently --
 *      one host thread per handle runs nmpc_ipm_solve, the persistent kernels of the handles overlap on the device (bound
 *      their grids with options.grid_limit so that they share the SMs).  warm_host: count flags or NULL (all cold);
 *      y_inout_dev_host: HOST array of count DEVICE pointers (each n doubles) or NULL; stats_host: count records or NULL.
 *      Every instance computes exactly what nmpc_ipm_solve on its handle alone computes (bitwise).  Returns NMPC_OK or the
 *      first status that is not NMPC_OK (every instance is run to its end either way).                                  */
nmpc_status nmpc_ipm_solve_batch(nmpc_handle* handles_host, int32_t count, const int32_t* warm_host,
                                 double* const* y_inout_dev_host, nmpc_stats* stats_host);

/* ---- current primal-dual iterate z (DEVICE outputs; any pointer may be NULL): s+,s-,w+,w- length m; zL,zU n */
nmpc_status nmpc_get_iterate(nmpc_handle h, double* y_dev, double* sp_dev, double* sm_dev, double* wp_dev,
                             double* wm_dev, double* zL_dev, double* zU_dev);
/* ---- overwrite the stored iterate (the paper's warmstart_backend_start_values; Alg. 1 line 10): DEVICE
 *      inputs, all seven required, strictly interior (s, w > 0; z > 0 where the bound is finite).  The next
 *      nmpc_ipm_solve(warm = 1) starts from it.  Async.                                                      */
nmpc_status nmpc_set_iterate(nmpc_handle h, const double* y_dev, const double* sp_dev, const double* sm_dev,
                             const double* wp_dev, const double* wm_dev, const double* zL_dev, const double* zU_dev);
/* ---- model evaluation at (y, lam) with the current parameters (DEVICE outputs, any may be NULL):
 *      c[m], gradf[n], Jval[nnzJ], Wval[nnzW]; and the assembled K values (pattern order) for given Sigma_x[n],
 *      q[m], eta.  Used by the parity tests of steps a2/a3.                                                  */
nmpc_status nmpc_model_eval(nmpc_handle h, const double* y_dev, const double* lam_dev, double* c_dev,
                            double* gradf_dev, double* Jval_dev, double* Wval_dev);
nmpc_status nmpc_assemble(nmpc_handle h, const double* Jval_dev, const double* Wval_dev, const double* sigma_x_dev,
                          const double* q_dev, double eta, double* Kval_dev);
/* ---- patterns of J (CSR, m x n) and W (lower CSR, n x n) in the value order of nmpc_model_eval (HOST out).
 *      Two-call protocol as nmpc_symbolic_pattern.                                                           */
nmpc_status nmpc_get_jac_pattern(nmpc_handle h, int64_t* nnz, int64_t* rowptr, int32_t* colind);
nmpc_status nmpc_get_hess_pattern(nmpc_handle h, int64_t* nnz, int64_t* rowptr, int32_t* colind);
nmpc_status nmpc_get_kkt_pattern(nmpc_handle h, int64_t* nnz, int64_t* rowptr, int32_t* colind);

nmpc_status nmpc_get_info(nmpc_handle h, nmpc_sym_info* out_host);
/* ---- copy of the factor for tests: the panels of all supernodes, one after the other, to a HOST buffer.  Panel of
 *      supernode s: column-major r_s x w_s with leading dimension r_s rounded up to even (rows = nmpc_sym_info.rows). */
nmpc_status nmpc_get_factor(nmpc_handle h, double* panels_host /* panel_doubles */);
/* ---- kernel launches issued by this handle since creation (graph replays count their kernel nodes)        */
int64_t     nmpc_launch_count(nmpc_handle h);
/* ---- message of the last error of this handle (string owned by the handle).  h == NULL: message of the last failed
 *      nmpc_analyze on the calling thread (thread-local; the library prints nothing).                          */
const char* nmpc_last_error(nmpc_handle h);
void        nmpc_destroy(nmpc_handle h);

#ifdef __cplusplus
}
#endif
#endif /* NMPC_H */
