// device.h -- device-side data layout and kernel launch wrappers shared by factor.cu / ipm.cu / api.cu.
//
// HBM layout (all owned by the handle, allocated once in nmpc_analyze):
//   L   : one dense column-major panel per supernode s, r_s x w_s (leading dimension r_s), at panel_ptr[s]
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
    int32_t* fail_col = nullptr;  // first failing pivot position (INT_MAX = none)
    const double* eta = nullptr;  // device scalar: diagonal shift eta_y of Eq. (13)/(17), read by the assembly kernels
};

constexpr int BIG_NB = 64;        // block size of the tiled (global-memory) front path

struct BigItem { int32_t sn, a, b, c; };   // work item of the tiled path: supernode + tile coordinates

// ---- factor.cu ----
void launch_front_small(const DevSym& D, const int32_t* sn_list, int count, int max_r, const double* Kval, cudaStream_t st);
void launch_big_assemble(const DevSym& D, const BigItem* items, int count, const double* Kval, cudaStream_t st);
void launch_big_potrf(const DevSym& D, const BigItem* items, int count, cudaStream_t st);
void launch_big_trsm(const DevSym& D, const BigItem* items, int count, cudaStream_t st);
void launch_big_syrk(const DevSym& D, const BigItem* items, int count, cudaStream_t st);
void launch_solve_fwd(const DevSym& D, const int32_t* sn_list, int count, int max_r, double* x, cudaStream_t st);
void launch_solve_bwd(const DevSym& D, const int32_t* sn_list, int count, int max_r, double* x, cudaStream_t st);
void launch_permute_in(const DevSym& D, const double* b, double* x, cudaStream_t st);     // x[i] = b[perm[i]]
void launch_permute_out(const DevSym& D, const double* x, double* b, cudaStream_t st);    // b[perm[i]] = x[i]
void launch_reset_flag(const DevSym& D, double* eta_dev, double eta, cudaStream_t st);   // fail_col = INT_MAX, *eta_dev = eta
size_t small_front_smem_bytes(int max_r);
cudaError_t configure_factor_kernels(int max_smem_bytes);

// ---- ipm.cu ----
struct DevModel {                 // device copies of the model maps (symbolic.h: ModelMaps) + parameters
    ModelDesc desc;
    int64_t n = 0, m = 0, nnzJ = 0, nnzW = 0, nnzK = 0;
    const int64_t* J_ptr = nullptr; const int32_t* J_idx = nullptr;
    const int64_t* jt_ptr = nullptr; const int32_t* jt_idx = nullptr; const int32_t* jt_row = nullptr;
    const int64_t* trip_ptr = nullptr; const int32_t* trip_a = nullptr; const int32_t* trip_b = nullptr; const int32_t* trip_r = nullptr;
    const int32_t* k_w = nullptr; const int32_t* k_diag = nullptr;
    const double* lb = nullptr; const double* ub = nullptr;             // n, +-inf allowed
    double* x0 = nullptr; double* ref = nullptr;                       // parameters p = (x0, ref)
};

struct IpmVectors {               // primal-dual iterate and work vectors (device)
    double *y, *sp, *sm, *wp, *wm, *zL, *zU;                 // z = (y, s+, s-, w+, w-, zL, zU)
    double *c, *gradf, *Jval, *Wval, *Kval;                  // model evaluation + assembled K values
    double *r_pp, *r_pm, *q, *t, *sigx, *b, *dy;             // residuals, Sigma, rhs, step
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
void launch_sigma_rhs(const DevModel& M, const IpmVectors& V, double mu, cudaStream_t st);
void launch_step(const DevModel& M, const IpmVectors& V, double mu, double tau, cudaStream_t st);
void launch_update(const DevModel& M, const IpmVectors& V, cudaStream_t st);
void launch_objective(const DevModel& M, const IpmVectors& V, cudaStream_t st);

}  // namespace nmpc
