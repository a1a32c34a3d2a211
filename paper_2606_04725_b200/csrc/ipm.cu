// ipm.cu -- model/derivative evaluation (step a2), condensed lifted KKT assembly (step a3, Eq. 14/17)
// and the fused IPM vector kernels (step a6: residuals of Eq. 9/11, right-hand side of Eq. 17, eliminated directions of
// Eq. 10/14, fraction-to-the-boundary min-reductions, Eq. 26 update, error norms of Eq. 27-28).
//
// Reductions use a FIXED grid (RED_BLOCKS x 256 threads, grid-stride) and a fixed shuffle/shared-memory tree; the block that
// takes the last ticket (last_block_arrives) reduces the per-block partials in block order, so there is no separate finalize
// launch and results are bitwise reproducible run to run.  No floating-point atomics anywhere.
// Compiled with -fmad=false: the element-wise expressions below round like the plain fp64 statements of the method.
#include <algorithm>
#include <cfloat>
#include <climits>

#include "device.h"

namespace nmpc {

namespace {

constexpr int NT = 256;
constexpr int GV = 8;                   // lanes that share one column of J in the J^T products (residual, right-hand side)
constexpr int GK = 4;                   // lanes that share one entry of K in the condensed assembly
constexpr double INF = __builtin_huge_val();

struct LamDiff { const double* p; const double* m; __device__ __forceinline__ double operator[](int i) const { return p[i] - m[i]; } };

// ------------------------------------------------------------------------------------------------------------
// a2: one thread per Jacobian row / per variable / per Hessian entry
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(NT) model_eval_kernel(DevModel M, const double* __restrict__ y, const double* __restrict__ wp,
                                                        const double* __restrict__ wm, const double* __restrict__ lam_in,
                                                        double* __restrict__ c_out, double* __restrict__ gradf,
                                                        double* __restrict__ Jval, double* __restrict__ Wval) {
    const ModelDesc& D = M.desc;
    const int nx = D.nx, nv = D.nv;
    const int hc = hess_count(D);
    const int64_t nW = (int64_t)D.N * hc;
    const int64_t idx = blockIdx.x * (int64_t)NT + threadIdx.x;
    if (idx >= M.m_dyn && idx < M.m) {                           // general linear row: c = G_r y, constant Jacobian row
        if (!c_out && !Jval) return;
        const double* gv = M.g_val - M.J_ptr[M.m_dyn];
        double acc = 0.0;
        for (int64_t p = M.J_ptr[idx]; p < M.J_ptr[idx + 1]; ++p) { const double v = gv[p]; acc += v * y[M.J_idx[p]]; if (Jval) Jval[p] = v; }
        if (c_out) c_out[idx] = acc;
    } else if (idx < M.m) {                                      // constraint row (k, c): h and its Jacobian row
        if (!c_out && !Jval) return;
        const int k = (int)(idx / nx), c = (int)(idx - (int64_t)k * nx);
        const double* x = y + (int64_t)k * nv;
        const double* u = x + nx;
        int64_t pos = M.J_ptr[idx];
        double xprev;
        if (k > 0) { xprev = y[(int64_t)(k - 1) * nv + c]; if (Jval) Jval[pos] = -1.0; ++pos; }
        else xprev = M.x0[c];
        const double F = model_row(D, c, x, u, [&](int, double v) { if (Jval) Jval[pos] = v; ++pos; });
        if (c_out) c_out[idx] = x[c] - xprev - D.dt * F;
    } else if (idx < M.m + M.n) {                                // gradient entry
        if (!gradf) return;
        const int64_t v = idx - M.m;
        const int k = (int)(v / nv), a = (int)(v - (int64_t)k * nv);
        const double* x = y + (int64_t)k * nv;
        gradf[v] = cost_grad(D, a, x, x + nx, M.ref + (int64_t)k * D.nr);
    } else if (idx < M.m + M.n + nW) {                           // Lagrangian Hessian entry, lam = w+ - w-
        if (!Wval) return;
        const int64_t q = idx - M.m - M.n;
        const int k = (int)(q / hc), e = (int)(q - (int64_t)k * hc);
        const double* x = y + (int64_t)k * nv;
        const int64_t r0 = (int64_t)k * nx;
        if (lam_in) { Wval[q] = hess_val(D, e, x, x + nx, lam_in + r0); return; }
        LamDiff lam{wp + r0, wm + r0};                           // lam = w+ - w- formed on the fly
        Wval[q] = hess_val(D, e, x, x + nx, lam);
    }
}

// ------------------------------------------------------------------------------------------------------------
// a3: K = W + diag(Sigma_x + eta) + J^T diag(q) J on the fixed pattern, one thread per K entry (gather form)
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(NT) assemble_K_kernel(DevModel M, const double* __restrict__ Jval, const double* __restrict__ Wval,
                                                        const double* __restrict__ sigx, const double* __restrict__ q,
                                                        double eta, double* __restrict__ Kval) {
    const int64_t gtid = blockIdx.x * (int64_t)NT + threadIdx.x;
    const int64_t e = gtid / GK;                         // GK lanes per K entry walk its triple list, fixed butterfly order
    const int gl = (int)(gtid % GK);
    const bool valid = e < M.nnzK;
    double acc = 0.0;
    if (valid) {
#pragma unroll 4
        for (int64_t p = M.trip_ptr[e] + gl; p < M.trip_ptr[e + 1]; p += GK)
            acc += Jval[M.trip_a[p]] * q[M.trip_r[p]] * Jval[M.trip_b[p]];
    }
#pragma unroll
    for (int o = 1; o < GK; o <<= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (!valid || gl != 0) return;
    const int wi = M.k_w[e], di = M.k_diag[e];
    if (wi >= 0) acc += Wval[wi];
    if (di >= 0) acc += sigx[di] + eta;
    Kval[e] = acc;
}

// y = (K + eta I) x from the full symmetric CSR (ptr/idx index the lower-pattern value array through src)
__global__ void __launch_bounds__(NT) kkt_multiply_kernel(int64_t n, const int64_t* __restrict__ ptr, const int32_t* __restrict__ idx,
                                                          const int32_t* __restrict__ src, const double* __restrict__ Kval,
                                                          double eta, const double* __restrict__ x, double* __restrict__ y) {
    const int64_t i = blockIdx.x * (int64_t)NT + threadIdx.x;
    if (i >= n) return;
    double acc = eta * x[i];
    for (int64_t p = ptr[i]; p < ptr[i + 1]; ++p) acc += Kval[src[p]] * x[idx[p]];
    y[i] = acc;
}

// ------------------------------------------------------------------------------------------------------------
// block reductions (fixed tree)
// ------------------------------------------------------------------------------------------------------------
template <int NV>
struct Red { double v[NV]; };

// op codes per slot: 0 = max, 1 = min, 2 = sum
template <int NV>
__device__ __forceinline__ void block_reduce(Red<NV>& a, const int* ops, double* out /* NV */) {
    __shared__ double sh[NV][NT / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < NV; ++k) {
        double v = a.v[k];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const double w = __shfl_xor_sync(0xffffffffu, v, o);
            v = ops[k] == 0 ? fmax(v, w) : (ops[k] == 1 ? fmin(v, w) : v + w);
        }
        if (lane == 0) sh[k][warp] = v;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int k = 0; k < NV; ++k) {
            double v = sh[k][0];
            for (int w2 = 1; w2 < NT / 32; ++w2) v = ops[k] == 0 ? fmax(v, sh[k][w2]) : (ops[k] == 1 ? fmin(v, sh[k][w2]) : v + sh[k][w2]);
            out[k] = v;
        }
    }
}

// The block whose ticket is the last one finishes the reduction over the per-block partials (fixed order over the blocks, so the
// result does not depend on which block that is) -- saves the one-block finalize launch.  Tickets live in scal[12..14].
__device__ __forceinline__ bool last_block_arrives(double* ticket_slot) {
    __shared__ int s_last;
    unsigned* ticket = reinterpret_cast<unsigned*>(ticket_slot);
    __syncthreads();                                     // thread 0 has written this block's partials (block_reduce)
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned t = atomicAdd(ticket, 1u);
        s_last = (t == gridDim.x - 1);
        if (s_last) { *ticket = 0u; __threadfence(); }
    }
    __syncthreads();
    return s_last != 0;
}

// ------------------------------------------------------------------------------------------------------------
// S1 cold start: push y0 into the interior, slacks from c, multipliers mu0/(.)
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(NT) cold_y_kernel(DevModel M, IpmVectors V, const double* __restrict__ u_init, int use_y0,
                                                    double kp, double mu0) {
    const int64_t i = blockIdx.x * (int64_t)NT + threadIdx.x;
    if (i >= M.n) return;
    const int nv = M.desc.nv, nx = M.desc.nx;
    const int a = (int)(i % nv);
    double y = use_y0 ? V.y[i] : (a < nx ? M.x0[a] : u_init[a - nx]);
    const double lb = M.lb[i], ub = M.ub[i];
    const bool hasL = lb > -INF, hasU = ub < INF;
    double pL = kp * fmax(1.0, fabs(lb)), pU = kp * fmax(1.0, fabs(ub));
    if (hasL && hasU) { pL = fmin(pL, kp * (ub - lb)); pU = fmin(pU, kp * (ub - lb)); }
    if (hasL) y = fmax(y, lb + pL);
    if (hasU) y = fmin(y, ub - pU);
    V.y[i] = y;
    V.zL[i] = hasL ? mu0 / (y - lb) : 0.0;
    V.zU[i] = hasU ? mu0 / (ub - y) : 0.0;
}

__global__ void __launch_bounds__(NT) cold_s_kernel(DevModel M, IpmVectors V, double gamma, double s_floor, double mu0) {
    const int64_t r = blockIdx.x * (int64_t)NT + threadIdx.x;
    if (r >= M.m) return;
    (void)gamma;                                         // the tube is part of the row interval [cl, cu] (api.cu)
    const double c = V.c[r], cl = M.cl[r], cu = M.cu[r];
    const bool hasU = cu < INF, hasL = cl > -INF;
    const double sp = hasU ? fmax(cu - c, s_floor) : 1.0, sm = hasL ? fmax(c - cl, s_floor) : 1.0;
    V.sp[r] = sp; V.sm[r] = sm; V.wp[r] = hasU ? mu0 / sp : 0.0; V.wm[r] = hasL ? mu0 / sm : 0.0;
}

__global__ void __launch_bounds__(NT) warm_push_kernel(DevModel M, IpmVectors V, double wpush) {
    const int64_t i = blockIdx.x * (int64_t)NT + threadIdx.x;
    if (i >= M.n) return;
    double y = V.y[i];
    const double lb = M.lb[i], ub = M.ub[i];
    if (lb > -INF) y = fmax(y, lb + wpush);
    if (ub < INF) y = fmin(y, ub - wpush);
    V.y[i] = y;
}

// ------------------------------------------------------------------------------------------------------------
// S2: residuals of the smoothed KKT system (Eq. 9) and the ingredients of E_mu (Eq. 27/28)
//   partial[b][0..6] = max|r_d|, max|r_p+|, max|r_p-|, max comp product, min comp product, sum multipliers, #non-finite
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(NT) residual_kernel(DevModel M, IpmVectors V, double gamma) {
    (void)gamma;                                         // part of the row intervals [cl, cu]
    Red<7> a;
    a.v[0] = a.v[1] = a.v[2] = 0.0; a.v[3] = -INF; a.v[4] = INF; a.v[5] = 0.0; a.v[6] = 0.0;
    // variables: GV lanes share one column of J (the input columns hold 2 nx entries), fixed butterfly order
    const int64_t gthreads = (int64_t)gridDim.x * NT, gtid = blockIdx.x * (int64_t)NT + threadIdx.x;
    const int gl = (int)(gtid % GV);
    for (int64_t i0 = 0; i0 < M.n; i0 += gthreads / GV) {
        const int64_t i = i0 + gtid / GV;
        const bool valid = i < M.n;
        double jt = 0.0;
        if (valid) {
#pragma unroll 4
            for (int64_t p = M.jt_ptr[i] + gl; p < M.jt_ptr[i + 1]; p += GV) { const int r = M.jt_row[p]; jt += V.Jval[M.jt_idx[p]] * (V.wp[r] - V.wm[r]); }
        }
#pragma unroll
        for (int o = 1; o < GV; o <<= 1) jt += __shfl_xor_sync(0xffffffffu, jt, o);
        if (valid && gl == 0) {
            const double lb = M.lb[i], ub = M.ub[i], y = V.y[i];
            const bool hasL = lb > -INF, hasU = ub < INF;
            const double zL = hasL ? V.zL[i] : 0.0, zU = hasU ? V.zU[i] : 0.0;
            const double rd = V.gradf[i] + jt - zL + zU;
            a.v[0] = fmax(a.v[0], fabs(rd));
            if (!isfinite(rd) || !isfinite(y)) a.v[6] += 1.0;
            if (hasL) { const double cp = (y - lb) * zL; a.v[3] = fmax(a.v[3], cp); a.v[4] = fmin(a.v[4], cp); a.v[5] += zL; }
            if (hasU) { const double cp = (ub - y) * zU; a.v[3] = fmax(a.v[3], cp); a.v[4] = fmin(a.v[4], cp); a.v[5] += zU; }
        }
    }
    for (int64_t r = gtid; r < M.m; r += gthreads) {
        const double c = V.c[r], sp = V.sp[r], sm = V.sm[r], wp = V.wp[r], wm = V.wm[r];
        const double cl = M.cl[r], cu = M.cu[r];
        const bool hasU = cu < INF, hasL = cl > -INF;     // a row side without a bound: s = 1, w = 0, out of every formula
        const double rpp = hasU ? c - cu + sp : 0.0, rpm = hasL ? -c + cl + sm : 0.0;
        V.r_pp[r] = rpp; V.r_pm[r] = rpm;
        a.v[1] = fmax(a.v[1], fabs(rpp)); a.v[2] = fmax(a.v[2], fabs(rpm));
        if (!isfinite(rpp) || !isfinite(rpm)) a.v[6] += 1.0;
        if (hasU) { const double c1 = sp * wp; a.v[3] = fmax(a.v[3], c1); a.v[4] = fmin(a.v[4], c1); a.v[5] += wp; }
        if (hasL) { const double c2 = sm * wm; a.v[3] = fmax(a.v[3], c2); a.v[4] = fmin(a.v[4], c2); a.v[5] += wm; }
    }
    const int ops[7] = {0, 0, 0, 0, 1, 2, 2};
    block_reduce<7>(a, ops, V.partial + (int64_t)blockIdx.x * 8);
    if (!last_block_arrives(V.scal + 12)) return;
    a.v[0] = a.v[1] = a.v[2] = 0.0; a.v[3] = -INF; a.v[4] = INF; a.v[5] = 0.0; a.v[6] = 0.0;
    for (int b = threadIdx.x; b < (int)gridDim.x; b += NT) {
        const double* p = V.partial + (int64_t)b * 8;
        a.v[0] = fmax(a.v[0], __ldcg(p)); a.v[1] = fmax(a.v[1], __ldcg(p + 1)); a.v[2] = fmax(a.v[2], __ldcg(p + 2));
        a.v[3] = fmax(a.v[3], __ldcg(p + 3)); a.v[4] = fmin(a.v[4], __ldcg(p + 4)); a.v[5] += __ldcg(p + 5); a.v[6] += __ldcg(p + 6);
    }
    block_reduce<7>(a, ops, V.scal);
}

// ------------------------------------------------------------------------------------------------------------
// S6: Sigma, q, t (rows) then Sigma_x and the right-hand side b of Eq. 17 (variables)
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(NT) sigma_rows_kernel(DevModel M, IpmVectors V, double mu, const double* __restrict__ par) {
    if (par) mu = par[0];                                // graph replay: the barrier parameter comes from device memory
    const int64_t r = blockIdx.x * (int64_t)NT + threadIdx.x;
    if (r >= M.m) return;
    const double sp = V.sp[r], sm = V.sm[r];
    const bool hasU = M.cu[r] < INF, hasL = M.cl[r] > -INF;
    const double qp = V.wp[r] / sp, qm = V.wm[r] / sm;   // 0 for a side without a bound (w = 0, s = 1)
    V.q[r] = qp + qm;
    V.t[r] = qp * V.r_pp[r] + (hasU ? mu / sp : 0.0) - qm * V.r_pm[r] - (hasL ? mu / sm : 0.0);
}

__global__ void __launch_bounds__(NT) sigma_vars_kernel(DevModel M, IpmVectors V, double mu, const double* __restrict__ par) {
    if (par) mu = par[0];
    const int64_t gtid = blockIdx.x * (int64_t)NT + threadIdx.x;
    const int64_t i = gtid / GV;                         // GV lanes per variable for the J^T t product
    const int gl = (int)(gtid % GV);
    const bool valid = i < M.n;
    double jt = 0.0;
    if (valid) {
#pragma unroll 4
        for (int64_t p = M.jt_ptr[i] + gl; p < M.jt_ptr[i + 1]; p += GV) jt += V.Jval[M.jt_idx[p]] * V.t[M.jt_row[p]];
    }
#pragma unroll
    for (int o = 1; o < GV; o <<= 1) jt += __shfl_xor_sync(0xffffffffu, jt, o);
    if (!valid || gl != 0) return;
    const double lb = M.lb[i], ub = M.ub[i], y = V.y[i];
    const bool hasL = lb > -INF, hasU = ub < INF;
    const double dL = hasL ? y - lb : 1.0, dU = hasU ? ub - y : 1.0;
    V.sigx[i] = (hasL ? V.zL[i] / dL : 0.0) + (hasU ? V.zU[i] / dU : 0.0);
    V.b[i] = -(V.gradf[i] - (hasL ? mu / dL : 0.0) + (hasU ? mu / dU : 0.0) + jt);
}

// ------------------------------------------------------------------------------------------------------------
// S8 + S9: eliminated directions (Eq. 10/14) and fraction-to-the-boundary step lengths
//   partial[b][0..1] = min primal step, min dual step
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ double max_step(double v, double dv, double tau) { return dv < 0.0 ? fmin(1.0, -tau * v / dv) : 1.0; }

__global__ void __launch_bounds__(NT) step_kernel(DevModel M, IpmVectors V, double mu, double tau, const double* __restrict__ par) {
    if (par) { mu = par[0]; tau = par[1]; }
    Red<2> a; a.v[0] = 1.0; a.v[1] = 1.0;
    const int64_t total = M.n + M.m;
    for (int64_t idx = blockIdx.x * (int64_t)NT + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * NT) {
        if (idx < M.n) {
            const int64_t i = idx;
            const double lb = M.lb[i], ub = M.ub[i], y = V.y[i], dy = V.dy[i];
            const bool hasL = lb > -INF, hasU = ub < INF;
            double dzL = 0.0, dzU = 0.0;
            if (hasL) {
                const double dL = y - lb, zL = V.zL[i];
                dzL = -(zL - mu / dL) - zL / dL * dy;
                a.v[0] = fmin(a.v[0], max_step(dL, dy, tau)); a.v[1] = fmin(a.v[1], max_step(zL, dzL, tau));
            }
            if (hasU) {
                const double dU = ub - y, zU = V.zU[i];
                dzU = -(zU - mu / dU) + zU / dU * dy;
                a.v[0] = fmin(a.v[0], max_step(dU, -dy, tau)); a.v[1] = fmin(a.v[1], max_step(zU, dzU, tau));
            }
            V.dzL[i] = dzL; V.dzU[i] = dzU;
        } else {
            const int64_t r = idx - M.n;
            double jdy = 0.0;
            for (int64_t p = M.J_ptr[r]; p < M.J_ptr[r + 1]; ++p) jdy += V.Jval[p] * V.dy[M.J_idx[p]];
            const double sp = V.sp[r], sm = V.sm[r], wp = V.wp[r], wm = V.wm[r];
            const bool hasU = M.cu[r] < INF, hasL = M.cl[r] > -INF;
            const double dsp = hasU ? -V.r_pp[r] - jdy : 0.0, dsm = hasL ? -V.r_pm[r] + jdy : 0.0;
            const double dwp = hasU ? -(wp - mu / sp) - wp / sp * dsp : 0.0, dwm = hasL ? -(wm - mu / sm) - wm / sm * dsm : 0.0;
            V.dsp[r] = dsp; V.dsm[r] = dsm; V.dwp[r] = dwp; V.dwm[r] = dwm;
            a.v[0] = fmin(a.v[0], fmin(max_step(sp, dsp, tau), max_step(sm, dsm, tau)));
            a.v[1] = fmin(a.v[1], fmin(max_step(wp, dwp, tau), max_step(wm, dwm, tau)));
        }
    }
    const int ops[2] = {1, 1};
    block_reduce<2>(a, ops, V.partial + (int64_t)blockIdx.x * 8);
    if (!last_block_arrives(V.scal + 13)) return;
    a.v[0] = 1.0; a.v[1] = 1.0;
    for (int b = threadIdx.x; b < (int)gridDim.x; b += NT) { a.v[0] = fmin(a.v[0], __ldcg(V.partial + (int64_t)b * 8)); a.v[1] = fmin(a.v[1], __ldcg(V.partial + (int64_t)b * 8 + 1)); }
    block_reduce<2>(a, ops, V.scal + 7);
}

// S10: Eq. (26) with the step lengths read from device memory
__global__ void __launch_bounds__(NT) update_kernel(DevModel M, IpmVectors V, const int32_t* __restrict__ fail_col) {
    if (fail_col && *fail_col != INT_MAX) return;        // the factorization behind this step met a bad pivot: keep the iterate
    const double apr = V.scal[7], adu = V.scal[8];
    const int64_t idx = blockIdx.x * (int64_t)NT + threadIdx.x;
    if (idx < M.n) {
        V.y[idx] += apr * V.dy[idx]; V.zL[idx] += adu * V.dzL[idx]; V.zU[idx] += adu * V.dzU[idx];
    } else if (idx < M.n + M.m) {
        const int64_t r = idx - M.n;
        V.sp[r] += apr * V.dsp[r]; V.sm[r] += apr * V.dsm[r]; V.wp[r] += adu * V.dwp[r]; V.wm[r] += adu * V.dwm[r];
    }
}

__global__ void __launch_bounds__(NT) objective_kernel(DevModel M, IpmVectors V) {
    Red<1> a; a.v[0] = 0.0;
    const int nv = M.desc.nv, nx = M.desc.nx;
    for (int64_t i = blockIdx.x * (int64_t)NT + threadIdx.x; i < M.n; i += (int64_t)gridDim.x * NT) {
        const int k = (int)(i / nv), e = (int)(i - (int64_t)k * nv);
        const double* x = V.y + (int64_t)k * nv;
        a.v[0] += cost_value_entry(M.desc, e, x, x + nx, M.ref + (int64_t)k * M.desc.nr);
    }
    const int ops[1] = {2};
    block_reduce<1>(a, ops, V.partial + (int64_t)blockIdx.x * 8);
    if (!last_block_arrives(V.scal + 14)) return;
    a.v[0] = 0.0;
    for (int b = threadIdx.x; b < (int)gridDim.x; b += NT) a.v[0] += __ldcg(V.partial + (int64_t)b * 8);
    block_reduce<1>(a, ops, V.scal + 9);
}

// ------------------------------------------------------------------------------------------------------------
// Iterative refinement of the Newton direction (options.refine_steps): residual of the FIRST block row of the un-condensed
// system Eq. (10) at the current (dy, dw+-, dz) -- r_d expanded, so the multipliers enter as w + dw, z + dz:
//   rho = grad f + J^T((w+ + dw+) - (w- + dw-)) - (zL + dzL) + (zU + dzU) + (W + eta I) dy;      V.rho <- -rho
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(NT) refine_residual_kernel(DevModel M, IpmVectors V, double eta, const int32_t* __restrict__ fail_col) {
    if (fail_col && *fail_col != INT_MAX) return;
    const int64_t gtid = blockIdx.x * (int64_t)NT + threadIdx.x;
    const int64_t i = gtid / GV;
    const int gl = (int)(gtid % GV);
    const bool valid = i < M.n;
    double acc = 0.0;
    if (valid) {
#pragma unroll 4
        for (int64_t p = M.jt_ptr[i] + gl; p < M.jt_ptr[i + 1]; p += GV) {
            const int r = M.jt_row[p];
            acc += V.Jval[M.jt_idx[p]] * ((V.wp[r] + V.dwp[r]) - (V.wm[r] + V.dwm[r]));
        }
        for (int64_t q = M.wf_ptr[i] + gl; q < M.wf_ptr[i + 1]; q += GV) acc += V.Wval[M.wf_src[q]] * V.dy[M.wf_idx[q]];
    }
#pragma unroll
    for (int o = 1; o < GV; o <<= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (!valid || gl != 0) return;
    const bool hasL = M.lb[i] > -INF, hasU = M.ub[i] < INF;
    const double zl = hasL ? V.zL[i] + V.dzL[i] : 0.0, zu = hasU ? V.zU[i] + V.dzU[i] : 0.0;
    V.rho[i] = -(V.gradf[i] + acc - zl + zu + eta * V.dy[i]);
}

__global__ void __launch_bounds__(NT) add_correction_kernel(DevModel M, IpmVectors V, const int32_t* __restrict__ fail_col) {
    if (fail_col && *fail_col != INT_MAX) return;
    const int64_t i = blockIdx.x * (int64_t)NT + threadIdx.x;
    if (i < M.n) V.dy[i] += V.rho[i];
}

// ------------------------------------------------------------------------------------------------------------
// Filter line search of ref. [17] (options.globalization): the two measures of a trial point (y + alpha dy, s + alpha ds)
//   theta = |c - cu + s+|_1 + |-c + cl + s-|_1 (row sides with a bound),   phi_mu = f - mu (sum ln s+ + sum ln s- + sum ln(y - lb) + sum ln(ub - y))
// reduced with the fixed tree; scal[0..4] = theta, sum of logs, f, #arguments <= 0, grad phi_mu^T d (alpha = 0 call only)
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(NT) trial_point_kernel(DevModel M, IpmVectors V, double alpha) {
    const int64_t i = blockIdx.x * (int64_t)NT + threadIdx.x;
    if (i < M.n) V.yt[i] = alpha != 0.0 ? V.y[i] + alpha * V.dy[i] : V.y[i];
}

__global__ void __launch_bounds__(NT) merit_kernel(DevModel M, IpmVectors V, double alpha, double mu, double gamma, int with_grad) {
    (void)gamma;                                         // part of the row intervals [cl, cu]
    Red<5> a;
#pragma unroll
    for (int k = 0; k < 5; ++k) a.v[k] = 0.0;
    const bool step = alpha != 0.0;
    const int nv = M.desc.nv, nx = M.desc.nx;
    const int64_t total = M.n + M.m;
    for (int64_t idx = blockIdx.x * (int64_t)NT + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * NT) {
        if (idx < M.n) {
            const int64_t i = idx;
            const double lb = M.lb[i], ub = M.ub[i], yt = V.yt[i];
            const int k = (int)(i / nv), e = (int)(i - (int64_t)k * nv);
            const double* x = V.yt + (int64_t)k * nv;
            a.v[2] += cost_value_entry(M.desc, e, x, x + nx, M.ref + (int64_t)k * M.desc.nr);
            if (lb > -INF) { const double d = yt - lb; if (d > 0.0) a.v[1] += log(d); else a.v[3] += 1.0; }
            if (ub < INF) { const double d = ub - yt; if (d > 0.0) a.v[1] += log(d); else a.v[3] += 1.0; }
            if (with_grad) {
                const double dy = V.dy[i], y = V.y[i];
                double g = V.gradf[i] * dy;
                if (lb > -INF) g -= mu * (dy / (y - lb));
                if (ub < INF) g += mu * (dy / (ub - y));
                a.v[4] += g;
            }
        } else {
            const int64_t r = idx - M.n;
            const double c = V.ct[r];
            const double sp = step ? V.sp[r] + alpha * V.dsp[r] : V.sp[r], sm = step ? V.sm[r] + alpha * V.dsm[r] : V.sm[r];
            const double cl = M.cl[r], cu = M.cu[r];
            const bool hasU = cu < INF, hasL = cl > -INF;
            a.v[0] += (hasU ? fabs(c - cu + sp) : 0.0) + (hasL ? fabs(-c + cl + sm) : 0.0);
            if (hasU) { if (sp > 0.0) a.v[1] += log(sp); else a.v[3] += 1.0; }
            if (hasL) { if (sm > 0.0) a.v[1] += log(sm); else a.v[3] += 1.0; }
            if (with_grad) a.v[4] -= mu * (V.dsp[r] / V.sp[r] + V.dsm[r] / V.sm[r]);   // 0 / 1 for a side without a bound
        }
    }
    const int ops[5] = {2, 2, 2, 2, 2};
    block_reduce<5>(a, ops, V.partial + (int64_t)blockIdx.x * 8);
    if (!last_block_arrives(V.scal + 15)) return;
#pragma unroll
    for (int k = 0; k < 5; ++k) a.v[k] = 0.0;
    for (int b = threadIdx.x; b < (int)gridDim.x; b += NT) {
        const double* p = V.partial + (int64_t)b * 8;
#pragma unroll
        for (int k = 0; k < 5; ++k) a.v[k] += __ldcg(p + k);
    }
    block_reduce<5>(a, ops, V.scal);
}

inline unsigned blocks_for(int64_t work) { return (unsigned)((work + NT - 1) / NT); }
inline int red_blocks(int64_t work) { return (int)std::min<int64_t>(RED_BLOCKS, (work + NT - 1) / NT); }

}  // namespace

void launch_model_eval(const DevModel& M, const double* y, const double* wp, const double* wm, const double* lam,
                       double* c, double* gradf, double* Jval, double* Wval, cudaStream_t st) {
    const int64_t work = M.m + M.n + (int64_t)M.desc.N * hess_count(M.desc);
    model_eval_kernel<<<blocks_for(work), NT, 0, st>>>(M, y, wp, wm, lam, c, gradf, Jval, Wval);
}
void launch_assemble_K(const DevModel& M, const double* Jval, const double* Wval, const double* sigx, const double* q,
                       double eta, double* Kval, cudaStream_t st) {
    assemble_K_kernel<<<blocks_for(M.nnzK * GK), NT, 0, st>>>(M, Jval, Wval, sigx, q, eta, Kval);
}
void launch_kkt_multiply(int64_t n, const int64_t* ptr, const int32_t* idx, const int32_t* src, const double* Kval, double eta,
                         const double* x, double* y, cudaStream_t st) {
    kkt_multiply_kernel<<<blocks_for(n), NT, 0, st>>>(n, ptr, idx, src, Kval, eta, x, y);
}
void launch_cold_init_y(const DevModel& M, const IpmVectors& V, const double* u_init, int use_y0, double kappa_push, double mu0, cudaStream_t st) {
    cold_y_kernel<<<blocks_for(M.n), NT, 0, st>>>(M, V, u_init, use_y0, kappa_push, mu0);
}
void launch_cold_init_s(const DevModel& M, const IpmVectors& V, double gamma, double s_floor, double mu0, cudaStream_t st) {
    cold_s_kernel<<<blocks_for(M.m), NT, 0, st>>>(M, V, gamma, s_floor, mu0);
}
void launch_warm_push(const DevModel& M, const IpmVectors& V, double warm_push, cudaStream_t st) {
    warm_push_kernel<<<blocks_for(M.n), NT, 0, st>>>(M, V, warm_push);
}
void launch_residuals(const DevModel& M, const IpmVectors& V, double gamma, cudaStream_t st) {
    const int nb = red_blocks(M.n * GV + M.m);
    residual_kernel<<<nb, NT, 0, st>>>(M, V, gamma);
}
void launch_sigma_rhs(const DevModel& M, const IpmVectors& V, double mu, const double* par, cudaStream_t st) {
    sigma_rows_kernel<<<blocks_for(M.m), NT, 0, st>>>(M, V, mu, par);
    sigma_vars_kernel<<<blocks_for(M.n * GV), NT, 0, st>>>(M, V, mu, par);
}
void launch_step(const DevModel& M, const IpmVectors& V, double mu, double tau, const double* par, cudaStream_t st) {
    const int nb = red_blocks(M.n + M.m);
    step_kernel<<<nb, NT, 0, st>>>(M, V, mu, tau, par);
}
void launch_update(const DevModel& M, const IpmVectors& V, const int32_t* fail_col, cudaStream_t st) {
    update_kernel<<<blocks_for(M.n + M.m), NT, 0, st>>>(M, V, fail_col);
}
void launch_refine_residual(const DevModel& M, const IpmVectors& V, double eta, const int32_t* fail_col, cudaStream_t st) {
    refine_residual_kernel<<<blocks_for(M.n * GV), NT, 0, st>>>(M, V, eta, fail_col);
}
void launch_add_correction(const DevModel& M, const IpmVectors& V, const int32_t* fail_col, cudaStream_t st) {
    add_correction_kernel<<<blocks_for(M.n), NT, 0, st>>>(M, V, fail_col);
}
void launch_trial_point(const DevModel& M, const IpmVectors& V, double alpha, cudaStream_t st) {
    trial_point_kernel<<<blocks_for(M.n), NT, 0, st>>>(M, V, alpha);
}
void launch_merit(const DevModel& M, const IpmVectors& V, double alpha, double mu, double gamma, int with_grad, cudaStream_t st) {
    merit_kernel<<<red_blocks(M.n + M.m), NT, 0, st>>>(M, V, alpha, mu, gamma, with_grad);
}
void launch_objective(const DevModel& M, const IpmVectors& V, cudaStream_t st) {
    const int nb = red_blocks(M.n);
    objective_kernel<<<nb, NT, 0, st>>>(M, V);
}

}  // namespace nmpc
