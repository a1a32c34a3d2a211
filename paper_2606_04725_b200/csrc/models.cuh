// models.cuh -- per-stage model and derivative enumerators of the three built-in OCP models (step a2 of the hot
// path: the paper's K_SIMD derivative kernels, re-done as hand-derived per-model CUDA).
//
// Every function is __host__ __device__: the device kernels call them to produce VALUES, the host symbolic
// analysis calls the same enumerators to produce the fixed PATTERN (column of every emitted entry), so the
// value order of J and W can never drift from the analysed pattern.
//
// Transcription (Problem 5, implicit Euler): stage k = 0..N-1 holds v_k = (x_k, u_k),
//   h_k = x_k - x_{k-1} - dt F(x_k, u_k),  x_{-1} = x0 (parameter),   f = sum_k l(x_k, u_k; ref_k).
// J row (k,c) = [ -1 at x_{k-1,c} | e_c - dt dF_c/dx_k | -dt dF_c/du_k ]  (emitted in increasing column order)
// W stage block (lower) = Hess l - dt sum_c lam_{k,c} Hess F_c,  lam = w+ - w-.
//
// Model statements: VdP  BASELINE.json:configs[0];  distillation  Problem (29) PAPER.md:451-473 as read in
// DESIGN.md section 3 (G12) with the vapour composition eliminated;  plate  BASELINE.json:configs[2].
#pragma once
#include <cstdint>

#ifdef __CUDACC__
#define NMPC_HD __host__ __device__ __forceinline__
#else
#define NMPC_HD inline
#endif

namespace nmpc {

enum { MODEL_NONE = 0, MODEL_VDP = 1, MODEL_DISTILL = 2, MODEL_PLATE = 3 };
constexpr int MAX_JROW = 8;      // max entries of one Jacobian row over all models

struct ModelDesc {
    int model, N, nx, nu, nr, nv;
    double dt;
    double p[12];
};

// ------------------------------------------------------------------------------------------------------------
// Van der Pol:  F = (x2, (1 - x1^2) x2 - x1 + u),  l = w_x |x - r|^2 + w_u u^2        p = [w_x, w_u]
// ------------------------------------------------------------------------------------------------------------
template <class Emit>
NMPC_HD double vdp_row(const ModelDesc& M, int c, const double* x, const double* u, Emit emit) {
    const double dt = M.dt;
    if (c == 0) {
        emit(0, 1.0);
        emit(1, -dt);
        return x[1];
    }
    emit(0, -dt * (-2.0 * x[0] * x[1] - 1.0));
    emit(1, 1.0 - dt * (1.0 - x[0] * x[0]));
    emit(2, -dt);
    return (1.0 - x[0] * x[0]) * x[1] - x[0] + u[0];
}

// ------------------------------------------------------------------------------------------------------------
// Binary distillation column, state 0 = condenser, 1..nx-2 trays, nx-1 = reboiler, y(x) = alpha x/(1+(alpha-1)x)
//   p = [alpha, D, F_feed, x_feed, A_c, A_t, A_r, feed_index, u_bar, w_u];   L = u D, V = L + D, S = L + F_feed
// ------------------------------------------------------------------------------------------------------------
NMPC_HD double vle(double al, double x) { return al * x / (1.0 + (al - 1.0) * x); }
NMPC_HD double dvle(double al, double x) { double d = 1.0 + (al - 1.0) * x; return al / (d * d); }
NMPC_HD double d2vle(double al, double x) { double d = 1.0 + (al - 1.0) * x; return -2.0 * al * (al - 1.0) / (d * d * d); }
NMPC_HD double distill_holdup(const ModelDesc& M, int c) { return c == 0 ? M.p[4] : (c == M.nx - 1 ? M.p[6] : M.p[5]); }

template <class Emit>
NMPC_HD double distill_row(const ModelDesc& M, int c, const double* x, const double* u, Emit emit) {
    const double al = M.p[0], D = M.p[1], Ff = M.p[2], xf = M.p[3], Ac = M.p[4], At = M.p[5], Ar = M.p[6];
    const int f = (int)M.p[7], n = M.nx;
    const double dt = M.dt;
    const double L = u[0] * D, V = L + D, S = L + Ff;
    if (c == 0) {                                           // condenser: A_c x0' = V (y1 - x0)
        const double y1 = vle(al, x[1]);
        emit(0, 1.0 + dt * V / Ac);
        emit(1, -dt * V * dvle(al, x[1]) / Ac);
        emit(n, -dt * D * (y1 - x[0]) / Ac);
        return V * (y1 - x[0]) / Ac;
    }
    if (c == n - 1) {                                       // reboiler: A_r x' = S x_{n-2} - (F - D) x_{n-1} - V y_{n-1}
        const double yn = vle(al, x[n - 1]);
        emit(n - 2, -dt * S / Ar);
        emit(n - 1, 1.0 - dt * (-(Ff - D) - V * dvle(al, x[n - 1])) / Ar);
        emit(n, -dt * D * (x[n - 2] - yn) / Ar);
        return (S * x[n - 2] - (Ff - D) * x[n - 1] - V * yn) / Ar;
    }
    // tray c: A_t x' = lin x_{c-1} - lout x_c - V (y_c - y_{c+1}) (+ F x_f on the feed tray)
    const double lin = (c <= f) ? L : S, lout = (c < f) ? L : S;
    const double yc = vle(al, x[c]), yp = vle(al, x[c + 1]);
    emit(c - 1, -dt * lin / At);
    emit(c, 1.0 - dt * (-lout - V * dvle(al, x[c])) / At);
    emit(c + 1, -dt * V * dvle(al, x[c + 1]) / At);
    emit(n, -dt * D * ((x[c - 1] - x[c]) - (yc - yp)) / At);
    double F = (lin * x[c - 1] - lout * x[c] - V * (yc - yp)) / At;
    if (c == f) F += Ff * xf / At;
    return F;
}

// ------------------------------------------------------------------------------------------------------------
// 2-D heated plate, cell c = i*g + j, 5-point Laplacian with insulated edges, radiative loss, edge heaters
//   p = [g, a, kappa_r, T_amb, b, nseg, w_T, w_u];   F_c = a sum_nbr (T_nbr - T_c) - kr (T_c^4 - Tamb^4) + b sum_h u_h
//   heater index of edge e (0: i=0, 1: i=g-1, 2: j=0, 3: j=g-1), segment floor(t*nseg/g) along the edge
// ------------------------------------------------------------------------------------------------------------
template <class Emit>
NMPC_HD double plate_row(const ModelDesc& M, int c, const double* x, const double* u, Emit emit) {
    const int g = (int)M.p[0], nseg = (int)M.p[5], nx = M.nx;
    const double a = M.p[1], kr = M.p[2], Tamb = M.p[3], b = M.p[4], dt = M.dt;
    const int i = c / g, j = c - i * g;
    const double T = x[c];
    double lap = 0.0;
    const int deg = (i > 0) + (j > 0) + (j < g - 1) + (i < g - 1);
    if (i > 0)     { emit(c - g, -dt * a); lap += x[c - g] - T; }
    if (j > 0)     { emit(c - 1, -dt * a); lap += x[c - 1] - T; }
    emit(c, 1.0 - dt * (-(double)deg * a - 4.0 * kr * T * T * T));
    if (j < g - 1) { emit(c + 1, -dt * a); lap += x[c + 1] - T; }
    if (i < g - 1) { emit(c + g, -dt * a); lap += x[c + g] - T; }
    double heat = 0.0;
    if (i == 0)     { int h = 0 * nseg + (j * nseg) / g; emit(nx + h, -dt * b); heat += u[h]; }
    if (i == g - 1) { int h = 1 * nseg + (j * nseg) / g; emit(nx + h, -dt * b); heat += u[h]; }
    if (j == 0)     { int h = 2 * nseg + (i * nseg) / g; emit(nx + h, -dt * b); heat += u[h]; }
    if (j == g - 1) { int h = 3 * nseg + (i * nseg) / g; emit(nx + h, -dt * b); heat += u[h]; }
    const double T2 = T * T, Ta2 = Tamb * Tamb;
    return a * lap - kr * (T2 * T2 - Ta2 * Ta2) + b * heat;
}

// Jacobian row (k-local): emits (local column in [0,nv), value) in increasing column order, returns F_c(x,u).
template <class Emit>
NMPC_HD double model_row(const ModelDesc& M, int c, const double* x, const double* u, Emit emit) {
    switch (M.model) {
        case MODEL_VDP: return vdp_row(M, c, x, u, emit);
        case MODEL_DISTILL: return distill_row(M, c, x, u, emit);
        default: return plate_row(M, c, x, u, emit);
    }
}

// ------------------------------------------------------------------------------------------------------------
// Stage cost gradient entry a in [0,nv):  d l / d v_a
// ------------------------------------------------------------------------------------------------------------
NMPC_HD double cost_grad(const ModelDesc& M, int a, const double* x, const double* u, const double* ref) {
    switch (M.model) {
        case MODEL_VDP:
            return a < 2 ? 2.0 * M.p[0] * (x[a] - ref[a]) : 2.0 * M.p[1] * u[0];
        case MODEL_DISTILL:
            if (a == 0) return 2.0 * (x[0] - ref[0]);
            if (a == M.nx) return 2.0 * M.p[9] * (u[0] - M.p[8]);
            return 0.0;
        default:
            return a < M.nx ? 2.0 * M.p[6] * (x[a] - ref[a]) : 2.0 * M.p[7] * u[a - M.nx];
    }
}

NMPC_HD double cost_value_entry(const ModelDesc& M, int a, const double* x, const double* u, const double* ref) {
    switch (M.model) {
        case MODEL_VDP: { double d = a < 2 ? x[a] - ref[a] : u[0]; return (a < 2 ? M.p[0] : M.p[1]) * d * d; }
        case MODEL_DISTILL:
            if (a == 0) { double d = x[0] - ref[0]; return d * d; }
            if (a == M.nx) { double d = u[0] - M.p[8]; return M.p[9] * d * d; }
            return 0.0;
        default: { double d = a < M.nx ? x[a] - ref[a] : u[a - M.nx]; return (a < M.nx ? M.p[6] : M.p[7]) * d * d; }
    }
}

// ------------------------------------------------------------------------------------------------------------
// Lagrangian Hessian, stage-local lower triangle, enumerated by entry e in [0, hess_count): position (a,b), a>=b,
// sorted by (a,b); value = Hess l - dt sum_c lam_c Hess F_c.
// ------------------------------------------------------------------------------------------------------------
NMPC_HD int hess_count(const ModelDesc& M) {
    switch (M.model) {
        case MODEL_VDP: return 4;
        case MODEL_DISTILL: return 2 * M.nx + 1;
        default: return M.nv;
    }
}

NMPC_HD void hess_pos(const ModelDesc& M, int e, int* a, int* b) {
    switch (M.model) {
        case MODEL_VDP: { const int A[4] = {0, 1, 1, 2}, B[4] = {0, 0, 1, 2}; *a = A[e]; *b = B[e]; return; }
        case MODEL_DISTILL:
            if (e < M.nx) { *a = e; *b = e; }
            else { *a = M.nx; *b = e - M.nx; }
            return;
        default: *a = e; *b = e; return;
    }
}

template <class LamT>
NMPC_HD double hess_val(const ModelDesc& M, int e, const double* x, const double* u, const LamT& lam) {
    const double dt = M.dt;
    switch (M.model) {
        case MODEL_VDP:
            // only F_2 is nonlinear: d2F2/dx1^2 = -2 x2, d2F2/dx1dx2 = -2 x1
            if (e == 0) return 2.0 * M.p[0] - dt * lam[1] * (-2.0 * x[1]);
            if (e == 1) return -dt * lam[1] * (-2.0 * x[0]);
            if (e == 2) return 2.0 * M.p[0];
            return 2.0 * M.p[1];
        case MODEL_DISTILL: {
            const double al = M.p[0], D = M.p[1];
            const int n = M.nx;
            const double V = u[0] * D + D;
            if (e < n) {                    // (j,j): y''_j V ( lam_{j-1}/A_{j-1} - lam_j/A_j ),  j >= 1
                const int j = e;
                double h = (j == 0) ? 2.0 : 0.0;                    // Hess l: (x0 - r)^2
                if (j >= 1) {
                    const double s = lam[j - 1] / distill_holdup(M, j - 1) - lam[j] / distill_holdup(M, j);
                    h -= dt * d2vle(al, x[j]) * V * s;
                }
                return h;
            }
            if (e == 2 * n) return 2.0 * M.p[9];                    // (u,u)
            const int j = e - n;                                    // (u, x_j): every flow has d/du = D
            double s = 0.0;
            if (j + 1 <= n - 1) s += lam[j + 1] / distill_holdup(M, j + 1);              // lin x_{c-1}, c = j+1
            if (j == 0) s -= lam[0] / distill_holdup(M, 0);                              // V (y1 - x0)
            else if (j == n - 1) s -= lam[j] / distill_holdup(M, j) * dvle(al, x[j]);    // -V y_{n-1}
            else s += lam[j] / distill_holdup(M, j) * (-1.0 - dvle(al, x[j]));           // -lout x_j - V y_j
            if (j >= 1) s += lam[j - 1] / distill_holdup(M, j - 1) * dvle(al, x[j]);     // +V y_{c+1}, c = j-1
            return -dt * D * s;
        }
        default:
            if (e < M.nx) return 2.0 * M.p[6] - dt * lam[e] * (-12.0 * M.p[2] * x[e] * x[e]);
            return 2.0 * M.p[7];
    }
}

}  // namespace nmpc
