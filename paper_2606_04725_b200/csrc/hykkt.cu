// hykkt.cu -- vector kernels of the HyKKT variant of Algorithm 2 ("the system can be reformulated using either
// Lifted-KKT or HyKKT ... a hybrid direct-iterative approach based on an augmented Lagrangian formulation"; reading G21 of
// DESIGN.md section 3).  The equalities h(y) = 0 are kept exact (no gamma tube, no slacks):
//
//     K_g = W + Sigma_x + eta I + gamma_h J^T J            assembled by assemble_K_kernel with q == gamma_h, factored and solved
//                                                           by the same kernels as the lifted K of Eq. (17)
//     S dlam = J K_g^-1 (r1 + gamma_h J^T r2) - r2          conjugate gradients on S = J K_g^-1 J^T, one K_g solve per iteration
//     dy     = K_g^-1 (r1 + gamma_h J^T r2 - J^T dlam),     r1 = -(grad f + J^T lam - mu/(y-lb) + mu/(ub-y)),  r2 = -c
//
// State mapping onto the IPM vectors: lam = V.wp (V.wm == 0, so the model evaluation's lam = w+ - w- is lam), dlam = V.dwp,
// CG residual / direction / S p = V.r_pp / V.r_pm / V.t, V.q == gamma_h, n-vector scratch = V.rho.  The CG scalars (alpha, beta)
// are host scalars: two reductions are read back per CG iteration.  Compiled with -fmad=false like ipm.cu.
#include <climits>

#include "device.h"

namespace nmpc {

namespace {

constexpr int NT = 256;
constexpr int GV = 8;
constexpr double INF = __builtin_huge_val();

template <int NV>
struct Red { double v[NV]; };

template <int NV>
__device__ __forceinline__ void block_reduce(Red<NV>& a, const int* ops, double* out) {     // 0 max, 1 min, 2 sum; fixed tree
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

__device__ __forceinline__ bool last_block_arrives(double* ticket_slot) {
    __shared__ int s_last;
    unsigned* ticket = reinterpret_cast<unsigned*>(ticket_slot);
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned t = atomicAdd(ticket, 1u);
        s_last = (t == gridDim.x - 1);
        if (s_last) { *ticket = 0u; __threadfence(); }
    }
    __syncthreads();
    return s_last != 0;
}

// J^T v for variable i, GV lanes per variable (fixed butterfly order); every lane of the group returns the sum
__device__ __forceinline__ double jt_dot(const DevModel& M, const double* __restrict__ Jval, const double* __restrict__ v, int64_t i, int gl, bool valid) {
    double acc = 0.0;
    if (valid) {
#pragma unroll 4
        for (int64_t p = M.jt_ptr[i] + gl; p < M.jt_ptr[i + 1]; p += GV) acc += Jval[M.jt_idx[p]] * v[M.jt_row[p]];
    }
#pragma unroll
    for (int o = 1; o < GV; o <<= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    return acc;
}

// residuals of the primal-dual system and the ingredients of E_mu, same slots as ipm.cu: residual_kernel
//   scal[0..6] = max|r_d|, max|c|, 0, max comp product, min comp product, |lam|_1 + sum z, #non-finite
__global__ void __launch_bounds__(NT) hk_residual_kernel(DevModel M, IpmVectors V) {
    Red<7> a;
    a.v[0] = a.v[1] = a.v[2] = 0.0; a.v[3] = -INF; a.v[4] = INF; a.v[5] = 0.0; a.v[6] = 0.0;
    const int64_t gthreads = (int64_t)gridDim.x * NT, gtid = blockIdx.x * (int64_t)NT + threadIdx.x;
    const int gl = (int)(gtid % GV);
    for (int64_t i0 = 0; i0 < M.n; i0 += gthreads / GV) {
        const int64_t i = i0 + gtid / GV;
        const bool valid = i < M.n;
        const double jt = jt_dot(M, V.Jval, V.wp, i, gl, valid);
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
        const double c = V.c[r], lam = V.wp[r];
        a.v[1] = fmax(a.v[1], fabs(c));
        if (!isfinite(c) || !isfinite(lam)) a.v[6] += 1.0;
        a.v[5] += fabs(lam);
    }
    const int ops[7] = {0, 0, 0, 0, 1, 2, 2};
    block_reduce<7>(a, ops, V.partial + (int64_t)blockIdx.x * 8);
    if (!last_block_arrives(V.scal + 12)) return;
    a.v[0] = a.v[1] = a.v[2] = 0.0; a.v[3] = -INF; a.v[4] = INF; a.v[5] = 0.0; a.v[6] = 0.0;
    for (int b = threadIdx.x; b < (int)gridDim.x; b += NT) {
        const double* p = V.partial + (int64_t)b * 8;
        a.v[0] = fmax(a.v[0], __ldcg(p)); a.v[1] = fmax(a.v[1], __ldcg(p + 1));
        a.v[3] = fmax(a.v[3], __ldcg(p + 3)); a.v[4] = fmin(a.v[4], __ldcg(p + 4)); a.v[5] += __ldcg(p + 5); a.v[6] += __ldcg(p + 6);
    }
    block_reduce<7>(a, ops, V.scal);
}

// Sigma_x and the right-hand side b_g = r1 + gamma_h J^T r2 = -(grad f + J^T lam - mu/(y-lb) + mu/(ub-y)) - gamma_h J^T c
__global__ void __launch_bounds__(NT) hk_rhs_kernel(DevModel M, IpmVectors V, double mu, double gamma_h) {
    const int64_t gtid = blockIdx.x * (int64_t)NT + threadIdx.x;
    const int64_t i = gtid / GV;
    const int gl = (int)(gtid % GV);
    const bool valid = i < M.n;
    const double jl = jt_dot(M, V.Jval, V.wp, i, gl, valid), jc = jt_dot(M, V.Jval, V.c, i, gl, valid);
    if (!valid || gl != 0) return;
    const double lb = M.lb[i], ub = M.ub[i], y = V.y[i];
    const bool hasL = lb > -INF, hasU = ub < INF;
    const double dL = hasL ? y - lb : 1.0, dU = hasU ? ub - y : 1.0;
    V.sigx[i] = (hasL ? V.zL[i] / dL : 0.0) + (hasU ? V.zU[i] / dU : 0.0);
    const double r1 = -(V.gradf[i] + jl - (hasL ? mu / dL : 0.0) + (hasU ? mu / dU : 0.0));
    V.b[i] = r1 - gamma_h * jc;
}

// out_n = a_n - J^T v_m   (a may be null: out = -J^T v ... used as out = J^T v with sign = +1)
__global__ void __launch_bounds__(NT) hk_jt_kernel(DevModel M, const double* __restrict__ Jval, const double* __restrict__ v,
                                                   const double* __restrict__ a, double sign, double* __restrict__ out) {
    const int64_t gtid = blockIdx.x * (int64_t)NT + threadIdx.x;
    const int64_t i = gtid / GV;
    const int gl = (int)(gtid % GV);
    const bool valid = i < M.n;
    const double jt = jt_dot(M, Jval, v, i, gl, valid);
    if (valid && gl == 0) out[i] = (a ? a[i] : 0.0) + sign * jt;
}

// out_m = J u_n + shift_m (shift may be null); scal[0] = p . out (p may be null), scal[1] = out . out
__global__ void __launch_bounds__(NT) hk_j_kernel(DevModel M, IpmVectors V, const double* __restrict__ u, const double* __restrict__ shift,
                                                  const double* __restrict__ p, double* __restrict__ out) {
    Red<2> a; a.v[0] = 0.0; a.v[1] = 0.0;
    for (int64_t r = blockIdx.x * (int64_t)NT + threadIdx.x; r < M.m; r += (int64_t)gridDim.x * NT) {
        double acc = 0.0;
        for (int64_t q = M.J_ptr[r]; q < M.J_ptr[r + 1]; ++q) acc += V.Jval[q] * u[M.J_idx[q]];
        if (shift) acc += shift[r];
        out[r] = acc;
        if (p) a.v[0] += p[r] * acc;
        a.v[1] += acc * acc;
    }
    const int ops[2] = {2, 2};
    block_reduce<2>(a, ops, V.partial + (int64_t)blockIdx.x * 8);
    if (!last_block_arrives(V.scal + 13)) return;
    a.v[0] = 0.0; a.v[1] = 0.0;
    for (int b = threadIdx.x; b < (int)gridDim.x; b += NT) { a.v[0] += __ldcg(V.partial + (int64_t)b * 8); a.v[1] += __ldcg(V.partial + (int64_t)b * 8 + 1); }
    block_reduce<2>(a, ops, V.scal);
}

// CG update: x += alpha p, r -= alpha Sp, scal[1] = r . r
__global__ void __launch_bounds__(NT) hk_cg_update_kernel(DevModel M, IpmVectors V, double alpha, double* __restrict__ x, double* __restrict__ r,
                                                          const double* __restrict__ p, const double* __restrict__ Sp) {
    Red<2> a; a.v[0] = 0.0; a.v[1] = 0.0;
    for (int64_t k = blockIdx.x * (int64_t)NT + threadIdx.x; k < M.m; k += (int64_t)gridDim.x * NT) {
        x[k] += alpha * p[k];
        const double rk = r[k] - alpha * Sp[k];
        r[k] = rk;
        a.v[1] += rk * rk;
    }
    const int ops[2] = {2, 2};
    block_reduce<2>(a, ops, V.partial + (int64_t)blockIdx.x * 8);
    if (!last_block_arrives(V.scal + 13)) return;
    a.v[0] = 0.0; a.v[1] = 0.0;
    for (int b = threadIdx.x; b < (int)gridDim.x; b += NT) a.v[1] += __ldcg(V.partial + (int64_t)b * 8 + 1);
    block_reduce<2>(a, ops, V.scal);
}

// p = r + beta p   (beta = 0: p = r);  x = 0 when init
__global__ void __launch_bounds__(NT) hk_cg_dir_kernel(DevModel M, double beta, const double* __restrict__ r, double* __restrict__ p, double* __restrict__ x, int init) {
    const int64_t k = blockIdx.x * (int64_t)NT + threadIdx.x;
    if (k >= M.m) return;
    p[k] = init ? r[k] : r[k] + beta * p[k];
    if (init) x[k] = 0.0;
}

__device__ __forceinline__ double max_step(double v, double dv, double tau) { return dv < 0.0 ? fmin(1.0, -tau * v / dv) : 1.0; }

// eliminated bound-multiplier directions and the fraction-to-the-boundary step lengths: scal[7] = alpha_pr, scal[8] = alpha_du
__global__ void __launch_bounds__(NT) hk_step_kernel(DevModel M, IpmVectors V, double mu, double tau) {
    Red<2> a; a.v[0] = 1.0; a.v[1] = 1.0;
    for (int64_t i = blockIdx.x * (int64_t)NT + threadIdx.x; i < M.n; i += (int64_t)gridDim.x * NT) {
        const double lb = M.lb[i], ub = M.ub[i], y = V.y[i], dy = V.dy[i];
        double dzL = 0.0, dzU = 0.0;
        if (lb > -INF) {
            const double dL = y - lb, zL = V.zL[i];
            dzL = -(zL - mu / dL) - zL / dL * dy;
            a.v[0] = fmin(a.v[0], max_step(dL, dy, tau)); a.v[1] = fmin(a.v[1], max_step(zL, dzL, tau));
        }
        if (ub < INF) {
            const double dU = ub - y, zU = V.zU[i];
            dzU = -(zU - mu / dU) + zU / dU * dy;
            a.v[0] = fmin(a.v[0], max_step(dU, -dy, tau)); a.v[1] = fmin(a.v[1], max_step(zU, dzU, tau));
        }
        V.dzL[i] = dzL; V.dzU[i] = dzU;
    }
    const int ops[2] = {1, 1};
    block_reduce<2>(a, ops, V.partial + (int64_t)blockIdx.x * 8);
    if (!last_block_arrives(V.scal + 13)) return;
    a.v[0] = 1.0; a.v[1] = 1.0;
    for (int b = threadIdx.x; b < (int)gridDim.x; b += NT) { a.v[0] = fmin(a.v[0], __ldcg(V.partial + (int64_t)b * 8)); a.v[1] = fmin(a.v[1], __ldcg(V.partial + (int64_t)b * 8 + 1)); }
    block_reduce<2>(a, ops, V.scal + 7);
}

// y += alpha_pr dy, lam += alpha_pr dlam, z += alpha_du dz
__global__ void __launch_bounds__(NT) hk_update_kernel(DevModel M, IpmVectors V) {
    const double apr = V.scal[7], adu = V.scal[8];
    const int64_t idx = blockIdx.x * (int64_t)NT + threadIdx.x;
    if (idx < M.n) { V.y[idx] += apr * V.dy[idx]; V.zL[idx] += adu * V.dzL[idx]; V.zU[idx] += adu * V.dzU[idx]; }
    else if (idx < M.n + M.m) { const int64_t r = idx - M.n; V.wp[r] += apr * V.dwp[r]; }
}

__global__ void __launch_bounds__(NT) hk_fill_kernel(int64_t n, double v, double* __restrict__ out) {
    const int64_t i = blockIdx.x * (int64_t)NT + threadIdx.x;
    if (i < n) out[i] = v;
}

inline unsigned blocks_for(int64_t work) { return (unsigned)((work + NT - 1) / NT); }
inline int red_blocks(int64_t work) { return (int)(work + NT - 1) / NT < RED_BLOCKS ? (int)((work + NT - 1) / NT) : RED_BLOCKS; }

}  // namespace

void launch_hk_residuals(const DevModel& M, const IpmVectors& V, cudaStream_t st) {
    hk_residual_kernel<<<red_blocks(M.n * GV + M.m), NT, 0, st>>>(M, V);
}
void launch_hk_rhs(const DevModel& M, const IpmVectors& V, double mu, double gamma_h, cudaStream_t st) {
    hk_rhs_kernel<<<blocks_for(M.n * GV), NT, 0, st>>>(M, V, mu, gamma_h);
}
void launch_hk_jt(const DevModel& M, const IpmVectors& V, const double* v_m, const double* a_n, double sign, double* out_n, cudaStream_t st) {
    hk_jt_kernel<<<blocks_for(M.n * GV), NT, 0, st>>>(M, V.Jval, v_m, a_n, sign, out_n);
}
void launch_hk_j(const DevModel& M, const IpmVectors& V, const double* u_n, const double* shift_m, const double* p_m, double* out_m, cudaStream_t st) {
    hk_j_kernel<<<red_blocks(M.m), NT, 0, st>>>(M, V, u_n, shift_m, p_m, out_m);
}
void launch_hk_cg_update(const DevModel& M, const IpmVectors& V, double alpha, double* x, double* r, const double* p, const double* Sp, cudaStream_t st) {
    hk_cg_update_kernel<<<red_blocks(M.m), NT, 0, st>>>(M, V, alpha, x, r, p, Sp);
}
void launch_hk_cg_dir(const DevModel& M, double beta, const double* r, double* p, double* x, int init, cudaStream_t st) {
    hk_cg_dir_kernel<<<blocks_for(M.m), NT, 0, st>>>(M, beta, r, p, x, init);
}
void launch_hk_step(const DevModel& M, const IpmVectors& V, double mu, double tau, cudaStream_t st) {
    hk_step_kernel<<<red_blocks(M.n), NT, 0, st>>>(M, V, mu, tau);
}
void launch_hk_update(const DevModel& M, const IpmVectors& V, cudaStream_t st) {
    hk_update_kernel<<<blocks_for(M.n + M.m), NT, 0, st>>>(M, V);
}
void launch_fill(int64_t n, double v, double* out, cudaStream_t st) {
    if (n > 0) hk_fill_kernel<<<blocks_for(n), NT, 0, st>>>(n, v, out);
}

}  // namespace nmpc
