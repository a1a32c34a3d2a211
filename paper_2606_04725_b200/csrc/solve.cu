// solve.cu -- supernodal triangular solves (step a5, Eq. (22)-(25)) on the factor produced by factor.cu:
// L v = P b (leaves -> root), L^T Omega = v (root -> leaves), dy = P^T Omega.  fp64, fixed summation order.
#include "device.h"

namespace nmpc {

namespace {

constexpr int NT = 256;

// =============================================================================================================
// triangular solves, one CTA per supernode, levels leaves->root (forward) and root->leaves (backward)
// =============================================================================================================
// forward (Eq. 23): t = [x[cols]; 0] + sum_children extend(ctr_child);  L11 y = t1;  t2 -= L21 y;  x[cols] = y; ctr = t2
__global__ void __launch_bounds__(NT) solve_fwd_kernel(DevSym D, const int32_t* __restrict__ sn_list, double* __restrict__ x) {
    extern __shared__ double sm[];
    double* t = sm;                                  // r
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int s = sn_list[blockIdx.x];
    const int c0 = D.sn_start[s], w = D.sn_start[s + 1] - c0;
    const int r = (int)(D.rows_ptr[s + 1] - D.rows_ptr[s]), ld = ld_even(r);
    double (*Ld)[BIG_NB + 1] = reinterpret_cast<double (*)[BIG_NB + 1]>(sm + ((r + 1) & ~1));
    const double* __restrict__ P = D.L + D.panel_ptr[s];
    for (int i = tid; i < r; i += NT) t[i] = (i < w) ? x[c0 + i] : 0.0;
    for (int ci = D.child_ptr[s]; ci < D.child_ptr[s + 1]; ++ci) {
        const int c = D.child_idx[ci];
        const int mc = (int)(D.rel_ptr[c + 1] - D.rel_ptr[c]);
        const double* __restrict__ cc = D.ctr + D.rel_ptr[c];
        const int32_t* __restrict__ rel = D.rel + D.rel_ptr[c];
        __syncthreads();
        for (int a = tid; a < mc; a += NT) t[rel[a]] += cc[a];
    }
    __syncthreads();
    for (int j0 = 0; j0 < w; j0 += BIG_NB) {
        const int nb = min(BIG_NB, w - j0);
        for (int idx = tid; idx < nb * nb; idx += NT) {
            const int i = idx % nb, c = idx / nb;
            if (i >= c) Ld[i][c] = P[(j0 + i) + (int64_t)(j0 + c) * ld];
        }
        __syncthreads();
        if (warp == 0) {                             // one warp: in-block forward substitution, no block barriers
            for (int j = 0; j < nb; ++j) {
                const double v = t[j0 + j] / Ld[j][j];
                __syncwarp();
                if (lane == 0) t[j0 + j] = v;
                for (int i = j + 1 + lane; i < nb; i += 32) t[j0 + i] -= Ld[i][j] * v;
                __syncwarp();
            }
        }
        __syncthreads();
        // rows below the block: t[i] -= sum_k L[i, j0+k] y[k]
        for (int i = j0 + nb + tid; i < r; i += NT) {
            double acc = 0.0;
            const double* __restrict__ Pi = P + i + (int64_t)j0 * ld;
            for (int k = 0; k < nb; ++k) acc = fma(Pi[(int64_t)k * ld], t[j0 + k], acc);
            t[i] -= acc;
        }
        __syncthreads();
    }
    for (int i = tid; i < w; i += NT) x[c0 + i] = t[i];
    double* __restrict__ co = D.ctr + D.rel_ptr[s];
    for (int i = w + tid; i < r; i += NT) co[i - w] = t[i];
}

// backward (Eq. 24): t2 = x[rows below];  L11^T z = y - L21^T t2;  x[cols] = z
__global__ void __launch_bounds__(NT) solve_bwd_kernel(DevSym D, const int32_t* __restrict__ sn_list, double* __restrict__ x) {
    extern __shared__ double sm[];
    double* t = sm;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarp = NT / 32;
    const int s = sn_list[blockIdx.x];
    const int c0 = D.sn_start[s], w = D.sn_start[s + 1] - c0;
    const int r = (int)(D.rows_ptr[s + 1] - D.rows_ptr[s]), ld = ld_even(r);
    double (*Ld)[BIG_NB + 1] = reinterpret_cast<double (*)[BIG_NB + 1]>(sm + ((r + 1) & ~1));
    const double* __restrict__ P = D.L + D.panel_ptr[s];
    const int32_t* __restrict__ rows = D.rows + D.rows_ptr[s];
    for (int i = tid; i < r; i += NT) t[i] = x[rows[i]];
    __syncthreads();
    const int nblk = (w + BIG_NB - 1) / BIG_NB;
    for (int bk = nblk - 1; bk >= 0; --bk) {
        const int j0 = bk * BIG_NB, nb = min(BIG_NB, w - j0);
        for (int idx = tid; idx < nb * nb; idx += NT) {
            const int i = idx % nb, c = idx / nb;
            if (i >= c) Ld[i][c] = P[(j0 + i) + (int64_t)(j0 + c) * ld];
        }
        // t[j] -= sum_{i >= j0+nb} L[i,j] t[i] : one warp per column, lanes over rows (coalesced), fixed shuffle tree
        for (int j = warp; j < nb; j += nwarp) {
            const double* __restrict__ Pj = P + (int64_t)(j0 + j) * ld;
            double acc = 0.0;
            for (int i = j0 + nb + lane; i < r; i += 32) acc = fma(Pj[i], t[i], acc);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
            if (lane == 0) t[j0 + j] -= acc;
        }
        __syncthreads();
        if (warp == 0) {                             // in-block backward substitution with L11^T
            for (int j = nb - 1; j >= 0; --j) {
                const double v = t[j0 + j] / Ld[j][j];
                __syncwarp();
                if (lane == 0) t[j0 + j] = v;
                for (int i = lane; i < j; i += 32) t[j0 + i] -= Ld[j][i] * v;
                __syncwarp();
            }
        }
        __syncthreads();
    }
    for (int i = tid; i < w; i += NT) x[c0 + i] = t[i];
}

__global__ void permute_in_kernel(int64_t n, const int32_t* __restrict__ perm, const double* __restrict__ b, double* __restrict__ x) {
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i < n) x[i] = b[perm[i]];
}
__global__ void permute_out_kernel(int64_t n, const int32_t* __restrict__ perm, const double* __restrict__ x, double* __restrict__ b) {
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i < n) b[perm[i]] = x[i];
}

}  // namespace

static size_t solve_smem_bytes(int max_r) { return ((size_t)((max_r + 1) & ~1) + (size_t)BIG_NB * (BIG_NB + 1)) * sizeof(double); }

cudaError_t configure_solve_kernels(int max_smem_bytes) {
    cudaError_t e = cudaFuncSetAttribute(solve_fwd_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem_bytes);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(solve_bwd_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem_bytes);
}
void launch_solve_fwd(const DevSym& D, const int32_t* sn_list, int count, int max_r, double* x, cudaStream_t st) {
    if (count > 0) solve_fwd_kernel<<<count, NT, solve_smem_bytes(max_r), st>>>(D, sn_list, x);
}
void launch_solve_bwd(const DevSym& D, const int32_t* sn_list, int count, int max_r, double* x, cudaStream_t st) {
    if (count > 0) solve_bwd_kernel<<<count, NT, solve_smem_bytes(max_r), st>>>(D, sn_list, x);
}
void launch_permute_in(const DevSym& D, const double* b, double* x, cudaStream_t st) {
    permute_in_kernel<<<(unsigned)((D.n + 255) / 256), 256, 0, st>>>(D.n, D.perm, b, x);
}
void launch_permute_out(const DevSym& D, const double* x, double* b, cudaStream_t st) {
    permute_out_kernel<<<(unsigned)((D.n + 255) / 256), 256, 0, st>>>(D.n, D.perm, x, b);
}

}  // namespace nmpc
