// factor.cu -- numeric multifrontal supernodal Cholesky (step a4, NumCholesky Eq. (20)-(21)) and the
// supernodal triangular solves (step a5, Eq. (22)-(25)) on the fixed structure S_L produced once by
// symbolic.cpp.  fp64 throughout, no atomics on floating-point data, fixed summation order -> bitwise reproducible.
//
// Two kernel families, chosen per supernode at analysis time by the front size r:
//   small  (r <= smem_front_max): ONE CTA assembles the whole r x r front in shared memory (K entries through the
//          scatter map + extend-add of the children's update matrices, pulled in fixed child order), factors its w
//          pivot columns (Eq. 21 column by column), and writes the r x w panel of L and the (r-w)^2 update matrix.
//   big    (r >  smem_front_max): the front lives in HBM (panel + update storage are the front); a column-slice
//          assembly kernel, then per 64-column block step: POTRF of the diagonal block, TRSM of the block column,
//          SYRK/GEMM update of the trailing front.  Launches are batched over all big fronts of a tree level.
#include <climits>
#include <cstdio>

#include "device.h"

namespace nmpc {

namespace {

constexpr int NT = 256;                 // threads per CTA for every kernel in this file

struct FrontView {                      // the r x r front of a supernode, split over panel (cols < w) and update storage
    double* P; double* Uu; int r, w, m;
    __device__ __forceinline__ double* at(int i, int c) const {
        return c < w ? P + (i + (int64_t)c * r) : Uu + ((i - w) + (int64_t)(c - w) * m);
    }
};

__device__ __forceinline__ FrontView front_view(const DevSym& D, int s) {
    FrontView F;
    F.w = D.sn_start[s + 1] - D.sn_start[s];
    F.r = (int)(D.rows_ptr[s + 1] - D.rows_ptr[s]);
    F.m = F.r - F.w;
    F.P = D.L + D.panel_ptr[s];
    F.Uu = D.U + D.upd_ptr[s];
    return F;
}

__device__ __forceinline__ bool bad_pivot(double d) { return !(d > 0.0) || isinf(d); }

// =============================================================================================================
// small fronts: whole front in shared memory
// =============================================================================================================
__global__ void __launch_bounds__(NT) front_small_kernel(DevSym D, const int32_t* __restrict__ sn_list,
                                                         const double* __restrict__ Kval) {
    extern __shared__ double F[];
    const double eta = *D.eta;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarp = NT / 32;
    const int s = sn_list[blockIdx.x];
    const int c0 = D.sn_start[s], w = D.sn_start[s + 1] - c0;
    const int r = (int)(D.rows_ptr[s + 1] - D.rows_ptr[s]);
    // 1. zero
    for (int idx = tid; idx < r * r; idx += NT) F[idx] = 0.0;
    __syncthreads();
    // 2. K entries of the pivot columns (scatter map: kent_dst = i + j*r)
    for (int64_t q = D.kent_ptr[s] + tid; q < D.kent_ptr[s + 1]; q += NT) F[D.kent_dst[q]] = Kval[D.kent_src[q]];
    __syncthreads();
    if (eta != 0.0) for (int j = tid; j < w; j += NT) F[j + j * r] += eta;
    // 3. extend-add of the children's update matrices, fixed child order
    for (int ci = D.child_ptr[s]; ci < D.child_ptr[s + 1]; ++ci) {
        const int c = D.child_idx[ci];
        const int mc = (int)(D.rel_ptr[c + 1] - D.rel_ptr[c]);
        const double* __restrict__ Uc = D.U + D.upd_ptr[c];
        const int32_t* __restrict__ rel = D.rel + D.rel_ptr[c];
        __syncthreads();
        for (int b = warp; b < mc; b += nwarp) {
            const int cb = rel[b] * r;
            for (int a = b + lane; a < mc; a += 32) F[rel[a] + cb] += Uc[a + (int64_t)b * mc];
        }
    }
    __syncthreads();
    // 4. partial Cholesky of the first w columns, right-looking (Eq. 21)
    for (int j = 0; j < w; ++j) {
        double* Fj = F + j * r;
        const double d = Fj[j];
        const bool bad = bad_pivot(d);
        const double dj = bad ? 1.0 : sqrt(d);
        __syncthreads();
        if (tid == 0) { Fj[j] = dj; if (bad) atomicMin(D.fail_col, c0 + j); }
        for (int i = j + 1 + tid; i < r; i += NT) Fj[i] /= dj;
        __syncthreads();
        for (int c = j + 1 + warp; c < r; c += nwarp) {
            const double lc = Fj[c];
            double* Fc = F + c * r;
            for (int i = c + lane; i < r; i += 32) Fc[i] -= Fj[i] * lc;
        }
        __syncthreads();
    }
    // 5. write the panel of L and the update matrix
    double* __restrict__ P = D.L + D.panel_ptr[s];
    for (int j = warp; j < w; j += nwarp)
        for (int i = j + lane; i < r; i += 32) P[i + (int64_t)j * r] = F[i + j * r];
    const int m = r - w;
    double* __restrict__ Uo = D.U + D.upd_ptr[s];
    for (int j = warp; j < m; j += nwarp)
        for (int i = j + lane; i < m; i += 32) Uo[i + (int64_t)j * m] = F[(i + w) + (j + w) * r];
}

// =============================================================================================================
// big fronts: tiled path in global memory
// =============================================================================================================
// item = (sn, c_lo, c_hi, -): this CTA owns front columns [c_lo, c_hi): zero, K entries, children, all in order.
__global__ void __launch_bounds__(NT) big_assemble_kernel(DevSym D, const BigItem* __restrict__ items,
                                                          const double* __restrict__ Kval) {
    const double eta = *D.eta;
    const BigItem it = items[blockIdx.x];
    const int s = it.sn, c_lo = it.a, c_hi = it.b;
    const FrontView F = front_view(D, s);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarp = NT / 32;
    for (int c = c_lo + warp; c < c_hi; c += nwarp)
        for (int i = c + lane; i < F.r; i += 32) *F.at(i, c) = 0.0;
    __syncthreads();
    if (c_lo < F.w) {
        // K entries are sorted by column: binary search the first entry with column >= c_lo and >= c_hi
        const int64_t q0 = D.kent_ptr[s], q1 = D.kent_ptr[s + 1];
        auto lower = [&](int col) {
            int64_t a = q0, b = q1;
            while (a < b) { int64_t mid = (a + b) >> 1; if (D.kent_dst[mid] / F.r < col) a = mid + 1; else b = mid; }
            return a;
        };
        const int64_t qa = lower(c_lo), qb = lower(c_hi);
        for (int64_t q = qa + tid; q < qb; q += NT) F.P[D.kent_dst[q]] = Kval[D.kent_src[q]];
        __syncthreads();
        if (eta != 0.0) for (int j = c_lo + tid; j < c_hi && j < F.w; j += NT) F.P[j + (int64_t)j * F.r] += eta;
    }
    for (int ci = D.child_ptr[s]; ci < D.child_ptr[s + 1]; ++ci) {
        const int c = D.child_idx[ci];
        const int mc = (int)(D.rel_ptr[c + 1] - D.rel_ptr[c]);
        const double* __restrict__ Uc = D.U + D.upd_ptr[c];
        const int32_t* __restrict__ rel = D.rel + D.rel_ptr[c];
        auto lower = [&](int col) { int a = 0, b = mc; while (a < b) { int mid = (a + b) >> 1; if (rel[mid] < col) a = mid + 1; else b = mid; } return a; };
        const int b0 = lower(c_lo), b1 = lower(c_hi);
        __syncthreads();
        for (int b = b0 + warp; b < b1; b += nwarp) {
            const int cb = rel[b];
            for (int a = b + lane; a < mc; a += 32) *F.at(rel[a], cb) += Uc[a + (int64_t)b * mc];
        }
    }
}

// item = (sn, j0): Cholesky of the diagonal block [j0, j0+nb) of the panel, one CTA.
__global__ void __launch_bounds__(NT) big_potrf_kernel(DevSym D, const BigItem* __restrict__ items) {
    __shared__ double A[BIG_NB][BIG_NB + 1];
    const BigItem it = items[blockIdx.x];
    const FrontView F = front_view(D, it.sn);
    const int j0 = it.a, nb = min(BIG_NB, F.w - j0);
    const int tid = threadIdx.x;
    const int c0 = D.sn_start[it.sn];
    for (int idx = tid; idx < nb * nb; idx += NT) {
        const int i = idx % nb, c = idx / nb;
        A[i][c] = (i >= c) ? F.P[(j0 + i) + (int64_t)(j0 + c) * F.r] : 0.0;
    }
    __syncthreads();
    for (int j = 0; j < nb; ++j) {
        const double d = A[j][j];
        const bool bad = bad_pivot(d);
        const double dj = bad ? 1.0 : sqrt(d);
        __syncthreads();
        if (tid == 0) { A[j][j] = dj; if (bad) atomicMin(D.fail_col, c0 + j0 + j); }
        for (int i = j + 1 + tid; i < nb; i += NT) A[i][j] /= dj;
        __syncthreads();
        for (int idx = tid; idx < (nb - j - 1) * (nb - j - 1); idx += NT) {
            const int i = j + 1 + idx % (nb - j - 1), c = j + 1 + idx / (nb - j - 1);
            if (i >= c) A[i][c] -= A[i][j] * A[c][j];
        }
        __syncthreads();
    }
    for (int idx = tid; idx < nb * nb; idx += NT) {
        const int i = idx % nb, c = idx / nb;
        if (i >= c) F.P[(j0 + i) + (int64_t)(j0 + c) * F.r] = A[i][c];
    }
}

// item = (sn, j0, i0): X = A D^-T for the 64-row tile starting at front row i0 of block column j0.
__global__ void __launch_bounds__(NT) big_trsm_kernel(DevSym D, const BigItem* __restrict__ items) {
    extern __shared__ double sm[];
    double (*Dg)[BIG_NB + 1] = reinterpret_cast<double (*)[BIG_NB + 1]>(sm);
    double (*X)[BIG_NB + 1] = reinterpret_cast<double (*)[BIG_NB + 1]>(sm + BIG_NB * (BIG_NB + 1));   // X[c][i]: column c of the tile
    const BigItem it = items[blockIdx.x];
    const FrontView F = front_view(D, it.sn);
    const int j0 = it.a, i0 = it.b, nb = min(BIG_NB, F.w - j0), nr = min(BIG_NB, F.r - i0);
    const int tid = threadIdx.x;
    for (int idx = tid; idx < nb * nb; idx += NT) {
        const int i = idx % nb, c = idx / nb;
        Dg[i][c] = (i >= c) ? F.P[(j0 + i) + (int64_t)(j0 + c) * F.r] : 0.0;
    }
    for (int idx = tid; idx < nr * nb; idx += NT) {
        const int i = idx % nr, c = idx / nr;
        X[c][i] = F.P[(i0 + i) + (int64_t)(j0 + c) * F.r];
    }
    __syncthreads();
    for (int c = 0; c < nb; ++c) {
        const double dc = Dg[c][c];
        for (int i = tid; i < nr; i += NT) X[c][i] /= dc;
        __syncthreads();
        for (int idx = tid; idx < nr * (nb - c - 1); idx += NT) {
            const int i = idx % nr, k = c + 1 + idx / nr;
            X[k][i] -= X[c][i] * Dg[k][c];
        }
        __syncthreads();
    }
    for (int idx = tid; idx < nr * nb; idx += NT) {
        const int i = idx % nr, c = idx / nr;
        F.P[(i0 + i) + (int64_t)(j0 + c) * F.r] = X[c][i];
    }
}

// item = (sn, j0, I0, J0): C[I0.., J0..] -= X[I0.., :] X[J0.., :]^T on the lower triangle, X = block column j0 of the panel.
__global__ void __launch_bounds__(NT) big_syrk_kernel(DevSym D, const BigItem* __restrict__ items) {
    extern __shared__ double sm[];
    double (*XI)[BIG_NB] = reinterpret_cast<double (*)[BIG_NB]>(sm);                       // [k][i]
    double (*XJ)[BIG_NB] = reinterpret_cast<double (*)[BIG_NB]>(sm + BIG_NB * BIG_NB);
    const BigItem it = items[blockIdx.x];
    const FrontView F = front_view(D, it.sn);
    const int j0 = it.a, I0 = it.b, J0 = it.c;
    const int nb = min(BIG_NB, F.w - j0), ni = min(BIG_NB, F.r - I0), nj = min(BIG_NB, F.r - J0);
    const int tid = threadIdx.x;
    for (int idx = tid; idx < BIG_NB * nb; idx += NT) {
        const int i = idx % BIG_NB, k = idx / BIG_NB;
        XI[k][i] = (i < ni) ? F.P[(I0 + i) + (int64_t)(j0 + k) * F.r] : 0.0;
        XJ[k][i] = (i < nj) ? F.P[(J0 + i) + (int64_t)(j0 + k) * F.r] : 0.0;
    }
    __syncthreads();
    const int tx = tid & 15, ty = tid >> 4;         // thread computes rows ty*4.., cols tx*4..
    double acc[4][4];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) acc[a][b] = 0.0;
    for (int k = 0; k < nb; ++k) {
        double av[4], bv[4];
#pragma unroll
        for (int a = 0; a < 4; ++a) { av[a] = XI[k][ty * 4 + a]; bv[a] = XJ[k][tx * 4 + a]; }
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = 0; b < 4; ++b) acc[a][b] = fma(av[a], bv[b], acc[a][b]);
    }
#pragma unroll
    for (int b = 0; b < 4; ++b) {
        const int c = J0 + tx * 4 + b;
        if (tx * 4 + b >= nj) continue;
#pragma unroll
        for (int a = 0; a < 4; ++a) {
            const int i = I0 + ty * 4 + a;
            if (ty * 4 + a < ni && i >= c) *F.at(i, c) -= acc[a][b];
        }
    }
}

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
    const int r = (int)(D.rows_ptr[s + 1] - D.rows_ptr[s]);
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
            if (i >= c) Ld[i][c] = P[(j0 + i) + (int64_t)(j0 + c) * r];
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
            const double* __restrict__ Pi = P + i + (int64_t)j0 * r;
            for (int k = 0; k < nb; ++k) acc = fma(Pi[(int64_t)k * r], t[j0 + k], acc);
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
    const int r = (int)(D.rows_ptr[s + 1] - D.rows_ptr[s]);
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
            if (i >= c) Ld[i][c] = P[(j0 + i) + (int64_t)(j0 + c) * r];
        }
        // t[j] -= sum_{i >= j0+nb} L[i,j] t[i] : one warp per column, lanes over rows (coalesced), fixed shuffle tree
        for (int j = warp; j < nb; j += nwarp) {
            const double* __restrict__ Pj = P + (int64_t)(j0 + j) * r;
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
__global__ void reset_flag_kernel(int32_t* f, double* eta_dev, double eta) { *f = INT_MAX; *eta_dev = eta; }

}  // namespace

constexpr size_t TRSM_SMEM = 2 * BIG_NB * (BIG_NB + 1) * sizeof(double);
constexpr size_t SYRK_SMEM = 2 * BIG_NB * BIG_NB * sizeof(double);
size_t small_front_smem_bytes(int max_r) { return (size_t)max_r * max_r * sizeof(double); }
static size_t solve_smem_bytes(int max_r) { return ((size_t)((max_r + 1) & ~1) + (size_t)BIG_NB * (BIG_NB + 1)) * sizeof(double); }

cudaError_t configure_factor_kernels(int max_smem_bytes) {
    cudaError_t e = cudaFuncSetAttribute(front_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem_bytes);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(big_trsm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TRSM_SMEM);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(big_syrk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SYRK_SMEM);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(solve_fwd_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem_bytes);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(solve_bwd_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem_bytes);
}

void launch_front_small(const DevSym& D, const int32_t* sn_list, int count, int max_r, const double* Kval, cudaStream_t st) {
    if (count > 0) front_small_kernel<<<count, NT, small_front_smem_bytes(max_r), st>>>(D, sn_list, Kval);
}
void launch_big_assemble(const DevSym& D, const BigItem* items, int count, const double* Kval, cudaStream_t st) {
    if (count > 0) big_assemble_kernel<<<count, NT, 0, st>>>(D, items, Kval);
}
void launch_big_potrf(const DevSym& D, const BigItem* items, int count, cudaStream_t st) {
    if (count > 0) big_potrf_kernel<<<count, NT, 0, st>>>(D, items);
}
void launch_big_trsm(const DevSym& D, const BigItem* items, int count, cudaStream_t st) {
    if (count > 0) big_trsm_kernel<<<count, NT, TRSM_SMEM, st>>>(D, items);
}
void launch_big_syrk(const DevSym& D, const BigItem* items, int count, cudaStream_t st) {
    if (count > 0) big_syrk_kernel<<<count, NT, SYRK_SMEM, st>>>(D, items);
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
void launch_reset_flag(const DevSym& D, double* eta_dev, double eta, cudaStream_t st) { reset_flag_kernel<<<1, 1, 0, st>>>(D.fail_col, eta_dev, eta); }

}  // namespace nmpc
