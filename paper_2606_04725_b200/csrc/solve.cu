// solve.cu -- supernodal triangular solves (step a5, Eq. (22)-(25)) on the factor produced by factor.cu:
// L v = P b (leaves -> root), L^T Omega = v (root -> leaves), dy = P^T Omega, as ONE persistent task-DAG kernel.
//
// Tasks (host-ordered, claimed in order, waiting on epoch-valued completion flags):
//   forward,  small supernode: t = [b[P cols]; 0] + children's contribution vectors (fixed order); L11 y = t1 in 32-column
//             blocks (one warp substitutes, all threads update the rows below); x[cols] = y; contribution = t2 - L21 y.
//   forward,  block row I of a tiled supernode (left-looking): t_I = init_I - sum_{k<I} L(I,k) y_k, waiting for each y_k as it
//             is reached; then L(I,I) y_I = t_I by one warp (64-step substitution on the staged diagonal tile).
//   backward, small supernode / block column J of a tiled supernode: x_J = L(J,J)^-T (y_J - sum_{I>J} L(I,J)^T x_I), rows
//             taken from the ancestors' finished x first, then from this supernode's later blocks as their flags arrive.
// The permutations are fused: forward tasks read b[perm[.]], backward tasks write b[perm[.]] (in place, no hazard: a
// supernode's entries of b are read by its own forward task only).  Divisions by L_jj are multiplications by the reciprocals
// the factorization stored (dinv).  fp64, fixed summation order -> bitwise reproducible.
#include "device.h"

namespace nmpc {

namespace {

constexpr int NT = 256;
constexpr int DLD = 65;                 // leading dimension of the staged 64x64 diagonal tile
constexpr int SLD = 33;                 // ... of the 32x32 diagonal block of a small supernode
// shared memory (doubles): vec[256] | ys[64] | part[4*64] | Ld[64*65]
constexpr int OFF_YS = 256, OFF_PART = OFF_YS + 64, OFF_LD = OFF_PART + 256, SOLVE_SMEM_DOUBLES = OFF_LD + TILE * DLD;
constexpr unsigned FULL = 0xffffffffu;

__device__ __forceinline__ uint32_t ld_acquire(const uint32_t* p) {
    uint32_t v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release(uint32_t* p, uint32_t v) {
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void red_release_add(uint32_t* p, uint32_t v) {
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void spin_until_ge(const uint32_t* p, uint32_t target) {
    while (ld_acquire(p) < target) __nanosleep(40);
}

struct Sn {                             // per-supernode scalars every task needs
    int c0, w, r, ld;
    const double* P;
    const int32_t* rows;
};
__device__ __forceinline__ Sn sn_of(const DevSym& D, int s) {
    Sn q;
    q.c0 = D.sn_start[s]; q.w = D.sn_start[s + 1] - q.c0;
    q.r = (int)(D.rows_ptr[s + 1] - D.rows_ptr[s]); q.ld = ld_even(q.r);
    q.P = D.L + D.panel_ptr[s]; q.rows = D.rows + D.rows_ptr[s];
    return q;
}

// ---------------- forward, whole small supernode ----------------
__device__ __forceinline__ void fwd_small(const DevSym& D, const DagPlan& F, int s, const double* b, double* x, uint32_t epoch, double* sm) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const Sn q = sn_of(D, s);
    double* t = sm;
    double* Lb = sm + OFF_LD;
    for (int i = tid; i < q.r; i += NT) t[i] = (i < q.w) ? b[D.perm[q.c0 + i]] : 0.0;
    const int ch0 = D.child_ptr[s], ch1 = D.child_ptr[s + 1];
    for (int ci = ch0 + tid; ci < ch1; ci += NT) { const int c = D.child_idx[ci]; spin_until_ge(F.sol_done_f + c, epoch * (uint32_t)F.target_f[c]); }
    for (int ci = ch0; ci < ch1; ++ci) {
        const int c = D.child_idx[ci];
        const int mc = (int)(D.rel_ptr[c + 1] - D.rel_ptr[c]);
        const double* cc = D.ctr + D.rel_ptr[c];
        const int32_t* __restrict__ rel = D.rel + D.rel_ptr[c];
        __syncthreads();
        for (int a = tid; a < mc; a += NT) t[rel[a]] += __ldcg(cc + a);
    }
    __syncthreads();
    for (int j0 = 0; j0 < q.w; j0 += 32) {
        const int nb = min(32, q.w - j0);
        for (int idx = tid; idx < nb * nb; idx += NT) {
            const int i = idx % nb, c = idx / nb;
            if (i >= c) Lb[c * SLD + i] = __ldcg(q.P + (j0 + i) + (int64_t)(j0 + c) * q.ld);
        }
        __syncthreads();
        if (warp == 0) {
            double tv = lane < nb ? t[j0 + lane] : 0.0;
            const double dv = lane < nb ? __ldcg(D.dinv + q.c0 + j0 + lane) : 1.0;
            for (int j = 0; j < nb; ++j) {
                const double yj = __shfl_sync(FULL, tv * dv, j);
                if (lane == j) tv = yj;
                else if (lane > j && lane < nb) tv = fma(-Lb[j * SLD + lane], yj, tv);
            }
            if (lane < nb) t[j0 + lane] = tv;
        }
        __syncthreads();
        for (int i = j0 + nb + tid; i < q.r; i += NT) {
            const double* Pi = q.P + i + (int64_t)j0 * q.ld;
            double acc = 0.0;
#pragma unroll 8
            for (int k = 0; k < nb; ++k) acc = fma(__ldcg(Pi + (int64_t)k * q.ld), t[j0 + k], acc);
            t[i] -= acc;
        }
        __syncthreads();
    }
    for (int i = tid; i < q.w; i += NT) x[q.c0 + i] = t[i];
    double* co = D.ctr + D.rel_ptr[s];
    for (int i = q.w + tid; i < q.r; i += NT) co[i - q.w] = t[i];
    __threadfence();
    __syncthreads();
    if (tid == 0) red_release_add(F.sol_done_f + s, 1u);
}

// ---------------- forward, block row I of a tiled supernode ----------------
__device__ __forceinline__ void fwd_tiled(const DevSym& D, const DagPlan& F, int s, int I, const double* b, double* x, uint32_t epoch, double* sm) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const Sn q = sn_of(D, s);
    const int nbp = tile_nbp(q.w);
    const int i0 = tile_bound(I, q.w, q.r, nbp), ni = tile_bound(I + 1, q.w, q.r, nbp) - i0;
    double* tI = sm; double* ys = sm + OFF_YS; double* part = sm + OFF_PART; double* Ld = sm + OFF_LD;
    uint32_t* bf = F.blk_f + F.bbase[s];
    const bool pivot = I < nbp;
    if (pivot)
        for (int idx = tid; idx < ni * ni; idx += NT) {
            const int i = idx % ni, c = idx / ni;
            if (i >= c) Ld[c * DLD + i] = __ldcg(q.P + (i0 + i) + (int64_t)(i0 + c) * q.ld);
        }
    if (tid < TILE) tI[tid] = (pivot && tid < ni) ? b[D.perm[q.c0 + i0 + tid]] : 0.0;
    const int ch0 = D.child_ptr[s], ch1 = D.child_ptr[s + 1];
    if (I == 0)                                          // block rows I > 0 inherit this through the flag of y_0
        for (int ci = ch0 + tid; ci < ch1; ci += NT) { const int c = D.child_idx[ci]; spin_until_ge(F.sol_done_f + c, epoch * (uint32_t)F.target_f[c]); }
    const int mrow = tid & 63, cg = tid >> 6;
    const int nk = min(I, nbp);
    double acc = 0.0;
    for (int kb = 0; kb < nk; ++kb) {
        if (tid == 0) spin_until_ge(bf + kb, epoch);
        __syncthreads();
        const int k0 = kb * TILE, nkk = min(TILE, q.w - k0);
        if (tid < TILE) ys[tid] = tid < nkk ? __ldcg(x + q.c0 + k0 + tid) : 0.0;
        __syncthreads();
        if (mrow < ni) {
            const double* Pm = q.P + (i0 + mrow) + (int64_t)k0 * q.ld;
#pragma unroll 8
            for (int kk = cg; kk < nkk; kk += 4) acc = fma(__ldcg(Pm + (int64_t)kk * q.ld), ys[kk], acc);
        }
    }
    part[cg * TILE + mrow] = acc;
    for (int ci = ch0; ci < ch1; ++ci) {             // children are complete: waited above (I == 0) or through the flag of y_0
        const int c = D.child_idx[ci];
        const int32_t* cb = F.cbnd + F.cb_ptr[c];
        const int a0 = cb[I], a1 = cb[I + 1];
        if (a0 == a1) continue;
        const double* cc = D.ctr + D.rel_ptr[c];
        const int32_t* __restrict__ rel = D.rel + D.rel_ptr[c];
        __syncthreads();
        for (int a = a0 + tid; a < a1; a += NT) tI[rel[a] - i0] += __ldcg(cc + a);
    }
    __syncthreads();
    if (tid < TILE) tI[tid] -= (part[tid] + part[TILE + tid]) + (part[2 * TILE + tid] + part[3 * TILE + tid]);
    __syncthreads();
    if (pivot) {
        if (warp == 0) {
            const bool h1 = lane + 32 < ni;
            double t0 = tI[lane], t1 = tI[lane + 32];
            const double d0 = lane < ni ? __ldcg(D.dinv + q.c0 + i0 + lane) : 1.0, d1 = h1 ? __ldcg(D.dinv + q.c0 + i0 + lane + 32) : 1.0;
            const int n0 = min(ni, 32);
            for (int j = 0; j < n0; ++j) {
                const double yj = __shfl_sync(FULL, t0 * d0, j);
                if (lane == j) t0 = yj;
                else if (lane > j && lane < ni) t0 = fma(-Ld[j * DLD + lane], yj, t0);
                if (h1) t1 = fma(-Ld[j * DLD + lane + 32], yj, t1);
            }
            for (int j = 32; j < ni; ++j) {
                const double yj = __shfl_sync(FULL, t1 * d1, j - 32);
                if (lane + 32 == j) t1 = yj;
                else if (lane + 32 > j && h1) t1 = fma(-Ld[j * DLD + lane + 32], yj, t1);
            }
            if (lane < ni) x[q.c0 + i0 + lane] = t0;
            if (h1) x[q.c0 + i0 + lane + 32] = t1;
        }
        __threadfence();
        __syncthreads();
        if (tid == 0) { st_release(bf + I, epoch); red_release_add(F.sol_done_f + s, 1u); }
    } else {
        double* co = D.ctr + D.rel_ptr[s];
        if (tid < ni) co[i0 + tid - q.w] = tI[tid];
        __threadfence();
        __syncthreads();
        if (tid == 0) red_release_add(F.sol_done_f + s, 1u);
    }
}

// ---------------- backward, whole small supernode ----------------
__device__ __forceinline__ void bwd_small(const DevSym& D, const DagPlan& F, int s, double* b, double* x, uint32_t epoch, double* sm) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarp = NT / 32;
    const Sn q = sn_of(D, s);
    double* t = sm;
    double* Lb = sm + OFF_LD;
    if (tid == 0) {
        spin_until_ge(F.sol_done_f + s, epoch * (uint32_t)F.target_f[s]);
        const int p = F.sn_parent[s];
        if (p >= 0) spin_until_ge(F.sol_done_b + p, epoch * (uint32_t)F.target_b[p]);
    }
    __syncthreads();
    for (int i = tid; i < q.r; i += NT) t[i] = __ldcg(x + q.rows[i]);
    __syncthreads();
    const int nblk = (q.w + 31) / 32;
    for (int bk = nblk - 1; bk >= 0; --bk) {
        const int j0 = bk * 32, nb = min(32, q.w - j0);
        for (int idx = tid; idx < nb * nb; idx += NT) {
            const int i = idx % nb, c = idx / nb;
            if (i >= c) Lb[c * SLD + i] = __ldcg(q.P + (j0 + i) + (int64_t)(j0 + c) * q.ld);
        }
        for (int c = warp; c < nb; c += nwarp) {         // z_c = y_c - sum_{i >= j0+nb} L[i, j0+c] t_i
            const double* Pc = q.P + (int64_t)(j0 + c) * q.ld;
            double acc = 0.0;
            for (int i = j0 + nb + lane; i < q.r; i += 32) acc = fma(__ldcg(Pc + i), t[i], acc);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(FULL, acc, o);
            if (lane == 0) t[j0 + c] -= acc;
        }
        __syncthreads();
        if (warp == 0) {
            double zv = lane < nb ? t[j0 + lane] : 0.0;
            const double dv = lane < nb ? __ldcg(D.dinv + q.c0 + j0 + lane) : 1.0;
            for (int j = nb - 1; j >= 0; --j) {
                const double xj = __shfl_sync(FULL, zv * dv, j);
                if (lane == j) zv = xj;
                else if (lane < j) zv = fma(-Lb[lane * SLD + j], xj, zv);
            }
            if (lane < nb) t[j0 + lane] = zv;
        }
        __syncthreads();
    }
    for (int i = tid; i < q.w; i += NT) { x[q.c0 + i] = t[i]; b[D.perm[q.c0 + i]] = t[i]; }
    __threadfence();
    __syncthreads();
    if (tid == 0) red_release_add(F.sol_done_b + s, 1u);
}

// ---------------- backward, block column J of a tiled supernode ----------------
__device__ __forceinline__ void bwd_tiled(const DevSym& D, const DagPlan& F, int s, int J, double* b, double* x, uint32_t epoch, double* sm) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const Sn q = sn_of(D, s);
    const int nbp = tile_nbp(q.w), nbt = nbp + tile_nbu(q.w, q.r);
    const int j0 = J * TILE, nj = min(TILE, q.w - j0);
    double* xs = sm + OFF_YS; double* zs = sm; double* Ld = sm + OFF_LD;
    uint32_t* bb = F.blk_b + F.bbase[s];
    for (int idx = tid; idx < nj * nj; idx += NT) {
        const int i = idx % nj, c = idx / nj;
        if (i >= c) Ld[c * DLD + i] = __ldcg(q.P + (j0 + i) + (int64_t)(j0 + c) * q.ld);
    }
    if (tid == 0) {
        spin_until_ge(F.sol_done_f + s, epoch * (uint32_t)F.target_f[s]);
        const int p = F.sn_parent[s];
        if (p >= 0) spin_until_ge(F.sol_done_b + p, epoch * (uint32_t)F.target_b[p]);   // the rows below belong to finished ancestors
    }
    double acc[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) acc[e] = 0.0;
    for (int I = nbt - 1; I > J; --I) {
        if (I < nbp && tid == 0) spin_until_ge(bb + I, epoch);
        __syncthreads();
        const int i0 = tile_bound(I, q.w, q.r, nbp), ni = tile_bound(I + 1, q.w, q.r, nbp) - i0;
        if (tid < TILE) xs[tid] = tid < ni ? __ldcg(x + q.rows[i0 + tid]) : 0.0;
        __syncthreads();
#pragma unroll
        for (int e = 0; e < 8; ++e) {
            const int c = warp * 8 + e;
            if (c < nj) {
                const double* Pc = q.P + i0 + (int64_t)(j0 + c) * q.ld;
                if (lane < ni) acc[e] = fma(__ldcg(Pc + lane), xs[lane], acc[e]);
                if (lane + 32 < ni) acc[e] = fma(__ldcg(Pc + lane + 32), xs[lane + 32], acc[e]);
            }
        }
    }
    __syncthreads();                                     // also orders thread 0's waits when the loop above is empty
#pragma unroll
    for (int e = 0; e < 8; ++e) {
        double v = acc[e];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
        const int c = warp * 8 + e;
        if (lane == 0 && c < nj) zs[c] = __ldcg(x + q.c0 + j0 + c) - v;
    }
    __syncthreads();
    if (warp == 0) {
        const bool h1 = lane + 32 < nj;
        double z0 = lane < nj ? zs[lane] : 0.0, z1 = h1 ? zs[lane + 32] : 0.0;
        const double d0 = lane < nj ? __ldcg(D.dinv + q.c0 + j0 + lane) : 1.0, d1 = h1 ? __ldcg(D.dinv + q.c0 + j0 + lane + 32) : 1.0;
        for (int j = nj - 1; j >= 32; --j) {
            const double xj = __shfl_sync(FULL, z1 * d1, j - 32);
            if (lane + 32 == j) z1 = xj;
            else if (lane + 32 < j) z1 = fma(-Ld[(lane + 32) * DLD + j], xj, z1);
            z0 = fma(-Ld[lane * DLD + j], xj, z0);
        }
        for (int j = min(nj, 32) - 1; j >= 0; --j) {
            const double xj = __shfl_sync(FULL, z0 * d0, j);
            if (lane == j) z0 = xj;
            else if (lane < j) z0 = fma(-Ld[lane * DLD + j], xj, z0);
        }
        if (lane < nj) { x[q.c0 + j0 + lane] = z0; b[D.perm[q.c0 + j0 + lane]] = z0; }
        if (h1) { x[q.c0 + j0 + lane + 32] = z1; b[D.perm[q.c0 + j0 + lane + 32]] = z1; }
    }
    __threadfence();
    __syncthreads();
    if (tid == 0) { st_release(bb + J, epoch); red_release_add(F.sol_done_b + s, 1u); }
}

__global__ void __launch_bounds__(NT) solve_dag_kernel(DevSym D, DagPlan F, double* b, double* x, uint32_t epoch) {
    extern __shared__ __align__(16) double sm[];
    __shared__ int s_task;
    const uint32_t base = (epoch - 1u) * (uint32_t)(F.n_stasks + (int)gridDim.x);
    while (true) {
        __syncthreads();
        if (threadIdx.x == 0) s_task = (int)(atomicAdd(F.sync + 1, 1u) - base);
        __syncthreads();
        const int t = s_task;
        if (t >= F.n_stasks) break;
        const int4 tk = F.stasks[t];
        unsigned long long* tr = F.strace ? F.strace + (size_t)t * 8 : nullptr;
        if (tr && threadIdx.x == 0) { unsigned long long g; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g)); tr[0] = g; }
        if (tk.w == 0) { if (tk.x == 0) fwd_small(D, F, tk.y, b, x, epoch, sm); else fwd_tiled(D, F, tk.y, tk.z, b, x, epoch, sm); }
        else           { if (tk.x == 0) bwd_small(D, F, tk.y, b, x, epoch, sm); else bwd_tiled(D, F, tk.y, tk.z, b, x, epoch, sm); }
        if (tr && threadIdx.x == 0) { unsigned long long g; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g)); tr[4] = g; }
    }
}

}  // namespace

cudaError_t configure_solve_kernels(int max_smem_bytes, int* ctas_per_sm, size_t* smem_bytes) {
    const size_t bytes = (size_t)SOLVE_SMEM_DOUBLES * sizeof(double);
    if (bytes > (size_t)max_smem_bytes) return cudaErrorInvalidValue;
    cudaError_t e = cudaFuncSetAttribute(solve_dag_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e != cudaSuccess) return e;
    int occ = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, solve_dag_kernel, NT, bytes);
    if (e != cudaSuccess) return e;
    *ctas_per_sm = occ < 1 ? 1 : occ;
    *smem_bytes = bytes;
    return cudaSuccess;
}

void launch_solve(const DevSym& D, const DagPlan& F, double* rhs_inout, double* x, uint32_t epoch, cudaStream_t st) {
    if (F.n_stasks > 0) solve_dag_kernel<<<F.sgrid, NT, F.ssmem, st>>>(D, F, rhs_inout, x, epoch);
}

}  // namespace nmpc
