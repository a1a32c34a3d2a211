// solve.cu -- supernodal triangular solves (step a5, Eq. (22)-(25)) on the factor produced by factor.cu:
// L v = P b (leaves -> root), L^T Omega = v (root -> leaves), dy = P^T Omega, as ONE persistent task-DAG kernel.
//
// Tasks (host-ordered, claimed in order, waiting on epoch-valued completion flags):
//   forward,  small supernode: t = [b[P cols]; 0] + children's contribution vectors (child table and relative indices fetched
//             before the wait, contributions loaded in one round trip, added in fixed child order); the panel streams through
//             shared memory in 32-column blocks (cp.async, requested before the task waits); L11 y = t1 by pre-scaled warp
//             substitution (only shuffle + fma on the chain), one thread per row for the block below; contribution = t2 - L21 y.
//   forward,  block row I of a tiled supernode (left-looking): t_I = init_I - sum_{k<I} L(I,k) y_k; the 64x64 tile L(I,k+1)
//             is in registers before the task waits for y_k; then L(I,I) y_I = t_I by one warp on the staged diagonal tile.
//   backward, small supernode / block column J of a tiled supernode: x_J = L(J,J)^-T (y_J - sum_{I>J} L(I,J)^T x_I).  For a
//             tiled supernode the rows of the ANCESTORS (block rows I >= nbp, known as soon as the parent is done) are taken by
//             separate chunk tasks (BWD_CH tiles each, all block columns and chunks in parallel) that leave partial sums.  The
//             chain of the nbp diagonal blocks runs in ONE CTA (bwd_chain): per block column J it applies L(J+1,J)^T x_{J+1} from
//             registers and substitutes with L(J,J) in shared memory, while its other warps prepare block J-1 (the product
//             L(J+1,J-1)^T x_{J+1} from a tile staged with cp.async, the next diagonal tile, v, the partial sums) -- no flag
//             round trip between consecutive blocks.  The blocks further away, S_J = sum_{I >= J+3} L(I,J)^T x_I, come from one
//             helper task per block column (bwd_sum) that follows the chain two blocks behind.
// The permutations are fused: forward tasks read b[perm[.]], backward tasks write b[perm[.]] (in place, no hazard: a
// supernode's entries of b are read by its own forward task only).  Divisions by L_jj are multiplications by the reciprocals
// the factorization stored (dinv).  fp64, fixed summation order -> bitwise reproducible.
// Right-hand-side row (options.fuse_rhs, symbolic.h): the structure has one extra last variable whose row of L holds
// v = L^-1 P b of the b that went through the factorization.  A FUSED solve runs the backward tasks only and takes v from that
// row (the last row of every panel); a general solve treats the extra variable's right-hand side and solution as 0.
#include <algorithm>

#include "device.h"

namespace nmpc {

namespace {

constexpr int NT = 256;
constexpr int DLD = 65;                 // leading dimension of the staged 64x64 diagonal tile
constexpr int SLD = 33;                 // ... of the transposed-access copy of a 32x32 diagonal block (small supernodes)
constexpr int SB = 32;                  // column block of the small-supernode solves
constexpr int SCH = 16, SREL = 1024;    // children / total relative indices a forward task keeps in shared memory (else: one by one)
constexpr int FWD_WORK_DOUBLES = (SCH * 8 + (SCH + 4) * 4 + 7) / 8 + 2;   // child table behind the staging buffers
// shared memory (doubles): vec[256] | ys[64] | part[4*64] | dv[2*32] | Lbt[32*33] | buf[2][DagPlan::sbuf]
// (one staged column block: rows [j0, ld) x 32 columns; tiled tasks: Ld[64*65] aliases buf)
constexpr int OFF_YS = 256, OFF_PART = OFF_YS + 64, OFF_DV = OFF_PART + 256, OFF_LBT = OFF_DV + 2 * SB, OFF_BUF = OFF_LBT + SB * SLD,
              OFF_LD = OFF_BUF;
constexpr unsigned FULL = 0xffffffffu;

__device__ __forceinline__ uint32_t ld_acquire(const uint32_t* p) {
    uint32_t v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
// relaxed flag updates: always issued right after the publishing thread's __threadfence() (fence + relaxed store = release pattern)
__device__ __forceinline__ void st_release(uint32_t* p, uint32_t v) {
    asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void red_release_add(uint32_t* p, uint32_t v) {
    asm volatile("red.relaxed.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void spin_until_ge(const uint32_t* p, uint32_t target) {
    while (ld_acquire(p) < target) __nanosleep(40);
}

__device__ __forceinline__ void cp_async16(double* dst_smem, const double* src) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(dst_smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async8(double* dst_smem, const double* src) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(dst_smem);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

__device__ __forceinline__ double rhs_at(const DevSym& D, const double* b, int col) {      // P b at pivot position col
    return col == D.aug_col ? 0.0 : b[D.perm[col]];
}
__device__ __forceinline__ void put_solution(const DevSym& D, double* b, int col, double v) {
    if (col != D.aug_col) b[D.perm[col]] = v;
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

// ---------------- small supernodes: column blocks of the panel are staged in shared memory ----------------
// Column block k (columns [32k, 32k+nb), rows [32k, ld)) is copied with cp.async into buf[k & 1] (leading dimension
// ld - 32k, 16-byte chunks: 32k and ld are even) together with the pivot reciprocals of its columns.  The first two blocks
// are requested BEFORE the task waits for its dependencies, later ones two blocks ahead: no load from L sits on the
// dependency chain of the solve.
__device__ __forceinline__ void stage_block(const DevSym& D, const Sn& q, int k, double* sm, int sbuf) {
    const int j0 = k * SB, nb = min(SB, q.w - j0), ldb = q.ld - j0, half = ldb >> 1;
    double* buf = sm + OFF_BUF + (k & 1) * sbuf;
    const double* src = q.P + j0 + (int64_t)j0 * q.ld;
    for (int idx = threadIdx.x; idx < nb * half; idx += NT) {
        const int c = idx / half, h = idx - c * half;
        cp_async16(buf + c * ldb + 2 * h, src + (int64_t)c * q.ld + 2 * h);
    }
    if (threadIdx.x < nb) cp_async8(sm + OFF_DV + (k & 1) * SB + threadIdx.x, D.dinv + q.c0 + j0 + threadIdx.x);
    cp_async_commit();
}

#ifdef NMPC_TRACE_BUILD
#define STRACE(slot) do { if (tr && threadIdx.x == 0) { unsigned long long g_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g_)); tr[slot] = g_; } } while (0)
#else
#define STRACE(slot) do { (void)tr; } while (0)
#endif
#ifdef NMPC_TRACE_BUILD                     // measurement build: time accumulated per phase of the chain task
#define CHT0() unsigned long long cht_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(cht_))
#define CHT1(slot) do { if (tr) { unsigned long long g_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g_)); tr[slot] += g_ - cht_; } } while (0)
#else
#define CHT0() do {} while (0)
#define CHT1(slot) do { (void)tr; } while (0)
#endif
__device__ __forceinline__ void fwd_small(const DevSym& D, const DagPlan& F, int s, const double* b, double* x, uint32_t epoch, double* sm, unsigned long long* tr) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const Sn q = sn_of(D, s);
    double* t = sm;
    const int nblk = (q.w + SB - 1) / SB;
    stage_block(D, q, 0, sm, F.sbuf);
    if (nblk > 1) stage_block(D, q, 1, sm, F.sbuf);
    for (int i = tid; i < q.r; i += NT) t[i] = (i < q.w) ? rhs_at(D, b, q.c0 + i) : 0.0;
    const int ch0 = D.child_ptr[s], ch1 = D.child_ptr[s + 1], nch = ch1 - ch0;
    // child table + the relative indices of all children: fetched BEFORE the children are waited for (static data); the
    // contributions are then loaded in one round trip and added child by child (fixed order)
    long long* chRp = reinterpret_cast<long long*>(sm + OFF_BUF + 2 * F.sbuf);   // [SCH] rel_ptr of the child (= offset of its ctr)
    int* chOff = reinterpret_cast<int*>(chRp + SCH);                              // [SCH + 1] offset of its list in relS
    int myc = -1;
    if (tid < nch) {
        myc = D.child_idx[ch0 + tid];
        if (nch <= SCH) { const long long rp0 = D.rel_ptr[myc]; chRp[tid] = rp0; chOff[tid + 1] = (int)(D.rel_ptr[myc + 1] - rp0); }
    }
    __syncthreads();
    if (tid == 0 && nch <= SCH) { int off = 0; for (int i = 0; i < nch; ++i) { const int mc = chOff[i + 1]; chOff[i] = off; off += mc; } chOff[nch] = off; }
    __syncthreads();
    const bool fast = nch <= SCH && chOff[nch <= SCH ? nch : 0] <= SREL;
    const int tot = fast ? chOff[nch] : 0;
    int who[SREL / NT], dst[SREL / NT];
    long long src[SREL / NT];
#pragma unroll
    for (int k = 0; k < SREL / NT; ++k) {
        const int idx = tid + k * NT;
        who[k] = -1; dst[k] = 0; src[k] = 0;
        if (idx < tot) {
            int i = 0;
            while (idx >= chOff[i + 1]) ++i;
            who[k] = i; src[k] = chRp[i] + (idx - chOff[i]); dst[k] = D.rel[src[k]];
        }
    }
    for (int ci = tid; ci < nch; ci += NT) {
        const int c = (ci == tid && myc >= 0) ? myc : D.child_idx[ch0 + ci];
        spin_until_ge(F.sol_done_f + c, epoch * (uint32_t)F.target_f[c]);
    }
    __syncthreads();
    STRACE(1);
    if (fast) {
        double v[SREL / NT];
#pragma unroll
        for (int k = 0; k < SREL / NT; ++k) v[k] = who[k] >= 0 ? __ldcg(D.ctr + src[k]) : 0.0;
        for (int i = 0; i < nch; ++i) {
#pragma unroll
            for (int k = 0; k < SREL / NT; ++k)
                if (who[k] == i) t[dst[k]] += v[k];
            __syncthreads();
        }
    } else {
        for (int ci = ch0; ci < ch1; ++ci) {
            const int c = D.child_idx[ci];
            const int64_t rp0 = D.rel_ptr[c];
            const int mc = (int)(D.rel_ptr[c + 1] - rp0);
            const double* cc = D.ctr + rp0;
            const int32_t* __restrict__ rel = D.rel + rp0;
            if (ci > ch0) __syncthreads();
            for (int a = tid; a < mc; a += NT) t[rel[a]] += __ldcg(cc + a);
        }
    }
    STRACE(2);
    for (int k = 0; k < nblk; ++k) {
        const int j0 = k * SB, nb = min(SB, q.w - j0), ldb = q.ld - j0;
        const double* Bk = sm + OFF_BUF + (k & 1) * F.sbuf;
        const double* dv = sm + OFF_DV + (k & 1) * SB;
        if (k + 1 < nblk) cp_async_wait<1>(); else cp_async_wait<0>();
        __syncthreads();                                 // block k has landed; t is complete up to the previous block's update
        if (warp == 0) {                                 // L11 y = t1 on the diagonal block, one lane per row
            double tv = lane < nb ? t[j0 + lane] : 0.0;
            const double dvl = lane < nb ? dv[lane] : 1.0;
            // pre-scaled substitution: s_i = d_i t_i, s_i -= (d_i L_ij) y_j; only (shuffle, fma) on the chain, the scaled
            // column entries are loaded 8 columns ahead
            tv *= dvl;
            const int lcl = min(lane, ldb - 1);
            for (int jb = 0; jb < nb; jb += 8) {
                double lj[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) lj[e] = Bk[min(jb + e, nb - 1) * ldb + lcl] * dvl;
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const int j = jb + e;
                    const double yj = __shfl_sync(FULL, tv, j & 31);
                    tv = (lane > j && j < nb) ? fma(-lj[e], yj, tv) : tv;
                }
            }
            if (lane < nb) { t[j0 + lane] = tv; x[q.c0 + j0 + lane] = tv; }
        }
        __syncthreads();
        for (int i = j0 + nb + tid; i < q.r; i += NT) {  // t2 -= L21 y
            const double* Bi = Bk + (i - j0);
            double a0 = 0.0, a1 = 0.0;
            int c = 0;
            for (; c + 1 < nb; c += 2) { a0 = fma(Bi[c * ldb], t[j0 + c], a0); a1 = fma(Bi[(c + 1) * ldb], t[j0 + c + 1], a1); }
            if (c < nb) a0 = fma(Bi[c * ldb], t[j0 + c], a0);
            t[i] -= a0 + a1;
        }
        if (k + 2 < nblk) {
            __syncthreads();                             // everyone is done with buf[k & 1]
            stage_block(D, q, k + 2, sm, F.sbuf);
        }
    }
    __syncthreads();
    STRACE(3);
    double* co = D.ctr + D.rel_ptr[s];
    for (int i = q.w + tid; i < q.r; i += NT) co[i - q.w] = t[i];
    __syncthreads();
    if (tid == 0) { __threadfence(); red_release_add(F.sol_done_f + s, 1u); }
}

// ---------------- forward, block row I of a tiled supernode ----------------
// Left-looking over the finished y_k.  Nothing that can be fetched early sits on the dependency chain: the children's
// contributions are gathered first, the diagonal tile and the pivot reciprocals are staged at task start, and the 64x64
// tile L(I,k+1) is loaded into registers BEFORE the task waits for y_k.
__device__ __forceinline__ void fwd_tiled(const DevSym& D, const DagPlan& F, int s, int I, const double* b, double* x, uint32_t epoch, double* sm) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const Sn q = sn_of(D, s);
    const int nbp = tile_nbp(q.w);
    const int i0 = tile_bound(I, q.w, q.r, nbp), ni = tile_bound(I + 1, q.w, q.r, nbp) - i0;
    double* tI = sm; double* ys = sm + OFF_YS; double* part = sm + OFF_PART; double* Ld = sm + OFF_LD;
    uint32_t* bf = F.blk_f + F.bbase[s];
    const bool pivot = I < nbp;
    double d0 = 1.0, d1 = 1.0;
    if (pivot) {
        for (int idx = tid; idx < TILE * TILE; idx += NT) {
            const int i = idx & (TILE - 1), c = idx >> 6;
            if (i >= c && i < ni) Ld[c * DLD + i] = __ldg(q.P + (i0 + i) + (int64_t)(i0 + c) * q.ld);
        }
        if (warp == 0) {
            if (lane < ni) d0 = __ldcg(D.dinv + q.c0 + i0 + lane);
            if (lane + 32 < ni) d1 = __ldcg(D.dinv + q.c0 + i0 + lane + 32);
        }
    }
    if (tid < TILE) tI[tid] = (pivot && tid < ni) ? rhs_at(D, b, q.c0 + i0 + tid) : 0.0;
    const int ch0 = D.child_ptr[s], ch1 = D.child_ptr[s + 1];
    if (I == 0) {                                        // block rows I > 0 inherit this through the flag of y_0
        for (int ci = ch0 + tid; ci < ch1; ci += NT) { const int c = D.child_idx[ci]; spin_until_ge(F.sol_done_f + c, epoch * (uint32_t)F.target_f[c]); }
    } else if (tid == 0) {
        spin_until_ge(bf, epoch);
    }
    for (int ci = ch0; ci < ch1; ++ci) {
        const int c = D.child_idx[ci];
        const int32_t* cb = F.cbnd + F.cb_ptr[c];
        const int a0 = cb[I], a1 = cb[I + 1];
        __syncthreads();                                 // orders the waits above / the previous child's additions
        if (a0 == a1) continue;
        const double* cc = D.ctr + D.rel_ptr[c];
        const int32_t* __restrict__ rel = D.rel + D.rel_ptr[c];
        for (int a = a0 + tid; a < a1; a += NT) tI[rel[a] - i0] += __ldcg(cc + a);
    }
    const int mrow = tid & 63, cg = tid >> 6;
    const int nk = min(I, nbp);
    const bool rowok = mrow < ni;
    double acc = 0.0;
    double cur[16], nxt[16];
    auto load_tile = [&](int kb, double (&v)[16]) {
        const int k0 = kb * TILE, nkk = min(TILE, q.w - k0);
        const double* Pm = q.P + (i0 + (rowok ? mrow : 0)) + (int64_t)k0 * q.ld;
#pragma unroll
        for (int e = 0; e < 16; ++e) { const int kk = cg + 4 * e; v[e] = (rowok && kk < nkk) ? __ldg(Pm + (int64_t)kk * q.ld) : 0.0; }
    };
    if (nk > 0) load_tile(0, cur);
    for (int kb = 0; kb < nk; ++kb) {
        if (kb + 1 < nk) load_tile(kb + 1, nxt);
        if (tid < TILE) {
            if (lane == 0) spin_until_ge(bf + kb, epoch);
            __syncwarp();
            const int k0 = kb * TILE;
            ys[tid] = (k0 + tid < q.w) ? __ldcg(x + q.c0 + k0 + tid) : 0.0;
        }
        __syncthreads();
#pragma unroll
        for (int e = 0; e < 16; ++e) acc = fma(cur[e], ys[cg + 4 * e], acc);
        __syncthreads();
#pragma unroll
        for (int e = 0; e < 16; ++e) cur[e] = nxt[e];
    }
    part[cg * TILE + mrow] = acc;
    __syncthreads();
    if (tid < TILE) tI[tid] -= (part[tid] + part[TILE + tid]) + (part[2 * TILE + tid] + part[3 * TILE + tid]);
    __syncthreads();
    if (pivot) {
        if (warp == 0) {
            const bool h1 = lane + 32 < ni;
            double t0 = tI[lane], t1 = tI[lane + 32];
            const int n0 = min(ni, 32);
            // pre-scaled substitution (s_i = d_i t_i): only (shuffle, fma) on the chain, scaled entries loaded 8 columns ahead
            t0 = lane < ni ? t0 * d0 : 0.0;
            t1 = h1 ? t1 * d1 : 0.0;
            const int r0 = min(lane, ni - 1), r1 = min(lane + 32, ni - 1);
            for (int jb = 0; jb < n0; jb += 8) {
                double la[8], lb[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) { const int jc = min(jb + e, ni - 1); la[e] = Ld[jc * DLD + r0] * d0; lb[e] = Ld[jc * DLD + r1] * d1; }
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const int j = jb + e;
                    const double yj = __shfl_sync(FULL, t0, j & 31);
                    const bool on = j < n0;
                    t0 = (on && lane > j && lane < ni) ? fma(-la[e], yj, t0) : t0;
                    t1 = (on && h1) ? fma(-lb[e], yj, t1) : t1;
                }
            }
            for (int jb = 32; jb < ni; jb += 8) {
                double lb[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) lb[e] = Ld[min(jb + e, ni - 1) * DLD + r1] * d1;
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const int j = jb + e;
                    const double yj = __shfl_sync(FULL, t1, (j - 32) & 31);
                    t1 = (j < ni && lane + 32 > j && h1) ? fma(-lb[e], yj, t1) : t1;
                }
            }
            if (lane < ni) x[q.c0 + i0 + lane] = t0;
            if (h1) x[q.c0 + i0 + lane + 32] = t1;
            __syncwarp();
            if (lane == 0) { __threadfence(); st_release(bf + I, epoch); red_release_add(F.sol_done_f + s, 1u); }
        }
    } else {
        double* co = D.ctr + D.rel_ptr[s];
        if (tid < ni) co[i0 + tid - q.w] = tI[tid];
        __syncthreads();
        if (tid == 0) { __threadfence(); red_release_add(F.sol_done_f + s, 1u); }
    }
}

// ---------------- backward, whole small supernode ----------------
__device__ __forceinline__ void bwd_small(const DevSym& D, const DagPlan& F, int s, double* b, double* x, uint32_t ef, uint32_t epoch, bool fused, double* sm, unsigned long long* tr) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarp = NT / 32;
    const Sn q = sn_of(D, s);
    double* t = sm;
    double* Lbt = sm + OFF_LBT;
    const int nblk = (q.w + SB - 1) / SB;
    stage_block(D, q, nblk - 1, sm, F.sbuf);
    if (nblk > 1) stage_block(D, q, nblk - 2, sm, F.sbuf);
    const int myrow = tid < q.r ? q.rows[tid] : 0;       // q.r <= SMALL_ROWS_MAX < NT: one front row per thread
    if (tid == 0) {
        if (!fused) spin_until_ge(F.sol_done_f + s, ef * (uint32_t)F.target_f[s]);
        const int p = F.sn_parent[s];
        if (p >= 0) spin_until_ge(F.sol_done_b + p, epoch * (uint32_t)F.target_b[p]);
    }
    __syncthreads();
    STRACE(1);
    // own columns: v from the forward solve, or (fused) from the right-hand-side row of the panel; rows below: the ancestors' x
    if (tid < q.r) t[tid] = myrow == D.aug_col ? 0.0 : (fused && tid < q.w) ? __ldcg(q.P + (q.r - 1) + (int64_t)tid * q.ld) : __ldcg(x + myrow);
    STRACE(2);
    for (int k = nblk - 1; k >= 0; --k) {
        const int j0 = k * SB, nb = min(SB, q.w - j0), ldb = q.ld - j0;
        const double* Bk = sm + OFF_BUF + (k & 1) * F.sbuf;
        const double* dv = sm + OFF_DV + (k & 1) * SB;
        if (k > 0) cp_async_wait<1>(); else cp_async_wait<0>();
        __syncthreads();                                 // block k has landed; t holds y1 and the finished x below
        for (int idx = tid; idx < nb * SB; idx += NT) {  // padded copy of the diagonal block for the row-wise accesses below
            const int c = idx >> 5, i = idx & 31;
            if (i >= c && i < nb) Lbt[c * SLD + i] = Bk[c * ldb + i];
        }
        {   // z_c = y_c - sum_{i >= j0+nb} L[i, j0+c] x_i: a warp takes columns warp, warp+8, warp+16, warp+24 TOGETHER (lanes over the
            // rows), so that the four butterfly reductions interleave
            double a[4] = {0.0, 0.0, 0.0, 0.0};
            const double* Bc[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) Bc[e] = Bk + min(warp + nwarp * e, nb - 1) * ldb - j0;
            for (int i = j0 + nb + lane; i < q.r; i += 32) {
                const double ti = t[i];
#pragma unroll
                for (int e = 0; e < 4; ++e) a[e] = fma(Bc[e][i], ti, a[e]);
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1)
#pragma unroll
                for (int e = 0; e < 4; ++e) a[e] += __shfl_xor_sync(FULL, a[e], o);
#pragma unroll
            for (int e = 0; e < 4; ++e)
                if (lane == 0 && warp + nwarp * e < nb) t[j0 + warp + nwarp * e] -= a[e];
        }
        __syncthreads();
        if (warp == 0) {                                 // L11^T x1 = z on the diagonal block
            double zv = lane < nb ? t[j0 + lane] : 0.0;
            const double dvl = lane < nb ? dv[lane] : 1.0;
            zv *= dvl;                                   // pre-scaled: s_i = d_i z_i, s_i -= (d_i L_ji) x_j for i < j
            for (int jb = ((nb - 1) >> 3) << 3; jb >= 0; jb -= 8) {
                double lj[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) lj[e] = Lbt[lane * SLD + min(jb + e, nb - 1)] * dvl;
#pragma unroll
                for (int e = 7; e >= 0; --e) {
                    const int j = jb + e;
                    const double xj = __shfl_sync(FULL, zv, j & 31);
                    zv = (lane < j && j < nb) ? fma(-lj[e], xj, zv) : zv;
                }
            }
            if (lane < nb) t[j0 + lane] = zv;
        }
        if (k >= 2) {
            __syncthreads();                             // everyone is done with buf[k & 1]
            stage_block(D, q, k - 2, sm, F.sbuf);
        }
    }
    __syncthreads();
    STRACE(3);
    for (int i = tid; i < q.w; i += NT) { x[q.c0 + i] = t[i]; put_solution(D, b, q.c0 + i, t[i]); }
    __syncthreads();
    if (tid == 0) { __threadfence(); red_release_add(F.sol_done_b + s, 1u); }
}

// ---------------- backward, tiled supernode ----------------
// load_tile: the 64x64 tile L(I,J) into registers, warp w holds columns 8w..8w+7, lanes over the rows (two per lane)
struct BwdTile {
    const Sn& q; int nbp, j0, nj;
    __device__ __forceinline__ void load(int I, double (&v)[16]) const {
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
        const int i0 = tile_bound(I, q.w, q.r, nbp), ni = tile_bound(I + 1, q.w, q.r, nbp) - i0;
#pragma unroll
        for (int e = 0; e < 8; ++e) {
            const int c = warp * 8 + e;
            const double* Pc = q.P + i0 + (int64_t)(j0 + min(c, nj - 1)) * q.ld;
            v[2 * e] = (c < nj && lane < ni) ? __ldg(Pc + lane) : 0.0;
            v[2 * e + 1] = (c < nj && lane + 32 < ni) ? __ldg(Pc + lane + 32) : 0.0;
        }
    }
};

// chunk task (s, J, c): partial[c][J] = sum over the ancestors' block rows I in chunk c of L(I,J)^T x_I.  It waits for exactly the
// pieces of x its rows touch (the analysis lists their flags: blocks of the ancestors' chains, small ancestors), so the chunk
// tasks of a supernode run WHILE the chain of its parent is still going down its blocks
// Everything that does not depend on x is in flight before the task waits: the row indices of the chunk and the first three
// tiles (cp.async into a three-slot ring in shared memory).  After the wait the <= 512 values of x are gathered in ONE round trip;
// the tiles are then consumed from the ring, each freed slot refilled three tiles ahead.
constexpr int UPD_RING = BWD_CH * TILE, UPD_END = UPD_RING + 3 * TILE * TILE;
__device__ __forceinline__ void bwd_upd(const DevSym& D, const DagPlan& F, int s, int J, int c, const double* x, uint32_t epoch, double* sm) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const Sn q = sn_of(D, s);
    const int nbp = tile_nbp(q.w), nbt = nbp + tile_nbu(q.w, q.r);
    const int j0 = J * TILE, nj = min(TILE, q.w - j0);
    const int Ia = nbp + c * BWD_CH, nt = min(nbt, Ia + BWD_CH) - Ia;
    double* xs = sm;                                     // [BWD_CH][64]: x of the chunk's rows, zero padded per tile
    double* ring = sm + UPD_RING;
    auto stage = [&](int k) {                            // tile Ia + k: 64 columns x 64 rows from the even row at or before its start
        if (k < nt) {
            const int ia = tile_bound(Ia + k, q.w, q.r, nbp) & ~1;
            double* dst = ring + (k % 3) * TILE * TILE;
            for (int idx = tid; idx < TILE * TILE / 2; idx += NT) {
                const int cc = idx >> 5, h = idx & 31;
                cp_async16(dst + cc * TILE + 2 * h, q.P + ia + 2 * h + (int64_t)(j0 + min(cc, nj - 1)) * q.ld);
            }
        }
        cp_async_commit();                               // one group per call, empty past the chunk: wait_group<2> below counts them
    };
    stage(0); stage(1); stage(2);
    int g[2];
#pragma unroll
    for (int e = 0; e < 2; ++e) {                        // slot tid + 256 e = (tile, row)
        const int slot = tid + NT * e, k = slot >> 6, r = slot & (TILE - 1);
        g[e] = -1;
        if (k < nt) {
            const int i0 = tile_bound(Ia + k, q.w, q.r, nbp), ni = tile_bound(Ia + k + 1, q.w, q.r, nbp) - i0;
            if (r < ni) g[e] = q.rows[i0 + r];
        }
    }
    {
        const int64_t d0 = F.cdep_ptr[F.cbase[s] + c], d1 = F.cdep_ptr[F.cbase[s] + c + 1];
        for (int64_t k = d0 + tid; k < d1; k += NT) spin_until_ge(F.sync + F.cdep[k], epoch);
    }
    __syncthreads();
#pragma unroll
    for (int e = 0; e < 2; ++e) xs[tid + NT * e] = g[e] >= 0 ? __ldcg(x + g[e]) : 0.0;
    double acc[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) acc[e] = 0.0;
    for (int k = 0; k < nt; ++k) {
        cp_async_wait<2>();                              // tile k has landed (two younger groups may still fly)
        __syncthreads();                                 // ... for everybody; k = 0: xs is complete
        const int di = tile_bound(Ia + k, q.w, q.r, nbp) & 1;   // the tile starts one row into its staged copy when its first row is odd
        const double* tk = ring + (k % 3) * TILE * TILE;
        const double xa = xs[k * TILE + lane], xb = xs[k * TILE + lane + 32];
#pragma unroll
        for (int e = 0; e < 8; ++e) {
            const double* tc = tk + (warp * 8 + e) * TILE;
            acc[e] = fma(tc[min(lane + 32 + di, TILE - 1)], xb, fma(tc[lane + di], xa, acc[e]));   // row 63 + di = 64 only meets xb = 0
        }
        __syncthreads();                                 // the slot is free
        stage(k + 3);
    }
    double* out = F.bpart + F.pbase[s] + (int64_t)c * q.w + j0;
#pragma unroll
    for (int e = 0; e < 8; ++e) {
        double v = acc[e];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
        const int cc = warp * 8 + e;
        if (lane == 0 && cc < nj) out[cc] = v;
    }
    cp_async_wait<0>();
    __syncthreads();
    if (tid == 0) { __threadfence(); red_release_add(F.blk_u + F.bbase[s] + J, 1u); }
}

// helper (s, J), J <= nbp - 4: S_J = sum_{I = nbp-1 .. J+3} L(I,J)^T x_I, each x_I taken as the chain publishes it (the tile
// L(I-1,J) is in registers before the task waits for x_I); two blocks of slack before the chain needs S_J
__device__ __forceinline__ void bwd_sum(const DevSym& D, const DagPlan& F, int s, int J, const double* x, uint32_t epoch, double* sm) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const Sn q = sn_of(D, s);
    const int nbp = tile_nbp(q.w);
    const int j0 = J * TILE, nj = min(TILE, q.w - j0);
    double* xs = sm + OFF_YS;
    uint32_t* bb = F.blk_b + F.bbase[s];
    const BwdTile T{q, nbp, j0, nj};
    double cur[16], nxt[16];
    T.load(nbp - 1, cur);
    double acc[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) acc[e] = 0.0;
    for (int I = nbp - 1; I >= J + 3; --I) {
        if (I - 1 >= J + 3) T.load(I - 1, nxt);
        const int i0 = I * TILE, ni = min(TILE, q.w - i0);
        if (tid < TILE) {
            if (lane == 0) spin_until_ge(bb + I, epoch);
            __syncwarp();
            xs[tid] = tid < ni ? __ldcg(x + q.c0 + i0 + tid) : 0.0;
        }
        __syncthreads();
#pragma unroll
        for (int e = 0; e < 8; ++e) acc[e] = fma(cur[2 * e + 1], xs[lane + 32], fma(cur[2 * e], xs[lane], acc[e]));
        __syncthreads();
#pragma unroll
        for (int e = 0; e < 16; ++e) cur[e] = nxt[e];
    }
    double* out = F.bsum + q.c0 + j0;
#pragma unroll
    for (int e = 0; e < 8; ++e) {
        double v = acc[e];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
        const int cc = warp * 8 + e;
        if (lane == 0 && cc < nj) out[cc] = v;
    }
    __syncthreads();
    if (tid == 0) { __threadfence(); st_release(F.blk_s + F.bbase[s] + J, epoch); }
}

// the chain of a tiled supernode: x_J = L(J,J)^-T (v_J - anc_J - S_J - L(J+2,J)^T x_{J+2} - L(J+1,J)^T x_{J+1}), J = nbp-1 .. 0, in one CTA.
// Per block ("hop"): all warps apply L(J+1,J)^T x_{J+1} from the staged tile T1; then
//   warp 0      substitutes with the staged L(J,J)^T (the factorization leaves it in the upper triangle of the diagonal tile:
//               row j of L(J,J) is a contiguous column there; staged packed, lanes read consecutive words);
//   warps 1, 2  write x_{J+1} to global memory and announce it, fetch S_{J-1} from the helper and v - anc of block J-2;
//   warps 3..7  compute L(J+1,J-1)^T x_{J+1} from the staged tile T2 and request the three tiles of the next hop (cp.async).
// Shared memory (doubles): zs[64] | pre[2][64] | xs[2][64] | dv[2][64] | Ld[2][2048] | T1[64*64] | T2[64*64]
constexpr int LDP = TILE * TILE / 2;                                // packed L(J,J)^T: column j (rows 0 .. j-1, rounded up to even) at j*j/2
constexpr int CH_PRE = 64, CH_XS = CH_PRE + 2 * TILE, CH_DV = CH_XS + 2 * TILE, CH_LD = CH_DV + 2 * TILE, CH_T1 = CH_LD + 2 * LDP,
              CH_T2 = CH_T1 + TILE * TILE, CH_END = CH_T2 + TILE * TILE;
__device__ __forceinline__ void bar_named(int id, int count) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory"); }
__device__ __forceinline__ void bwd_chain(const DevSym& D, const DagPlan& F, int s, double* b, double* x, uint32_t ef, uint32_t epoch, bool fused, double* sm, unsigned long long* tr) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const Sn q = sn_of(D, s);
    const int nbp = tile_nbp(q.w), nbt = nbp + tile_nbu(q.w, q.r);
    const int nchunk = (nbt - nbp + BWD_CH - 1) / BWD_CH;
    double* zs = sm;
    uint32_t* bb = F.blk_b + F.bbase[s];
    const uint32_t* bu = F.blk_u + F.bbase[s];
    const uint32_t* bs = F.blk_s + F.bbase[s];
    // v - anc for column t of block Jb: v from the right-hand-side row of the panel (fused) or from the forward solve; anc = the
    // chunk tasks' partial sums in chunk order (the caller has seen their flag)
    auto va_of = [&](int Jb, int t) {
        const int c = Jb * TILE + t, col = q.c0 + c;
        double a = col == D.aug_col ? 0.0 : fused ? __ldcg(q.P + (q.r - 1) + (int64_t)c * q.ld) : __ldcg(x + col);
        const double* pp = F.bpart + F.pbase[s] + c;
#pragma unroll 4
        for (int k = 0; k < nchunk; ++k) a -= __ldcg(pp + (int64_t)k * q.w);
        return a;
    };
    auto stage_diag = [&](int J, int buf, int t0, int nthr) {       // L(J,J)^T packed + pivot reciprocals, cp.async
        const int j0 = J * TILE, nj = min(TILE, q.w - j0);
        double* Ld = sm + CH_LD + buf * LDP;
        for (int idx = t0; idx < TILE * TILE / 2; idx += nthr) {
            const int j = idx >> 5, h = idx & 31;
            if (j < nj && 2 * h < j) cp_async16(Ld + ((j * j) >> 1) + 2 * h, q.P + j0 + 2 * h + (int64_t)(j0 + j) * q.ld);
        }
        if (t0 < nj) cp_async8(sm + CH_DV + buf * TILE + t0, D.dinv + q.c0 + j0 + t0);
    };
    auto stage_tile = [&](int off, int I, int Jc, int t0, int nthr) {   // L(I,Jc): 64 columns x the 64 rows from the start of block
        const double* src = q.P + I * TILE + (int64_t)(Jc * TILE) * q.ld;   // I (rows past a ragged block meet zeros of xs), 16 B
        for (int idx = t0; idx < TILE * TILE / 2; idx += nthr) {
            const int c = idx >> 5, h = idx & 31;
            cp_async16(sm + off + c * TILE + 2 * h, src + (int64_t)c * q.ld + 2 * h);
        }
    };
    int J = nbp - 1;
    stage_diag(J, J & 1, tid, NT);
    cp_async_commit();
    if (tid < 2 * TILE) sm[CH_XS + tid] = 0.0;
    // dependencies: the forward half (two-sided solve) and the chunk tasks of the first block (the later blocks' chunk tasks are
    // checked two hops ahead of their use).  The chain itself reads nothing of the ancestors: the chunk tasks carry that
    // dependency (a supernode without rows below its pivots has no ancestors).
    if (tid == 0) {
        if (!fused) spin_until_ge(F.sol_done_f + s, ef * (uint32_t)F.target_f[s]);
        if (nchunk > 0) spin_until_ge(bu + J, epoch * (uint32_t)nchunk);
    }
    __syncthreads();
    double va_next = 0.0;                                           // threads 32..95: v - anc of the block the NEXT hop prepares
    {
        const int nj = min(TILE, q.w - J * TILE);
        if (tid < TILE) sm[CH_PRE + (J & 1) * TILE + tid] = tid < nj ? va_of(J, tid) : 0.0;
        if (J >= 1 && tid >= 32 && tid < 32 + TILE) {
            if (nchunk > 0) spin_until_ge(bu + J - 1, epoch * (uint32_t)nchunk);
            va_next = va_of(J - 1, tid - 32);
        }
    }
    cp_async_wait<0>();                                             // the first diagonal tile has landed
    __syncthreads();
#ifdef NMPC_TRACE_BUILD
    if (tr && tid == 0) { tr[2] = 0; tr[3] = 0; tr[5] = 0; tr[6] = 0; tr[7] = 0; }
#endif
    STRACE(1);
    for (; J >= 0; --J) {
        const int j0 = J * TILE, nj = min(TILE, q.w - j0);
        const double* pre = sm + CH_PRE + (J & 1) * TILE;
        const double* xprev = sm + CH_XS + ((J + 1) & 1) * TILE;    // x_{J+1} (zero padded)
        double* xcur = sm + CH_XS + (J & 1) * TILE;
        // A: z_J = pre_J - L(J+1,J)^T x_{J+1}  (block J is a full block when J + 1 < nbp)
        if (J + 1 < nbp) {
            const double* T1 = sm + CH_T1;
            const double xa = xprev[lane], xb = xprev[lane + 32];
            double v[8];
#pragma unroll
            for (int e = 0; e < 8; ++e) { const double* tc = T1 + (warp * 8 + e) * TILE; v[e] = fma(tc[lane + 32], xb, tc[lane] * xa); }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1)
#pragma unroll
                for (int e = 0; e < 8; ++e) v[e] += __shfl_xor_sync(FULL, v[e], o);
            double mine = v[0];
#pragma unroll
            for (int e = 1; e < 8; ++e) mine = lane == e ? v[e] : mine;
            if (lane < 8) zs[warp * 8 + lane] = pre[warp * 8 + lane] - mine;
        } else if (tid < TILE) {
            zs[tid] = pre[tid];
        }
        __syncthreads();
        const int Jn = J - 1;
        double* pren = sm + CH_PRE + (Jn & 1) * TILE;
        if (warp == 0) {
            // chain: L(J,J)^T x_J = z_J, pre-scaled substitution (s_i = d_i z_i): only (shuffle, fma) on the chain
            CHT0();
            const double* Ld = sm + CH_LD + (J & 1) * LDP;
            const double* dv = sm + CH_DV + (J & 1) * TILE;
            const bool h1 = lane + 32 < nj;
            const double d0 = lane < nj ? dv[lane] : 1.0, d1 = h1 ? dv[lane + 32] : 1.0;
            double z0 = lane < nj ? zs[lane] : 0.0, z1 = h1 ? zs[lane + 32] : 0.0;
            z0 *= d0; z1 *= d1;
            // packed column jr of L(J,J)^T = row jr of L(J,J): entries (jr, lane) and (jr, lane + 32) where they lie below the diagonal
            for (int jb = ((nj - 1) >> 3) << 3; jb >= 32; jb -= 8) {
                double la[8], lb[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const int jr = min(jb + e, nj - 1);
                    const double* row = Ld + ((jr * jr) >> 1);
                    la[e] = row[lane] * d0; lb[e] = row[min(lane + 32, jr - 1)] * d1;
                }
#pragma unroll
                for (int e = 7; e >= 0; --e) {
                    const int j = jb + e;
                    const double xj = __shfl_sync(FULL, z1, (j - 32) & 31);
                    const bool on = j < nj;
                    z1 = (on && lane + 32 < j) ? fma(-lb[e], xj, z1) : z1;
                    z0 = (on && lane < nj) ? fma(-la[e], xj, z0) : z0;
                }
            }
            for (int jb = ((min(nj, 32) - 1) >> 3) << 3; jb >= 0; jb -= 8) {
                double la[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const int jr = min(jb + e, nj - 1);
                    la[e] = Ld[((jr * jr) >> 1) + min(lane, max(jr - 1, 0))] * d0;
                }
#pragma unroll
                for (int e = 7; e >= 0; --e) {
                    const int j = jb + e;
                    const double xj = __shfl_sync(FULL, z0, j & 31);
                    z0 = (j < min(nj, 32) && lane < j) ? fma(-la[e], xj, z0) : z0;
                }
            }
            xcur[lane] = lane < nj ? z0 : 0.0;
            xcur[lane + 32] = h1 ? z1 : 0.0;
            if (lane == 0) CHT1(2);                                 // substitution
        } else if (warp <= 2) {
            // warps 1, 2 (thread t = column): publication of x_{J+1}, then S_{J-1} and v - anc of block J-2
            const int t = tid - 32;
            CHT0();
            double va2 = 0.0;
            if (J >= 2) {                                           // no dependency on the chain: used in the next hop
                if (nchunk > 0) spin_until_ge(bu + J - 2, epoch * (uint32_t)nchunk);
                va2 = va_of(J - 2, t);
            }
            if (J + 1 < nbp) {
                const int jp = (J + 1) * TILE, njp = min(TILE, q.w - jp);
                if (t < njp) { x[q.c0 + jp + t] = xprev[t]; put_solution(D, b, q.c0 + jp + t, xprev[t]); }
                bar_named(2, 2 * 32);
                if (t == 0) { __threadfence(); st_release(bb + J + 1, epoch); }   // for the helpers (nobody on the chain reads it)
            }
            if (J >= 1) {
                if (Jn + 3 <= nbp - 1) {                            // block J-1 is a full block
                    CHT0();
                    spin_until_ge(bs + Jn, epoch);
                    if (t == 0) CHT1(5);                            // waiting for the helper sum
                    va_next -= __ldcg(F.bsum + q.c0 + Jn * TILE + t);
                }
                bar_named(1, NT - 32);                              // warps 3..7 have written pren = - L(J+1,J-1)^T x_{J+1}
                pren[t] += va_next;
                va_next = va2;
            }
            if (t == 1) CHT1(6);
        } else {
            // warps 3..7: the product with T2 for block J-1, then the requests for the tiles of the next hop
            if (J >= 1) {
                const int ht = tid - 96, hn = NT - 96;
                CHT0();
                stage_tile(CH_T1, J, Jn, ht, hn);                   // next hop: L(J,J-1)^T x_J (T1 is free since the barrier after A)
                stage_diag(Jn, Jn & 1, ht, hn);
                cp_async_commit();
                if (J + 1 < nbp) {                                  // thirteen columns per warp, butterflies interleaved
                    const double* T2 = sm + CH_T2;
                    const double xa = xprev[lane], xb = xprev[lane + 32];
#pragma unroll
                    for (int kb = 0; kb < 13; kb += 5) {
                        double v[5];
#pragma unroll
                        for (int e = 0; e < 5; ++e) {
                            const int c = min(warp - 3 + 5 * (kb + e), TILE - 1);
                            v[e] = fma(T2[c * TILE + lane + 32], xb, T2[c * TILE + lane] * xa);
                        }
#pragma unroll
                        for (int o = 16; o > 0; o >>= 1)
#pragma unroll
                            for (int e = 0; e < 5; ++e) v[e] += __shfl_xor_sync(FULL, v[e], o);
#pragma unroll
                        for (int e = 0; e < 5; ++e) {
                            const int c = warp - 3 + 5 * (kb + e);
                            if (lane == 0 && kb + e < 13 && c < TILE) pren[c] = -v[e];
                        }
                    }
                } else if (ht < TILE) {
                    pren[ht] = 0.0;
                }
                bar_named(3, NT - 96);                              // the T2 buffer is free
                if (J >= 2) stage_tile(CH_T2, J, J - 2, ht, hn);    // next hop: L(J,J-2)^T x_J
                cp_async_commit();
                if (ht == 0) CHT1(3);
                bar_named(1, NT - 32);                              // pren is complete for warps 1, 2
                cp_async_wait<0>();                                 // the tiles of the next hop have landed
                if (ht == 0) CHT1(7);
            }
        }
        __syncthreads();
    }
    {
        const double* x0s = sm + CH_XS;                             // x_0
        const int nj0 = min(TILE, q.w);
        if (tid < nj0) { x[q.c0 + tid] = x0s[tid]; put_solution(D, b, q.c0 + tid, x0s[tid]); }
    }
    __syncthreads();
    if (tid == 0) { __threadfence(); st_release(bb, epoch); red_release_add(F.sol_done_b + s, 1u); }
}

__global__ void __launch_bounds__(NT, 2) solve_dag_kernel(DevSym D, DagPlan F, double* b, double* x, uint32_t ef, uint32_t eb,
                                                             const uint32_t* __restrict__ epoch_dev, int fused) {
    extern __shared__ __align__(16) double sm[];
    __shared__ int s_task, s_phase;
    if (epoch_dev) { ef = epoch_dev[0]; eb = epoch_dev[1]; }   // graph replay: the call numbers come from device memory
    const int n_fwd = F.n_sfwd, n_bwd = F.n_stasks - F.n_sfwd;
    const uint32_t base_f = (ef - 1u) * (uint32_t)(n_fwd + (int)gridDim.x), base_b = (eb - 1u) * (uint32_t)(n_bwd + (int)gridDim.x);
    if (threadIdx.x == 0) s_phase = fused ? 1 : 0;
    while (true) {
        __syncthreads();
        if (threadIdx.x == 0) {
            // the forward list is drained first (every CTA overshoots its counter exactly once), then the backward list
            int t = -1;
            if (s_phase == 0) {
                t = (int)(atomicAdd(F.sync + 1, 1u) - base_f);
                if (t < 0 || t >= n_fwd) { s_phase = 1; t = -1; }
            }
            if (s_phase == 1) {
                t = (int)(atomicAdd(F.sync + 2, 1u) - base_b);
                t = (t < 0 || t >= n_bwd) ? -1 : n_fwd + t;
            }
            s_task = t;
        }
        __syncthreads();
        const int t = s_task;
        if (t < 0) break;
        const int4 tk = F.stasks[t];
#ifdef NMPC_TRACE_BUILD
        unsigned long long* tr = F.strace ? F.strace + (size_t)t * 8 : nullptr;
        if (tr && threadIdx.x == 0) { unsigned long long g; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g)); tr[0] = g; }
#else
        unsigned long long* tr = nullptr;
#endif
        if (tk.w == 0) { if (tk.x == 0) fwd_small(D, F, tk.y, b, x, ef, sm, tr); else fwd_tiled(D, F, tk.y, tk.z, b, x, ef, sm); }
        else if (tk.x == 0) bwd_small(D, F, tk.y, b, x, ef, eb, fused != 0, sm, tr);
        else if (tk.x == 1) bwd_sum(D, F, tk.y, tk.z, x, eb, sm);
        else if (tk.x == 3) bwd_chain(D, F, tk.y, b, x, ef, eb, fused != 0, sm, tr);
        else                bwd_upd(D, F, tk.y, tk.z & 0xffff, tk.z >> 16, x, eb, sm);
        STRACE(4);
    }
}

}  // namespace

cudaError_t configure_solve_kernels(int max_smem_bytes, int small_max_r, int* ctas_per_sm, size_t* smem_bytes, int* sbuf_doubles) {
    int sbuf = ld_even(small_max_r) * SB;
    if (2 * sbuf < TILE * DLD) sbuf = (TILE * DLD + 1) / 2 + 1;      // the staged diagonal tile of the tiled tasks aliases the buffers
    sbuf = (sbuf + 1) & ~1;
    size_t bytes = (size_t)(OFF_BUF + 2 * sbuf + FWD_WORK_DOUBLES) * sizeof(double);
    bytes = std::max(bytes, (size_t)std::max(CH_END, UPD_END) * sizeof(double));   // the chain / chunk tasks of the backward solve
    if (bytes > (size_t)max_smem_bytes) return cudaErrorInvalidValue;
    cudaError_t e = cudaFuncSetAttribute(solve_dag_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem_bytes - 256);
    if (e != cudaSuccess) return e;
    int occ = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, solve_dag_kernel, NT, bytes);
    if (e != cudaSuccess) return e;
    *ctas_per_sm = occ < 1 ? 1 : occ;
    *smem_bytes = bytes;
    *sbuf_doubles = sbuf;
    return cudaSuccess;
}

void launch_solve(const DevSym& D, const DagPlan& F, double* rhs_inout, double* x, uint32_t epoch_f, uint32_t epoch_b,
                  const uint32_t* epoch_dev, bool fused, cudaStream_t st) {
    if (F.n_stasks > 0) solve_dag_kernel<<<F.sgrid, NT, F.ssmem, st>>>(D, F, rhs_inout, x, epoch_f, epoch_b, epoch_dev, fused ? 1 : 0);
}

}  // namespace nmpc
