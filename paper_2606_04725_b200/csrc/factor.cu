// factor.cu -- numeric multifrontal supernodal Cholesky (step a4, NumCholesky Eq. (20)-(21)) on the fixed
// structure S_L produced once by symbolic.cpp, as ONE persistent task-DAG kernel.
//
// The host analysis emits a topologically ordered task list (api.cu: build_plan).  CTAs claim tasks in order from an atomic
// counter and wait on completion flags (acquire/release at gpu scope) instead of kernel boundaries:
//   task type 0, small front (r <= small_max_r): ONE CTA assembles the whole front in shared memory (packed lower triangle):
//          K entries through the scatter map (before it waits for its children), extend-add of the children's update matrices
//          (child tables and relative indices fetched before the wait; small children loaded as one group, added in fixed
//          child order); panel-blocked partial Cholesky of its w pivot columns (partial_chol); publishes the (r-w)^2 update
//          matrix, then writes the panel of L.
//   task type 1, tile (I,J) of a tiled front (r > small_max_r; the front lives in HBM as panel + update storage), LEFT-looking:
//          assembles its tile first (K entries + children's contributions); acc = sum_k X(I,k) X(J,k)^T over the finished
//          tiles of block rows I and J (fp64 DMMA mma.sync.m8n8k4, operands streamed with cp.async.cg through a 4-stage
//          shared-memory ring; a chunk is multiplied before the warps wait for the flags of the chunk three ahead); C -= acc;
//          then POTRF (I == J; every finished 8-column block of L_JJ is stored and announced at once) or TRSM (I > J; streams
//          those blocks and runs one sub-step behind the POTRF) in shared memory; each tile is written exactly once.
// In-order claiming of a topological order cannot deadlock: the lowest-numbered unfinished task depends only on finished ones.
// fp64 throughout, no floating-point atomics, fixed summation order -> bitwise reproducible.
#include <climits>
#include <type_traits>

#include "device.h"

namespace nmpc {

namespace {

constexpr int NT = 256;                 // threads per CTA
constexpr int MAXCH = 24;               // children whose tables a small-front task keeps in shared memory (else: one by one)
constexpr int RELCAP = 2048;            // total relative indices of those children
constexpr int SMALL_WORK_DOUBLES = (2 * MAXCH * 8 + (2 * MAXCH + 4) * 4 + RELCAP * 4 + 7) / 8;
constexpr int KC = 16;                  // k-columns per pipeline stage
constexpr int ALD = 68;                 // leading dimension of an operand stage  (68 mod 16 == 4: conflict-free DMMA fragment loads)
constexpr int CLD = 66;                 // leading dimension of the C / L_JJ tile (2*66 mod 16 == 4: conflict-free fragment stores)
constexpr int NSTAGE = 4;
constexpr int TCH = 128;                // children whose tables a tile task fetches at once
constexpr int STAGE_DOUBLES = 2 * KC * ALD;
constexpr int PIPE_DOUBLES = NSTAGE * STAGE_DOUBLES;          // 8704
constexpr int CT_DOUBLES = TILE * CLD;                        // 4224
constexpr int TILE_SMEM_DOUBLES = PIPE_DOUBLES + CT_DOUBLES;  // 12928 doubles = 103424 B
static_assert(CT_DOUBLES + TILE <= PIPE_DOUBLES, "L_JJ tile + reciprocals alias the operand ring");

// ---- gpu-scope acquire / release on the completion flags ----
// Publishing: all threads store, CTA barrier, then ONE thread fences and releases the flag (the release is cumulative over
// what the barrier ordered before it -- the pattern of a grid-wide barrier).  Consuming: one thread acquires, CTA barrier
// (or __syncwarp), then everybody reads the produced data with ld.global.cg.
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
__device__ __forceinline__ void red_release_max(uint32_t* p, uint32_t v) {
    asm volatile("red.relaxed.gpu.global.max.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
#ifdef NMPC_TRACE_BUILD                     // measurement build: timestamps per task + the time thread 0 spends waiting on flags
__device__ __forceinline__ unsigned long long gtime() { unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }
__shared__ unsigned long long s_wait_ns;
#define TRACE(slot) do { if (tr && threadIdx.x == 0) { tr[slot] = gtime(); if ((slot) == 4) tr[6] = s_wait_ns; } } while (0)
__device__ __forceinline__ void spin_until_ge(const uint32_t* p, uint32_t target) {
    if (threadIdx.x != 0) { while (ld_acquire(p) < target) __nanosleep(40); return; }
    const unsigned long long t0 = gtime();
    while (ld_acquire(p) < target) __nanosleep(40);
    s_wait_ns += gtime() - t0;
}
#else
#define TRACE(slot) do { (void)tr; } while (0)
__device__ __forceinline__ void spin_until_ge(const uint32_t* p, uint32_t target) {
    while (ld_acquire(p) < target) __nanosleep(40);
}
#endif
__device__ __forceinline__ void cp_async16(double* dst_smem, const double* src, int src_bytes) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(dst_smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(d), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
// mbarrier helpers (shared-memory arrive / wait objects): the operand ring of the tile product hands its stages over with a
// "full" word per stage (every thread's cp.async group arrives on it when it has landed) and an "empty" word (one arrival per
// warp that has finished multiplying the stage), so no CTA-wide barrier sits in the product loop and the warps may drift by a chunk.
__device__ __forceinline__ unsigned smem_addr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* b, int n) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(b)), "r"(n) : "memory"); }
__device__ __forceinline__ void mbar_arrive(uint64_t* b) { asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_addr(b)) : "memory"); }
__device__ __forceinline__ void mbar_cp_async_arrive(uint64_t* b) { asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_addr(b)) : "memory"); }
__device__ __forceinline__ void mbar_wait(uint64_t* b, uint32_t parity) {
    asm volatile("{\n.reg .pred p;\nMBW: mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n@p bra MBD;\nbra MBW;\nMBD:\n}" ::"r"(smem_addr(b)), "r"(parity) : "memory");
}
// the same on shared-window addresses (the product loop converts its pointers once per tile, not once per instruction)
__device__ __forceinline__ void mbar_arrive_s(unsigned a) { asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(a) : "memory"); }
__device__ __forceinline__ void mbar_cp_async_arrive_s(unsigned a) { asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(a) : "memory"); }
__device__ __forceinline__ void mbar_wait_s(unsigned a, uint32_t parity) {
    asm volatile("{\n.reg .pred p;\nMBWS: mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n@!p bra MBWS;\n}" ::"r"(a), "r"(parity) : "memory");
}
// two 16-byte copies 256 bytes apart on both sides (one k-column of an operand is 512 contiguous bytes): immediate offsets, one address each
template <int DOFF>
__device__ __forceinline__ void cp_async16x2_s(unsigned d, const double* src) {
    asm volatile("cp.async.cg.shared.global [%0+%2], [%1], 16;\n\tcp.async.cg.shared.global [%0+%3], [%1+256], 16;" ::"r"(d), "l"(src), "n"(DOFF), "n"(DOFF + 256) : "memory");
}
// 1/sqrt(d) for a normal d > 0: hardware approximation (rsqrt.approx.f64, ~2^-22) + two Newton steps -> rounding level
__device__ __forceinline__ double rsqrt_newton(double d) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(d));
    const double h = 0.5 * d;
    double e = fma(-h * y, y, 0.5);
    y = fma(y, e, y);
    e = fma(-h * y, y, 0.5);
    y = fma(y, e, y);
    return y;
}
__device__ __forceinline__ void dmma(double (&c)[2], double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}

// =============================================================================================================
// Blocked partial Cholesky of the first w columns of an r x r lower-stored matrix in shared memory (Eq. 21).
// colp(j)[i] addresses element (i,j), i >= j.  Two-level blocking: panels of 32 columns, sub-steps of 8 columns, and the
// factorization of the NEXT 8x8 diagonal block is software-pipelined into the update of the current sub-step:
//   row solve:   thread t solves row j0+t of the block column against the finished diagonal block (x = f L_D^-T); barrier;
//   update:      rank-8 DMMA update of the rest of the panel (<= 24 columns); at a panel end the rank-32 DMMA update of the
//                trailing columns (8 chained mma.m8n8k4 per 8x8 tile).  Warp 0 takes the tile that holds the next diagonal
//                block first and then factors that block in registers (serial pivot chain: hardware rsqrt + two Newton
//                steps, L_jj = d * rsqrt(d)) while warps 1..7 work through the other tiles, two in flight per warp; barrier.
// DMMA operands come straight from the finished columns of the front, loads are unconditional with clamped indices
// (no divergence).  Requires r <= NT.  A pivot <= 0 or non-finite (reading G11) is replaced by 1 and reported.
// =============================================================================================================
template <class ColFn>
__device__ __forceinline__ void factor_diag8(ColFn colp, int j0, int jb, int c0, int aug_col, int32_t* fail_col, double* dinv, double* s_inv) {
    // The 8x8 block is spread over the warp: lane (i << 2) | q holds the entries (i, q) and (i, q + 4); operands are broadcast with
    // shuffles (measurements behind this form: profiles/r02b_potrf_phases.md).
    const int lane = threadIdx.x & 31, i = lane >> 2, q = lane & 3;
    const unsigned FULLM = 0xffffffffu;
    double a0, a1;                                       // entries (i, q), (i, q + 4); outside the block / above the diagonal: 0 (diagonal 1)
    {
        const int il = min(i, jb - 1);
        const double v0 = colp(j0 + min(q, jb - 1))[j0 + il], v1 = colp(j0 + min(q + 4, jb - 1))[j0 + il];
        a0 = (i < jb && q < jb && i >= q) ? v0 : ((i == q && i >= jb) ? 1.0 : 0.0);
        a1 = (i < jb && q + 4 < jb && i >= q + 4) ? v1 : ((i == q + 4 && i >= jb) ? 1.0 : 0.0);
    }
    // The pivots are a serial chain, and every dependent fp64 operation on it costs ~30 cycles behind the neighbour CTA's DMMA stream.
    // The elimination is therefore square-root free with the columns left UNSCALED: a_ik -= (a_ic a_kc) (1 / d_c), the products formed
    // while 1 / d_c (approximation + one cubic step) is on its way, so a pivot costs a shuffle, the reciprocal and one fma on the
    // chain.  The scaling L_ic = a_ic / sqrt(d_c) happens once at the end, the eight reciprocal square roots side by side in lanes 0..7.
    int badc = 8;
    double myd = 1.0;                                    // lane c keeps the pivot d_c (1 for a bad one)
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        const double src = (c < 4) ? a0 : a1;            // the half that holds column c
        double d = __shfl_sync(FULLM, src, (c << 2) | (c & 3));
        // the right-hand-side row (device.h: aug_col) is the last pivot of all: taken as 1, never tested
        if (c0 + j0 + c == aug_col) d = 1.0;
        const bool bad = !(d >= 2.2250738585072014e-308) || isinf(d);          // <= 0, non-finite (or subnormal): reading G11
        if (bad && c < jb && badc == 8) badc = c;
        if (bad || c0 + j0 + c == aug_col) {             // the pivot becomes 1: the column below it stays as it is
            d = 1.0;
            if (lane == ((c << 2) | (c & 3))) { if (c < 4) a0 = 1.0; else a1 = 1.0; }
        }
        myd = (lane == c) ? d : myd;
        const double lic = __shfl_sync(FULLM, src, (lane & ~3) | (c & 3));
        const double lk0 = __shfl_sync(FULLM, src, (q << 2) | (c & 3));
        const double lk1 = __shfl_sync(FULLM, src, ((q + 4) << 2) | (c & 3));
        const double p0 = lic * lk0, p1 = lic * lk1;     // before 1 / d is known
        double rc;
        asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(rc) : "d"(d));
        const double e = fma(-d, rc, 1.0);
        rc = fma(rc, fma(e, e, e), rc);                  // one cubic step: rc (1 + e + e^2), error e^3 ~ 2^-66 before rounding
        if (q > c && i >= q) a0 = fma(-p0, rc, a0);
        if (q + 4 > c && i >= q + 4) a1 = fma(-p1, rc, a1);
    }
    const double myinv = rsqrt_newton(myd);              // lanes 0..7: 1 / sqrt(d_lane)
    a0 *= __shfl_sync(FULLM, myinv, q);                  // L_iq = a_iq / sqrt(d_q); the diagonal: d / sqrt(d)
    a1 *= __shfl_sync(FULLM, myinv, q + 4);
    if (badc < 8 && lane == 0) atomicMin(fail_col, c0 + j0 + badc);
    if (lane < jb) { dinv[c0 + j0 + lane] = myinv; s_inv[lane] = myinv; }
    if (i < jb) {                                        // every lane stores its own entries of the factored block
        if (q < jb && i >= q) colp(j0 + q)[j0 + i] = a0;
        if (q + 4 < jb && i >= q + 4) colp(j0 + q + 4)[j0 + i] = a1;
    }
}

#ifdef NMPC_TRACE_BUILD
// measurement build: clock cycles thread 0 spends per phase of the POTRF of diagonal tiles (partial_chol with CW = 4), summed
// over all such tasks: [0] waiting for the row solve, [1] its tile update, [2] factor_diag8, [3] waiting at the end of the update,
// [4] sub-steps, [5] whole partial_chol
__device__ unsigned long long g_potrf_cycles[8];
#define PCLK(v) const long long v = clock64()
#define PACC(slot, a, b) do { if (r == w && r <= TILE && tid == 0) atomicAdd(&g_potrf_cycles[slot], (unsigned long long)((b) - (a))); } while (0)
#else
#define PCLK(v) do {} while (0)
#define PACC(slot, a, b) do {} while (0)
#endif
__shared__ uint64_t s_full[NSTAGE], s_empty[NSTAGE];    // operand ring of the tile product (initialised once per kernel)
__shared__ double s_inv8[8];                            // reciprocal pivots of the current 8 x 8 diagonal block (partial_chol)
__shared__ int s_all;                                   // trsm_tile: L_JJ was complete when the task looked
struct NoPublish { __device__ __forceinline__ void operator()(int, int) const {} };
// pub(j0, jb) is called by all threads right after the barrier that ends the row solve of columns [j0, j0 + jb): those columns
// are final from then on (the diagonal tile of a tiled front streams them to the TRSM tiles of its block column)
// CW = number of warps that COMPUTE (warp 0 .. CW-1; requires r <= 32 CW: one row-solving thread per row).  The diagonal tile of
// a tiled front runs with CW = 4: warps 4..7 only publish (store the finished columns, fence, flag); they meet the computing warps
// at the barrier after each row solve and stay out of the update and of the barrier that ends it, so the ~1 us of the
// publishing thread's fence overlaps the next update / row solve instead of sitting on the chain of every sub-step.
// RW > 0: r = w = RW at compile time (the full 64 x 64 diagonal tile of a tiled front: every clamp, mask and ragged-edge test of
// the general code folds away on the chain of the front).
template <class ColFn, class Pub = NoPublish, int CW = NT / 32, int RW = 0>
__device__ __forceinline__ void partial_chol(ColFn colp, int r_in, int w_in, int c0, int aug_col, int32_t* fail_col, double* dinv, Pub pub = Pub()) {
    const int r = RW ? RW : r_in, w = RW ? RW : w_in;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, gid = lane >> 2, tig = lane & 3;
    constexpr int NW1 = CW - 1;                          // warps 1..CW-1 share the tiles warp 0 does not take
    auto end_of_update = [&]() {
        if (CW == NT / 32) __syncthreads();
        else if (warp < CW) asm volatile("bar.sync 2, %0;" ::"n"(CW * 32) : "memory");
    };
    double* const s_inv = s_inv8;
    const int rl = r - 1;
    PCLK(pc_begin);
    if (warp == 0) factor_diag8(colp, 0, min(8, w), c0, aug_col, fail_col, dinv, s_inv);
    __syncthreads();
    for (int p0 = 0; p0 < w; p0 += 32) {
        const int p1 = min(w, p0 + 32);
        for (int j0 = p0; j0 < p1; j0 += 8) {
            const int jb = min(8, p1 - j0);
            const int t0 = j0 + jb;
            PCLK(pc0);
            if (tid >= jb && j0 + tid < r) {             // a row below the diagonal block: x = f L_D^-T (right-looking over the 8 columns)
                const int i = j0 + tid;
                double x[8], Lk[8][8], inv[8];
                if (jb == 8) {
#pragma unroll
                    for (int c = 0; c < 8; ++c) {
                        const double* cp = colp(j0 + c);
                        x[c] = cp[i];
                        inv[c] = s_inv[c];
#pragma unroll
                        for (int k = c + 1; k < 8; ++k) Lk[k][c] = cp[j0 + k];
                    }
                } else {
#pragma unroll
                    for (int c = 0; c < 8; ++c) {
                        const double* cp = colp(j0 + min(c, jb - 1));
                        const double xv = cp[i], iv = s_inv[min(c, jb - 1)];
                        x[c] = (c < jb) ? xv : 0.0;
                        inv[c] = (c < jb) ? iv : 1.0;
#pragma unroll
                        for (int k = c + 1; k < 8; ++k) { const double v = cp[j0 + min(k, jb - 1)]; Lk[k][c] = (k < jb) ? v : 0.0; }
                    }
                }
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    x[k] *= inv[k];
#pragma unroll
                    for (int c = k + 1; c < 8; ++c) x[c] = fma(-x[k], Lk[c][k], x[c]);
                }
#pragma unroll
                for (int c = 0; c < 8; ++c)
                    if (c < jb) colp(j0 + c)[i] = x[c];
            }
            __syncthreads();
            PCLK(pc1);
            PACC(0, pc0, pc1); PACC(4, 0, 1);
            pub(j0, jb);
            const bool has_next = t0 < w;
            if (t0 < p1) {                               // rank-8 update of the panel's remaining columns [t0, p1)
                const bool k0 = tig < jb, k1 = tig + 4 < jb;
                const double* ck0 = colp(j0 + (k0 ? tig : 0));
                const double* ck1 = colp(j0 + (k1 ? tig + 4 : 0));
                const int TU = (r - t0 + 7) >> 3, TV = (p1 - t0 + 7) >> 3, ntile = TU * TV;
                const float rTU = 1.0f / (float)TU;       // V = q / TU as (q + 0.5) * (1 / TU): exact for q < 2^12, three instructions
                auto pair = [&](int qa, int qb, auto cnt) {
                    constexpr int NE = decltype(cnt)::value;      // 2: two tiles in flight; 1: warp 0, whose one tile is on the chain
                    double acc[2][2], cold[2][2];
                    double* pc[2][2];
                    bool ok[2][2];
#pragma unroll
                    for (int e = 0; e < NE; ++e) {
                        const int qq = e ? qb : qa;
                        const int q = min(qq, ntile - 1);
                        const int V = (int)(((float)q + 0.5f) * rTU), U = q - V * TU;
                        const int u = t0 + 8 * U + gid, vb = t0 + 8 * V + gid, vc = t0 + 8 * V + 2 * tig;
                        const bool live = qq < ntile && U >= V;
                        const int ucl = min(u, rl), vbl = min(vb, rl);
                        const double a0 = ck0[ucl], a1 = ck1[ucl], b0 = ck0[vbl], b1 = ck1[vbl];
                        ok[e][0] = live && u < r && vc < p1 && u >= vc;
                        ok[e][1] = live && u < r && vc + 1 < p1 && u >= vc + 1;
                        pc[e][0] = colp(min(vc, rl)) + ucl;
                        pc[e][1] = colp(min(vc + 1, rl)) + ucl;
                        cold[e][0] = *pc[e][0];
                        cold[e][1] = *pc[e][1];
                        acc[e][0] = acc[e][1] = 0.0;
                        dmma(acc[e], (live && k0) ? a0 : 0.0, k0 ? b0 : 0.0);
                        dmma(acc[e], (live && k1) ? a1 : 0.0, k1 ? b1 : 0.0);
                    }
#pragma unroll
                    for (int e = 0; e < NE; ++e) {
                        if (ok[e][0]) *pc[e][0] = cold[e][0] - acc[e][0];
                        if (ok[e][1]) *pc[e][1] = cold[e][1] - acc[e][1];
                    }
                };
                if (warp == 0) {
                    pair(0, ntile, std::integral_constant<int, 1>());   // the tile of the next diagonal block, then that block's factorization
                    __syncwarp();
                    PCLK(pc2);
                    factor_diag8(colp, t0, min(8, p1 - t0), c0, aug_col, fail_col, dinv, s_inv);
                    PCLK(pc3);
                    PACC(1, pc1, pc2); PACC(2, pc2, pc3);
                } else if (warp < CW) {
                    for (int q = warp; q < ntile; q += 2 * NW1) pair(q, q + NW1, std::integral_constant<int, 2>());
                }
            } else if (p1 < r) {                         // panel end: rank-(p1-p0) update of the trailing columns [p1, r)
                const double* ck[8];
                bool kv[8];
#pragma unroll
                for (int s8 = 0; s8 < 8; ++s8) { const int kc = p0 + 4 * s8 + tig; kv[s8] = kc < p1; ck[s8] = colp(kv[s8] ? kc : p0); }
                const int T = (r - p1 + 7) >> 3, ntile = (T * (T + 1)) >> 1;
                auto pair = [&](int qa, int qb, auto cnt) {
                    constexpr int NE = decltype(cnt)::value;
                    double acc[2][2], cold[2][2];
                    double* pc[2][2];
                    bool ok[2][2];
                    int ucl[2], vbl[2];
#pragma unroll
                    for (int e = 0; e < NE; ++e) {
                        const int qq = e ? qb : qa;
                        const int q = min(qq, ntile - 1);
                        int U = (int)((sqrtf(8.0f * (float)q + 1.0f) - 1.0f) * 0.5f);
                        U += (((U + 1) * (U + 2)) >> 1 <= q) - (((U * (U + 1)) >> 1) > q);      // float rounding: off by at most one
                        const int V = q - ((U * (U + 1)) >> 1);
                        const bool live = qq < ntile;
                        const int u = p1 + 8 * U + gid, vb = p1 + 8 * V + gid, vc = p1 + 8 * V + 2 * tig;
                        ucl[e] = min(u, rl); vbl[e] = min(vb, rl);
                        ok[e][0] = live && u < r && vc < r && u >= vc;
                        ok[e][1] = live && u < r && vc + 1 < r && u >= vc + 1;
                        pc[e][0] = colp(min(vc, rl)) + ucl[e];
                        pc[e][1] = colp(min(vc + 1, rl)) + ucl[e];
                        cold[e][0] = *pc[e][0];
                        cold[e][1] = *pc[e][1];
                        acc[e][0] = acc[e][1] = 0.0;
                    }
#pragma unroll
                    for (int s8 = 0; s8 < 8; ++s8) {
                        double a[2], b[2];
#pragma unroll
                        for (int e = 0; e < NE; ++e) { a[e] = ck[s8][ucl[e]]; b[e] = ck[s8][vbl[e]]; }
#pragma unroll
                        for (int e = 0; e < NE; ++e) dmma(acc[e], kv[s8] ? a[e] : 0.0, kv[s8] ? b[e] : 0.0);
                    }
#pragma unroll
                    for (int e = 0; e < NE; ++e) {
                        if (ok[e][0]) *pc[e][0] = cold[e][0] - acc[e][0];
                        if (ok[e][1]) *pc[e][1] = cold[e][1] - acc[e][1];
                    }
                };
                if (warp == 0) {
                    pair(0, ntile, std::integral_constant<int, 1>());
                    __syncwarp();
                    PCLK(pc2);
                    if (has_next) factor_diag8(colp, p1, min(8, w - p1), c0, aug_col, fail_col, dinv, s_inv);
                    PCLK(pc3);
                    PACC(1, pc1, pc2); PACC(2, pc2, pc3);
                } else if (warp < CW) {
                    for (int q = warp; q < ntile; q += 2 * NW1) pair(q, q + NW1, std::integral_constant<int, 2>());
                }
            }
            PCLK(pc4);
            end_of_update();
            PCLK(pc5);
            PACC(3, pc4, pc5);
        }
    }
    PCLK(pc_end);
    PACC(5, pc_begin, pc_end);
}

// X = C L^-T for an ni x nj tile C (column-major, CLD) against the nj x nj lower-triangular Ls (column-major, CLD), in
// place, same panel scheme: thread i substitutes 8 columns of row i, the rest of the 32-column panel gets a rank-8 DMMA
// update, the columns after the panel a rank-32 one.  Rows >= ni / columns >= nj of the tiles are finite padding.
// The columns of L_JJ arrive in 8-column blocks as the diagonal task publishes them (sub[0] counts them, `sbase` = value before
// this call's first block): block k is fetched from the panel in global memory (Lg, leading dimension ldg) right before
// sub-step k needs it, so the TRSM runs one sub-step behind the POTRF instead of after it.  Xg: the tile of the panel that
// receives X (same leading dimension ldg); finished entries are stored by the thread that solved them.
template <bool FULL>                                    // FULL: ni = nj = TILE at compile time (no ragged-edge masks)
__device__ __forceinline__ void trsm_tile(double* Cs, double* Ls, double* rinv, int ni_in, int nj_in, const uint32_t* sub, uint32_t sbase,
                                          const double* __restrict__ Lg, int ldg, const double* __restrict__ dinv_g, double* __restrict__ Xg) {
    const int ni = FULL ? TILE : ni_in, nj = FULL ? TILE : nj_in;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, gid = lane >> 2, tig = lane & 3;
    constexpr int NW = NT / 32;
    const int TU = (ni + 7) >> 3;
    const float rTU = 1.0f / (float)TU;                  // q / TU as (q + 0.5) * (1 / TU): exact for q < 2^12
    // a tile that is not right behind its POTRF finds L_JJ complete: one fetch of the whole triangle instead of one round trip
    // to L2 per sub-step
    if (tid == 0) s_all = ld_acquire(sub) >= sbase + (uint32_t)((nj + 7) >> 3);
    __syncthreads();
    const bool all = s_all != 0;
    if (all) {
        {
            const int ii = tid & (TILE - 1);
            if (ii < nj)
                for (int cc0 = tid >> 6; cc0 <= ii; cc0 += 8 * (NT / TILE)) {   // eight loads in flight
                    double v[8];
#pragma unroll
                    for (int e = 0; e < 8; ++e) { const int cc = cc0 + e * (NT / TILE); v[e] = cc <= ii ? __ldcg(Lg + ii + (int64_t)cc * ldg) : 0.0; }
#pragma unroll
                    for (int e = 0; e < 8; ++e) { const int cc = cc0 + e * (NT / TILE); if (cc <= ii) Ls[cc * CLD + ii] = v[e]; }
                }
        }
        if (tid < nj) rinv[tid] = __ldcg(dinv_g + tid);
        __syncthreads();
    }
    for (int p0 = 0; p0 < nj; p0 += 32) {
        const int p1 = min(nj, p0 + 32);
        for (int j0 = p0; j0 < p1; j0 += 8) {
            const int jb = min(8, p1 - j0), t0 = j0 + jb;
            if (!all) {   // fetch columns [j0, j0 + jb) of L_JJ (rows j0 .. nj-1) and their pivot reciprocals
                if (lane == 0) spin_until_ge(sub, sbase + (uint32_t)(j0 >> 3) + 1u);
                __syncwarp();
                const int nr = nj - j0;
                if (warp < jb)                           // one warp per column of the block
                    for (int ii = lane; ii < nr; ii += 32) Ls[(j0 + warp) * CLD + j0 + ii] = __ldcg(Lg + (j0 + ii) + (int64_t)(j0 + warp) * ldg);
                if (tid < jb) rinv[j0 + tid] = __ldcg(dinv_g + j0 + tid);
                __syncthreads();
            }
            if (tid < ni) {
                double x[8], Lk[8][8], inv[8];
#pragma unroll
                for (int c = 0; c < 8; ++c) {
                    const int cc = j0 + min(c, jb - 1);
                    const double xv = Cs[cc * CLD + tid], iv = rinv[cc];
                    x[c] = (c < jb) ? xv : 0.0;
                    inv[c] = (c < jb) ? iv : 1.0;
#pragma unroll
                    for (int k = c + 1; k < 8; ++k) { const double v = Ls[cc * CLD + j0 + min(k, jb - 1)]; Lk[k][c] = (k < jb) ? v : 0.0; }
                }
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    x[k] *= inv[k];
#pragma unroll
                    for (int c = k + 1; c < 8; ++c) x[c] = fma(-x[k], Lk[c][k], x[c]);
                }
#pragma unroll
                for (int c = 0; c < 8; ++c)
                    if (c < jb) { Cs[(j0 + c) * CLD + tid] = x[c]; Xg[tid + (int64_t)(j0 + c) * ldg] = x[c]; }   // final: straight to the panel
            }
            __syncthreads();
            if (t0 < p1) {
                const bool k0 = tig < jb, k1 = tig + 4 < jb;
                const int kc0 = j0 + (k0 ? tig : 0), kc1 = j0 + (k1 ? tig + 4 : 0);
                const int TV = (p1 - t0 + 7) >> 3;
                for (int q = warp; q < TU * TV; q += NW) {
                    const int V = (int)(((float)q + 0.5f) * rTU), U = q - V * TU;
                    const int u = 8 * U + gid, v0 = t0 + 8 * V + 2 * tig, vb = min(t0 + 8 * V + gid, TILE - 1);
                    const double a0 = Cs[kc0 * CLD + u], a1 = Cs[kc1 * CLD + u];
                    const double b0 = Ls[kc0 * CLD + vb], b1 = Ls[kc1 * CLD + vb];
                    const bool ok0 = v0 < p1, ok1 = v0 + 1 < p1;
                    double* pc = Cs + min(v0, TILE - 2) * CLD + u;
                    const double c0v = pc[0], c1v = pc[CLD];
                    double acc[2] = {0.0, 0.0};
                    dmma(acc, k0 ? a0 : 0.0, k0 ? b0 : 0.0);
                    dmma(acc, k1 ? a1 : 0.0, k1 ? b1 : 0.0);
                    if (ok0) pc[0] = c0v - acc[0];
                    if (ok1) pc[CLD] = c1v - acc[1];
                }
                __syncthreads();
            }
        }
        if (p1 < nj) {
            const int TV = (nj - p1 + 7) >> 3;
            for (int q = warp; q < TU * TV; q += NW) {
                const int V = (int)(((float)q + 0.5f) * rTU), U = q - V * TU;
                const int u = 8 * U + gid, v0 = p1 + 8 * V + 2 * tig, vb = min(p1 + 8 * V + gid, TILE - 1);
                const bool ok0 = v0 < nj, ok1 = v0 + 1 < nj;
                double* pc = Cs + min(v0, TILE - 2) * CLD + u;
                const double c0v = pc[0], c1v = pc[CLD];
                double acc[2] = {0.0, 0.0};
#pragma unroll
                for (int s8 = 0; s8 < 8; ++s8) {
                    const int kc = p0 + 4 * s8 + tig;
                    const bool kv = kc < p1;
                    const int kcl = kv ? kc : p0;
                    dmma(acc, kv ? Cs[kcl * CLD + u] : 0.0, kv ? Ls[kcl * CLD + vb] : 0.0);
                }
                if (ok0) pc[0] = c0v - acc[0];
                if (ok1) pc[CLD] = c1v - acc[1];
            }
            __syncthreads();
        }
    }
}

// =============================================================================================================
// task type 0: whole front in shared memory, packed lower triangle: element (i,j), i >= j, at j*r - j(j-1)/2 + (i-j)
// =============================================================================================================
__device__ __forceinline__ void small_front_task(const DevSym& D, const DagPlan& F, int s, const double* __restrict__ Kval,
                                                 double eta, uint32_t epoch, double* sm, unsigned long long* tr) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarp = NT / 32;
    const int c0 = D.sn_start[s], w = D.sn_start[s + 1] - c0;
    const int r = (int)(D.rows_ptr[s + 1] - D.rows_ptr[s]);
    const int ch0 = D.child_ptr[s], ch1 = D.child_ptr[s + 1];
    const int64_t kq0 = D.kent_ptr[s], kq1 = D.kent_ptr[s + 1];
    uint32_t* front_done = F.fac_done;
    auto colp = [sm, r](int j) { return sm + (j * r - ((j * (j - 1)) >> 1) - j); };
    const int ntri = (r * (r + 1)) >> 1;
    // work area behind the front: child table + the relative indices of ALL children (fetched before the children are waited for)
    long long* chRp = reinterpret_cast<long long*>(sm + ((ntri + 1) & ~1));   // [MAXCH] rel_ptr of the child
    long long* chUp = chRp + MAXCH;                                           // [MAXCH] upd_ptr of the child
    int* chMc = reinterpret_cast<int*>(chUp + MAXCH);                         // [MAXCH] rows of the child's update matrix
    int* chOff = chMc + MAXCH;                                                // [MAXCH + 1] offset of its list in relS
    int* relS = chOff + MAXCH + 2;                                            // [RELCAP] (fast path) / 2 x NT (fallback)
    const int nch = ch1 - ch0;
    // everything that does not depend on the children first: zero, K entries, eta, child table, relative indices
    for (int idx = tid; idx < ntri; idx += NT) sm[idx] = 0.0;
    int myc = -1;
    if (tid < nch) {
        myc = D.child_idx[ch0 + tid];
        if (nch <= MAXCH) {
            const long long rp0 = D.rel_ptr[myc];
            chRp[tid] = rp0; chMc[tid] = (int)(D.rel_ptr[myc + 1] - rp0); chUp[tid] = D.upd_ptr[myc];
        }
    }
    __syncthreads();
    for (int64_t q = kq0 + tid; q < kq1; q += NT) sm[D.kent_dst[q]] = Kval[D.kent_src[q]];
    if (tid == 0 && nch <= MAXCH) { int off = 0; for (int i = 0; i < nch; ++i) { chOff[i] = off; off += chMc[i]; } chOff[nch] = off; }
    __syncthreads();
    if (eta != 0.0) for (int j = tid; j < w; j += NT) colp(j)[j] += eta;
    const bool fast = nch <= MAXCH && chOff[nch <= MAXCH ? nch : 0] <= RELCAP;
    if (fast) {
        const int tot_rel = chOff[nch];
#pragma unroll 4
        for (int idx = tid; idx < tot_rel; idx += NT) {
            int i = 0;
            while (idx >= chOff[i + 1]) ++i;
            relS[idx] = D.rel[chRp[i] + (idx - chOff[i])];
        }
    }
    for (int ci = tid; ci < nch; ci += NT) {             // wait for the children (thread ci < NT holds its child in myc)
        const int c = ci == tid && myc >= 0 ? myc : D.child_idx[ch0 + ci];
        spin_until_ge(front_done + c, epoch * (uint32_t)F.target[c]);
    }
    __syncthreads();
    TRACE(1);
    auto entry = [&](int mc, const int* rb, const double* Uc, int f, double& v, int& dst) {
        // columns b and mc-1-b of a child's lower triangle together hold mc+1 entries: a balanced flat index space
        const int per = mc + 1;
        const int p = f / per, e = f - p * per;
        int a, b2;
        if (e < mc - p) { b2 = p; a = p + e; }
        else { b2 = mc - 1 - p; a = b2 + (e - (mc - p)); }
        dst = -1; v = 0.0;
        if (b2 != p || e < mc - p) {                     // the middle column of an odd mc is its own partner: count it once
            const int j = rb[b2], i = rb[a];
            dst = j * r - ((j * (j - 1)) >> 1) + (i - j);
            v = __ldcg(Uc + a + (int64_t)b2 * mc);
        }
    };
    if (fast) {
        // children are taken in their fixed order.  Consecutive small children whose entries together fit one batch (8 per
        // thread) are LOADED together (one round trip to L2 for the group) and ADDED one child after the other (a barrier
        // between children: two children may hit the same entry of the front, the order of the additions is fixed).
        int i = 0;
        while (i < nch) {
            const int mci = chMc[i];
            const int toti = ((mci + 1) >> 1) * (mci + 1);
            if (toti > 8 * NT) {                         // a big child on its own, several batches
                const int* rb = relS + chOff[i];
                const double* Uc = D.U + chUp[i];
                for (int f0 = tid; f0 < toti; f0 += 8 * NT) {
                    double v[8];
                    int dst[8];
#pragma unroll
                    for (int k = 0; k < 8; ++k) { dst[k] = -1; v[k] = 0.0; if (f0 + k * NT < toti) entry(mci, rb, Uc, f0 + k * NT, v[k], dst[k]); }
#pragma unroll
                    for (int k = 0; k < 8; ++k)
                        if (dst[k] >= 0) sm[dst[k]] += v[k];
                }
                __syncthreads();
                ++i;
                continue;
            }
            int e = i, gtot = 0;                         // group [i, e): cumulative entry counts in cum[]
            int cum[9];
            cum[0] = 0;
#pragma unroll
            for (int g = 0; g < 8; ++g) {
                int tg = 0;
                if (e < nch && e == i + g) { const int m2 = chMc[e]; tg = ((m2 + 1) >> 1) * (m2 + 1); if (gtot + tg <= 8 * NT) { gtot += tg; ++e; } }
                cum[g + 1] = gtot;
            }
            double v[8];
            int dst[8], who[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const int Fk = tid + k * NT;
                dst[k] = -1; v[k] = 0.0; who[k] = -1;
                if (Fk < gtot) {
                    int g = 0;
#pragma unroll
                    for (int t2 = 1; t2 < 8; ++t2) g += (Fk >= cum[t2] && i + t2 < e) ? 1 : 0;
                    who[k] = g;
                    entry(chMc[i + g], relS + chOff[i + g], D.U + chUp[i + g], Fk - cum[g], v[k], dst[k]);
                }
            }
            for (int g = 0; g < e - i; ++g) {
#pragma unroll
                for (int k = 0; k < 8; ++k)
                    if (who[k] == g && dst[k] >= 0) sm[dst[k]] += v[k];
                __syncthreads();
            }
            i = e;
        }
    } else {
        for (int ci = ch0; ci < ch1; ++ci) {             // many / large children: one by one, relative indices per child
            const int c = D.child_idx[ci];
            const int64_t rp0 = D.rel_ptr[c];
            const int mc = (int)(D.rel_ptr[c + 1] - rp0);
            const double* Uc = D.U + D.upd_ptr[c];
            int* rb = relS + NT * ((ci - ch0) & 1);
            if (tid < mc) rb[tid] = D.rel[rp0 + tid];
            __syncthreads();                             // also orders the previous child's additions
            const int tot = ((mc + 1) >> 1) * (mc + 1);
            for (int f0 = tid; f0 < tot; f0 += 8 * NT) {
                double v[8];
                int dst[8];
#pragma unroll
                for (int k = 0; k < 8; ++k) { dst[k] = -1; v[k] = 0.0; if (f0 + k * NT < tot) entry(mc, rb, Uc, f0 + k * NT, v[k], dst[k]); }
#pragma unroll
                for (int k = 0; k < 8; ++k)
                    if (dst[k] >= 0) sm[dst[k]] += v[k];
            }
        }
    }
    __syncthreads();
    TRACE(2);
    partial_chol(colp, r, w, c0, D.aug_col, D.fail_col, D.dinv);
    TRACE(3);
    const int ld = ld_even(r), m = r - w;
    double* Uo = D.U + D.upd_ptr[s];                     // the update matrix first: it is all the parent waits for
    for (int j = warp; j < m; j += nwarp) {
        const double* cj = colp(j + w) + w;
        for (int i = j + lane; i < m; i += 32) Uo[i + (int64_t)j * m] = cj[i];
    }
    __syncthreads();
    if (tid == 0) { __threadfence(); red_release_add(front_done + s, 1u); }
    TRACE(4);
    double* P = D.L + D.panel_ptr[s];                    // the panel of L is read by the solves only (after the kernel)
    for (int j = warp; j < w; j += nwarp) {
        const double* cj = colp(j);
        for (int i = j + lane; i < r; i += 32) P[i + (int64_t)j * ld] = cj[i];
    }
}

// =============================================================================================================
// tiles of a tiled front (left-looking): tile_build (assembly + product), then tile_task / pair_task
// =============================================================================================================
// Tile (I,J) of a tiled front up to the point where only its own column block is missing: Cs <- assembled tile (K entries, eta,
// children's update matrices) - sum_{k < Kend} X(I,k) X(J,k)^T.  NST = stages of the operand ring in `pipe` (4 for a tile task,
// 2 for the pair task that keeps two C tiles in shared memory).
template <int NST>
__device__ __forceinline__ void tile_build(const DevSym& D, const DagPlan& F, int s, int I, int J, int Kend, const double* __restrict__ Kval,
                                           double eta, uint32_t epoch, double* pipe, double* Cs, unsigned long long* tr, uint32_t& gchunk) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int gid = lane >> 2, tig = lane & 3, wm = warp >> 1, wn = warp & 1;
    static_assert(NST == NSTAGE && (NST & (NST - 1)) == 0, "ring stages: the mbarrier words are sized for NSTAGE, a power of two");
    const uint32_t gbase = gchunk;                       // chunks this CTA has multiplied so far (same in every thread): stage and phase of chunk c follow from gbase + c
    const int c0 = D.sn_start[s], w = D.sn_start[s + 1] - c0;
    const int r = (int)(D.rows_ptr[s + 1] - D.rows_ptr[s]), ld = ld_even(r);
    const int nbp = tile_nbp(w), nbt = nbp + tile_nbu(w, r);
    const int i0 = tile_bound(I, w, r, nbp);
    const int j0 = tile_bound(J, w, r, nbp), j1 = tile_bound(J + 1, w, r, nbp), nj = j1 - j0;
    const int ia = i0 & ~1, ja = j0 & ~1, di = i0 - ia, dj = j0 - ja;
    double* P = D.L + D.panel_ptr[s];
    uint32_t* front_done = F.fac_done;
    uint32_t* tdone = F.tile_done + F.tbase[s];
    // row progress: the panel tiles of a block row finish in the order of their block columns (each waits for the ones to its
    // left), so ONE word per block row, (call number << 12) | finished tiles, tells a left-looking product how far it can run
    uint32_t* rowp = tdone + nbp * nbt + 1;
    (void)c0;

    // ---- 1. assemble the tile first (independent of the tiles to the left): zero, K entries, eta, children's update
    //         matrices in fixed child order ----
    for (int idx = tid; idx < CT_DOUBLES; idx += NT) Cs[idx] = 0.0;
    const int ch0 = D.child_ptr[s], ch1 = D.child_ptr[s + 1];
    // the child tables of the first batch are static data: fetched BEFORE the task waits (three dependent index loads per child)
    int* ctab = reinterpret_cast<int*>(pipe);                            // [TCH][4]: a0, a1, b0, b1
    long long* cptr = reinterpret_cast<long long*>(pipe + TCH * 2);      // [TCH][3]: update offset, rel offset, rows of the update matrix
    auto fetch_tables = [&](int base, int nbat) {
        if (tid < nbat) {
            const int c = D.child_idx[base + tid];
            const int32_t* cb = F.cbnd + F.cb_ptr[c];
            ctab[4 * tid] = cb[I]; ctab[4 * tid + 1] = cb[I + 1]; ctab[4 * tid + 2] = cb[J]; ctab[4 * tid + 3] = cb[J + 1];
            const long long rp0 = D.rel_ptr[c];
            cptr[3 * tid] = D.upd_ptr[c]; cptr[3 * tid + 1] = rp0; cptr[3 * tid + 2] = D.rel_ptr[c + 1] - rp0;
        }
    };
    fetch_tables(ch0, min(TCH, ch1 - ch0));
    // the K entries of the tile depend on nothing the task waits for: their (index, index, value) chain of loads runs before /
    // during the wait, two entries per thread in registers; they are stored after the barrier that ends the zero fill
    int64_t kq0 = 0, kq1 = 0;
    int kdst[2] = {-1, -1};
    double kval[2] = {0.0, 0.0};
    if (J < nbp) {
        kq0 = F.tile_kptr[F.tbase[s] + J * nbt + I]; kq1 = F.tile_kptr[F.tbase[s] + J * nbt + I + 1];
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const int64_t qq = kq0 + tid + NT * e;
            if (qq < kq1) { kdst[e] = D.kent_dst[qq]; kval[e] = Kval[D.kent_src[qq]]; }
        }
    }
    if (J == 0) {                                        // tiles with J > 0 inherit this through the flag of tile (I,0)
        for (int ci = ch0 + tid; ci < ch1; ci += NT) { const int c = D.child_idx[ci]; spin_until_ge(front_done + c, epoch * (uint32_t)F.target[c]); }
    } else if (tid == 0) {
        spin_until_ge(tdone + I, epoch);
    }
    __syncthreads();
    if (J < nbp) {
#pragma unroll
        for (int e = 0; e < 2; ++e)
            if (kdst[e] >= 0) Cs[kdst[e]] = kval[e];
        for (int64_t qq = kq0 + 2 * NT + tid; qq < kq1; qq += NT) Cs[D.kent_dst[qq]] = Kval[D.kent_src[qq]];
        __syncthreads();
        if (I == J && eta != 0.0) for (int nn = tid; nn < nj; nn += NT) Cs[nn * CLD + nn] += eta;
    }
    // Children's update matrices, in fixed child order (two children may add into the same entry).  The child tables (block
    // boundaries inside this front, offsets) are fetched for up to TCH children at once, one child per thread, so the
    // dependent index loads cost one round trip per batch instead of one per child; a child that meets the tile stages its
    // <= 64 + 64 relative indices in shared memory and its <= 64 x 64 values are then loaded eight per thread in flight.
    {
        int* relA = reinterpret_cast<int*>(pipe + TCH * 5);                  // [64] row of the tile, [64] column offset in the tile
        int* relB = relA + TILE;
        for (int base = ch0; base < ch1; base += TCH) {
            const int nbat = min(TCH, ch1 - base);
            if (base > ch0) { __syncthreads(); fetch_tables(base, nbat); }
            __syncthreads();
            for (int k = 0; k < nbat; ++k) {
                const int a0 = ctab[4 * k], a1 = ctab[4 * k + 1], b0 = ctab[4 * k + 2], b1 = ctab[4 * k + 3];
                if (a0 == a1 || b0 == b1) continue;      // uniform over the CTA
                const int na = a1 - a0, nb = b1 - b0;
                const double* Uc = D.U + cptr[3 * k];
                const int32_t* __restrict__ rel = D.rel + cptr[3 * k + 1];
                const long long mc = cptr[3 * k + 2];
                __syncthreads();                         // the previous child's additions are done, relA / relB are free
                if (tid < na) relA[tid] = rel[a0 + tid] - i0;
                else if (tid >= NT / 2 && tid - NT / 2 < nb) relB[tid - NT / 2] = (rel[b0 + tid - NT / 2] - j0) * CLD;
                __syncthreads();
                // flat index f = bb * na + aa over the na x nb block, NT apart per step: (aa, bb) advance by the CTA-uniform
                // (NT % na, NT / na) with one carry -- one division per thread and child instead of one per entry
                if (na == TILE) {
                    // the child covers all 64 rows of the tile (the usual case inside a large front): thread = (row, column mod 4),
                    // no index carry, the row's offset read once
                    const int aa = tid & (TILE - 1), da = relA[aa], adl = a0 + aa - b0;
                    const double* Ua = Uc + (a0 + aa) + (long long)b0 * mc;
                    for (int bb0 = tid >> 6; bb0 < nb; bb0 += 8 * (NT / TILE)) {
                        double v[8];
                        int dst[8];
#pragma unroll
                        for (int e = 0; e < 8; ++e) {
                            const int bb = bb0 + e * (NT / TILE);
                            const bool on = bb < nb && adl >= bb;
                            v[e] = on ? __ldcg(Ua + (long long)bb * mc) : 0.0;
                            dst[e] = on ? relB[on ? bb : 0] + da : -1;
                        }
#pragma unroll
                        for (int e = 0; e < 8; ++e)
                            if (dst[e] >= 0) Cs[dst[e]] += v[e];
                    }
                    continue;
                }
                const int tot = na * nb, qa = NT / na, ra = NT - qa * na;
                int bb = tid / na, aa = tid - bb * na;
                for (int f0 = tid; f0 < tot; f0 += 8 * NT) {
                    double v[8];
                    int dst[8];
#pragma unroll
                    for (int e = 0; e < 8; ++e) {
                        const bool on = bb < nb && a0 + aa >= b0 + bb;       // the child's update matrix is stored as a lower triangle
                        v[e] = on ? __ldcg(Uc + (a0 + aa) + (long long)(b0 + bb) * mc) : 0.0;
                        dst[e] = on ? relB[on ? bb : 0] + relA[aa] : -1;
                        aa += ra; bb += qa;
                        if (aa >= na) { aa -= na; ++bb; }
                    }
#pragma unroll
                    for (int e = 0; e < 8; ++e)
                        if (dst[e] >= 0) Cs[dst[e]] += v[e];
                }
            }
        }
        if (ch1 > ch0) __syncthreads();                  // the tables alias the operand ring the GEMM fills next
    }
    TRACE(1);

    // ---- 2. acc = sum_{k < Kend} X(I,k) X(J,k)^T ----
    double acc[2][4][2];
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) acc[a][b][0] = acc[a][b][1] = 0.0;
    const int nch = (Kend + KC - 1) / KC;
    int safe = 0;                                        // per warp: block columns [0, safe) of rows I and J are known to be finished
    auto wait_flags = [&](int c) {                       // every warp: the 64-column block that chunk c starts must be finished
        if (c < nch && ((c * KC) & (TILE - 1)) == 0) {
            const int kb = (c * KC) / TILE;
            if (kb >= safe) {                            // at the frontier only: one acquire per row says how far both rows are
                int got = 0;
                if (lane == 0) {
                    const uint32_t need = (epoch << 12) | (uint32_t)(kb + 1);
                    uint32_t vi, vj;
                    while ((vi = ld_acquire(rowp + I)) < need) __nanosleep(40);
                    vj = vi;
                    if (J != I) while ((vj = ld_acquire(rowp + J)) < need) __nanosleep(40);
                    got = (int)(min(vi, vj) & 4095u);
                }
                safe = __shfl_sync(0xffffffffu, got, 0);
            }
        }
    };
    // operand copies of a chunk: thread = (k-column tid >> 4, 16-byte segments tid & 15 and that + 16) of operand A and of operand B.
    // Everything that does not change from chunk to chunk is formed once per tile (shared-window addresses, the thread's source
    // pointer in chunk 0); a full chunk is then four copies at fixed offsets, and only a ragged last chunk takes the clamped form.
    const unsigned pipe_s = smem_addr(pipe), full_s = smem_addr(s_full), empty_s = smem_addr(s_empty);
    const unsigned dst0 = pipe_s + (unsigned)(((tid >> 4) * ALD + 2 * (tid & 15)) * 8);
    const double* const src0 = P + ia + 2 * (tid & 15) + (int64_t)(tid >> 4) * ld;
    const int64_t dAB = (int64_t)ja - ia;
    auto issue = [&](int c) {
        if (c < nch) {
            const int kc = c * KC;
            const uint32_t g = gbase + (uint32_t)c, sg = g & (NST - 1);
            if (g >= (uint32_t)NST) mbar_wait_s(empty_s + 8 * sg, ((g / NST) - 1u) & 1u);   // every warp is done with the chunk that was here
            if (kc + KC <= Kend) {
                const unsigned d = dst0 + sg * (unsigned)(STAGE_DOUBLES * 8);
                const double* sa = src0 + (int64_t)kc * ld;
                cp_async16x2_s<0>(d, sa);
                cp_async16x2_s<KC * ALD * 8>(d, sa + dAB);
            } else {
                double* st = pipe + sg * STAGE_DOUBLES;
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const int p = tid + NT * q;
                    const int op = p >> 9, rem = p & 511, kk = rem >> 5, seg = rem & 31;
                    const int k = kc + kk;
                    const int kcl = k < Kend ? k : Kend - 1;
                    const double* src = P + (op ? ja : ia) + 2 * seg + (int64_t)kcl * ld;
                    cp_async16(st + op * (KC * ALD) + kk * ALD + 2 * seg, src, k < Kend ? 16 : 0);
                }
            }
            mbar_cp_async_arrive_s(full_s + 8 * sg);
        }
    };
    // chunk c is multiplied BEFORE the warps wait for the flags of chunk c+3 (and request it): when a flag is late, the chunks
    // already in shared memory are finished first and the newly released columns only add their own latency
#pragma unroll
    for (int c = 0; c < NST - 1; ++c) { wait_flags(c); issue(c); }
    for (int c = 0; c < nch; ++c) {
        const uint32_t g = gbase + (uint32_t)c, sg = g & (NST - 1);
        mbar_wait_s(full_s + 8 * sg, (g / NST) & 1u);     // all 256 threads' copies of this chunk have landed
        const double* As = pipe + sg * STAGE_DOUBLES + wm * 16 + gid + di;
        const double* Bs = pipe + sg * STAGE_DOUBLES + KC * ALD + wn * 32 + gid + dj;
#pragma unroll
        for (int ks = 0; ks < KC; ks += 4) {
            double a[2], b[4];
#pragma unroll
            for (int mt = 0; mt < 2; ++mt) a[mt] = As[(ks + tig) * ALD + mt * 8];
#pragma unroll
            for (int nt = 0; nt < 4; ++nt) b[nt] = Bs[(ks + tig) * ALD + nt * 8];
#pragma unroll
            for (int mt = 0; mt < 2; ++mt)
#pragma unroll
                for (int nt = 0; nt < 4; ++nt) dmma(acc[mt][nt], a[mt], b[nt]);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive_s(empty_s + 8 * sg);
        wait_flags(c + NST - 1); issue(c + NST - 1);     // that stage held chunk c-1: refilled once every warp has left it
    }
    gchunk = gbase + (uint32_t)nch;
    TRACE(2);

    __syncthreads();
#pragma unroll
    for (int mt = 0; mt < 2; ++mt)
#pragma unroll
        for (int nt = 0; nt < 4; ++nt)
#pragma unroll
            for (int e = 0; e < 2; ++e) Cs[(wn * 32 + nt * 8 + 2 * tig + e) * CLD + wm * 16 + mt * 8 + gid] -= acc[mt][nt][e];
    __syncthreads();

}

// =============================================================================================================
// task type 1: tile (I,J) of a tiled front, left-looking
// =============================================================================================================
__device__ __forceinline__ void tile_task(const DevSym& D, const DagPlan& F, int s, int I, int J, const double* __restrict__ Kval,
                                          double eta, uint32_t epoch, double* sm, unsigned long long* tr, uint32_t& gchunk) {
    const int tid = threadIdx.x;
    const int c0 = D.sn_start[s], w = D.sn_start[s + 1] - c0;
    const int r = (int)(D.rows_ptr[s + 1] - D.rows_ptr[s]), ld = ld_even(r), m = r - w;
    const int nbp = tile_nbp(w), nbt = nbp + tile_nbu(w, r);
    const int i0 = tile_bound(I, w, r, nbp), i1 = tile_bound(I + 1, w, r, nbp), ni = i1 - i0;
    const int j0 = tile_bound(J, w, r, nbp), j1 = tile_bound(J + 1, w, r, nbp), nj = j1 - j0;
    double* P = D.L + D.panel_ptr[s];
    uint32_t* front_done = F.fac_done;
    uint32_t* tdone = F.tile_done + F.tbase[s];
    uint32_t* rowp = tdone + nbp * nbt + 1;
    double* pipe = sm;
    double* Cs = sm + PIPE_DOUBLES;
    tile_build<NSTAGE>(D, F, s, I, J, (J < nbp) ? j0 : w, Kval, eta, epoch, pipe, Cs, tr, gchunk);

    // ---- 3. finish: POTRF / TRSM for panel tiles, then store (each tile is written once) ----
    if (J < nbp) {
        uint32_t* sub = F.sub_done + F.bbase[s] + J;     // counts the published 8-column blocks of L_JJ: (epoch-1)*16 + blocks
        const uint32_t sbase = (epoch - 1u) * 16u;
        if (I == J) {
            // every finished 8-column block of L_JJ is stored and announced at once: the TRSM tiles of this block column
            // run one sub-step behind this POTRF instead of after it (the chain POTRF -> TRSM -> POTRF of the front)
            auto colf = [Cs](int j) { return Cs + j * CLD; };
            auto pub = [&](int js, int jbs) {
                if (tid >= NT / 2) {                     // warps 4..7 store, warp 0 goes on with the next diagonal block
                    const int nr = nj - js;
                    const int cc = (tid - NT / 2) >> 4;  // 16 threads per column of the block
                    for (int ii = (tid & 15); ii < nr && cc < jbs; ii += 16) {
                        if (ii >= cc) {
                            const double v = Cs[(js + cc) * CLD + js + ii];
                            P[(j0 + js + ii) + (int64_t)(j0 + js + cc) * ld] = v;
                            // the unused upper triangle of the diagonal tile receives L_JJ^T: row j of L_JJ becomes a contiguous
                            // column, which is what the backward substitution of solve.cu (bwd_chain) streams
                            if (ii > cc) P[(j0 + js + cc) + (int64_t)(j0 + js + ii) * ld] = v;
                        }
                    }
                    asm volatile("bar.sync 1, %0;" ::"n"(NT / 2) : "memory");
                    if (tid == NT - 1) { __threadfence(); st_release(sub, sbase + (uint32_t)(js >> 3) + 1u); }
                }
            };
            if (nj == TILE) partial_chol<decltype(colf), decltype(pub), NT / 32, TILE>(colf, nj, nj, c0 + j0, D.aug_col, D.fail_col, D.dinv, pub);
            else partial_chol(colf, nj, nj, c0 + j0, D.aug_col, D.fail_col, D.dinv, pub);
            TRACE(3);
        } else {
            double* Ls = pipe;
            double* rinv = pipe + CT_DOUBLES;
            if (ni == TILE && nj == TILE) trsm_tile<true>(Cs, Ls, rinv, ni, nj, sub, sbase, P + j0 + (int64_t)j0 * ld, ld, D.dinv + c0 + j0, P + i0 + (int64_t)j0 * ld);
            else trsm_tile<false>(Cs, Ls, rinv, ni, nj, sub, sbase, P + j0 + (int64_t)j0 * ld, ld, D.dinv + c0 + j0, P + i0 + (int64_t)j0 * ld);
            TRACE(3);                                    // every row-solving thread has already stored its finished entries
        }
        __syncthreads();
        if (tid == 0) { __threadfence(); red_release_max(rowp + I, (epoch << 12) | (uint32_t)(J + 1)); st_release(tdone + J * nbt + I, epoch); red_release_add(front_done + s, 1u); }
    } else {
        double* Uo = D.U + D.upd_ptr[s];
        TRACE(3);
        {
            const int mm = tid & (TILE - 1), n0 = tid >> 6;
            if (mm < ni) {
                double* po = Uo + (i0 + mm - w) + (int64_t)(j0 + n0 - w) * m;
                const double* pc = Cs + n0 * CLD + mm;
                const int64_t so = (int64_t)(NT / TILE) * m;
                for (int nn = n0; nn < nj; nn += NT / TILE, po += so, pc += (NT / TILE) * CLD)
                    if (I != J || mm >= nn) *po = *pc;
            }
        }
        __syncthreads();
        if (tid == 0) { __threadfence(); red_release_add(front_done + s, 1u); }
    }
    TRACE(4);
}

__global__ void __launch_bounds__(NT, 2) factor_dag_kernel(DevSym D, DagPlan F, const double* __restrict__ Kval, double eta, uint32_t epoch,
                                                              const uint32_t* __restrict__ epoch_dev) {
    extern __shared__ __align__(16) double sm[];
    __shared__ int s_task;
    if (epoch_dev) epoch = epoch_dev[0];                 // graph replay: the call number comes from device memory
    const uint32_t base = (epoch - 1u) * (uint32_t)(F.n_ftasks + (int)gridDim.x);
    if (threadIdx.x == 0) {
        for (int q = 0; q < NSTAGE; ++q) { mbar_init(&s_full[q], NT); mbar_init(&s_empty[q], NT / 32); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    uint32_t gchunk = 0;                                 // chunks of tile products this CTA has run (stage / phase bookkeeping of the ring)
    while (true) {
        __syncthreads();
        if (threadIdx.x == 0) s_task = (int)(atomicAdd(F.sync, 1u) - base);
        __syncthreads();
        const int t = s_task;
        if (t < 0 || t >= F.n_ftasks) break;             // t < 0: a call number that does not match the counters (never on a consistent handle)
        const int4 tk = F.ftasks[t];
#ifdef NMPC_TRACE_BUILD
        unsigned long long* tr = F.ftrace ? F.ftrace + (size_t)t * 8 : nullptr;
        if (threadIdx.x == 0) s_wait_ns = 0;
        if (tr && threadIdx.x == 0) { tr[0] = gtime(); unsigned sid; asm volatile("mov.u32 %0, %%smid;" : "=r"(sid)); tr[5] = sid; }
#else
        unsigned long long* tr = nullptr;
#endif
        if (tk.x == 0) small_front_task(D, F, tk.y, Kval, eta, epoch, sm, tr);
        else tile_task(D, F, tk.y, tk.z, tk.w, Kval, eta, epoch, sm, tr, gchunk);
    }
}

__global__ void reset_fail_kernel(int32_t* fail_col) { *fail_col = INT_MAX; }


}  // namespace

cudaError_t configure_factor_kernels(int max_smem_bytes, bool one_cta_per_sm, int* ctas_per_sm, size_t* smem_bytes, int* small_max_r) {
    // two CTAs per SM: half of the SM's shared memory each (minus the 1 KB per-CTA reservation), at least the tile layout;
    // latency mode: one CTA per SM with all of it, so that fronts up to SMALL_ROWS_MAX rows stay in shared memory
    size_t bytes = (size_t)TILE_SMEM_DOUBLES * sizeof(double);
    const size_t half = ((size_t)max_smem_bytes + 1024) / 2 - 1024 - 256;       // 256 B of slack for the kernel's static shared memory
    const size_t avail = one_cta_per_sm ? (size_t)max_smem_bytes - 256 : half;
    if (avail > bytes) bytes = avail & ~(size_t)15;
    if (bytes > (size_t)max_smem_bytes) return cudaErrorInvalidValue;
    cudaError_t e = cudaFuncSetAttribute(factor_dag_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem_bytes - 256);
    if (e != cudaSuccess) return e;
    int occ = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, factor_dag_kernel, NT, bytes);
    if (e != cudaSuccess) return e;
    *ctas_per_sm = occ < 1 ? 1 : occ;
    *smem_bytes = bytes;
    int rmax = 1;                                        // largest r with the packed front + the relative-index buffers in `bytes`
    while (rmax < NT && rmax + 2 <= SMALL_ROWS_MAX && ((size_t)(rmax + 1) * (rmax + 2) / 2 + 1 + SMALL_WORK_DOUBLES) * sizeof(double) <= bytes) ++rmax;   // front + work area
    *small_max_r = rmax;
    return cudaSuccess;
}

void launch_factor(const DevSym& D, const DagPlan& F, const double* Kval, double eta, uint32_t epoch, const uint32_t* epoch_dev,
                   cudaStream_t st) {
    if (F.n_ftasks > 0) factor_dag_kernel<<<F.fgrid, NT, F.fsmem, st>>>(D, F, Kval, eta, epoch, epoch_dev);
}
void launch_reset_fail(const DevSym& D, cudaStream_t st) { reset_fail_kernel<<<1, 1, 0, st>>>(D.fail_col); }
#ifdef NMPC_TRACE_BUILD
cudaError_t read_potrf_cycles(unsigned long long* out8, bool reset) {
    cudaError_t e = cudaMemcpyFromSymbol(out8, g_potrf_cycles, sizeof(unsigned long long) * 8);
    if (e == cudaSuccess && reset) { unsigned long long z[8] = {0, 0, 0, 0, 0, 0, 0, 0}; e = cudaMemcpyToSymbol(g_potrf_cycles, z, sizeof(z)); }
    return e;
}
#endif

}  // namespace nmpc
