// peak.cu -- measured fp64 roofline denominators.  MEASURED_PEAKS.json holds only the HBM copy bandwidth and the bf16
// GEMM rate; the numeric factorization (step a4) is fp64, so bench.py measures the chip's sustained DFMA (vector pipe)
// and DMMA (mma.sync m8n8k4 f64 tensor path) rates with these two register-resident kernels and reports the factor
// kernels against them.  Not on the hot path.
#include <cuda_runtime.h>

#include <cstdint>

#include "../../include/nmpc_aids.h"

namespace {

constexpr int PEAK_NT = 256;
constexpr int PEAK_ILP = 8;
constexpr int PEAK_INNER = 512;

__global__ void __launch_bounds__(PEAK_NT) dfma_peak_kernel(double* out, int iters, double a0) {
    double acc[PEAK_ILP];
#pragma unroll
    for (int k = 0; k < PEAK_ILP; ++k) acc[k] = threadIdx.x * 1e-3 + k;
    const double a = a0, b = 1e-9;
    for (int it = 0; it < iters; ++it) {
#pragma unroll 8
        for (int j = 0; j < PEAK_INNER; ++j) {
#pragma unroll
            for (int k = 0; k < PEAK_ILP; ++k) acc[k] = fma(acc[k], a, b);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < PEAK_ILP; ++k) s += acc[k];
    if (s == 123.456) out[blockIdx.x * PEAK_NT + threadIdx.x] = s;      // keeps the loop alive, never true in practice
}

__global__ void __launch_bounds__(PEAK_NT) dmma_peak_kernel(double* out, int iters, double a0) {
    double c[PEAK_ILP][2];
#pragma unroll
    for (int k = 0; k < PEAK_ILP; ++k) { c[k][0] = threadIdx.x * 1e-3 + k; c[k][1] = 0.5 * k; }
    const double a = a0, b = 1e-9 * (threadIdx.x & 3);
    for (int it = 0; it < iters; ++it) {
#pragma unroll 4
        for (int j = 0; j < PEAK_INNER; ++j) {
#pragma unroll
            for (int k = 0; k < PEAK_ILP; ++k)
                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                             : "+d"(c[k][0]), "+d"(c[k][1]) : "d"(a), "d"(b));
        }
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < PEAK_ILP; ++k) s += c[k][0] + c[k][1];
    if (s == 123.456) out[blockIdx.x * PEAK_NT + threadIdx.x] = s;
}

// ---- the left-looking tile GEMM of factor.cu (tile_task, step 2) in isolation: one 64 x 64 tile per CTA, 256 threads, fp64
//      DMMA m8n8k4 (2 x 4 accumulator tiles per thread), operands streamed from a column-major panel with cp.async.cg through
//      a 4-stage ring of 16 columns handed over with mbarrier words -- same tile shape, ring and fragment mapping as the factorization, no flags, no assembly,
//      no POTRF / TRSM.  CTA b multiplies the rows of block b with the rows of block b + 1 of one tall panel. ----
constexpr int G_TILE = 64, G_KC = 16, G_ALD = 68, G_NSTAGE = 4, G_STAGE = 2 * G_KC * G_ALD;

__device__ __forceinline__ unsigned g_saddr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void g_mbar_wait(uint64_t* b, uint32_t parity) {
    asm volatile("{\n.reg .pred p;\nGW: mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n@p bra GD;\nbra GW;\nGD:\n}" ::"r"(g_saddr(b)), "r"(parity) : "memory");
}

__global__ void __launch_bounds__(PEAK_NT, 2) tile_gemm_kernel(const double* __restrict__ P, int ld, int K, int nblocks, double* __restrict__ out) {
    extern __shared__ __align__(16) double pipe[];
    __shared__ uint64_t full[G_NSTAGE], empty[G_NSTAGE];  // the ring is handed over as in factor.cu: cp.async arrivals / one arrival per warp
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, gid = lane >> 2, tig = lane & 3, wm = warp >> 1, wn = warp & 1;
    const int ia = (int)(blockIdx.x % nblocks) * G_TILE, ja = (int)((blockIdx.x + 1) % nblocks) * G_TILE;
    double acc[2][4][2];
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) acc[a][b][0] = acc[a][b][1] = 0.0;
    if (tid == 0) {
        for (int q = 0; q < G_NSTAGE; ++q) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(g_saddr(&full[q])), "r"(PEAK_NT) : "memory");
            asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(g_saddr(&empty[q])), "r"(PEAK_NT / 32) : "memory");
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const int nch = K / G_KC;
    auto issue = [&](int c) {
        if (c < nch) {
            const int sg = c % G_NSTAGE;
            if (c >= G_NSTAGE) g_mbar_wait(&empty[sg], (uint32_t)((c / G_NSTAGE) - 1) & 1u);
            double* st = pipe + sg * G_STAGE;
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int p = tid + PEAK_NT * q;
                const int op = p >> 9, rem = p & 511, kk = rem >> 5, seg = rem & 31;
                const double* src = P + (op ? ja : ia) + 2 * seg + (int64_t)(c * G_KC + kk) * ld;
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(g_saddr(st + op * (G_KC * G_ALD) + kk * G_ALD + 2 * seg)), "l"(src) : "memory");
            }
            asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(g_saddr(&full[sg])) : "memory");
        }
    };
    issue(0); issue(1); issue(2);
    for (int c = 0; c < nch; ++c) {
        const int sg = c % G_NSTAGE;
        g_mbar_wait(&full[sg], (uint32_t)(c / G_NSTAGE) & 1u);
        const double* As = pipe + sg * G_STAGE + wm * 16 + gid;
        const double* Bs = pipe + sg * G_STAGE + G_KC * G_ALD + wn * 32 + gid;
#pragma unroll
        for (int ks = 0; ks < G_KC; ks += 4) {
            double a[2], b[4];
#pragma unroll
            for (int mt = 0; mt < 2; ++mt) a[mt] = As[(ks + tig) * G_ALD + mt * 8];
#pragma unroll
            for (int nt = 0; nt < 4; ++nt) b[nt] = Bs[(ks + tig) * G_ALD + nt * 8];
#pragma unroll
            for (int mt = 0; mt < 2; ++mt)
#pragma unroll
                for (int nt = 0; nt < 4; ++nt)
                    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                                 : "+d"(acc[mt][nt][0]), "+d"(acc[mt][nt][1]) : "d"(a[mt]), "d"(b[nt]));
        }
        __syncwarp();
        if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(g_saddr(&empty[sg])) : "memory");
        issue(c + 3);
    }
    double s = 0.0;
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) s += acc[a][b][0] + acc[a][b][1];
    out[blockIdx.x * PEAK_NT + tid] = s;
}

}  // namespace

extern "C" nmpc_status nmpc_tile_gemm_peak(int32_t K, int32_t repeats, double* tflops_out, double* ms_out) {
    if (!tflops_out || K < 64 || (K % G_KC) || repeats < 1) return NMPC_E_ARG;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) { cudaGetLastError(); return NMPC_E_CUDA; }
    // NMPC_GEMM_CTAS_PER_SM=1: one CTA per SM (how fast a LONE tile product runs while its SM neighbour is in a non-GEMM phase)
    const char* env = getenv("NMPC_GEMM_CTAS_PER_SM");
    const int blocks = sms * ((env && env[0] == '1') ? 1 : 2), ld = blocks * G_TILE;
    const size_t smem = (size_t)G_NSTAGE * G_STAGE * sizeof(double) + 34 * 1024;   // + the C tile the factorization keeps beside the ring
    double *P = nullptr, *out = nullptr;
    if (cudaMalloc((void**)&P, sizeof(double) * (size_t)ld * K) != cudaSuccess || cudaMalloc((void**)&out, sizeof(double) * (size_t)blocks * PEAK_NT) != cudaSuccess) {
        cudaGetLastError(); cudaFree(P); return NMPC_E_ALLOC;
    }
    cudaMemset(P, 0, sizeof(double) * (size_t)ld * K);
    cudaFuncSetAttribute(tile_gemm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    double best_ms = 1e300;
    for (int r = 0; r < repeats + 1; ++r) {
        cudaEventRecord(e0);
        tile_gemm_kernel<<<blocks, PEAK_NT, smem>>>(P, ld, K, blocks, out);
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (r > 0 && ms < best_ms) best_ms = ms;
    }
    cudaError_t err = cudaGetLastError();
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(P); cudaFree(out);
    if (err != cudaSuccess) return NMPC_E_CUDA;
    *tflops_out = 2.0 * G_TILE * G_TILE * (double)K * blocks / (best_ms * 1e-3) / 1e12;
    if (ms_out) *ms_out = best_ms;
    return NMPC_OK;
}

extern "C" nmpc_status nmpc_fp64_peak(int32_t kind, int32_t repeats, double* tflops_out, double* ms_out) {
    if (!tflops_out || kind < 0 || kind > 1 || repeats < 1) return NMPC_E_ARG;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        cudaGetLastError();
        return NMPC_E_CUDA;
    }
    const int blocks = sms * 8, iters = 24;
    double* out = nullptr;
    if (cudaMalloc((void**)&out, sizeof(double) * (size_t)blocks * PEAK_NT) != cudaSuccess) { cudaGetLastError(); return NMPC_E_ALLOC; }
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    double best_ms = 1e300;
    for (int r = 0; r < repeats + 1; ++r) {                    // first pass is the warm-up
        cudaEventRecord(e0);
        if (kind == 0) dfma_peak_kernel<<<blocks, PEAK_NT>>>(out, iters, 0.999999);
        else dmma_peak_kernel<<<blocks, PEAK_NT>>>(out, iters, 0.999999);
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (r > 0 && ms < best_ms) best_ms = ms;
    }
    cudaError_t err = cudaGetLastError();
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out);
    if (err != cudaSuccess) return NMPC_E_CUDA;
    // flops per thread: DFMA 2 per fma;  DMMA m8n8k4 = 2*8*8*4 = 512 per warp instruction = 16 per thread
    const double per_thread = (kind == 0 ? 2.0 : 16.0) * PEAK_ILP * (double)PEAK_INNER * iters;
    const double flops = per_thread * (double)blocks * PEAK_NT;
    *tflops_out = flops / (best_ms * 1e-3) / 1e12;
    if (ms_out) *ms_out = best_ms;
    return NMPC_OK;
}
