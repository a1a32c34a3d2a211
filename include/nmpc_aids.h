/* include/nmpc_aids.h -- measurement aids, NOT part of the product library.
 *
 * libnmpc_b200_aids.so is the same source tree as libnmpc_b200.so compiled with -DNMPC_TRACE_BUILD (the persistent
 * factor / solve kernels then record per-task timestamps) plus csrc/peak.cu.  It exports everything include/nmpc.h
 * declares and the entry points below.  bench.py loads it for the live fp64 peak only; the per-task timelines
 * under profiles/ were recorded with it.  The product library contains neither the timestamps nor these symbols.
 */
#ifndef NMPC_AIDS_H
#define NMPC_AIDS_H

#include "nmpc.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Sustained fp64 rate of the current device in TFLOP/s, kind 0 = DFMA (vector pipe), 1 = DMMA (mma.sync m8n8k4 f64);
 * best of `repeats` launches of a register-resident kernel.  HOST outputs; ms_out may be NULL.  These are the live
 * cross-checks of the derived fp64 peak the factorization roofline uses.                     */
nmpc_status nmpc_fp64_peak(int32_t kind, int32_t repeats, double* tflops_out, double* ms_out);

/* The left-looking 64 x 64 tile GEMM of the factorization in isolation (same tile shape, cp.async ring and DMMA fragment
 * mapping; no flags, assembly, POTRF or TRSM): two CTAs per SM, each accumulating K columns (multiple of 16).  TFLOP/s of the
 * best of `repeats` launches: what the contraction alone reaches, the ceiling of factor_dag_kernel's tile tasks.       */
nmpc_status nmpc_tile_gemm_peak(int32_t K, int32_t repeats, double* tflops_out, double* ms_out);

/* Per-task timestamps of the last factorization (kind 0) / solve (kind 1).  tasks_host: 4 int32 per task (type,
 * supernode, I, J|dir); stamps_host: 8 uint64 per task (globaltimer ns: claimed, dependencies met / GEMM done,
 * assembled, factored, done; [5] = SM id).  Returns the number of tasks copied (<= cap), or the task count if a
 * pointer is NULL.                                                                                               */
int64_t nmpc_get_task_trace(nmpc_handle h, int32_t kind, int32_t* tasks_host, uint64_t* stamps_host, int64_t cap);

#ifdef __cplusplus
}
#endif
#endif /* NMPC_AIDS_H */
