#!/usr/bin/env python
"""bench.py -- headline measurement of the KKT hot path (BASELINE.json:metric) on synthetic OCPs.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C3] [--impl b200|reference] [--no-extra] [--no-cpu]

A STEP is one warm NMPC re-solve (Algorithm 1 lines 9-11 + Algorithm 2): parameter update a1, then
per IPM iteration model/derivative evaluation a2, Sigma update + condensed assembly a3, numeric supernodal Cholesky a4
(+ inertia retries a4'), triangular solves a5, fused IPM vector kernels a6, barrier/termination a7 -- every row of
SURVEY.md section 8(a); the symbolic analysis a0 is done once before the loop and reported separately (the reuse win).
The closed loop is Algorithm 1 with plant == model: x0 of step j+1 is x_1* of step j plus the seeded noise.

The default workload is C3 (plate-50, n = 125 800), the largest single-GPU configuration of BASELINE.json:configs (its
`metric` names no configuration).  The other four configurations and the C4 refactor sweep are measured the same way
(their own R re-solves, L2 flush, clock record, e2e leg, oracle sample) and reported under `other_workloads`.

value        = micro-seconds per IPM iteration (whole iteration, all phases), device-timed with CUDA events on the
               handle's stream, inputs resident in HBM;  ms_per_step = milli-seconds per NMPC re-solve.
               `per_iteration` adds median / p95 over all IPM iterations of all timed re-solves (per-iteration CUDA
               events recorded by the library, nmpc_trace_row.ms_iter) and the same per phase (a separate pass with
               options.time_phases).
e2e          = the same through nmpc_ipm_solve_host: HOST x0/ref in, HOST y out, copies inside the timed region.
roofline     = the numeric Cholesky (the dominant kernel, factor_dag_kernel): sum_j cc_j^2 flops / average factorization
               time against the fp64 peak (derived 148 SM x 64 DFMA/clk x 2 x 1.965 GHz; the live DFMA / DMMA
               microbenchmarks are printed beside it).  roofline_solve = solve_dag_kernel against the measured HBM copy
               bandwidth.  `traffic` = dram bytes per launch from the committed ncu raw export under profiles/.
cpu_baseline = the oracle (oracle/, as it stands) on a bounded sample of the same workload on the host cores.

N > 1: replicas only: each rank solves an independent replica of the OCP (own x0 stream), no
data-path collective; value = max-over-ranks time / all ranks' IPM iterations.
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from ocp_inputs import make_config  # noqa: E402

METRIC = "kkt_refactor_solve_us_per_ipm_iteration"
UNIT = "us/IPM-iteration"
FP64_DERIVED_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12      # 64 DFMA lanes/SM at clocks.max.sm
NCU_RAW = os.path.join("profiles", "r02d_c3_ncu_raw.csv")  # `ncu --page raw --csv` export of the --set full capture (C3)
C3_SAMPLE_N = 4                                           # stages of the sub-horizon instance the oracle is timed on for C3


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="C3", choices=["C0", "C1", "C2", "C3", "C4"])
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-extra", action="store_true", help="skip the other four workloads and the C4 refactor sweep")
    ap.add_argument("--no-cpu", action="store_true", help="skip every oracle (cpu_baseline) leg, e.g. for profiling runs")
    ap.add_argument("--main-only", action="store_true", help="device-resident loop of the main workload only (ncu runs)")
    return ap.parse_args()


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy bandwidth)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def profiled_traffic(kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel`, averaged over the launches captured in the
    committed ncu raw export NCU_RAW (the file's .md sibling names the command); None when the file or kernel is absent."""
    path = os.path.join(ROOT, NCU_RAW)
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
    try:
        with open(path, newline="") as f:
            rows = [r for r in csv.reader(f) if r]
        hdr = rows[0]
        units = rows[1]
        ik = hdr.index("Kernel Name")
        ir, iw = hdr.index("dram__bytes_read.sum"), hdr.index("dram__bytes_write.sum")
        vals = [float(r[ir].replace(",", "")) * scale[units[ir]] + float(r[iw].replace(",", "")) * scale[units[iw]]
                for r in rows[2:] if kernel in r[ik]]
        if vals:
            return {"bytes_per_launch": float(np.mean(vals)), "launches": len(vals), "source": NCU_RAW}
    except (OSError, ValueError, KeyError, IndexError):
        pass
    return None


def replica_x0(cfg, rank):
    """Rank r > 0 starts its replica from a seeded perturbation of the config's x0 (plain data, no method arithmetic)."""
    if rank == 0:
        return np.array(cfg.x0, dtype=np.float64)
    rng = np.random.default_rng(20260604 + 7919 * rank)
    sd = {1: 0.05, 2: 0.002, 3: 2.0}[cfg.model]
    return np.clip(cfg.x0 + rng.normal(0.0, sd, cfg.nx), cfg.x0_clip[0], cfg.x0_clip[1])


def aggregate_over_ranks(dist, world, device, dev_ms, host_ms, n_it, n_f, steps, launches):
    """Replicas only: the job's time is the MAX over ranks, its work the SUM over ranks.  Returns
    (dev_ms_max, host_ms_max, total_iters, total_factorizations, total_steps, total_launches).  `dist` is
    torch.distributed (nccl on the GPU box, gloo in the CPU tests); no data-path collective exists besides this one."""
    if world <= 1:
        return dev_ms, host_ms, int(n_it), int(n_f), int(steps), int(launches)
    import torch
    t = torch.tensor([dev_ms, host_ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    c = torch.tensor([n_it, n_f, steps, launches], dtype=torch.float64, device=device)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    tot = [int(v) for v in c.tolist()]
    return float(t[0]), float(t[1]), tot[0], tot[1], tot[2], tot[3]


def dist_stats(us):
    """mean / median / p95 of a list of per-iteration micro-seconds."""
    if not len(us):
        return None
    a = np.asarray(us, dtype=np.float64)
    return {"mean": float(a.mean()), "median": float(np.median(a)), "p95": float(np.percentile(a, 95)), "count": int(a.size)}


# ======================================================================================================================
# the CPU oracle, as it stands (cpu_baseline leg and the reference arm)
# ======================================================================================================================
def oracle_threads():
    try:
        from threadpoolctl import threadpool_info
        return max([1] + [int(p.get("num_threads", 1)) for p in threadpool_info()])
    except Exception:
        return 1


def oracle_loop(cfg, n_steps, warmup, budget_s, x0=None, linsolve="sparse"):
    """Oracle closed loop: cold solve, `warmup` untimed warm re-solves, then up to n_steps timed ones (stops early once
    budget_s is spent, keeping at least one timed step).
    Returns (seconds, IPM iterations, count) of the timed re-solves, cold seconds, cold iterations."""
    from oracle.ipm import LiftedIPM
    ipm = LiftedIPM(cfg, linsolve=linsolve)
    x0 = np.array(cfg.x0 if x0 is None else x0, dtype=np.float64)
    t_all = time.perf_counter()
    warm_s, warm_it, warm_n, cold_s, cold_it = 0.0, 0, 0, 0.0, 0
    for j in range(1 + warmup + n_steps):
        ipm.nlp.set_params(x0, cfg.ref_for_solve(j))
        t0 = time.perf_counter()
        res = ipm.solve(warm=(j > 0))
        dt = time.perf_counter() - t0
        if j == 0:
            cold_s, cold_it = dt, res["iters"]
        elif j > warmup:
            warm_s += dt; warm_it += res["iters"]; warm_n += 1
        x0 = np.clip(res["state"].y[: cfg.nx] + cfg.noise_for_solve(j), cfg.x0_clip[0], cfg.x0_clip[1])
        if time.perf_counter() - t_all > budget_s and warm_n >= 1:
            break
    return warm_s, warm_it, warm_n, cold_s, cold_it


def oracle_single_iterations(cfg, linsolve, n_iter, warmup=0):
    """`warmup + n_iter` single IPM iterations of the oracle (LiftedIPM with max_iter = 1: evaluate, assemble, factor, solve,
    step, evaluate; the first from the cold start, the next ones continuing from the stored iterate); returns the list of
    seconds of the last n_iter and the number of factorizations they ran."""
    from oracle.ipm import LiftedIPM
    ipm = LiftedIPM(cfg, linsolve=linsolve, max_iter=1)
    ipm.nlp.set_params(cfg.x0, cfg.ref_for_solve(0))
    secs, facts = [], 0
    for k in range(warmup + n_iter):
        t0 = time.perf_counter()
        res = ipm.solve(warm=(k > 0))
        if k >= warmup:
            secs.append(time.perf_counter() - t0); facts += res["factorizations"]
    return secs, facts


def oracle_sample(name, x0=None, steps=3):
    """cpu_baseline of one workload: the oracle as it stands on a bounded sample (about 10-30 s of CPU work for the largest,
    less for the small ones).  C0/C1/C4: O1 (plain-C scalar sparse Cholesky, 1 thread) on warm re-solves of the same closed
    loop.  C2: O1 on the first IPM iterations of the cold solve (one factorization takes seconds).  C3: O2 (block-tridiagonal
    dense Cholesky, LAPACK with 4 BLAS threads) on a sub-horizon instance of C3_SAMPLE_N of the 50 stages, scaled by
    50 / C3_SAMPLE_N: every per-iteration cost of the oracle (model evaluation, assembly, block factorization, solves) is
    linear in the number of stages."""
    cfg = make_config(name)
    cores_avail = os.cpu_count()
    if name == "C3":
        cs = make_config(name, N=C3_SAMPLE_N)
        secs, facts = oracle_single_iterations(cs, "blocktri", n_iter=4, warmup=1)
        scale = cfg.N / cs.N
        us = float(np.mean(secs)) * scale * 1e6
        return {"value": us, "unit": UNIT, "cores": min(4, oracle_threads()), "kind": "oracle", "host_cores_available": cores_avail,
                "sample": f"{len(secs)} IPM iterations ({facts} factorizations) of the plate-50 OCP cut to N={cs.N} of {cfg.N} stages "
                          f"(blocks of {cs.nv}), oracle linsolve=blocktri (O2, LAPACK, 4 BLAS threads), per-iteration time x {scale:g} "
                          f"(every oracle step is linear in the stage count); measured {float(np.mean(secs)):.2f} s per sample iteration"}
    if name == "C2":
        secs, facts = oracle_single_iterations(cfg, "sparse", n_iter=1, warmup=0)
        return {"value": float(np.mean(secs)) * 1e6, "unit": UNIT, "cores": 1, "kind": "oracle", "host_cores_available": cores_avail,
                "sample": f"the first IPM iteration of the cold solve ({facts} factorizations, includes the oracle's own symbolic "
                          f"analysis), oracle linsolve=sparse (O1, plain C, 1 thread)"}
    budget = {"C0": 3.0, "C1": 8.0, "C4": 12.0}[name]
    warm_s, warm_it, warm_n, cold_s, cold_it = oracle_loop(cfg, steps, 0, budget, x0=x0, linsolve="sparse")
    return {"value": warm_s * 1e6 / max(1, warm_it), "unit": UNIT, "cores": 1, "kind": "oracle", "host_cores_available": cores_avail,
            "ms_per_resolve": warm_s * 1e3 / max(1, warm_n),
            "sample": f"cold solve ({cold_it} it, {cold_s:.2f} s, not in value) + {warm_n} warm re-solves ({warm_it} IPM iterations) "
                      f"of the same closed loop, oracle linsolve=sparse (O1, plain C, 1 thread)"}


def oracle_sigma_sweep_sample(cfg, draws=2):
    """Oracle side of the C4 refactor sweep: O1 numeric refactorization + solve per draw (symbolic analysis reused)."""
    import scipy.sparse as sp
    from ocp_inputs import sigma_sweep_draws
    from oracle.linalg import SparseCholesky
    from oracle.nlp import TranscribedOCP
    nlp = TranscribedOCP(cfg)
    nlp.set_params(cfg.x0, cfg.ref_for_solve(0))
    y0 = cfg.y_cold(cfg.x0)
    J, W = nlp.jacobian(y0), nlp.hessian(y0, np.zeros(cfg.m))
    chol = SparseCholesky(nlp.K_pattern(), None)
    secs = []
    for sx, ss, b in sigma_sweep_draws(cfg, count=draws):
        K = (W + sp.diags(sx) + J.T @ sp.diags(ss) @ J).tocsc()
        t0 = time.perf_counter()
        chol.factor(K).solve(b)
        secs.append(time.perf_counter() - t0)
    return {"us_per_refactor_plus_solve": float(np.mean(secs)) * 1e6, "draws": draws, "cores": 1,
            "sample": "O1 numeric refactorization + both solves per draw, natural order, symbolic analysis reused"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = make_config(args.workload)
    K, W = max(1, args.steps), args.warmup
    if args.workload == "C3":
        cs = make_config("C3", N=C3_SAMPLE_N)
        secs, facts = oracle_single_iterations(cs, "blocktri", n_iter=K, warmup=W)
        scale = cfg.N / cs.N
        us = float(np.mean(secs)) * scale * 1e6
        ms_step, cores = float(np.mean(secs)) * scale * 1e3, min(4, oracle_threads())
        sample = (f"each step = ONE oracle IPM iteration of the plate-50 OCP cut to N={cs.N} of {cfg.N} stages (O2 block-tridiagonal "
                  f"dense Cholesky, LAPACK, 4 BLAS threads), time x {scale:g} (the oracle's per-iteration work is linear in the stage "
                  f"count); {W} warm-up + {len(secs)} timed iterations, {facts} factorizations, {float(np.mean(secs)):.2f} s per sample iteration")
        done = len(secs)
    else:
        ls = "sparse"
        warm_s, warm_it, warm_n, cold_s, cold_it = oracle_loop(cfg, K, W, budget_s=150.0, linsolve=ls)
        us, ms_step, cores, done = warm_s * 1e6 / max(1, warm_it), warm_s * 1e3 / max(1, warm_n), 1, warm_n
        sample = (f"cold solve ({cold_it} it, {cold_s:.2f} s, not in value) + {W} warm-up + {warm_n} timed warm re-solves "
                  f"({warm_it} IPM iterations), oracle linsolve={ls} (O1)")
    line = {
        "impl": "reference", "metric": METRIC, "value": us, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "steps_completed_within_budget": done, "ms_per_step": ms_step, "higher_is_better": False,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_label(cfg), "sample": sample},
        "cpu_baseline": {"value": us, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                         "host_cores_available": os.cpu_count()},
        "e2e": {"value": us, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def workload_label(cfg):
    return f"{cfg.name} {cfg.title} N={cfg.N} nx={cfg.nx} nu={cfg.nu} n={cfg.n} m={cfg.m}"


# ======================================================================================================================
# own arm
# ======================================================================================================================
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "100"], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush(); self.f.seek(0)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.f.read().splitlines():
            c = [x.strip() for x in ln.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1])); pw.append(float(c[2]))
            except ValueError:
                continue
            for k, nme in enumerate(names):
                if c[3 + k].lower().startswith("active"):
                    reasons.add(nme)
        self.f.close()
        try:
            os.unlink(self.f.name)
        except OSError:
            pass
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons), samples=len(sm),
                       power_w_max=float(max(pw)))
        return out


def closed_loop(nb, torch, cfg, h, stream, x0_first, n_steps, warmup, mode, flush_buf, record=None):
    """Cold solve + warm re-solves on handle h.  mode 'dev': device buffers + CUDA events on `stream`;
    mode 'host': nmpc_ipm_solve_host with HOST buffers, wall clock.  Steps j = 1..warmup are untimed warm-ups, the next
    n_steps are timed (per step; the L2 flush and the plant update between steps are outside the timed brackets).
    Returns dict(times_ms, iters, facts, iter_us, launches, x0s, bad)."""
    dev = torch.device("cuda", torch.cuda.current_device())
    y_dev = torch.zeros(cfg.n, dtype=torch.float64, device=dev)
    y_host = torch.zeros(cfg.n, dtype=torch.float64).pin_memory()
    x0_host = torch.zeros(cfg.nx, dtype=torch.float64).pin_memory()
    ref_host = torch.zeros(max(1, cfg.N * cfg.nr), dtype=torch.float64).pin_memory()
    noise = [torch.as_tensor(cfg.noise_for_solve(j), dtype=torch.float64, device=dev) for j in range(len(cfg.noise_seq))]
    lo, hi = float(cfg.x0_clip[0]), float(cfg.x0_clip[1])
    x0 = np.array(x0_first, dtype=np.float64)
    times, iters, facts, iter_us, x0s, status_bad, launches = [], [], [], [], [], 0, 0
    cold = {}
    total = 1 + warmup + n_steps
    for j in range(total):
        if record is not None:
            x0 = record[j]
        x0s.append(np.array(x0))
        ref = np.ascontiguousarray(cfg.ref_for_solve(j))
        timed = j > warmup
        if timed and flush_buf is not None:
            with torch.cuda.stream(stream):
                flush_buf.add_(1.0)                       # > L2 write between timed steps
            stream.synchronize()
        l0 = h.launch_count()
        if mode == "dev":
            with torch.cuda.stream(stream):
                x0_d = torch.as_tensor(x0, dtype=torch.float64).to(dev)
                ref_d = torch.as_tensor(ref, dtype=torch.float64).to(dev)
            stream.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            h.update_params(x0_d, ref_d)
            r = h.ipm_solve(int(j > 0), y_dev, check=False, trace_cap=256)
            e1.record(stream)
            e1.synchronize()
            ms = e0.elapsed_time(e1)
            y_np = None
        else:
            x0_host.copy_(torch.as_tensor(x0)); ref_host[: len(ref)].copy_(torch.as_tensor(ref))
            t0 = time.perf_counter()
            r = h.ipm_solve_host(int(j > 0), x0_host, ref_host, y_host, check=False)
            ms = (time.perf_counter() - t0) * 1e3
            y_np = y_host.numpy()
        if r["status"] != 0:
            status_bad += 1
        if j == 0:
            cold = {"ms": ms, "iters": r["iters"], "factorizations": r["factorizations"], "status": r["status"]}
        if timed:
            times.append(ms); iters.append(r["iters"]); facts.append(r["factorizations"])
            launches += h.launch_count() - l0
            iter_us += [t["ms_iter"] * 1e3 for t in r.get("trace", [])]
        # plant == model (Alg. 1 lines 6-9): x0 <- x_1* + noise_j, clipped
        if record is None:
            if y_np is None:
                x1 = y_dev[: cfg.nx] + noise[j % len(noise)]
                x0 = torch.clamp(x1, lo, hi).cpu().numpy()
            else:
                x0 = np.clip(y_np[: cfg.nx] + cfg.noise_for_solve(j), lo, hi)
    return dict(times_ms=times, iters=iters, facts=facts, iter_us=iter_us, launches=launches, x0s=x0s, bad=status_bad, cold=cold)


PHASES = ("eval", "assemble", "factor", "solve", "vector")


def phase_pass(nb, torch, cfg, stream, x0s, warmup):
    """Replay the recorded x0 sequence on a handle with CUDA-event phase timing switched on (time_phases = 1).  Returns the
    per-phase sums and the per-iteration phase times (micro-seconds) of the timed re-solves."""
    h = nb.Handle(None, nb.make_ocp(cfg), nb.default_options(time_phases=1), stream=stream.cuda_stream)
    dev = torch.device("cuda", torch.cuda.current_device())
    y = torch.zeros(cfg.n, dtype=torch.float64, device=dev)
    acc = dict(iters=0, facts=0, **{k: 0.0 for k in PHASES}, per_iter={k: [] for k in PHASES})
    for j, x0 in enumerate(x0s):
        with torch.cuda.stream(stream):
            x0_d = torch.as_tensor(x0, dtype=torch.float64).to(dev)
            ref_d = torch.as_tensor(np.ascontiguousarray(cfg.ref_for_solve(j)), dtype=torch.float64).to(dev)
        stream.synchronize()
        h.update_params(x0_d, ref_d)
        r = h.ipm_solve(int(j > 0), y, check=False, trace_cap=256)
        if j > warmup:
            for k in PHASES:
                acc[k] += r["ms_" + k]
                acc["per_iter"][k] += [t["ms_" + k] * 1e3 for t in r["trace"]]
            acc["iters"] += r["iters"]; acc["facts"] += r["factorizations"]
    h.close()
    return acc


def sigma_sweep(nb, torch, cfg, stream, count=200):
    """BASELINE.json:configs[4]: `count` numeric refactorizations + solves on the C4 pattern through nmpc_assemble /
    nmpc_factor / nmpc_solve with Sigma_x, Sigma_s redrawn log-uniform in [1e-8, 1e8] per call (J, grad^2 f frozen at
    the cold-start point; all draws resident in HBM before the timed loop; CUDA events on the handle's stream).  After the
    timed loop every draw is solved once more and its normwise backward error ||b - K x||_inf / (||K||_inf ||x||_inf + ||b||_inf)
    (reading G16) is evaluated on the device through nmpc_kkt_multiply; the worst of all `count` is reported."""
    from ocp_inputs import sigma_sweep_draws
    dev = torch.device("cuda", torch.cuda.current_device())
    with torch.cuda.stream(stream):
        h = nb.Handle(None, nb.make_ocp(cfg), nb.default_options(), stream=stream.cuda_stream)
        td = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).to(dev)   # noqa: E731
        h.update_params(td(cfg.x0), td(cfg.ref_for_solve(0)))
        jrp, _ = h.get_jac_pattern(cfg.m)
        wrp, _ = h.get_hess_pattern(cfg.n)
        krp, kci = h.get_kkt_pattern(cfg.n)
        c, g = torch.empty(cfg.m, dtype=torch.float64, device=dev), torch.empty(cfg.n, dtype=torch.float64, device=dev)
        Jv = torch.empty(int(jrp[-1]), dtype=torch.float64, device=dev)
        Wv = torch.empty(int(wrp[-1]), dtype=torch.float64, device=dev)
        Kv = torch.empty(int(krp[-1]), dtype=torch.float64, device=dev)
        h.model_eval(td(cfg.y_cold(cfg.x0)), td(np.zeros(cfg.m)), c, g, Jv, Wv)
        draws = [(td(sx), td(ss), td(b)) for sx, ss, b in sigma_sweep_draws(cfg, count=count)]
        rows = torch.as_tensor(np.repeat(np.arange(cfg.n), np.diff(krp)), device=dev)
        cols = torch.as_tensor(kci.astype(np.int64), device=dev)
    stream.synchronize()
    fails = 0
    for sx, ss, b in draws[:3]:                           # warm-up
        with torch.cuda.stream(stream):
            x = b.clone()
        h.assemble(Jv, Wv, sx, ss, 0.0, Kv); h.factor(Kv, 0.0, check=False); h.solve(x)
    times, times2 = [], []
    with torch.cuda.stream(stream):
        x = torch.empty(cfg.n, dtype=torch.float64, device=dev)
    for sx, ss, b in draws:                               # b known before the factorization: Eq. (22) inside it, Eq. (24) after it
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        h.assemble(Jv, Wv, sx, ss, 0.0, Kv)
        st, _ = h.factor_rhs(Kv, b, 0.0, check=False)
        h.solve_fused(x)
        e1.record(stream)
        e1.synchronize()
        fails += int(st != 0)
        times.append(e0.elapsed_time(e1) * 1e3)
    for sx, ss, b in draws[:40]:                          # the same with nmpc_factor + the two-sided nmpc_solve
        with torch.cuda.stream(stream):
            x2 = b.clone()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        h.assemble(Jv, Wv, sx, ss, 0.0, Kv)
        h.factor(Kv, 0.0, check=False)
        h.solve(x2)
        e1.record(stream)
        e1.synchronize()
        times2.append(e0.elapsed_time(e1) * 1e3)
    worst = 0.0
    with torch.cuda.stream(stream):                       # backward errors, untimed (measurement arithmetic, not the method's)
        for sx, ss, b in draws:
            h.assemble(Jv, Wv, sx, ss, 0.0, Kv)
            h.factor_rhs(Kv, b, 0.0, check=False)
            x = torch.empty_like(b)
            h.solve_fused(x)
            kx = torch.empty_like(x)
            h.kkt_multiply(x, kx)
            absrow = torch.zeros(cfg.n, dtype=torch.float64, device=dev)
            absrow.index_add_(0, rows, Kv.abs())
            off = rows != cols
            absrow.index_add_(0, cols[off], Kv.abs()[off])
            err = (b - kx).abs().max() / (absrow.max() * x.abs().max() + b.abs().max())
            worst = max(worst, float(err))
    h.close()
    return {"calls": count, "pivot_failures": fails, "us_per_refactor_plus_solve": dist_stats(times),
            "us_per_refactor_plus_two_sided_solve": dist_stats(times2),
            "worst_solve_backward_error": worst, "bar": 1e-10,
            "note": "assemble + numeric Cholesky with the right-hand-side row (nmpc_factor_rhs) + backward solve (nmpc_solve_fused) per call, "
                    "CUDA events per call, host synchronisation on the pivot flag included; us_per_refactor_plus_two_sided_solve: the first 40 "
                    "draws through nmpc_factor + nmpc_solve; backward error of every draw (fused path) evaluated after the timed loop"}


def batched_throughput(nb, torch, cfg, B, grid_limit, R):
    """B independent instances of one OCP structure (seeded x0 perturbations) on B handles / B streams,
    solved concurrently by nmpc_ipm_solve_batch, R warm re-solve rounds after a cold round.  Wall clock around the rounds
    (device idle before and after), parameter uploads included."""
    dev = torch.device("cuda", torch.cuda.current_device())
    td = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).to(dev)   # noqa: E731
    streams = [torch.cuda.Stream() for _ in range(B)]
    hs = [nb.Handle(None, nb.make_ocp(cfg), nb.default_options(grid_limit=grid_limit), stream=streams[b].cuda_stream) for b in range(B)]
    ys = [torch.zeros(cfg.n, dtype=torch.float64, device=dev) for _ in range(B)]
    x0 = [replica_x0(cfg, b) for b in range(B)]
    lo, hi = float(cfg.x0_clip[0]), float(cfg.x0_clip[1])
    iters, bad, t_timed = 0, 0, 0.0
    for j in range(R + 1):
        for b in range(B):
            with torch.cuda.stream(streams[b]):
                hs[b].update_params(td(x0[b]), td(cfg.ref_for_solve(j)))
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        stats = nb.ipm_solve_batch(hs, [int(j > 0)] * B, ys, check=False)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        if j > 0:
            t_timed += dt; iters += sum(s["iters"] for s in stats)
        bad += sum(int(s["status"] != 0) for s in stats)
        for b in range(B):
            x0[b] = np.clip(ys[b][: cfg.nx].cpu().numpy() + cfg.noise_for_solve(j), lo, hi)
    for h in hs:
        h.close()
    return {"instances": B, "grid_limit": grid_limit, "rounds": R, "resolves_per_s": B * R / t_timed,
            "us_per_ipm_iter_aggregate": t_timed * 1e6 / max(1, iters), "ipm_iters": iters, "not_converged": bad,
            "timing": "host wall clock around nmpc_ipm_solve_batch with the device idle on both sides; one host thread per instance"}


def hykkt_leg(nb, torch, cfg, stream, R):
    """the HyKKT variant (nmpc_hykkt_solve) on the same closed loop: cold solve + R warm re-solves, CUDA
    events around each call; per IPM iteration one factorization of K_g and 2 + #CG two-sided triangular solves."""
    dev = torch.device("cuda", torch.cuda.current_device())
    td = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).to(dev)   # noqa: E731
    h = nb.Handle(None, nb.make_ocp(cfg), nb.default_options(), stream=stream.cuda_stream)
    y = torch.zeros(cfg.n, dtype=torch.float64, device=dev)
    x0 = np.array(cfg.x0, dtype=np.float64)
    lo, hi = float(cfg.x0_clip[0]), float(cfg.x0_clip[1])
    ms, iters, cg, bad = 0.0, 0, 0, 0
    for j in range(R + 1):
        with torch.cuda.stream(stream):
            h.update_params(td(x0), td(cfg.ref_for_solve(j)))
        stream.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        r = h.hykkt_solve(int(j > 0), y, trace_cap=256, check=False)
        e1.record(stream)
        e1.synchronize()
        bad += int(r["status"] != 0)
        if j > 0:
            ms += e0.elapsed_time(e1); iters += r["iters"]; cg += int(sum(t["backtracks"] for t in r["trace"]))
        x0 = np.clip(y[: cfg.nx].cpu().numpy() + cfg.noise_for_solve(j), lo, hi)
    h.close()
    return {"warm_resolves": R, "ipm_iters": iters, "cg_iterations": cg, "not_converged": bad,
            "us_per_ipm_iter": ms * 1e3 / max(1, iters), "ms_per_resolve": ms / max(1, R),
            "note": "nmpc_hykkt_solve: K_g = W + Sigma_x + gamma_h J^T J factored once per IPM iteration, CG on the Schur complement "
                    "with one two-sided triangular solve per CG iteration; host-synchronous CG scalars"}


def measure_workload(nb, torch, cfg, stream, K, W, flush_buf, x0_first, gpu_index, sample_clocks=True):
    """Everything bench.py reports about one configuration: analysis (a0), the device-resident closed loop with L2 flush
    and clock record, the HOST-buffer (e2e) loop on the recorded x0 sequence, and the phase split."""
    t0 = time.perf_counter()
    h = nb.Handle(None, nb.make_ocp(cfg), nb.default_options(), stream=stream.cuda_stream)
    analyze_wall_ms = (time.perf_counter() - t0) * 1e3
    info = h.get_info()
    sampler = ClockSampler(gpu_index) if sample_clocks else None
    t_wall0 = time.perf_counter()
    res = closed_loop(nb, torch, cfg, h, stream, x0_first, K, W, "dev", flush_buf)
    torch.cuda.synchronize()
    wall_s = time.perf_counter() - t_wall0
    clocks = sampler.stop() if sampler else None
    h.close()
    h = nb.Handle(None, nb.make_ocp(cfg), nb.default_options(), stream=stream.cuda_stream)
    res_h = closed_loop(nb, torch, cfg, h, stream, x0_first, K, W, "host", flush_buf, record=res["x0s"])
    h.close()
    acc = phase_pass(nb, torch, cfg, stream, res["x0s"], W)
    return dict(cfg=cfg, info=info, analyze_wall_ms=analyze_wall_ms, res=res, res_h=res_h, acc=acc, clocks=clocks, wall_s=wall_s, K=K, W=W)


def solve_bytes(info):
    """Algorithmic bytes of one solve launch of an IPM iteration: with the right-hand-side row
    (options.fuse_rhs, the default for model handles) the forward solve happens inside the factorization and the launch is the
    backward solve only: every stored entry of L read once, 8 nnz(L); else both solves, 16 nnz(L)."""
    return (8.0 if info.get("fused_rhs") else 16.0) * info["nnz_L"]


def workload_report(mw, hbm_peak):
    """Per-configuration summary (the entries of `other_workloads`; the top-level line is built from the same fields)."""
    cfg, info, res, res_h, acc = mw["cfg"], mw["info"], mw["res"], mw["res_h"], mw["acc"]
    n_it, n_f = max(1, sum(res["iters"])), max(1, sum(res["facts"]))
    dev_ms, host_ms = float(sum(res["times_ms"])), float(sum(res_h["times_ms"]))
    factor_us = acc["factor"] * 1e3 / max(1, acc["facts"])
    solve_us = acc["solve"] * 1e3 / max(1, acc["iters"])
    flops = float(info["flops"])
    ms_res = dev_ms / max(1, mw["K"])
    return {
        "workload": workload_label(cfg), "warm_resolves": mw["K"], "warmup_resolves": mw["W"],
        "us_per_ipm_iter": dev_ms * 1e3 / n_it, "per_iteration_us": dist_stats(res["iter_us"]),
        "ms_per_resolve": ms_res, "ms_per_resolve_stats": dist_stats(res["times_ms"]),
        "ipm_iters": res["iters"], "factorizations": sum(res["facts"]), "eta_retries": sum(res["facts"]) - sum(res["iters"]),
        "not_converged": res["bad"], "cold_solve": res["cold"],
        "analyze_ms": float(info["analyze_ms"]), "analyze_wall_ms_incl_upload": mw["analyze_wall_ms"],
        "ms_per_resolve_plus_analysis": ms_res + mw["analyze_wall_ms"],
        "phase_us_per_ipm_iter": {k: dist_stats(acc["per_iter"][k]) for k in PHASES},
        "factor_us": factor_us, "solve_us": solve_us, "refactor_plus_solve_us": factor_us + solve_us,
        "symbolic": {"n": int(info["n"]), "nnz_K": int(info["nnz_K"]), "nnz_L": int(info["nnz_L"]), "flops": flops,
                     "supernodes": int(info["nsuper"]), "levels": int(info["nlevels"]), "max_front": int(info["max_front"])},
        "factor_tflops": flops / factor_us * 1e-6, "factor_frac_fp64": flops / factor_us * 1e-6 / FP64_DERIVED_TFLOPS,
        "solve_gbs": solve_bytes(info) / solve_us * 1e-3, "solve_frac_hbm": solve_bytes(info) / solve_us * 1e-3 / hbm_peak,
        "e2e_us_per_ipm_iter": host_ms * 1e3 / max(1, sum(res_h["iters"])), "e2e_ms_per_resolve": host_ms / max(1, mw["K"]),
        "e2e_same_iteration_counts": bool(res_h["iters"] == res["iters"]),
        "gpu_launches": res["launches"], "clocks": mw["clocks"],
        "l2": "flushed between timed re-solves (384 MB write, outside the per-step event brackets)",
    }


def run_own(args):
    import torch
    import torch.distributed as dist

    import paper_2606_04725_b200 as nb

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the numeric path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = make_config(args.workload)
    K, W = args.steps, max(3, args.warmup)
    stream = torch.cuda.Stream()
    hbm_peak, peak_src = measured_peaks()
    flush_buf = torch.zeros(48 * 1024 * 1024, dtype=torch.float64, device=dev)       # 384 MB > 126 MB L2
    x0_first = replica_x0(cfg, rank)

    if args.main_only:                                    # profiling runs: the device-resident loop only, nothing printed but a note
        h = nb.Handle(None, nb.make_ocp(cfg), nb.default_options(), stream=stream.cuda_stream)
        res = closed_loop(nb, torch, cfg, h, stream, x0_first, K, W, "dev", flush_buf)
        h.close()
        print(json.dumps({"main_only": True, "workload": workload_label(cfg), "iters": res["iters"],
                          "us_per_ipm_iter": sum(res["times_ms"]) * 1e3 / max(1, sum(res["iters"]))}), flush=True)
        return

    barrier()
    mw = measure_workload(nb, torch, cfg, stream, K, W, flush_buf, x0_first, local, sample_clocks=(rank == 0))
    barrier()
    res, res_h, acc, info = mw["res"], mw["res_h"], mw["acc"], mw["info"]
    dev_ms, host_ms = float(sum(res["times_ms"])), float(sum(res_h["times_ms"]))
    n_it, n_f = int(sum(res["iters"])), int(sum(res["facts"]))
    dfma_tf, _ = nb.fp64_peak(0, 3)                       # measurement build (libnmpc_b200_aids.so): live cross-check of the peak
    dmma_tf, _ = nb.fp64_peak(1, 3)
    gemm_tf, _ = nb.tile_gemm_peak(2048, 3)               # the factorization's tile GEMM loop in isolation

    # ---- max over ranks / totals ----
    dev_ms_max, host_ms_max, tot_it, tot_f, tot_steps, tot_launch = aggregate_over_ranks(
        dist, world, dev, dev_ms, host_ms, n_it, n_f, K, res["launches"])
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    rep = workload_report(mw, hbm_peak)
    value = dev_ms_max * 1e3 / max(1, tot_it)
    e2e = host_ms_max * 1e3 / max(1, tot_it)
    tr_f, tr_s = profiled_traffic("factor_dag_kernel"), profiled_traffic("solve_dag_kernel")
    if cfg.name != "C3":
        tr_f = tr_s = None                                # the committed capture is of C3
    ms_per_step = dev_ms_max / max(1, K)
    flops = float(info["flops"])
    factor_us, solve_us = rep["factor_us"], rep["solve_us"]
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_per_step, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_label(cfg),
                   "step": "one warm NMPC re-solve (closed loop, plant == model), all rows a1-a7 of the hot path",
                   "l2": "flushed between timed steps (384 MB write, outside the per-step event brackets)",
                   "parallelism": "single GPU" if world == 1 else f"{world} independent replicas, no collective",
                   "ordering": int(info["ordering_used"])},
        "per_iteration_us": rep["per_iteration_us"], "ms_per_resolve_stats": rep["ms_per_resolve_stats"],
        "ipm_iters_per_step": n_it / max(1, K), "ipm_iters_timed": tot_it, "factorizations_timed": tot_f,
        "eta_retries_timed": tot_f - tot_it, "not_converged_steps": res["bad"], "cold_solve": res["cold"],
        "ms_per_resolve": ms_per_step,
        "analyze_ms": float(info["analyze_ms"]), "analyze_wall_ms_incl_upload": mw["analyze_wall_ms"],
        "ms_per_resolve_plus_analysis": ms_per_step + mw["analyze_wall_ms"],
        "us_per_ipm_iter_plus_analysis": (dev_ms_max + K * mw["analyze_wall_ms"]) * 1e3 / max(1, tot_it),
        "phase_us_per_ipm_iter": rep["phase_us_per_ipm_iter"],
        "factor_us": factor_us, "solve_us": solve_us, "refactor_plus_solve_us": factor_us + solve_us,
        "symbolic": rep["symbolic"],
        "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": 8 * (cfg.nx + cfg.N * cfg.nr),
                "d2h_bytes_per_step": 8 * cfg.n, "ms_per_step": host_ms_max / max(1, K),
                "same_iteration_counts_as_device_run": rep["e2e_same_iteration_counts"],
                "note": "plus 88 B of reduced scalars + pivot flag read back per IPM iteration inside the library"},
        "gpu_launches": tot_launch,
        "wall_s_whole_loop": mw["wall_s"],
        "roofline": {"bound": "alu", "kernel": "factor_dag_kernel (numeric supernodal Cholesky, one launch per factorization)",
                     "achieved": flops / factor_us * 1e-6, "peak": FP64_DERIVED_TFLOPS, "unit": "TFLOP/s",
                     "frac": flops / factor_us * 1e-6 / FP64_DERIVED_TFLOPS,
                     "traffic": tr_f["bytes_per_launch"] if tr_f else None, "traffic_source": tr_f["source"] if tr_f else None,
                     "peak_source": "derived: 148 SM x 64 DFMA/clk x 2 x 1.965 GHz (DESIGN.md section 7); fp64 is not in MEASURED_PEAKS.json",
                     "peak_live_dfma_tflops": dfma_tf, "peak_live_dmma_tflops": dmma_tf, "tile_gemm_isolated_tflops": gemm_tf,
                     "flops_per_launch": flops, "avg_launch_us": factor_us,
                     "share_of_iteration": factor_us * n_f / max(1e-9, dev_ms * 1e3)},
        "roofline_solve": {"bound": "hbm", "kernel": "solve_dag_kernel (supernodal backward triangular solve; the forward solve of the "
                                                     "Newton system is carried through the factorization as a right-hand-side row)"
                                                     if info.get("fused_rhs") else "solve_dag_kernel (supernodal forward + backward triangular solves)",
                           "achieved": solve_bytes(info) / solve_us * 1e-3, "peak": hbm_peak, "unit": "GB/s",
                           "frac": solve_bytes(info) / solve_us * 1e-3 / hbm_peak,
                           "traffic": tr_s["bytes_per_launch"] if tr_s else None, "traffic_source": tr_s["source"] if tr_s else None,
                           "peak_source": peak_src, "bytes_per_launch": solve_bytes(info), "avg_launch_us": solve_us},
        "clocks": mw["clocks"],
    }

    # ---- CPU oracle on a bounded sample of the same workload (rank 0, N = 1 only), then the other configurations ----
    if world == 1:
        line["cpu_baseline"] = None if args.no_cpu else oracle_sample(cfg.name, x0=x0_first)
        if not args.no_extra:
            extra = {}
            for name in ("C0", "C1", "C2", "C4", "C3"):
                if name == args.workload:
                    continue
                try:
                    c2 = make_config(name)
                    m2 = measure_workload(nb, torch, c2, stream, c2.R, 3, flush_buf, c2.x0, local)
                    extra[name] = workload_report(m2, hbm_peak)
                    if not args.no_cpu:
                        extra[name]["cpu_baseline"] = oracle_sample(name)
                    if name in ("C0", "C1"):            # latency-bound single instances: what concurrent instances make of the GPU
                        extra[name]["batched"] = batched_throughput(nb, torch, c2, 16, 18 if name == "C1" else 9, 10)
                    if name in ("C1", "C2"):            # the HyKKT variant on the same closed loop
                        extra[name]["hykkt"] = hykkt_leg(nb, torch, c2, stream, 5)
                    if name == "C4":
                        extra[name]["sigma_sweep"] = sigma_sweep(nb, torch, c2, stream)
                        if not args.no_cpu:
                            extra[name]["sigma_sweep"]["cpu_baseline"] = oracle_sigma_sweep_sample(c2)
                except Exception as e:  # noqa: BLE001  (a summary must not take the bench line down)
                    extra[name] = {"error": repr(e)}
            # the same closed loop with general linear rows below the dynamics rows (control-horizon hold + input
            # move limits on the distillation column, hold + a one-sided total-input limit on the plate)
            for name, ov in (("C1", dict(Nc=60, move_limit=0.1)), ("C2", dict(Nc=30, power_limit=1.5))):
                try:
                    c2 = make_config(name, **ov)
                    m2 = measure_workload(nb, torch, c2, stream, min(c2.R, 10), 3, flush_buf, c2.x0, local, sample_clocks=False)
                    extra[name + "+rows"] = workload_report(m2, hbm_peak)
                    extra[name + "+rows"]["general_rows"] = dict(count=int(c2.m - c2.m_dyn), **{k: v for k, v in c2.path_rows.items() if v is not None})
                except Exception as e:  # noqa: BLE001
                    extra[name + "+rows"] = {"error": repr(e)}
            line["other_workloads"] = extra
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_own(args)


if __name__ == "__main__":
    main()
