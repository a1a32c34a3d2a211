#!/usr/bin/env python
"""Writes tests/golden/ipm_full_<config>.npz: the ORACLE's closed loop (Algorithm 1 + 2) at BASELINE size.

    python tests/golden/make_fullsize_ipm.py C3 [--resolves 2] [--linsolve blocktri]

Calls only `oracle/` and the seeded input generator `ocp_inputs.py` (never the CUDA path).  The stored values are what
`tests/test_gpu_fullsize.py` compares the CUDA path with where the oracle needs tens of minutes (C3: block-tridiagonal
dense Cholesky O2 over 50 stage blocks of 2516, SURVEY.md section 8(c) "Oracle linear algebra", BASELINE.md section 3:
"cold + 2 re-solves, results cached on disk").  Cache key = (config, master seed, oracle option defaults, linsolve):
stored in the file and checked by the test.

Per solve j = 0..R (0 = cold): x0, iteration / factorization counts, status, the per-iteration trace (mu, eta, E0,
alpha_pr, alpha_du), the converged primal y* and the full primal-dual iterate z* (float64).  Of the LAST solve additionally
the iterate BEFORE its last Newton step (a late-iteration KKT system: mu small, Sigma spread over many decades).
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from ocp_inputs import MASTER_SEED, make_config  # noqa: E402
from oracle.ipm import DEFAULTS, nmpc_closed_loop  # noqa: E402

STATE_FIELDS = ("y", "sp", "sm", "wp", "wm", "zL", "zU")


S0_KEYS = ("eps_outer", "eta_first", "eta_grow", "eta_grow_first", "eta_max", "eta_min", "eta_shrink", "gamma", "kappa_eps",
           "kappa_mu", "kappa_push", "max_iter", "mu0", "mu_warm", "s_floor", "s_max", "tau_min", "theta_mu", "warm_push")


def cache_key(name, linsolve, **overrides):
    """Key of a stored run: config, seed, the S0 constants of the oracle, the linear solver, and any option that is switched on."""
    opts = {k: DEFAULTS[k] for k in S0_KEYS}
    opts.update(overrides)
    blob = json.dumps(dict(config=name, seed=MASTER_SEED, options=opts, linsolve=linsolve), sort_keys=True, default=str)
    return hashlib.sha256(blob.encode()).hexdigest()[:16]


def golden_path(name, tag=""):
    return os.path.join(HERE, f"ipm_full_{name}{'_' + tag if tag else ''}.npz")


def slim(d, keep="last"):
    """keep = "last": the full primal-dual iterate z* of the LAST solve only; "none": no multipliers / slacks at all (y* of
    every solve always stays)."""
    last = int(d["n_solves"]) - 1
    drop = range(last) if keep == "last" else range(last + 1)
    out = {k: v for k, v in d.items() if not any(k == f"{f}_{j}" for f in STATE_FIELDS[1:] for j in drop)}
    if keep == "none":
        out = {k: v for k, v in out.items() if not k.startswith("late_")}
    return out


def run(name, resolves, linsolve, log=print, **overrides):
    cfg = make_config(name)
    t0 = time.perf_counter()
    out, ipm = nmpc_closed_loop(cfg, n_resolves=resolves, linsolve=linsolve, **overrides)
    wall = time.perf_counter() - t0
    d = dict(key=np.array(cache_key(name, linsolve, **overrides)), n_solves=np.array(len(out)), wall_seconds=np.array(wall),
             linsolve=np.array(linsolve))
    for j, o in enumerate(out):
        log(f"{name} solve {j}: status {o['status']} iters {o['iters']} factorizations {o['factorizations']}")
        d[f"x0_{j}"] = o["x0"]
        d[f"iters_{j}"] = np.array(o["iters"])
        d[f"fact_{j}"] = np.array(o["factorizations"])
        d[f"status_{j}"] = np.array(o["status"])
        d[f"trace_{j}"] = np.array([[t["mu"], t["eta"], t["E0"], t["alpha_pr"], t["alpha_du"]] for t in o["trace"]]).reshape(-1, 5)
        for f in STATE_FIELDS:
            d[f"{f}_{j}"] = getattr(o["state"], f)
    ls = ipm.last_step                                   # the iterate before the last Newton step of the last solve
    for f in STATE_FIELDS:
        d[f"late_{f}"] = getattr(ls["state"], f)
    d["late_mu"] = np.array(ls["mu"])
    d["late_eta"] = np.array(ls["eta"])
    d["late_dy"] = ls["dy"]
    return d


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("config", choices=["C1", "C2", "C3", "C4"])
    ap.add_argument("--resolves", type=int, default=2)
    ap.add_argument("--linsolve", default=None)
    ap.add_argument("--out", default=None)
    ap.add_argument("--states", default="all", choices=["all", "last", "none"], help="which solves keep their full iterate z*")
    ap.add_argument("--refine-steps", type=int, default=0, help="oracle option refine_steps (file tag refine<k>)")
    ap.add_argument("--globalization", default="none", choices=["none", "filter"], help="oracle option globalization (file tag filter)")
    a = ap.parse_args()
    linsolve = a.linsolve or ("blocktri" if a.config in ("C2", "C3") else "sparse")
    overrides = dict(refine_steps=a.refine_steps) if a.refine_steps else {}
    if a.globalization != "none":
        overrides["globalization"] = a.globalization
    d = run(a.config, a.resolves, linsolve, **overrides)
    if a.states != "all":
        d = slim(d, a.states)
    tag = "_".join(t for t in (f"refine{a.refine_steps}" if a.refine_steps else "", a.globalization if a.globalization != "none" else "") if t)
    path = a.out or golden_path(a.config, tag)
    np.savez_compressed(path, **d)
    print(f"wrote {path} ({os.path.getsize(path) / 1e6:.1f} MB) in {float(d['wall_seconds']):.1f} s of oracle time")


if __name__ == "__main__":
    main()
