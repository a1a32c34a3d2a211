"""Pins for oracle/hykkt.py, the HyKKT variant of the paper's IPM (reading G21 of DESIGN.md section 3).
CPU only.

  * the HyKKT step (Cholesky of K_g + CG on the Schur complement) against the dense solve of the saddle-point Newton
    system it condenses, and the CG against a dense solve of S;
  * the Riccati closed form on an unconstrained LQ instance: HyKKT keeps the equalities exact, so it must match to 1e-8
    (the lifted IPM only to O(gamma));
  * KKT conditions recomputed from the raw model functions at the converged point (|c| <= eps: no gamma tube);
  * the same limit point as the lifted IPM up to O(gamma) of the tube, fewer iterations, no inertia retries.
"""
import numpy as np
import pytest
import scipy.sparse as sp

from ocp_inputs import lq_instance, make_config
from oracle.hykkt import HyKKTIPM, hykkt_closed_loop
from oracle.ipm import LiftedIPM
from oracle.models import make_model


def test_hykkt_step_matches_the_saddle_point_system():
    cfg = make_config("C1", trays=4, N=5)
    ipm = HyKKTIPM(cfg, linsolve="dense", max_iter=3)
    ipm.solve()
    L = ipm.last_step
    n, m = cfg.n, cfg.m
    J = L["J"].toarray()
    K = L["W"].toarray() + np.diag(L["Sigma_x"]) + L["eta"] * np.eye(n)
    M = np.block([[K, J.T], [J, np.zeros((m, m))]])
    sol = np.linalg.solve(M, np.concatenate([L["r1"], L["r2"]]))
    assert np.abs(sol[:n] - L["dy"]).max() <= 1e-8 * max(1.0, np.abs(sol[:n]).max())
    assert np.abs(sol[n:] - L["dlam"]).max() <= 1e-8 * max(1.0, np.abs(sol[n:]).max())
    # the CG alone: S x = rhs against the dense Schur complement
    g = ipm.opt["gamma_h"]
    Kg = K + g * J.T @ J
    S = J @ np.linalg.solve(Kg, J.T)
    rhs = np.random.default_rng(0).normal(size=m)
    x, k = ipm._cg(sp.csr_matrix(J), rhs)
    assert k <= ipm.opt["cg_max_iter"]
    assert np.abs(S @ x - rhs).max() <= 1e-8 * np.abs(rhs).max()


def test_hykkt_riccati_closed_form_lq():
    """the backward Riccati recursion is the exact minimiser of the un-relaxed LQ problem."""
    cfg = lq_instance()
    A, B, Q, R = cfg.A, cfg.B, np.diag(cfg.q), np.diag(cfg.r)
    nx, N, dt = cfg.nx, cfg.N, cfg.dt
    Abar = np.linalg.inv(np.eye(nx) - dt * A)
    Bbar = dt * Abar @ B
    P = Q.copy()
    gains = [None] * N
    for k in range(N - 1, -1, -1):
        G = np.linalg.solve(R + Bbar.T @ P @ Bbar, Bbar.T @ P @ Abar)
        gains[k] = G
        P = (Q if k > 0 else 0 * Q) + Abar.T @ P @ (Abar - Bbar @ G)
    x = cfg.x0.copy()
    y_ric = []
    for k in range(N):
        u = -gains[k] @ x
        x = Abar @ x + Bbar @ u
        y_ric.append(np.concatenate([x, u]))
    y_ric = np.concatenate(y_ric)
    res = HyKKTIPM(cfg, linsolve="sparse", eps_outer=1e-10).solve()
    assert res["status"] == "converged" and res["iters"] <= 3              # a QP without inequalities: one Newton step
    assert np.linalg.norm(res["state"].y - y_ric, np.inf) <= 1e-8 * max(1.0, np.linalg.norm(y_ric, np.inf))


@pytest.mark.parametrize("name,ov", [("C0", {}), ("C1", dict(trays=8, N=12)), ("C2", dict(g=5, N=6))])
def test_hykkt_kkt_conditions_at_converged_point(name, ov):
    cfg = make_config(name, **ov)
    ipm = HyKKTIPM(cfg, linsolve="sparse")
    res = ipm.solve()
    assert res["status"] == "converged"
    assert res["factorizations"] == res["iters"]                           # no inertia correction was needed
    st, o = res["state"], ipm.opt
    mdl, nlp = make_model(cfg), ipm.nlp
    X0, N, nx, nv, dt = cfg.x0, cfg.N, cfg.nx, cfg.nv, cfg.dt

    def lagrangian(y):
        Y = y.reshape(N, nv)
        val = 0.0
        for k in range(N):
            x, u = Y[k, :nx], Y[k, nx:]
            xprev = X0 if k == 0 else Y[k - 1, :nx]
            val += mdl.cost(x, u, nlp._ref(k)) + st.lam[k * nx:(k + 1) * nx] @ (x - xprev - dt * mdl.F(x, u))
        return val

    g = np.zeros(cfg.n)
    for i in range(cfg.n):
        h = 1e-6 * max(1.0, abs(st.y[i]))
        e = np.zeros(cfg.n); e[i] = h
        g[i] = (lagrangian(st.y + e) - lagrangian(st.y - e)) / (2 * h)
    hasL, hasU = ipm.hasL, ipm.hasU
    stat = g - np.where(hasL, st.zL, 0) + np.where(hasU, st.zU, 0)
    l1 = np.abs(st.lam).sum() + st.zL[hasL].sum() + st.zU[hasU].sum()
    s_d = max(100.0, l1 / (cfg.m + hasL.sum() + hasU.sum())) / 100.0
    assert np.max(np.abs(stat)) / s_d <= 3 * o["eps_outer"]
    Y = st.y.reshape(N, nv)
    c_raw = np.concatenate([Y[k, :nx] - (X0 if k == 0 else Y[k - 1, :nx]) - dt * mdl.F(Y[k, :nx], Y[k, nx:]) for k in range(N)])
    assert np.max(np.abs(c_raw)) <= o["eps_outer"]                          # the equalities themselves, not a tube
    assert np.all(st.y[hasL] > ipm.lb[hasL]) and np.all(st.y[hasU] < ipm.ub[hasU])
    comp = max(np.max(((st.y - ipm.lb) * st.zL)[hasL], initial=0), np.max(((ipm.ub - st.y) * st.zU)[hasU], initial=0))
    assert comp / s_d <= o["eps_outer"]


@pytest.mark.parametrize("name,ov", [("C1", dict(trays=10, N=14)), ("C2", dict(g=6, N=5)), ("C4", dict(trays=20, N=15))])
def test_hykkt_and_lifted_agree_up_to_the_tube(name, ov):
    """Both variants solve Problem (6); the lifted one inside the 2 gamma tube.  Shrinking gamma moves the lifted solution
    towards the HyKKT one (linearly, until the termination tolerance is reached)."""
    cfg = make_config(name, **ov)
    yh = HyKKTIPM(cfg, linsolve="blocktri").solve()["state"].y
    d = []
    for gam in (1e-4, 1e-5):
        yl = LiftedIPM(cfg, linsolve="blocktri", gamma=gam).solve()["state"].y
        d.append(np.abs(yl - yh).max() / np.abs(yh).max())
    assert d[0] <= 5e-3 and d[1] <= max(0.35 * d[0], 2e-5)               # down to the termination tolerance eps_outer = 1e-5


def test_hykkt_closed_loop_warm_starts():
    cfg = make_config("C1", trays=8, N=12)
    out, ipm = hykkt_closed_loop(cfg, n_resolves=4, linsolve="sparse")
    assert all(o["status"] == "converged" for o in out)
    assert max(o["iters"] for o in out[1:]) <= out[0]["iters"]
    ipm.nlp.set_params(out[-1]["x0"], out[-1]["ref"])
    assert ipm.solve(warm=True)["iters"] == 0                              # unchanged problem: 0 iterations
