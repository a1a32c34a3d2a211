"""Pins for oracle/models.py, oracle/nlp.py and oracle/ipm.py (CPU only).

  * derivatives vs central finite differences of the raw F / cost functions
  * distillation steady state vs Table 1 -- sanity, tol 1e-3
  * condensation algebra: the condensed step (Eq. 14/17) reproduces the dense solve of the un-condensed
    Newton system (Eq. 10) written out with every block
  * inertia relation Eq. (15) on a tiny system, before and after the eta-correction of Eq. (13)
  * Riccati closed form on an unconstrained LQ instance
  * KKT conditions (8) recomputed from raw model functions at the converged point
  * NMPC invariants: unchanged problem re-solves in 0 iterations; warm <= cold; ordering independence
"""
import numpy as np
import pytest
import scipy.optimize as sopt
import scipy.sparse as sp

from ocp_inputs import lq_instance, make_config
from oracle.ipm import LiftedIPM, nmpc_closed_loop
from oracle.models import make_model
from oracle.nlp import TranscribedOCP

SMALL = [("C0", {}), ("C1", dict(trays=5, N=4)), ("C2", dict(g=4, N=3)), ("C3", dict(g=6, nseg=2, N=2))]


def _interior_point(cfg, rng):
    lo = np.where(np.isfinite(cfg.lb), cfg.lb, 280.0)
    hi = np.where(np.isfinite(cfg.ub), cfg.ub, 400.0)
    return np.concatenate([lo + (hi - lo) * rng.uniform(0.2, 0.8, cfg.nv) for _ in range(cfg.N)])


@pytest.mark.parametrize("name,ov", SMALL)
def test_jacobian_and_gradient_vs_finite_differences(name, ov):
    cfg = make_config(name, **ov)
    nlp = TranscribedOCP(cfg)
    rng = np.random.default_rng(1)
    y = _interior_point(cfg, rng)
    J = nlp.jacobian(y).toarray()
    g = nlp.gradient(y)
    Jfd = np.zeros_like(J)
    gfd = np.zeros_like(g)
    for i in range(cfg.n):
        h = 1e-6 * max(1.0, abs(y[i]))
        e = np.zeros(cfg.n)
        e[i] = h
        Jfd[:, i] = (nlp.constraints(y + e) - nlp.constraints(y - e)) / (2 * h)
        gfd[i] = (nlp.objective(y + e) - nlp.objective(y - e)) / (2 * h)
    assert np.max(np.abs(J - Jfd)) <= 1e-6 * max(1.0, np.abs(J).max())
    assert np.max(np.abs(g - gfd)) <= 1e-6 * max(1.0, np.abs(g).max())


@pytest.mark.parametrize("name,ov", SMALL)
def test_lagrangian_hessian_vs_finite_differences(name, ov):
    """W = Hess_yy (f + lam^T h) by central differences of grad f + J^T lam."""
    cfg = make_config(name, **ov)
    nlp = TranscribedOCP(cfg)
    rng = np.random.default_rng(2)
    y = _interior_point(cfg, rng)
    lam = rng.normal(0.0, 1.0, cfg.m)
    W = nlp.hessian(y, lam).toarray()
    assert np.allclose(W, W.T)
    Wfd = np.zeros_like(W)

    def glag(yy):
        return nlp.gradient(yy) + nlp.jacobian(yy).T @ lam

    for i in range(cfg.n):
        h = 1e-5 * max(1.0, abs(y[i]))
        e = np.zeros(cfg.n)
        e[i] = h
        Wfd[:, i] = (glag(y + e) - glag(y - e)) / (2 * h)
    assert np.max(np.abs(W - Wfd)) <= 1e-6 * max(1.0, np.abs(W).max())


def test_distillation_steady_state_table1():
    """Table 1: xbar = 0.8958 at ubar = 2.51459.  Sanity pin (tol 1e-3): the garbled
    Problem (29) is read as DESIGN.md G12; the steady state of that reading must land on the paper's value."""
    cfg = make_config("C1", trays=30, N=2)     # the paper's column: N = 32 states in all, feed at state 17
    mdl = make_model(cfg)
    assert cfg.nx == 32 and mdl.f + 1 == 17
    u = np.array([2.51459])
    x = sopt.fsolve(lambda x: mdl.F(x, u), np.linspace(0.9, 0.1, cfg.nx), xtol=1e-13)
    assert np.max(np.abs(mdl.F(x, u))) < 1e-10
    assert abs(x[0] - 0.8958) < 1e-3


def test_plate_model_closed_forms():
    """Uniform field at T_amb with heaters off is an equilibrium; a uniform field only feels the radiative term;
    each heater raises exactly its edge strip (corners get two)."""
    cfg = make_config("C3", g=8, nseg=2, N=2)
    mdl = make_model(cfg)
    g, a, kr, Tamb, b = 8, *cfg.model_params[1:5]
    assert np.allclose(mdl.F(np.full(64, Tamb), np.zeros(8)), 0.0)
    T = np.full(64, 400.0)
    assert np.allclose(mdl.F(T, np.zeros(8)), -kr * (400.0 ** 4 - Tamb ** 4))
    F1 = mdl.F(np.full(64, Tamb), np.ones(8)).reshape(g, g)
    cnt = np.zeros((g, g))
    cnt[0, :] += 1; cnt[-1, :] += 1; cnt[:, 0] += 1; cnt[:, -1] += 1
    assert np.allclose(F1, b * cnt)
    # one segment: edge i=0, second half (segment 1 of 2) -> cells (0, 4..7)
    u = np.zeros(8); u[1] = 1.0
    F2 = mdl.F(np.full(64, Tamb), u).reshape(g, g)
    exp = np.zeros((g, g)); exp[0, 4:] = b
    assert np.allclose(F2, exp)
    # 5-point Laplacian of a linear-in-i field vanishes in the interior, insulated at the edges
    Tlin = (300.0 + 10.0 * np.arange(g))[:, None] * np.ones((1, g))
    lap = (mdl.Lap @ Tlin.reshape(-1)).reshape(g, g)
    assert np.allclose(lap[1:-1, :], 0.0) and np.allclose(lap[0, :], 10.0) and np.allclose(lap[-1, :], -10.0)


def test_condensation_matches_uncondensed_newton_system():
    """Eq. (10) with the lifted inequalities and bound multipliers, every block written out and solved densely,
    must give the (dy, ds, dw, dz) that the condensed path Eq. (14)/(17) produces."""
    cfg = make_config("C1", trays=4, N=5)
    ipm = LiftedIPM(cfg, linsolve="dense", max_iter=3)
    ipm.solve()
    L = ipm.last_step
    st, mu = L["state"], L["mu"]
    n, m = cfg.n, cfg.m
    J, W = L["J"].toarray(), L["W"].toarray()
    lb, ub = ipm.lb, ipm.ub
    I_n, I_m, Z = np.eye(n), np.eye(m), np.zeros
    # unknowns: dy(n) ds+(m) ds-(m) dw+(m) dw-(m) dzL(n) dzU(n)
    rows = [
        [W + L["eta"] * I_n, Z((n, m)), Z((n, m)), J.T, -J.T, -I_n, I_n],            # stationarity in y
        [J, I_m, Z((m, m)), Z((m, m)), Z((m, m)), Z((m, n)), Z((m, n))],             # h - gamma + s+ = 0
        [-J, Z((m, m)), I_m, Z((m, m)), Z((m, m)), Z((m, n)), Z((m, n))],            # -h - gamma + s- = 0
        [Z((m, n)), np.diag(st.wp), Z((m, m)), np.diag(st.sp), Z((m, m)), Z((m, n)), Z((m, n))],   # S B = mu e
        [Z((m, n)), Z((m, m)), np.diag(st.wm), Z((m, m)), np.diag(st.sm), Z((m, n)), Z((m, n))],
        [np.diag(st.zL), Z((n, m)), Z((n, m)), Z((n, m)), Z((n, m)), np.diag(st.y - lb), Z((n, n))],
        [-np.diag(st.zU), Z((n, m)), Z((n, m)), Z((n, m)), Z((n, m)), Z((n, n)), np.diag(ub - st.y)],
    ]
    M = np.block(rows)
    rhs = -np.concatenate([L["r_d"], L["r_pp"], L["r_pm"], st.sp * st.wp - mu, st.sm * st.wm - mu,
                           (st.y - lb) * st.zL - mu, (ub - st.y) * st.zU - mu])
    sol = np.linalg.solve(M, rhs)
    parts = np.split(sol, np.cumsum([n, m, m, m, m, n]))
    for got, key in zip(parts, ["dy", "ds_p", "ds_m", "dw_p", "dw_m", "dzL", "dzU"]):
        ref = L[key]
        assert np.linalg.norm(got - ref, np.inf) <= 1e-8 * max(1.0, np.linalg.norm(ref, np.inf)), key


def test_inertia_relation_eq15_and_eta_correction():
    """Eq. (15): inertia(K_aug) = (n+m_g, 0, m_g+m_h)  <=>  inertia(K_c) = (n, 0, m_h); lifted: m_h = 0, so
    K_c^l must be PD exactly when K_aug^l has n+m_g positive and m_g negative eigenvalues (Eq. 12-13)."""
    cfg = make_config("C0")
    nlp = TranscribedOCP(cfg)
    rng = np.random.default_rng(4)
    y = _interior_point(cfg, rng)
    n, m = cfg.n, cfg.m
    J = nlp.jacobian(y).toarray()
    G = np.vstack([J, -J])                                   # lifted inequality Jacobian G^l
    mg = 2 * m
    q = rng.uniform(0.5, 2.0, mg)                            # Q_s = S^-1 B
    for lam_scale, expect_pd in ((0.0, True), (-400.0, False)):
        lam = lam_scale * np.ones(m)
        W = nlp.hessian(y, lam).toarray()
        for eta in (0.0, 1e4):
            Kaug = np.block([[W + eta * np.eye(n), np.zeros((n, mg)), G.T],
                             [np.zeros((mg, n)), np.diag(q), np.eye(mg)],
                             [G, np.eye(mg), np.zeros((mg, mg))]])
            ev = np.linalg.eigvalsh(Kaug)
            inertia_ok = (int((ev > 0).sum()), int((ev < 0).sum())) == (n + mg, mg)
            Kc = W + eta * np.eye(n) + G.T @ np.diag(q) @ G
            try:
                np.linalg.cholesky(Kc)
                pd = True
            except np.linalg.LinAlgError:
                pd = False
            assert pd == inertia_ok
            if eta == 0.0:
                assert pd == expect_pd
            else:
                assert pd                                    # eta_y "increased as needed" makes it PD


def test_ipm_inertia_correction_path_is_exercised():
    """A cold VdP solve from a poor multiplier guess needs eta > 0 at least once and still converges."""
    cfg = make_config("C0")
    ipm = LiftedIPM(cfg, linsolve="sparse")
    nlp = ipm.nlp
    st, mu = ipm.cold_start(cfg.y_cold(cfg.x0))
    st.wp[:] = 500.0                                         # lam = w+ - w- strongly positive -> W indefinite
    ipm.state = st
    res = ipm.solve(warm=True)
    assert res["status"] == "converged"
    assert any(t["eta"] > 0 for t in res["trace"])
    assert res["factorizations"] > res["iters"]


def test_riccati_closed_form_lq():
    """x_k = Abar x_{k-1} + Bbar u_k, backward Riccati recursion gives the exact minimiser
    of the un-relaxed LQ problem; the lifted IPM with gamma = 1e-8 must match it to 1e-6."""
    cfg = lq_instance()
    A, B, Q, R = cfg.A, cfg.B, np.diag(cfg.q), np.diag(cfg.r)
    nx, nu, N, dt = cfg.nx, cfg.nu, cfg.N, cfg.dt
    Abar = np.linalg.inv(np.eye(nx) - dt * A)
    Bbar = dt * Abar @ B
    P = Q.copy()
    gains = [None] * N
    for k in range(N - 1, -1, -1):                           # stage k+1 in 1-based counting
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
    res = LiftedIPM(cfg, linsolve="sparse", gamma=1e-8, eps_outer=1e-8).solve()
    assert res["status"] == "converged"
    assert np.linalg.norm(res["state"].y - y_ric, np.inf) <= 1e-6 * max(1.0, np.linalg.norm(y_ric, np.inf))


@pytest.mark.parametrize("name,ov", [("C0", {}), ("C1", dict(trays=8, N=12)), ("C2", dict(g=5, N=6))])
def test_kkt_conditions_at_converged_point(name, ov):
    """KKT (8) recomputed from the RAW model functions (F and stage cost only; gradient of the Lagrangian by
    central differences, no use of the oracle's derivative code)."""
    cfg = make_config(name, **ov)
    ipm = LiftedIPM(cfg, linsolve="sparse")
    res = ipm.solve()
    assert res["status"] == "converged"
    st, o = res["state"], ipm.opt
    mdl, nlp = make_model(cfg), ipm.nlp
    X0, N, nx, nu, nv, dt = cfg.x0, cfg.N, cfg.nx, cfg.nu, cfg.nv, cfg.dt
    lam = st.wp - st.wm

    def lagrangian(y):
        Y = y.reshape(N, nv)
        val = 0.0
        for k in range(N):
            x, u = Y[k, :nx], Y[k, nx:]
            xprev = X0 if k == 0 else Y[k - 1, :nx]
            val += mdl.cost(x, u, nlp._ref(k))
            val += lam[k * nx:(k + 1) * nx] @ (x - xprev - dt * mdl.F(x, u))
        return val

    g = np.zeros(cfg.n)
    for i in range(cfg.n):
        h = 1e-6 * max(1.0, abs(st.y[i]))
        e = np.zeros(cfg.n); e[i] = h
        g[i] = (lagrangian(st.y + e) - lagrangian(st.y - e)) / (2 * h)
    hasL, hasU = ipm.hasL, ipm.hasU
    stat = g - np.where(hasL, st.zL, 0) + np.where(hasU, st.zU, 0)
    l1 = st.wp.sum() + st.wm.sum() + st.zL[hasL].sum() + st.zU[hasU].sum()
    s_d = max(100.0, l1 / (2 * cfg.m + hasL.sum() + hasU.sum())) / 100.0
    assert np.max(np.abs(stat)) / s_d <= 3 * o["eps_outer"]           # stationarity (first row of (8))
    c = nlp.constraints(st.y)
    assert np.max(np.abs(c)) <= o["gamma"] * (1 + 1e-3) + o["eps_outer"]      # lifted feasibility, Eq. (16)
    assert np.all(st.y[hasL] > ipm.lb[hasL]) and np.all(st.y[hasU] < ipm.ub[hasU])
    assert min(st.wp.min(), st.wm.min(), st.sp.min(), st.sm.min()) > 0          # 0 <= s  _|_  beta >= 0
    assert np.all(st.zL[hasL] > 0) and np.all(st.zU[hasU] > 0)
    comp = max(np.max(st.sp * st.wp), np.max(st.sm * st.wm),
               np.max(((st.y - ipm.lb) * st.zL)[hasL], initial=0), np.max(((ipm.ub - st.y) * st.zU)[hasU], initial=0))
    assert comp / s_d <= o["eps_outer"]                                         # complementarity at mu = 0


def test_nmpc_invariants_warm_start_and_zero_iteration_resolve():
    cfg = make_config("C1", trays=8, N=15, R=3)
    out, ipm = nmpc_closed_loop(cfg)
    assert all(o["status"] == "converged" for o in out)
    assert ipm.n_symbolic == 1                        # SymCholesky once, reused by every re-solve (Alg. 1 line 4)
    assert max(o["iters"] for o in out[1:]) <= out[0]["iters"]
    # re-solving the unchanged problem from its own solution takes 0 iterations
    res = ipm.solve(warm=True)
    assert res["iters"] == 0 and res["status"] == "converged"


def test_ipm_result_independent_of_ordering_and_solver():
    cfg = make_config("C1", trays=6, N=10)
    rng = np.random.default_rng(8)
    ref = LiftedIPM(cfg, linsolve="sparse").solve()
    for kw in (dict(linsolve="sparse", perm=rng.permutation(cfg.n)), dict(linsolve="dense"), dict(linsolve="blocktri")):
        res = LiftedIPM(cfg, **kw).solve()
        assert res["iters"] == ref["iters"]
        assert np.linalg.norm(res["state"].y - ref["state"].y, np.inf) <= 1e-9 * np.linalg.norm(ref["state"].y, np.inf)


# ---------------------------------------------------------------------------------------------------------------
# options of SURVEY.md section 8(f) item 2: iterative refinement and the filter line search of ref. [17]
# ---------------------------------------------------------------------------------------------------------------
def _uncondensed_residual(L, st, mu, lb, ub):
    """Residual of all seven block rows of the un-condensed Newton system Eq. (10) at the recorded step."""
    J, W = L["J"], L["W"]
    r1 = W @ L["dy"] + L["eta"] * L["dy"] + J.T @ (L["dw_p"] - L["dw_m"]) - L["dzL"] + L["dzU"] + L["r_d"]
    r2 = J @ L["dy"] + L["ds_p"] + L["r_pp"]
    r3 = -(J @ L["dy"]) + L["ds_m"] + L["r_pm"]
    r4 = st.wp * L["ds_p"] + st.sp * L["dw_p"] + st.sp * st.wp - mu
    r5 = st.wm * L["ds_m"] + st.sm * L["dw_m"] + st.sm * st.wm - mu
    r6 = st.zL * L["dy"] + (st.y - lb) * L["dzL"] + (st.y - lb) * st.zL - mu
    r7 = -st.zU * L["dy"] + (ub - st.y) * L["dzU"] + (ub - st.y) * st.zU - mu
    # magnitudes of the terms summed in each eliminated row (the rows hold to rounding relative to these)
    aJdy = abs(J) @ np.abs(L["dy"])
    scales = (aJdy + np.abs(L["ds_p"]) + np.abs(L["r_pp"]), aJdy + np.abs(L["ds_m"]) + np.abs(L["r_pm"]),
              np.abs(st.wp * L["ds_p"]) + np.abs(st.sp * L["dw_p"]) + st.sp * st.wp + mu,
              np.abs(st.wm * L["ds_m"]) + np.abs(st.sm * L["dw_m"]) + st.sm * st.wm + mu,
              np.abs(st.zL * L["dy"]) + np.abs((st.y - lb) * L["dzL"]) + np.abs((st.y - lb) * st.zL) + mu,
              np.abs(st.zU * L["dy"]) + np.abs((ub - st.y) * L["dzU"]) + np.abs((ub - st.y) * st.zU) + mu)
    return r1, tuple(zip((r2, r3, r4, r5, r6, r7), scales))


@pytest.mark.parametrize("name,ov", [("C1", dict(trays=6, N=8)), ("C2", dict(g=5, N=6))])
def test_refinement_residual_is_the_uncondensed_first_row(name, ov):
    """refine_steps: the quantity the refinement drives to zero is the residual of the FIRST block row of Eq. (10) (the rows
    of the eliminated directions hold by construction).  At the recorded last step, refined or not, it is at the rounding level
    eps * |K| |dy| of a backward-stable solve -- a dropped term or a wrong sign in rho would leave an O(|b|) residual -- and the
    refined run takes the same number of iterations."""
    cfg = make_config(name, **ov)
    iters = {}
    for steps in (0, 2):
        ipm = LiftedIPM(cfg, linsolve="sparse", refine_steps=steps)
        out = ipm.solve()
        assert out["status"] == "converged"
        L = ipm.last_step
        r1, rest = _uncondensed_residual(L, L["state"], L["mu"], ipm.lb, ipm.ub)
        Kdy = abs(L["K0"]).max() * np.abs(L["dy"]).max()
        assert np.abs(L["b"]).max() >= 1e6 * np.finfo(float).eps * Kdy            # the check below can tell b from rounding
        assert np.abs(r1).max() <= 50.0 * np.finfo(float).eps * Kdy
        hasL, hasU = np.isfinite(cfg.lb_full()), np.isfinite(cfg.ub_full())
        for k, (r, sc) in enumerate(rest):                   # eliminated rows: rounding level by construction
            sel = hasL if k == 4 else (hasU if k == 5 else slice(None))
            assert np.all(np.abs(r[sel]) <= 1e-12 * sc[sel]), k
        iters[steps] = out["iters"]
    assert iters[0] == iters[2]


def test_refinement_makes_the_path_independent_of_the_linear_solver():
    """The point of the option: two backward-stable solvers with different elimination orders (stage
    block-tridiagonal LAPACK vs scalar sparse Cholesky in natural order) give step lengths that differ by cond(K) * eps
    without refinement and agree two orders of magnitude better with one step."""
    cfg = make_config("C2", g=8, N=10)
    gap = {}
    for steps in (0, 1):
        tr = {}
        for ls in ("blocktri", "sparse"):
            out = LiftedIPM(cfg, linsolve=ls, refine_steps=steps).solve()
            assert out["status"] == "converged"
            tr[ls] = np.array([[t["alpha_pr"], t["alpha_du"]] for t in out["trace"]])
        assert tr["blocktri"].shape == tr["sparse"].shape
        gap[steps] = np.abs(tr["blocktri"] - tr["sparse"]).max()
    assert gap[1] <= 0.1 * gap[0] + 1e-12


def test_merit_functions_against_their_definitions():
    """theta (1-norm of the lifted equality residuals) and phi_mu (barrier objective, [17] Eq. 3a with the native bounds of
    reading G1) recomputed term by term with Python loops on the tiny VdP instance."""
    import math
    cfg = make_config("C0")
    ipm = LiftedIPM(cfg, linsolve="dense", globalization="filter")
    st, mu = ipm.cold_start(cfg.y_cold(cfg.x0))
    rng = np.random.default_rng(3)
    st.sp *= rng.uniform(0.5, 2.0, cfg.m)
    st.sm *= rng.uniform(0.5, 2.0, cfg.m)
    c = ipm.nlp.constraints(st.y)
    g = ipm.opt["gamma"]
    theta = sum(abs(c[i] - g + st.sp[i]) + abs(-c[i] - g + st.sm[i]) for i in range(cfg.m))
    phi = ipm.nlp.objective(st.y)
    for i in range(cfg.m):
        phi -= mu * (math.log(st.sp[i]) + math.log(st.sm[i]))
    lbf, ubf = cfg.lb_full(), cfg.ub_full()
    for i in range(cfg.n):
        if np.isfinite(lbf[i]):
            phi -= mu * math.log(st.y[i] - lbf[i])
        if np.isfinite(ubf[i]):
            phi -= mu * math.log(ubf[i] - st.y[i])
    assert ipm._theta(st.y, st.sp, st.sm) == pytest.approx(theta, rel=1e-13)
    assert ipm._phi(st.y, st.sp, st.sm, mu) == pytest.approx(phi, rel=1e-13)


def test_filter_line_search_acceptance_rules():
    """[17] Algorithm A, steps A-5.3 / A-5.4 on a real direction of the tiny VdP instance: (i) with an empty filter the full
    fraction-to-the-boundary step of a Newton direction is accepted without backtracking; (ii) a filter entry that dominates
    every trial point forces max backtracks and the fallback of reading G20; (iii) an accepted step satisfies the sufficient
    decrease condition it was accepted under."""
    cfg = make_config("C0")
    ipm = LiftedIPM(cfg, linsolve="dense", globalization="filter", max_iter=2)
    ipm.solve()
    L = ipm.last_step
    st, mu = L["state"], L["mu"]
    o = ipm.opt
    th_k = ipm._theta(st.y, st.sp, st.sm)
    ph_k = ipm._phi(st.y, st.sp, st.sm, mu)
    from oracle.ipm import _max_step
    tau = max(o["tau_min"], 1.0 - mu)
    hasL, hasU = ipm.hasL, ipm.hasU
    a_max = min(_max_step(st.sp, L["ds_p"], tau), _max_step(st.sm, L["ds_m"], tau), _max_step((st.y - ipm.lb)[hasL], L["dy"][hasL], tau),
                _max_step((ipm.ub - st.y)[hasU], -L["dy"][hasU], tau))
    a, nback, augment, th_ret, ph_ret = ipm._filter_line_search(st, mu, L["dy"], L["ds_p"], L["ds_m"], a_max, L["gradf"], [(1e30, -np.inf)], 0.0)
    assert (th_ret, ph_ret) == (th_k, ph_k)
    th_t = ipm._theta(st.y + a * L["dy"], st.sp + a * L["ds_p"], st.sm + a * L["ds_m"])
    ph_t = ipm._phi(st.y + a * L["dy"], st.sp + a * L["ds_p"], st.sm + a * L["ds_m"], mu)
    assert th_t <= (1.0 - o["gamma_theta"]) * th_k or ph_t <= ph_k - o["gamma_phi"] * th_k + 1e-12 * abs(ph_k)      # (iii)
    assert nback == 0 and a == a_max                                                                               # (i)
    blocked = [(0.0, -np.inf)]                               # dominates everything: theta_t >= 0 and phi_t >= -inf always
    a2, nback2, augment2, _, _ = ipm._filter_line_search(st, mu, L["dy"], L["ds_p"], L["ds_m"], a_max, L["gradf"], blocked, 0.0)
    assert augment2 is None and nback2 == o["ls_max_backtracks"] + 1 and a2 == a_max                                # (ii)


@pytest.mark.parametrize("name,ov", [("C0", {}), ("C1", dict(trays=8, N=12)), ("C4", dict(trays=20, N=15))])
def test_filter_ipm_converges_to_the_same_point(name, ov):
    """With the filter line search the IPM converges to the same KKT point as with fraction-to-the-boundary steps alone (the
    limit point is unique on these convex-objective configs, reading G18); every accepted primal step length is the
    fraction-to-the-boundary length times a power of 1/2."""
    cfg = make_config(name, **ov)
    base = LiftedIPM(cfg, linsolve="blocktri").solve()
    flt = LiftedIPM(cfg, linsolve="blocktri", globalization="filter").solve()
    assert base["status"] == flt["status"] == "converged"
    assert np.abs(flt["state"].y - base["state"].y).max() <= 1e-4 * max(1.0, np.abs(base["state"].y).max())
    assert all(t["backtracks"] >= 0 for t in flt["trace"])
