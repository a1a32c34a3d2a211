"""Pins of the oracle's general rows (reading G22 of DESIGN.md section 3; Problem 5/6: inequality constraints g
and the control-horizon constraints y_c,u = y_c,u_c).  CPU only.

  * the un-condensed Newton system of Eq. (10) with ONE-sided and two-sided rows written out block by block (the slack /
    multiplier of a missing side simply absent) against the condensed path
  * KKT conditions (8) at the converged point with the rows' multipliers, recomputed from raw model functions and the raw CSR data
  * the converged solution against an independent solver (SciPy SLSQP on the exact, un-lifted problem) on a tiny instance
  * a case that reduces to something known: holding the input over the whole horizon (Nc = 1) gives a constant input, and the
    optimum over that one scalar found by a bounded scalar minimisation of the simulated cost
"""
import numpy as np
import pytest
import scipy.optimize as sopt
import scipy.sparse as sp

from ocp_inputs import make_config
from oracle.ipm import LiftedIPM
from oracle.models import make_model

CASES = [("C0", dict(Nc=25, move_limit=0.3)),
         ("C1", dict(trays=6, N=10, Nc=6, move_limit=0.2)),
         ("C2", dict(g=4, N=5, power_limit=1.2, Nc=4))]


def _G(cfg):
    g = cfg.g_rows
    return sp.csr_matrix((g["val"], g["colind"], g["rowptr"]), shape=(len(g["lo"]), cfg.n)), g["lo"], g["hi"]


def test_row_intervals_and_stacking():
    cfg = make_config("C2", g=4, N=5, power_limit=1.2, Nc=4)
    ipm = LiftedIPM(cfg, linsolve="dense")
    G, lo, hi = _G(cfg)
    gam = ipm.opt["gamma"]
    assert cfg.m == cfg.m_dyn + G.shape[0] and G.shape[0] == cfg.nu * (cfg.N - 4) + cfg.N
    # hold rows: u_k - u_{k-1} = 0 lifted to the gamma tube; power rows: one-sided, no lower side
    eq = lo == hi
    assert np.array_equal(ipm.rL[cfg.m_dyn:], np.isfinite(lo)) and np.all(ipm.rU[cfg.m_dyn:])
    assert np.allclose(ipm.cu[cfg.m_dyn:][eq], gam) and np.allclose(ipm.cl[cfg.m_dyn:][eq], -gam)
    assert np.allclose(ipm.cu[cfg.m_dyn:][~eq], 1.2) and not np.any(ipm.rL[cfg.m_dyn:][~eq])
    y = np.random.default_rng(0).uniform(0.1, 0.9, cfg.n)
    c = ipm.nlp.constraints(y)
    assert np.allclose(c[cfg.m_dyn:], G @ y)
    J = ipm.nlp.jacobian(y)
    assert abs(J[cfg.m_dyn:] - G).max() == 0.0
    # cold start: a missing side carries s = 1, w = 0 and never moves
    res = ipm.solve()
    st = res["state"]
    assert res["status"] == "converged"
    assert np.all(st.sm[~ipm.rL] == 1.0) and np.all(st.wm[~ipm.rL] == 0.0)


@pytest.mark.parametrize("name,ov", CASES)
def test_condensation_matches_uncondensed_newton_system_with_general_rows(name, ov):
    """Eq. (10) written out with every block; a row side without a bound has no slack and no multiplier (its unknowns are not
    in the system at all).  The condensed path of oracle/ipm.py must reproduce the dense solution."""
    cfg = make_config(name, **ov)
    ipm = LiftedIPM(cfg, linsolve="dense", max_iter=4)
    ipm.solve()
    L = ipm.last_step
    st, mu = L["state"], L["mu"]
    n = cfg.n
    J, W = L["J"].toarray(), L["W"].toarray()
    U, Lo = np.nonzero(ipm.rU)[0], np.nonzero(ipm.rL)[0]
    hL, hU = np.nonzero(ipm.hasL)[0], np.nonzero(ipm.hasU)[0]
    Ju, Jl = J[U], J[Lo]
    mu_, ml_, nl_, nu_ = len(U), len(Lo), len(hL), len(hU)
    EL, EU = np.eye(n)[:, hL], np.eye(n)[:, hU]
    Z = np.zeros
    # unknowns: dy (n), ds+ (rows with an upper side), ds- (rows with a lower side), dw+, dw-, dzL, dzU
    rows = [
        [W + L["eta"] * np.eye(n), Z((n, mu_)), Z((n, ml_)), Ju.T, -Jl.T, -EL, EU],
        [Ju, np.eye(mu_), Z((mu_, ml_)), Z((mu_, mu_)), Z((mu_, ml_)), Z((mu_, nl_)), Z((mu_, nu_))],       # c - cu + s+ = 0
        [-Jl, Z((ml_, mu_)), np.eye(ml_), Z((ml_, mu_)), Z((ml_, ml_)), Z((ml_, nl_)), Z((ml_, nu_))],      # -c + cl + s- = 0
        [Z((mu_, n)), np.diag(st.wp[U]), Z((mu_, ml_)), np.diag(st.sp[U]), Z((mu_, ml_)), Z((mu_, nl_)), Z((mu_, nu_))],
        [Z((ml_, n)), Z((ml_, mu_)), np.diag(st.wm[Lo]), Z((ml_, mu_)), np.diag(st.sm[Lo]), Z((ml_, nl_)), Z((ml_, nu_))],
        [np.diag(st.zL)[hL], Z((nl_, mu_)), Z((nl_, ml_)), Z((nl_, mu_)), Z((nl_, ml_)), np.diag((st.y - ipm.lb)[hL]), Z((nl_, nu_))],
        [-np.diag(st.zU)[hU], Z((nu_, mu_)), Z((nu_, ml_)), Z((nu_, mu_)), Z((nu_, ml_)), Z((nu_, nl_)), np.diag((ipm.ub - st.y)[hU])],
    ]
    c = L["c"]
    cl = np.where(ipm.rL, ipm.cl, 0.0); cu = np.where(ipm.rU, ipm.cu, 0.0)
    r_d = L["gradf"] + Ju.T @ st.wp[U] - Jl.T @ st.wm[Lo] - EL @ st.zL[hL] + EU @ st.zU[hU]
    rhs = -np.concatenate([r_d, (c - cu + st.sp)[U], (-c + cl + st.sm)[Lo], (st.sp * st.wp)[U] - mu, (st.sm * st.wm)[Lo] - mu,
                           ((st.y - ipm.lb) * st.zL)[hL] - mu, ((ipm.ub - st.y) * st.zU)[hU] - mu])
    sol = np.linalg.solve(np.block(rows), rhs)
    dy, dsp, dsm, dwp, dwm, dzL, dzU = np.split(sol, np.cumsum([n, mu_, ml_, mu_, ml_, nl_]))
    for got, ref, key in ((dy, L["dy"], "dy"), (dsp, L["ds_p"][U], "ds+"), (dsm, L["ds_m"][Lo], "ds-"), (dwp, L["dw_p"][U], "dw+"),
                          (dwm, L["dw_m"][Lo], "dw-"), (dzL, L["dzL"][hL], "dzL"), (dzU, L["dzU"][hU], "dzU")):
        # the plate's un-condensed system is badly scaled (temperatures ~3e2 next to multipliers ~1e-6): its dense LU solution
        # itself is only good to ~1e-6 relative; a dropped or mis-signed term would show at O(1)
        tol = 1e-5 if name == "C2" else 1e-8
        assert np.linalg.norm(got - ref, np.inf) <= tol * max(1.0, np.linalg.norm(ref, np.inf)), key
    # the sides that do not exist stay put
    assert np.all(L["ds_m"][~ipm.rL] == 0.0) and np.all(L["dw_m"][~ipm.rL] == 0.0)


@pytest.mark.parametrize("name,ov", CASES)
def test_kkt_conditions_with_general_rows(name, ov):
    """KKT (8) at the converged point, recomputed from the RAW model functions and the raw CSR rows (Lagrangian gradient by
    central differences): stationarity with the rows' multipliers, the row intervals, signs and complementarity."""
    cfg = make_config(name, **ov)
    ipm = LiftedIPM(cfg, linsolve="sparse")
    res = ipm.solve()
    assert res["status"] == "converged"
    st, o = res["state"], ipm.opt
    mdl, nlp = make_model(cfg), ipm.nlp
    G, lo, hi = _G(cfg)
    N, nx, nv, dt, md = cfg.N, cfg.nx, cfg.nv, cfg.dt, cfg.m_dyn
    lam = st.wp - st.wm

    def lagrangian(y):
        Y = y.reshape(N, nv)
        val = lam[md:] @ (G @ y)
        for k in range(N):
            x, u = Y[k, :nx], Y[k, nx:]
            xprev = cfg.x0 if k == 0 else Y[k - 1, :nx]
            val += mdl.cost(x, u, nlp._ref(k)) + lam[k * nx:(k + 1) * nx] @ (x - xprev - dt * mdl.F(x, u))
        return val

    g = np.zeros(cfg.n)
    for i in range(cfg.n):
        h = 1e-6 * max(1.0, abs(st.y[i]))
        e = np.zeros(cfg.n); e[i] = h
        g[i] = (lagrangian(st.y + e) - lagrangian(st.y - e)) / (2 * h)
    hasL, hasU = ipm.hasL, ipm.hasU
    stat = g - np.where(hasL, st.zL, 0) + np.where(hasU, st.zU, 0)
    nmult = ipm.rU.sum() + ipm.rL.sum() + hasL.sum() + hasU.sum()
    l1 = st.wp.sum() + st.wm.sum() + st.zL[hasL].sum() + st.zU[hasU].sum()
    s_d = max(100.0, l1 / nmult) / 100.0
    assert np.max(np.abs(stat)) / s_d <= 3 * o["eps_outer"]
    # feasibility: dynamics and equality rows inside the gamma tube, inequality rows inside their interval
    gy = G @ st.y
    eq = lo == hi
    tol = o["eps_outer"]
    assert np.max(np.abs(nlp.constraints(st.y)[:md])) <= o["gamma"] * (1 + 1e-3) + tol
    assert np.all(np.abs(gy[eq] - lo[eq]) <= o["gamma"] * (1 + 1e-3) + tol)
    assert np.all(gy[~eq] <= hi[~eq] + tol) and np.all(gy[~eq] >= lo[~eq] - tol)
    # multipliers: positive where the side exists, absent (0) where it does not; complementarity at mu = 0
    assert np.all(st.wp[ipm.rU] > 0) and np.all(st.wm[ipm.rL] > 0) and np.all(st.wm[~ipm.rL] == 0) and np.all(st.wp[~ipm.rU] == 0)
    comp = max(np.max((st.sp * st.wp)[ipm.rU]), np.max((st.sm * st.wm)[ipm.rL]))
    assert comp / s_d <= o["eps_outer"]
    # an inactive inequality row carries (almost) no multiplier
    slack = np.minimum(hi[~eq] - gy[~eq], np.where(np.isfinite(lo[~eq]), gy[~eq] - lo[~eq], np.inf))
    w_in = (st.wp + st.wm)[md:][~eq]
    assert np.all(w_in[slack > 1e-2] <= 1e-2)


def _vdp_problem(cfg):
    """Raw statement of the tiny VdP instance for SciPy: objective, dynamics equalities, general rows, bounds."""
    mdl = make_model(cfg)
    N, nx, nv, dt = cfg.N, cfg.nx, cfg.nv, cfg.dt
    ref = cfg.ref_for_solve(0)

    def f(y):
        Y = y.reshape(N, nv)
        return sum(mdl.cost(Y[k, :nx], Y[k, nx:], ref[k * cfg.nr:(k + 1) * cfg.nr]) for k in range(N))

    def h(y):
        Y = y.reshape(N, nv)
        out = []
        for k in range(N):
            xprev = cfg.x0 if k == 0 else Y[k - 1, :nx]
            out.append(Y[k, :nx] - xprev - dt * mdl.F(Y[k, :nx], Y[k, nx:]))
        return np.concatenate(out)
    return f, h


def test_solution_against_slsqp_on_the_exact_problem():
    """Tiny VdP instance with move limits and a control-horizon hold, solved by SciPy's SLSQP on the EXACT problem (equalities not
    lifted).  The lifted IPM with a small tube (gamma = 1e-7) must land on the same minimiser."""
    cfg = make_config("C0", Nc=6, move_limit=0.25)
    cfg.N = 10; cfg.n = cfg.N * cfg.nv                      # cut the horizon: rebuild the derived sizes and the rows
    cfg.ref_seq = [cfg.ref_seq[0][: cfg.N * cfg.nr]]
    cfg.m_dyn = cfg.N * cfg.nx; cfg.m = cfg.m_dyn; cfg.g_rows = None
    from ocp_inputs import add_path_rows
    add_path_rows(cfg, Nc=6, move_limit=0.25)
    G, lo, hi = _G(cfg)
    f, h = _vdp_problem(cfg)
    eq = lo == hi
    cons = [dict(type="eq", fun=h), dict(type="eq", fun=lambda y: (G @ y)[eq] - lo[eq]),
            dict(type="ineq", fun=lambda y: hi[~eq] - (G @ y)[~eq]), dict(type="ineq", fun=lambda y: (G @ y)[~eq] - lo[~eq])]
    y0 = cfg.y_cold(cfg.x0)
    ref = sopt.minimize(f, y0, method="SLSQP", constraints=cons, bounds=list(zip(cfg.lb_full(), cfg.ub_full())),
                        options=dict(maxiter=500, ftol=1e-14))
    assert ref.success
    res = LiftedIPM(cfg, linsolve="sparse", gamma=1e-7, eps_outer=1e-8).solve()
    assert res["status"] == "converged"
    y = res["state"].y
    assert abs(f(y) - ref.fun) <= 1e-5 * max(1.0, abs(ref.fun))
    assert np.abs(y - ref.x).max() <= 2e-4
    # the move limit is active somewhere and the hold is exact to the tube
    U = y.reshape(cfg.N, cfg.nv)[:, cfg.nx:]
    assert np.abs(np.diff(U[:6], axis=0)).max() >= 0.25 - 1e-5
    assert np.abs(np.diff(U[5:], axis=0)).max() <= 1e-6


def test_full_hold_reduces_to_a_scalar_input():
    """Nc = 1: the input is held over the whole horizon (PAPER.md:92 with t_c at the first step), i.e. ONE scalar decision.
    The optimum over that scalar, found by simulating the implicit-Euler dynamics for a given u and minimising the cost with a
    bounded scalar minimiser, must be what the IPM returns."""
    cfg = make_config("C0", Nc=1)
    mdl = make_model(cfg)
    N, nx, dt = cfg.N, cfg.nx, cfg.dt
    ref = cfg.ref_for_solve(0)

    def simulate(u):
        x, cost = np.array(cfg.x0), 0.0
        for k in range(N):
            xn = sopt.fsolve(lambda z: z - x - dt * mdl.F(z, np.array([u])), x, xtol=1e-13)
            cost += mdl.cost(xn, np.array([u]), ref[k * cfg.nr:(k + 1) * cfg.nr])
            x = xn
        return cost

    best = sopt.minimize_scalar(simulate, bounds=(cfg.lb[nx], cfg.ub[nx]), method="bounded", options=dict(xatol=1e-10))
    res = LiftedIPM(cfg, linsolve="sparse", gamma=1e-8, eps_outer=1e-8).solve()
    assert res["status"] == "converged"
    U = res["state"].y.reshape(N, cfg.nv)[:, nx]
    assert np.ptp(U) <= 1e-6
    assert abs(U.mean() - best.x) <= 1e-4
    assert abs(res["state"].y.reshape(N, cfg.nv)[:, :nx].max()) <= 3.0 + 1e-9
