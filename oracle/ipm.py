"""oracle/ipm.py -- TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).

Algorithm 2 (LiftedIPM) and Algorithm 1 (NMPC loop), step by step, in
the paper's order.  Where the paper is silent (constants, E_mu, mu update, step rule, inertia schedule) the
readings are those of DESIGN.md §3 (G1..G19); the step labels S0..S10 below are the ones used there.

Lifted problem (Eq. 16) with native variable bounds (reading G1):
    min f(y;p)   s.t.  h(y;p) - gamma + s+ = 0,  -h(y;p) - gamma + s- = 0,  s+- >= 0,  lb <= y <= ub
multipliers w+ , w- (omega of the lifted inequalities; beta == omega, reading G3), zL, zU for the bounds.

Newton step (Eq. 10 with the lifted G^l = [J; -J], condensed as Eq. 14/17):
    K dy = b,   K = W + eta I + Sigma_x + J^T (q+ + q-) J,      q+- = w+-/s+-   (Q_s = S^-1 B)
    b = -( grad f - mu/(y-lb) + mu/(ub-y) + J^T t ),  t = q+ r_p+ + mu/s+ - q- r_p- - mu/s-
which is -r_1^l - G^l^T (Q_s^l r_4^l - r_2^l) of Eq. 17 with r_2 = omega - mu S^-1 e (reading G2); the omega
terms of r_1 and r_2 cancel.
"""
from __future__ import annotations

import numpy as np
import scipy.sparse as sp

from .linalg import BlockTridiagCholesky, DenseCholesky, NotPositiveDefinite, SparseCholesky
from .nlp import TranscribedOCP

# S0 constants (every one an option; DESIGN.md §3 table "IPM constants")
DEFAULTS = dict(gamma=1e-4, eps_outer=1e-5, mu0=0.1, mu_warm=None,  # None -> eps_outer/10
                kappa_eps=10.0, kappa_mu=0.2, theta_mu=1.5, tau_min=0.99,
                kappa_push=1e-2, s_floor=1e-2, s_max=100.0, max_iter=200,
                eta_first=1e-4, eta_grow_first=100.0, eta_grow=8.0, eta_shrink=1.0 / 3.0,
                eta_min=1e-20, eta_max=1e40, warm_push=1e-10,
                # ---- globalisation and refinement (off by default: reading G8) ----
                # "line search with step size alpha" (Eq. 26) read as the filter line search of the paper's
                # IPM reference [17], Algorithm A steps A-5.1 .. A-5.10 without the second-order correction and
                # with the restoration phase replaced by taking the fraction-to-the-boundary step (reading G20, DESIGN.md
                # section 3).  Constants: the published defaults of [17] as recalled -- proposals, like S0.
                globalization="none",            # "none" | "filter"
                gamma_theta=1e-5, gamma_phi=1e-8, delta_sw=1.0, s_theta=1.1, s_phi=2.3, eta_phi=1e-8,
                theta_max_fact=1e4, theta_min_fact=1e-4, ls_max_backtracks=30,
                # iterative refinement of the Newton step on the UN-condensed first block row of Eq. (10):
                # rho = (W + eta I) dy + J^T(dw+ - dw-) - dzL + dzU + r_d  with dw, dz eliminated from dy; K ddy = -rho
                refine_steps=0)


class IPMState:
    """Primal-dual iterate z = (y, s+, s-, w+, w-, zL, zU) (PAPER.md:144 with beta == omega)."""

    def __init__(self, y, sp_, sm, wp, wm, zL, zU):
        self.y, self.sp, self.sm, self.wp, self.wm, self.zL, self.zU = y, sp_, sm, wp, wm, zL, zU

    def copy(self):
        return IPMState(*(v.copy() for v in (self.y, self.sp, self.sm, self.wp, self.wm, self.zL, self.zU)))


class LiftedIPM:
    def __init__(self, cfg, linsolve="sparse", perm=None, **options):
        self.cfg = cfg
        self.nlp = TranscribedOCP(cfg)
        self.opt = dict(DEFAULTS)
        self.opt.update(options)
        if self.opt["mu_warm"] is None:
            self.opt["mu_warm"] = self.opt["eps_outer"] / 10.0
        self.linsolve, self.perm = linsolve, perm
        self.chol = None                       # P, S_L = nothing (Alg. 1 line 4)
        self.n_symbolic = 0
        self.state = None
        n = self.nlp.n
        self.hasL, self.hasU = np.isfinite(self.nlp.lb), np.isfinite(self.nlp.ub)
        self.lb = np.where(self.hasL, self.nlp.lb, 0.0)
        self.ub = np.where(self.hasU, self.nlp.ub, 0.0)
        # Row intervals cl <= c(y) <= cu (oracle/nlp.py: row_bounds): the gamma tube of Eq. (16) for every equality row, the
        # stated bounds for the inequality rows g of Problem (6).  Slack form: c - cu + s+ = 0, -c + cl + s- = 0; a side that
        # is infinite has no slack and no multiplier (kept as s = 1, w = 0 and left out of every formula).  Reading G22.
        cl, cu = self.nlp.row_bounds(self.opt["gamma"])
        self.rL, self.rU = np.isfinite(cl), np.isfinite(cu)
        self.cl, self.cu = np.where(self.rL, cl, 0.0), np.where(self.rU, cu, 0.0)

    # ---------------------------------------------------------------------------------------------
    def _make_cholesky(self, K):
        """SymCholesky, Eq. (18): only when P, S_L = nothing (Alg. 2 lines 10-12)."""
        self.n_symbolic += 1
        if self.linsolve == "dense":
            return DenseCholesky(self.nlp.n)
        if self.linsolve == "blocktri":
            return BlockTridiagCholesky(self.nlp.N, self.nlp.nv)
        return SparseCholesky(self.nlp.K_pattern(), self.perm)

    # ---------------------------------------------------------------------------------------------
    def _errors(self, st, gradf, c, J, mu):
        """S2: residuals of the smoothed KKT system K_mu (Eq. 9) and the optimality error E_mu (Eq. 27/28)."""
        o = self.opt
        hasL, hasU = self.hasL, self.hasU
        dL, dU = st.y - self.lb, self.ub - st.y
        r_d = gradf + J.T @ (st.wp - st.wm) - np.where(hasL, st.zL, 0.0) + np.where(hasU, st.zU, 0.0)
        r_pp = np.where(self.rU, c - self.cu + st.sp, 0.0)
        r_pm = np.where(self.rL, -c + self.cl + st.sm, 0.0)
        comp = np.concatenate([(st.sp * st.wp - mu)[self.rU], (st.sm * st.wm - mu)[self.rL],
                               (dL * st.zL - mu)[hasL], (dU * st.zU - mu)[hasU]])
        nmult = int(self.rU.sum()) + int(self.rL.sum()) + int(hasL.sum()) + int(hasU.sum())
        l1 = st.wp.sum() + st.wm.sum() + st.zL[hasL].sum() + st.zU[hasU].sum()
        s_d = max(o["s_max"], l1 / nmult) / o["s_max"]
        E = max(np.max(np.abs(r_d)) / s_d, np.max(np.abs(r_pp)), np.max(np.abs(r_pm)),
                np.max(np.abs(comp)) / s_d)
        return E, r_d, r_pp, r_pm

    # ---------------------------------------------------------------------------------------------
    def _theta(self, y, s_p, s_m):
        """Constraint violation of the lifted equalities (the r_p rows of Eq. 9), 1-norm as in [17] Eq. (19)."""
        c = self.nlp.constraints(y)
        return float(np.sum(np.abs(c - self.cu + s_p)[self.rU]) + np.sum(np.abs(-c + self.cl + s_m)[self.rL]))

    def _phi(self, y, s_p, s_m, mu):
        """Barrier objective of the lifted problem with native bounds: f - mu sum ln(slacks, bound distances)  ([17] Eq. 3a)."""
        hasL, hasU = self.hasL, self.hasU
        if np.any(s_p[self.rU] <= 0.0) or np.any(s_m[self.rL] <= 0.0) or np.any((y - self.lb)[hasL] <= 0.0) or np.any((self.ub - y)[hasU] <= 0.0):
            return np.inf                                   # outside the domain of the barrier (never the case from alpha_max down)
        return float(self.nlp.objective(y) - mu * (np.sum(np.log(s_p[self.rU])) + np.sum(np.log(s_m[self.rL]))
                                                   + np.sum(np.log((y - self.lb)[hasL])) + np.sum(np.log((self.ub - y)[hasU]))))

    def _filter_line_search(self, st, mu, dy, ds_p, ds_m, a_max, gradf, flt, th_min):
        """[17] Algorithm A, step A-5 (backtracking line search with a filter) on (theta, phi_mu).  Returns the accepted primal
        step length, the number of halvings, and whether the filter has to be augmented (A-7)."""
        o = self.opt
        hasL, hasU = self.hasL, self.hasU
        th_k = self._theta(st.y, st.sp, st.sm)
        ph_k = self._phi(st.y, st.sp, st.sm, mu)
        dL, dU = st.y - self.lb, self.ub - st.y
        gphi_d = float(gradf @ dy - mu * (np.sum(ds_p / st.sp) + np.sum(ds_m / st.sm) + np.sum((dy / dL)[hasL]) - np.sum((dy / dU)[hasU])))
        tol = 10.0 * np.finfo(float).eps * abs(ph_k)                           # [17] Section 3.3: relax the comparisons by rounding
        alpha = a_max
        for nback in range(o["ls_max_backtracks"] + 1):
            y_t, sp_t, sm_t = st.y + alpha * dy, st.sp + alpha * ds_p, st.sm + alpha * ds_m
            th_t = self._theta(y_t, sp_t, sm_t)
            ph_t = self._phi(y_t, sp_t, sm_t, mu)
            in_filter = any(th_t >= tf and ph_t >= pf for tf, pf in flt)      # A-5.3
            switching = gphi_d < 0.0 and alpha * (-gphi_d) ** o["s_phi"] > o["delta_sw"] * th_k ** o["s_theta"]
            if not in_filter:
                if th_k <= th_min and switching:                               # A-5.4 case I: Armijo on phi
                    if ph_t - ph_k - tol <= o["eta_phi"] * alpha * gphi_d:
                        return alpha, nback, False, th_k, ph_k
                elif th_t <= (1.0 - o["gamma_theta"]) * th_k or ph_t - ph_k - tol <= -o["gamma_phi"] * th_k:   # case II
                    return alpha, nback, not switching or not (ph_t - ph_k - tol <= o["eta_phi"] * alpha * gphi_d), th_k, ph_k
            alpha *= 0.5                                                       # A-5.10
        # reading G20: no restoration phase -- take the fraction-to-the-boundary step and start a new filter
        return a_max, o["ls_max_backtracks"] + 1, None, th_k, ph_k

    # ---------------------------------------------------------------------------------------------
    def cold_start(self, y0):
        """S1 cold init."""
        o, nlp = self.opt, self.nlp
        y = np.array(y0, dtype=np.float64)
        kp = o["kappa_push"]
        both = self.hasL & self.hasU
        pL = np.where(both, np.minimum(kp * np.maximum(1.0, np.abs(self.lb)), kp * (self.ub - self.lb)),
                      kp * np.maximum(1.0, np.abs(self.lb)))
        pU = np.where(both, np.minimum(kp * np.maximum(1.0, np.abs(self.ub)), kp * (self.ub - self.lb)),
                      kp * np.maximum(1.0, np.abs(self.ub)))
        y = np.where(self.hasL, np.maximum(y, self.lb + pL), y)
        y = np.where(self.hasU, np.minimum(y, self.ub - pU), y)
        c = nlp.constraints(y)
        mu0 = o["mu0"]
        s_p = np.where(self.rU, np.maximum(self.cu - c, o["s_floor"]), 1.0)
        s_m = np.where(self.rL, np.maximum(c - self.cl, o["s_floor"]), 1.0)
        zL = np.where(self.hasL, mu0 / np.where(self.hasL, y - self.lb, 1.0), 0.0)
        zU = np.where(self.hasU, mu0 / np.where(self.hasU, self.ub - y, 1.0), 0.0)
        return IPMState(y, s_p, s_m, np.where(self.rU, mu0 / s_p, 0.0), np.where(self.rL, mu0 / s_m, 0.0), zL, zU), mu0

    def warm_start(self, prev):
        """S1 warm init: z_{k+1} <- z*_k verbatim (Alg. 1 line 10), smaller mu."""
        st = prev.copy()
        wpush = self.opt["warm_push"]
        st.y = np.where(self.hasL, np.maximum(st.y, self.lb + wpush), st.y)
        st.y = np.where(self.hasU, np.minimum(st.y, self.ub - wpush), st.y)
        return st, self.opt["mu_warm"]

    # ---------------------------------------------------------------------------------------------
    def solve(self, y0=None, warm=False, trace=None):
        """Algorithm 2.  Returns dict(status, iters, factorizations, state, trace)."""
        o, nlp = self.opt, self.nlp
        hasL, hasU = self.hasL, self.hasU
        if warm and self.state is not None:
            st, mu = self.warm_start(self.state)
        else:
            st, mu = self.cold_start(nlp.cfg.y_cold(nlp.x0) if y0 is None else y0)
        eta_last = 0.0
        nfact = 0
        tr = [] if trace is None else trace
        it = 0
        status = "maxiter"
        use_filter = o["globalization"] == "filter"
        if use_filter:                                      # [17] Eq. (21): theta_max, theta_min from the starting point
            th0 = self._theta(st.y, st.sp, st.sm)
            th_max, th_min = o["theta_max_fact"] * max(1.0, th0), o["theta_min_fact"] * max(1.0, th0)
            flt, flt_mu = [(th_max, -np.inf)], mu
        while True:
            # S2: evaluate (K_SIMD of the paper: f, grad f, c, J)            Alg. 2 line 5
            gradf = nlp.gradient(st.y)
            c = nlp.constraints(st.y)
            J = nlp.jacobian(st.y)
            E0, _, _, _ = self._errors(st, gradf, c, J, 0.0)
            # S3: outer test, Eq. (28)
            if E0 <= o["eps_outer"]:
                status = "converged"
                break
            if it >= o["max_iter"]:
                break
            # S4: barrier update while the inner test Eq. (27) holds with eps_inner = kappa_eps*mu  (Alg. 2 line 18)
            Emu, r_d, r_pp, r_pm = self._errors(st, gradf, c, J, mu)
            while Emu <= o["kappa_eps"] * mu and mu > o["eps_outer"] / 10.0:
                mu = max(o["eps_outer"] / 10.0, min(o["kappa_mu"] * mu, mu ** o["theta_mu"]))
                Emu, r_d, r_pp, r_pm = self._errors(st, gradf, c, J, mu)
            # S5
            tau = max(o["tau_min"], 1.0 - mu)
            # S6: condensed lifted KKT matrix and right-hand side (Eq. 17)      Alg. 2 lines 5-6
            dL = np.where(hasL, st.y - self.lb, 1.0)
            dU = np.where(hasU, self.ub - st.y, 1.0)
            Sigma_x = np.where(hasL, st.zL / dL, 0.0) + np.where(hasU, st.zU / dU, 0.0)
            q_p, q_m = st.wp / st.sp, st.wm / st.sm
            W = nlp.hessian(st.y, st.wp - st.wm)
            K0 = (W + sp.diags(Sigma_x) + J.T @ sp.diags(q_p + q_m) @ J).tocsc()
            t = q_p * r_pp + np.where(self.rU, mu / st.sp, 0.0) - q_m * r_pm - np.where(self.rL, mu / st.sm, 0.0)
            b = -(gradf - np.where(hasL, mu / dL, 0.0) + np.where(hasU, mu / dU, 0.0) + J.T @ t)
            # S7: inertia correction (Eq. 13/15) + NumCholesky      Alg. 2 lines 7-13
            if self.chol is None:
                self.chol = self._make_cholesky(K0)
            eta = 0.0
            while True:
                try:
                    nfact += 1
                    self.chol.factor(K0 + eta * sp.identity(nlp.n, format="csc") if eta > 0.0 else K0)
                    break
                except NotPositiveDefinite:
                    if eta == 0.0:
                        eta = o["eta_first"] if eta_last == 0.0 else max(o["eta_min"], o["eta_shrink"] * eta_last)
                    else:
                        eta = (o["eta_grow_first"] if eta_last == 0.0 else o["eta_grow"]) * eta
                    if eta > o["eta_max"]:
                        self.state = st
                        return dict(status="inertia", iters=it, factorizations=nfact, state=st, trace=tr)
            if eta > 0.0:
                eta_last = eta
            # S8: triangular solves Eq. (22)-(25), then the eliminated directions from Eq. (14)/(10)   line 14
            dy = self.chol.solve(b)

            def eliminated(dy_):
                Jdy = J @ dy_
                ds_p_ = np.where(self.rU, -r_pp - Jdy, 0.0)
                ds_m_ = np.where(self.rL, -r_pm + Jdy, 0.0)
                return (ds_p_, ds_m_, np.where(self.rU, -(st.wp - mu / st.sp) - q_p * ds_p_, 0.0),
                        np.where(self.rL, -(st.wm - mu / st.sm) - q_m * ds_m_, 0.0),
                        np.where(hasL, -(st.zL - mu / dL) - st.zL / dL * dy_, 0.0),
                        np.where(hasU, -(st.zU - mu / dU) + st.zU / dU * dy_, 0.0))

            ds_p, ds_m, dw_p, dw_m, dzL, dzU = eliminated(dy)
            for _ in range(o["refine_steps"]):              # iterative refinement on the un-condensed first row of Eq. (10)
                rho = W @ dy + eta * dy + J.T @ (dw_p - dw_m) - dzL + dzU + r_d
                dy = dy + self.chol.solve(-rho)
                ds_p, ds_m, dw_p, dw_m, dzL, dzU = eliminated(dy)
            # S9: fraction to the boundary, separate primal / dual steps (reading G8)
            a_pr = min(_max_step(st.sp, ds_p, tau), _max_step(st.sm, ds_m, tau),
                       _max_step(dL[hasL], dy[hasL], tau), _max_step(dU[hasU], -dy[hasU], tau))
            a_du = min(_max_step(st.wp, dw_p, tau), _max_step(st.wm, dw_m, tau),
                       _max_step(st.zL[hasL], dzL[hasL], tau), _max_step(st.zU[hasU], dzU[hasU], tau))
            nback = 0
            if use_filter:                                  # Eq. (26) "line search": filter line search of [17] on the primal step
                if mu != flt_mu:                            # a new barrier problem: the filter is re-initialised ([17] A-3)
                    flt, flt_mu = [(th_max, -np.inf)], mu
                a_pr, nback, augment, th_k, ph_k = self._filter_line_search(st, mu, dy, ds_p, ds_m, a_pr, gradf, flt, th_min)
                if augment is None:
                    flt = [(th_max, -np.inf)]
                elif augment:                               # A-7
                    flt.append(((1.0 - o["gamma_theta"]) * th_k, ph_k - o["gamma_phi"] * th_k))
            tr.append(dict(it=it, mu=mu, E0=E0, Emu=Emu, eta=eta, alpha_pr=a_pr, alpha_du=a_du, backtracks=nback))
            # kept for the pins (condensation algebra vs the un-condensed Newton system, Eq. 10)
            self.last_step = dict(state=st, mu=mu, eta=eta, gradf=gradf, c=c, J=J, W=W, K0=K0, b=b, dy=dy,
                                  ds_p=ds_p, ds_m=ds_m, dw_p=dw_p, dw_m=dw_m, dzL=dzL, dzU=dzU,
                                  r_d=r_d, r_pp=r_pp, r_pm=r_pm)
            # S10: Eq. (26)                                                     Alg. 2 line 15
            st = IPMState(st.y + a_pr * dy, st.sp + a_pr * ds_p, st.sm + a_pr * ds_m,
                          st.wp + a_du * dw_p, st.wm + a_du * dw_m, st.zL + a_du * dzL, st.zU + a_du * dzU)
            if not np.all(np.isfinite(st.y)):
                status = "step"
                break
            it += 1
        self.state = st
        return dict(status=status, iters=it, factorizations=nfact, state=st, trace=tr, E0=E0, mu=mu)


def _max_step(v, dv, tau):
    """Largest a in (0,1] with v + a dv >= (1-tau) v  (v > 0)."""
    neg = dv < 0.0
    if not np.any(neg):
        return 1.0
    return min(1.0, float(np.min(-tau * v[neg] / dv[neg])))


# ==================================================================================================
def nmpc_closed_loop(cfg, n_resolves=None, linsolve="sparse", perm=None, x0_sequence=None, **options):
    """Algorithm 1 with plant == model (SURVEY.md §8(d) "common"):
       solve j, extract u_1 / x_1 (line 6), x0^(j+1) = x_1* + noise_j (lines 8-9, clipped), z_{j+1} <- z*_j (line 10),
       update p (line 11).  Solve 0 is cold; the rest are warm re-solves on the cached P, S_L.
       If `x0_sequence` is given (replay mode) it overrides the closed-loop x0 of every solve."""
    R = cfg.R if n_resolves is None else n_resolves
    ipm = LiftedIPM(cfg, linsolve=linsolve, perm=perm, **options)
    x0 = np.array(cfg.x0, dtype=np.float64)
    out = []
    for j in range(R + 1):
        if x0_sequence is not None:
            x0 = np.array(x0_sequence[j], dtype=np.float64)
        ref = cfg.ref_for_solve(j)
        ipm.nlp.set_params(x0, ref)
        res = ipm.solve(warm=(j > 0))
        y = res["state"].y
        out.append(dict(solve=j, x0=x0.copy(), ref=ref, y=y.copy(), iters=res["iters"], status=res["status"],
                        factorizations=res["factorizations"], trace=res["trace"], E0=res.get("E0"),
                        state=res["state"].copy()))
        x1 = y[: cfg.nx]
        x0 = np.clip(x1 + cfg.noise_for_solve(j), cfg.x0_clip[0], cfg.x0_clip[1])
    return out, ipm
