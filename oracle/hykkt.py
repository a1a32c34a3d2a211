"""oracle/hykkt.py -- TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).

The HyKKT variant of the paper's interior-point method ("the system can be reformulated using either
Lifted-KKT or HyKKT [33] ... HyKKT is a hybrid direct-iterative approach based on an augmented Lagrangian formulation
[44, 45] ... the proposed framework and its implementation also support HyKKT"), step by step for the same transcribed OCPs:

    min f(y;p)   s.t.  h(y;p) = 0,   lb <= y <= ub          (Problem 6; the equalities are NOT relaxed: no gamma tube)

Primal-dual iterate (y, lam, zL, zU): lam the multipliers of h (free sign), zL / zU those of the bounds (reading G1).
Newton system after the elimination of dz (Eq. 12 with the equalities kept):

    [ W + Sigma_x + eta I   J^T ] [ dy  ]   [ r1 ]     r1 = -(grad f + J^T lam - mu/(y-lb) + mu/(ub-y))
    [ J                     0   ] [ dlam] = [ r2 ]     r2 = -c

HyKKT (reading G21, DESIGN.md section 3 -- the paper names the method and cites [44, 45] but prints no formula): add
gamma_h J^T times the second block row to the first,

    K_g = W + Sigma_x + eta I + gamma_h J^T J          (SPD for gamma_h large enough iff the reduced Hessian is: the same
                                                        inertia test by Cholesky as Eq. 15; same sparsity as Eq. 17's K)
    S dlam = J K_g^-1 (r1 + gamma_h J^T r2) - r2,      S = J K_g^-1 J^T   -- conjugate gradients, one K_g solve per iteration
    dy     = K_g^-1 (r1 + gamma_h J^T r2 - J^T dlam)

i.e. the direct part is exactly the paper's SymCholesky / NumCholesky / triangular solves (Eq. 18-25) applied to K_g, the
iterative part a CG on the Schur complement.  Everything else (mu rule, fraction to the boundary, inertia schedule, error
measure, warm start) is the reading of oracle/ipm.py with the slack rows removed; lam moves with the primal step length.
"""
from __future__ import annotations

import numpy as np
import scipy.sparse as sp

from .ipm import DEFAULTS, _max_step
from .linalg import BlockTridiagCholesky, DenseCholesky, NotPositiveDefinite, SparseCholesky
from .nlp import TranscribedOCP

HYKKT_DEFAULTS = dict(gamma_h=1e6, cg_tol=1e-10, cg_max_iter=50)


class HyKKTState:
    def __init__(self, y, lam, zL, zU):
        self.y, self.lam, self.zL, self.zU = y, lam, zL, zU

    def copy(self):
        return HyKKTState(self.y.copy(), self.lam.copy(), self.zL.copy(), self.zU.copy())


class HyKKTIPM:
    def __init__(self, cfg, linsolve="sparse", perm=None, **options):
        self.cfg = cfg
        self.nlp = TranscribedOCP(cfg)
        self.opt = dict(DEFAULTS)
        self.opt.update(HYKKT_DEFAULTS)
        self.opt.update(options)
        if self.opt["mu_warm"] is None:
            self.opt["mu_warm"] = self.opt["eps_outer"] / 10.0
        self.linsolve, self.perm = linsolve, perm
        self.chol = None
        self.state = None
        self.hasL, self.hasU = np.isfinite(self.nlp.lb), np.isfinite(self.nlp.ub)
        self.lb = np.where(self.hasL, self.nlp.lb, 0.0)
        self.ub = np.where(self.hasU, self.nlp.ub, 0.0)
        self.cg_iterations = 0

    def _make_cholesky(self):
        if self.linsolve == "dense":
            return DenseCholesky(self.nlp.n)
        if self.linsolve == "blocktri":
            return BlockTridiagCholesky(self.nlp.N, self.nlp.nv)
        return SparseCholesky(self.nlp.K_pattern(), self.perm)

    def _errors(self, st, gradf, c, J, mu):
        o, hasL, hasU = self.opt, self.hasL, self.hasU
        dL, dU = st.y - self.lb, self.ub - st.y
        r_d = gradf + J.T @ st.lam - np.where(hasL, st.zL, 0.0) + np.where(hasU, st.zU, 0.0)
        comp = np.concatenate([(dL * st.zL - mu)[hasL], (dU * st.zU - mu)[hasU], [0.0]])
        nmult = self.nlp.m + int(hasL.sum()) + int(hasU.sum())
        l1 = np.abs(st.lam).sum() + st.zL[hasL].sum() + st.zU[hasU].sum()
        s_d = max(o["s_max"], l1 / nmult) / o["s_max"]
        return max(np.max(np.abs(r_d)) / s_d, np.max(np.abs(c)), np.max(np.abs(comp)) / s_d), r_d

    def cold_start(self, y0):
        o = self.opt
        y = np.array(y0, dtype=np.float64)
        kp = o["kappa_push"]
        both = self.hasL & self.hasU
        pL = np.where(both, np.minimum(kp * np.maximum(1.0, np.abs(self.lb)), kp * (self.ub - self.lb)), kp * np.maximum(1.0, np.abs(self.lb)))
        pU = np.where(both, np.minimum(kp * np.maximum(1.0, np.abs(self.ub)), kp * (self.ub - self.lb)), kp * np.maximum(1.0, np.abs(self.ub)))
        y = np.where(self.hasL, np.maximum(y, self.lb + pL), y)
        y = np.where(self.hasU, np.minimum(y, self.ub - pU), y)
        mu0 = o["mu0"]
        zL = np.where(self.hasL, mu0 / np.where(self.hasL, y - self.lb, 1.0), 0.0)
        zU = np.where(self.hasU, mu0 / np.where(self.hasU, self.ub - y, 1.0), 0.0)
        return HyKKTState(y, np.zeros(self.nlp.m), zL, zU), mu0

    def warm_start(self, prev):
        st = prev.copy()
        w = self.opt["warm_push"]
        st.y = np.where(self.hasL, np.maximum(st.y, self.lb + w), st.y)
        st.y = np.where(self.hasU, np.minimum(st.y, self.ub - w), st.y)
        return st, self.opt["mu_warm"]

    def _cg(self, J, rhs):
        """Conjugate gradients on S = J K_g^-1 J^T (SPD), zero start, stop at |r|_2 <= cg_tol |rhs|_2."""
        o = self.opt
        x = np.zeros_like(rhs)
        r = rhs.copy()
        p = r.copy()
        rr = float(r @ r)
        stop = (o["cg_tol"] ** 2) * rr
        k = 0
        while k < o["cg_max_iter"] and rr > stop and rr > 0.0:
            Sp = J @ self.chol.solve(J.T @ p)
            a = rr / float(p @ Sp)
            x += a * p
            r -= a * Sp
            rr_new = float(r @ r)
            p = r + (rr_new / rr) * p
            rr = rr_new
            k += 1
        self.cg_iterations += k
        return x, k

    def solve(self, y0=None, warm=False):
        o, nlp = self.opt, self.nlp
        hasL, hasU = self.hasL, self.hasU
        if warm and self.state is not None:
            st, mu = self.warm_start(self.state)
        else:
            st, mu = self.cold_start(nlp.cfg.y_cold(nlp.x0) if y0 is None else y0)
        eta_last, nfact, it, status, tr = 0.0, 0, 0, "maxiter", []
        g = o["gamma_h"]
        while True:
            gradf, c, J = nlp.gradient(st.y), nlp.constraints(st.y), nlp.jacobian(st.y)
            E0, _ = self._errors(st, gradf, c, J, 0.0)
            if E0 <= o["eps_outer"]:
                status = "converged"
                break
            if it >= o["max_iter"]:
                break
            Emu, r_d = self._errors(st, gradf, c, J, mu)
            while Emu <= o["kappa_eps"] * mu and mu > o["eps_outer"] / 10.0:
                mu = max(o["eps_outer"] / 10.0, min(o["kappa_mu"] * mu, mu ** o["theta_mu"]))
                Emu, r_d = self._errors(st, gradf, c, J, mu)
            tau = max(o["tau_min"], 1.0 - mu)
            dL = np.where(hasL, st.y - self.lb, 1.0)
            dU = np.where(hasU, self.ub - st.y, 1.0)
            Sigma_x = np.where(hasL, st.zL / dL, 0.0) + np.where(hasU, st.zU / dU, 0.0)
            W = nlp.hessian(st.y, st.lam)
            Kg0 = (W + sp.diags(Sigma_x) + g * (J.T @ J)).tocsc()
            r1 = -(gradf + J.T @ st.lam - np.where(hasL, mu / dL, 0.0) + np.where(hasU, mu / dU, 0.0))
            r2 = -c
            if self.chol is None:
                self.chol = self._make_cholesky()
            eta = 0.0
            while True:
                try:
                    nfact += 1
                    self.chol.factor(Kg0 + eta * sp.identity(nlp.n, format="csc") if eta > 0.0 else Kg0)
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
            bg = r1 + g * (J.T @ r2)
            u = self.chol.solve(bg)
            dlam, ncg = self._cg(J, J @ u - r2)
            dy = self.chol.solve(bg - J.T @ dlam)
            dzL = np.where(hasL, -(st.zL - mu / dL) - st.zL / dL * dy, 0.0)
            dzU = np.where(hasU, -(st.zU - mu / dU) + st.zU / dU * dy, 0.0)
            a_pr = min(_max_step(dL[hasL], dy[hasL], tau), _max_step(dU[hasU], -dy[hasU], tau))
            a_du = min(_max_step(st.zL[hasL], dzL[hasL], tau), _max_step(st.zU[hasU], dzU[hasU], tau))
            tr.append(dict(it=it, mu=mu, E0=E0, Emu=Emu, eta=eta, alpha_pr=a_pr, alpha_du=a_du, cg=ncg))
            self.last_step = dict(state=st, mu=mu, eta=eta, J=J, W=W, Sigma_x=Sigma_x, r1=r1, r2=r2, dy=dy, dlam=dlam, dzL=dzL, dzU=dzU)
            st = HyKKTState(st.y + a_pr * dy, st.lam + a_pr * dlam, st.zL + a_du * dzL, st.zU + a_du * dzU)
            if not np.all(np.isfinite(st.y)):
                status = "step"
                break
            it += 1
        self.state = st
        return dict(status=status, iters=it, factorizations=nfact, state=st, trace=tr, E0=E0, mu=mu)


def hykkt_closed_loop(cfg, n_resolves=None, linsolve="sparse", **options):
    """Algorithm 1 with the HyKKT variant of Algorithm 2 (same loop as oracle.ipm.nmpc_closed_loop)."""
    R = cfg.R if n_resolves is None else n_resolves
    ipm = HyKKTIPM(cfg, linsolve=linsolve, **options)
    x0 = np.array(cfg.x0, dtype=np.float64)
    out = []
    for j in range(R + 1):
        ref = cfg.ref_for_solve(j)
        ipm.nlp.set_params(x0, ref)
        res = ipm.solve(warm=(j > 0))
        y = res["state"].y
        out.append(dict(solve=j, x0=x0.copy(), ref=ref, y=y.copy(), iters=res["iters"], status=res["status"],
                        factorizations=res["factorizations"], trace=res["trace"], state=res["state"].copy()))
        x0 = np.clip(y[: cfg.nx] + cfg.noise_for_solve(j), cfg.x0_clip[0], cfg.x0_clip[1])
    return out, ipm
