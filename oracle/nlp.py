"""oracle/nlp.py -- TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).

The transcribed parametric OCP  P_k(p_k)  of PAPER.md:98-126 (Problems 5/6) for the stage-structured
benchmark models: backward (implicit) Euler ("backward finite difference") with the
initial state x_0 = ybar_s(p) a PARAMETER, not a variable:

    y = [x_1,u_1, ..., x_N,u_N],      f(y;p) = sum_k l(x_k,u_k; ref_k),
    h_k(y;p) = x_k - x_{k-1} - dt F(x_k,u_k) = 0,  k = 1..N,      lb <= (x_k,u_k) <= ub.

J = dh/dy  (block lower bidiagonal:  [-I | I - dt A_k | -dt B_k]),
W = Hess f + sum_k lam_k Hess h_k = blockdiag( Hess l - dt sum_c lam_{k,c} Hess F_c ).
The parameter vector p = (x0, ref) is what changes between NMPC re-solves.

General rows (Problem 5/6: inequality constraints g and the control-horizon constraints
y_c,u = y_c,u_c; reading G22 of DESIGN.md section 3): linear rows  lo <= G y <= hi  stated by the configuration
(ocp_inputs.add_path_rows) are stacked BELOW the dynamics rows: c(y) = [h(y); G y], J = [dh/dy; G]; they are linear, so they
do not enter W.  `row_bounds(gamma)` gives the interval [cl, cu] of every row of c: the lifted equalities of Eq. (16),
-gamma <= h <= gamma, for the dynamics rows and for the equality rows of G (lo == hi: lo - gamma, hi + gamma), and [lo, hi]
itself (either side may be infinite) for the inequality rows.
"""
from __future__ import annotations

import numpy as np
import scipy.sparse as sp

from .models import make_model


class TranscribedOCP:
    def __init__(self, cfg):
        self.cfg = cfg
        self.model = make_model(cfg)
        self.N, self.nx, self.nu, self.nv = cfg.N, cfg.nx, cfg.nu, cfg.nx + cfg.nu
        self.n, self.m, self.dt = cfg.n, cfg.m, cfg.dt
        self.m_dyn = self.N * self.nx
        g = getattr(cfg, "g_rows", None)
        if g is not None:
            self.G = sp.csr_matrix((g["val"], g["colind"], g["rowptr"]), shape=(len(g["lo"]), self.n))
            self.glo, self.ghi = np.array(g["lo"], dtype=np.float64), np.array(g["hi"], dtype=np.float64)
        else:
            self.G = None
        assert self.m == self.m_dyn + (0 if self.G is None else self.G.shape[0])
        self.lb, self.ub = cfg.lb_full(), cfg.ub_full()
        self.x0 = np.array(cfg.x0, dtype=np.float64)
        self.ref = np.array(cfg.ref_for_solve(0), dtype=np.float64)
        # constant "-I" coupling of stage k to x_{k-1}
        rows = np.arange(self.nx, self.m_dyn)
        cols = ((rows // self.nx) - 1) * self.nv + (rows % self.nx)
        self._shift = sp.csr_matrix((np.ones(len(rows)), (rows, cols)), shape=(self.m_dyn, self.n))

    # ---- parameters p = (x0, ref): the only thing a re-solve changes ----
    def set_params(self, x0, ref):
        self.x0 = np.array(x0, dtype=np.float64)
        self.ref = np.array(ref, dtype=np.float64)

    def split(self, y):
        Y = np.asarray(y).reshape(self.N, self.nv)
        return Y[:, : self.nx], Y[:, self.nx:]

    def _ref(self, k):
        nr = self.cfg.nr
        return self.ref[k * nr:(k + 1) * nr]

    # ---- objective ----
    def objective(self, y):
        X, U = self.split(y)
        return sum(self.model.cost(X[k], U[k], self._ref(k)) for k in range(self.N))

    def gradient(self, y):
        X, U = self.split(y)
        return np.concatenate([self.model.cost_grad(X[k], U[k], self._ref(k)) for k in range(self.N)])

    # ---- constraint rows c(y;p) = [h(y;p); G y] ----
    def constraints(self, y):
        X, U = self.split(y)
        c = np.empty((self.N, self.nx))
        for k in range(self.N):
            xprev = self.x0 if k == 0 else X[k - 1]
            c[k] = X[k] - xprev - self.dt * self.model.F(X[k], U[k])
        c = c.reshape(-1)
        return c if self.G is None else np.concatenate([c, self.G @ np.asarray(y)])

    def row_bounds(self, gamma):
        """[cl, cu] of every row of c (module docstring)."""
        cl, cu = np.full(self.m_dyn, -gamma), np.full(self.m_dyn, gamma)
        if self.G is None:
            return cl, cu
        eq = self.glo == self.ghi
        return (np.concatenate([cl, np.where(eq, self.glo - gamma, self.glo)]),
                np.concatenate([cu, np.where(eq, self.ghi + gamma, self.ghi)]))

    def jacobian(self, y):
        X, U = self.split(y)
        blocks = []
        eye = sp.identity(self.nx, format="csr")
        for k in range(self.N):
            A, B = self.model.AB(X[k], U[k])
            blocks.append(sp.hstack([eye - self.dt * A, -self.dt * B], format="csr"))
        Jh = (sp.block_diag(blocks, format="csr") - self._shift).tocsr()
        return Jh if self.G is None else sp.vstack([Jh, self.G], format="csr")

    # ---- Hessian of the Lagrangian, lam = multiplier of h ----
    def hessian(self, y, lam):
        X, U = self.split(y)
        Lam = np.asarray(lam)[: self.m_dyn].reshape(self.N, self.nx)    # the general rows are linear
        Hl = self.model.cost_hess()
        blocks = [Hl - self.dt * self.model.hessF(X[k], U[k], Lam[k]) for k in range(self.N)]
        return sp.block_diag(blocks, format="csr")

    # ---- structural pattern of K = W + Sigma_x + J^T Q J  (values irrelevant, all entries positive) ----
    def K_pattern(self):
        rng = np.random.default_rng(12345)
        lo = np.where(np.isfinite(self.lb), self.lb, 250.0)
        hi = np.where(np.isfinite(self.ub), self.ub, lo + 100.0)
        y = lo + (hi - lo) * rng.uniform(0.2, 0.8, self.n)
        J = abs(self.jacobian(y))
        W = abs(self.hessian(y, rng.uniform(0.5, 1.5, self.m)))
        P = (J.T @ J + W + sp.identity(self.n)).tocsr()
        P.data[:] = 1.0
        return P
