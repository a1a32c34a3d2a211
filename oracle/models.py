"""oracle/models.py -- TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).

Stage models of the five benchmark OCPs: continuous-time right-hand side F(x,u), its Jacobians
A = dF/dx, B = dF/du, the multiplier-weighted second derivative  sum_c lam_c * Hess_{(x,u)} F_c,
and the stage cost l(x,u;ref) with gradient and (constant) Hessian.

All functions act on ONE stage (x: (nx,), u: (nu,)) and are written so that each line can be compared with the
model statement by eye; the stage loop lives in oracle/nlp.py.

Model statements followed:
  VdP      BASELINE.json:configs[0]:  x1' = x2,  x2' = (1-x1^2) x2 - x1 + u;  l = 10||x-r||^2 + 0.1 u^2
  distill  PAPER.md:451-473 (Problem 29) read as DESIGN.md §3 G12 / SURVEY.md §8(d) C1, with the vapour
           composition y_i eliminated (BASELINE.json:configs[1]: "one liquid composition state each")
  plate    BASELINE.json:configs[2]: 5-point heat equation, radiative loss, edge heaters
  LQ       F = A x + B u, l = x'Qx + u'Ru (Riccati pin)
"""
from __future__ import annotations

import numpy as np
import scipy.sparse as sp

from ocp_inputs import MODEL_DISTILL, MODEL_LQ, MODEL_PLATE, MODEL_VDP


# ======================================================================================================
# Van der Pol
# ======================================================================================================
class VdP:
    def __init__(self, cfg):
        self.nx, self.nu = 2, 1
        self.w_x, self.w_u = cfg.model_params[:2]

    def F(self, x, u):
        return np.array([x[1], (1.0 - x[0] ** 2) * x[1] - x[0] + u[0]])

    def AB(self, x, u):
        A = np.array([[0.0, 1.0],
                      [-2.0 * x[0] * x[1] - 1.0, 1.0 - x[0] ** 2]])
        B = np.array([[0.0], [1.0]])
        return sp.csr_matrix(A), sp.csr_matrix(B)

    def hessF(self, x, u, lam):
        # only F_2 is nonlinear: d2F2/dx1^2 = -2 x2 ; d2F2/dx1 dx2 = -2 x1
        H = np.zeros((3, 3))
        H[0, 0] = lam[1] * (-2.0 * x[1])
        H[0, 1] = H[1, 0] = lam[1] * (-2.0 * x[0])
        return sp.csr_matrix(H)

    def cost(self, x, u, ref):
        return self.w_x * np.sum((x - ref) ** 2) + self.w_u * u[0] ** 2

    def cost_grad(self, x, u, ref):
        return np.concatenate([2.0 * self.w_x * (x - ref), [2.0 * self.w_u * u[0]]])

    def cost_hess(self):
        return sp.diags([2.0 * self.w_x, 2.0 * self.w_x, 2.0 * self.w_u]).tocsr()


# ======================================================================================================
# Binary distillation column (condenser = state 0, trays 1..n-2, reboiler = state n-1)
# ======================================================================================================
class Distill:
    def __init__(self, cfg):
        p = cfg.model_params
        self.alpha, self.D, self.Ff, self.xf, self.Ac, self.At, self.Ar = p[:7]
        self.f = int(p[7])
        self.ubar, self.w_u = p[8], p[9]
        self.nx, self.nu = cfg.nx, 1

    # vapour-liquid equilibrium y = alpha x / (1 + (alpha-1) x) and its derivatives
    def vle(self, x):
        return self.alpha * x / (1.0 + (self.alpha - 1.0) * x)

    def dvle(self, x):
        return self.alpha / (1.0 + (self.alpha - 1.0) * x) ** 2

    def d2vle(self, x):
        return -2.0 * self.alpha * (self.alpha - 1.0) / (1.0 + (self.alpha - 1.0) * x) ** 3

    def flows(self, u):
        L = u[0] * self.D
        V = L + self.D
        S = L + self.Ff
        return L, V, S

    def _liquid_in_out(self, L, S):
        """Liquid flow entering / leaving tray i (1..n-2): (L,L) above the feed, (L,S) at it, (S,S) below."""
        i = np.arange(1, self.nx - 1)
        return i, np.where(i <= self.f, L, S), np.where(i < self.f, L, S)

    def F(self, x, u):
        n, f = self.nx, self.f
        L, V, S = self.flows(u)
        y = self.vle(x)
        dx = np.zeros(n)
        dx[0] = V * (y[1] - x[0]) / self.Ac                                           # condenser
        i, lin, lout = self._liquid_in_out(L, S)                                      # trays 1..n-2
        dx[i] = (lin * x[i - 1] - lout * x[i] - V * (y[i] - y[i + 1])) / self.At
        dx[f] += self.Ff * self.xf / self.At                                          # feed enters tray f
        dx[n - 1] = (S * x[n - 2] - (self.Ff - self.D) * x[n - 1] - V * y[n - 1]) / self.Ar   # reboiler
        return dx

    def AB(self, x, u):
        n, D = self.nx, self.D
        L, V, S = self.flows(u)
        y, dy = self.vle(x), self.dvle(x)
        A = np.zeros((n, n))
        B = np.zeros((n, 1))
        A[0, 0] = -V / self.Ac
        A[0, 1] = V * dy[1] / self.Ac
        B[0, 0] = D * (y[1] - x[0]) / self.Ac                      # dV/du = D
        i, lin, lout = self._liquid_in_out(L, S)
        A[i, i - 1] = lin / self.At
        A[i, i] = (-lout - V * dy[i]) / self.At
        A[i, i + 1] = V * dy[i + 1] / self.At
        # every flow (L, V, S) has derivative D with respect to u
        B[i, 0] = D * ((x[i - 1] - x[i]) - (y[i] - y[i + 1])) / self.At
        A[n - 1, n - 2] = S / self.Ar
        A[n - 1, n - 1] = (-(self.Ff - self.D) - V * dy[n - 1]) / self.Ar
        B[n - 1, 0] = D * (x[n - 2] - y[n - 1]) / self.Ar
        return sp.csr_matrix(A), sp.csr_matrix(B)

    def hessF(self, x, u, lam):
        n, D = self.nx, self.D
        L, V, S = self.flows(u)
        dy, d2y = self.dvle(x), self.d2vle(x)
        iu = n
        H = np.zeros((n + 1, n + 1))           # upper triangle accumulated, symmetrised at the end
        # condenser: F_0 = V (y_1 - x_0)/A_c
        H[1, 1] += lam[0] * V * d2y[1] / self.Ac
        H[0, iu] += lam[0] * (-D) / self.Ac
        H[1, iu] += lam[0] * D * dy[1] / self.Ac
        # trays: F_i = [flow_in x_{i-1} - flow_out x_i - V (y_i - y_{i+1}) (+ feed)]/A_t
        i = np.arange(1, n - 1)
        l = lam[i] / self.At
        np.add.at(H, (i, i), l * (-V * d2y[i]))
        np.add.at(H, (i + 1, i + 1), l * (V * d2y[i + 1]))
        np.add.at(H, (i - 1, iu), l * D)
        np.add.at(H, (i, iu), l * (-D - D * dy[i]))
        np.add.at(H, (i + 1, iu), l * D * dy[i + 1])
        # reboiler: F_{n-1} = [S x_{n-2} - (F-D) x_{n-1} - V y_{n-1}]/A_r
        l = lam[n - 1] / self.Ar
        H[n - 1, n - 1] += l * (-V * d2y[n - 1])
        H[n - 2, iu] += l * D
        H[n - 1, iu] += l * (-D * dy[n - 1])
        H = H + np.triu(H, 1).T
        return sp.csr_matrix(H)

    def cost(self, x, u, ref):
        return (x[0] - ref[0]) ** 2 + self.w_u * (u[0] - self.ubar) ** 2

    def cost_grad(self, x, u, ref):
        g = np.zeros(self.nx + 1)
        g[0] = 2.0 * (x[0] - ref[0])
        g[self.nx] = 2.0 * self.w_u * (u[0] - self.ubar)
        return g

    def cost_hess(self):
        d = np.zeros(self.nx + 1)
        d[0] = 2.0
        d[self.nx] = 2.0 * self.w_u
        return sp.diags(d).tocsr()


# ======================================================================================================
# 2-D heated plate, cell c = i*g + j, heaters on the four edges
# ======================================================================================================
class Plate:
    def __init__(self, cfg):
        p = cfg.model_params
        g = int(p[0])
        self.g, self.a, self.kr, self.Tamb, self.b = g, p[1], p[2], p[3], p[4]
        self.nseg = int(p[5])
        self.w_T, self.w_u = p[6], p[7]
        self.nx, self.nu = g * g, 4 * self.nseg
        # 5-point graph Laplacian, missing neighbours dropped (insulated edges)
        Lap = sp.lil_matrix((self.nx, self.nx))
        for i in range(g):
            for j in range(g):
                c = i * g + j
                for (ii, jj) in ((i - 1, j), (i + 1, j), (i, j - 1), (i, j + 1)):
                    if 0 <= ii < g and 0 <= jj < g:
                        Lap[c, ii * g + jj] += 1.0
                        Lap[c, c] -= 1.0
        self.Lap = Lap.tocsr()
        # heater incidence: edge e (0: i=0, 1: i=g-1, 2: j=0, 3: j=g-1), segment floor(t*nseg/g) along the edge
        Inc = sp.lil_matrix((self.nx, self.nu))
        for t in range(g):
            sgm = (t * self.nseg) // g
            Inc[0 * g + t, 0 * self.nseg + sgm] += 1.0
            Inc[(g - 1) * g + t, 1 * self.nseg + sgm] += 1.0
            Inc[t * g + 0, 2 * self.nseg + sgm] += 1.0
            Inc[t * g + (g - 1), 3 * self.nseg + sgm] += 1.0
        self.Inc = Inc.tocsr()

    def F(self, x, u):
        return self.a * (self.Lap @ x) - self.kr * (x ** 4 - self.Tamb ** 4) + self.b * (self.Inc @ u)

    def AB(self, x, u):
        A = self.a * self.Lap - sp.diags(4.0 * self.kr * x ** 3)
        return A.tocsr(), (self.b * self.Inc).tocsr()

    def hessF(self, x, u, lam):
        d = np.concatenate([lam * (-12.0 * self.kr * x ** 2), np.zeros(self.nu)])
        return sp.diags(d).tocsr()

    def cost(self, x, u, ref):
        return self.w_T * np.sum((x - ref) ** 2) + self.w_u * np.sum(u ** 2)

    def cost_grad(self, x, u, ref):
        return np.concatenate([2.0 * self.w_T * (x - ref), 2.0 * self.w_u * u])

    def cost_hess(self):
        return sp.diags(np.concatenate([np.full(self.nx, 2.0 * self.w_T), np.full(self.nu, 2.0 * self.w_u)])).tocsr()


# ======================================================================================================
# Linear-quadratic instance (Riccati pin)
# ======================================================================================================
class LQ:
    def __init__(self, cfg):
        self.nx, self.nu = cfg.nx, cfg.nu
        self.A, self.B, self.q, self.r = cfg.A, cfg.B, cfg.q, cfg.r

    def F(self, x, u):
        return self.A @ x + self.B @ u

    def AB(self, x, u):
        return sp.csr_matrix(self.A), sp.csr_matrix(self.B)

    def hessF(self, x, u, lam):
        return sp.csr_matrix((self.nx + self.nu, self.nx + self.nu))

    def cost(self, x, u, ref):
        return np.sum(self.q * x ** 2) + np.sum(self.r * u ** 2)

    def cost_grad(self, x, u, ref):
        return np.concatenate([2.0 * self.q * x, 2.0 * self.r * u])

    def cost_hess(self):
        return sp.diags(np.concatenate([2.0 * self.q, 2.0 * self.r])).tocsr()


def make_model(cfg):
    return {MODEL_VDP: VdP, MODEL_DISTILL: Distill, MODEL_PLATE: Plate, MODEL_LQ: LQ}[cfg.model](cfg)
