"""Seeded synthetic inputs for the five benchmark OCPs (C0..C4 of BASELINE.json:configs).

This module is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA path
(`paper_2606_04725_b200/`).  It holds no arithmetic of the method: no model function, no derivative,
no KKT assembly, no factorization, no IPM step.  It only states sizes, physical constants, bounds and the
seeded random data (initial states, setpoints / target fields, measurement-noise sequences) that both sides
receive as plain arrays.  No RNG is used inside either implementation.

The five configs stand in for the paper's Van der Pol tutorial-size problem, its distillation column
(Table 1 :443-447) and its 2-D heated plate (Table 2 :499-503); the recipe
is the one in SURVEY.md §8(d) and is restated in DESIGN.md §4.

Variable layout (both sides):  y = [x_1,u_1, x_2,u_2, ..., x_N,u_N]  (stage-major, nv = nx+nu per stage),
x_0 is a parameter.  Equality rows: stage k holds rows k*nx .. (k+1)*nx-1 of
h_k = x_k - x_{k-1} - dt*F(x_k,u_k).

General linear path rows (optional, `make_config(..., Nc=, move_limit=,
power_limit=)`): rows  lo <= G y <= hi  appended AFTER the N*nx dynamics rows, stated here as plain CSR data:
  * control-horizon hold:  u_k - u_{k-1} = 0 for the stages k >= Nc (lo = hi = 0),
  * input move limits:  -move_limit <= u_k - u_{k-1} <= move_limit for 1 <= k < Nc (two-sided inequality rows g),
  * total input limit:  sum_a u_{k,a} <= power_limit for every stage (one-sided inequality row g, lo = -inf).

Model parameter vectors (`model_params`, float64), by model id:
  MODEL_VDP     : [w_x, w_u]
  MODEL_DISTILL : [alpha, D, F_feed, x_feed, A_c, A_t, A_r, feed_index, u_bar, w_u]
  MODEL_PLATE   : [g, a, kappa_r, T_amb, b, nseg, w_T, w_u]
"""
from __future__ import annotations

import numpy as np

MASTER_SEED = 20260604

MODEL_NONE, MODEL_VDP, MODEL_DISTILL, MODEL_PLATE, MODEL_LQ = 0, 1, 2, 3, 4

CONFIG_NAMES = ("C0", "C1", "C2", "C3", "C4")

SIGMA_SB = 5.670374419e-8  # Stefan-Boltzmann constant, W m^-2 K^-4


class OCPConfig:
    """Plain record of one benchmark configuration (sizes, constants, seeded data)."""

    def __init__(self, **kw):
        self.__dict__.update(kw)
        self.nv = self.nx + self.nu
        self.n = self.N * self.nv
        self.m_dyn = self.N * self.nx          # dynamics rows h_k
        self.m = self.m_dyn                    # all constraint rows (dynamics + general linear rows, see add_path_rows)
        self.g_rows = None

    def __repr__(self):
        return (f"OCPConfig({self.name}: model={self.model} N={self.N} nx={self.nx} nu={self.nu} "
                f"n={self.n} m={self.m} R={self.R})")

    # ---- per-re-solve data (pure table look-ups, no arithmetic of the method) ----
    def ref_for_solve(self, j: int) -> np.ndarray:
        """Reference array (N*nr,) for NMPC solve j (j=0 is the cold solve)."""
        return self.ref_seq[min(j, len(self.ref_seq) - 1)]

    def noise_for_solve(self, j: int) -> np.ndarray:
        """Measurement noise (nx,) added to x_1* of solve j to obtain x0 of solve j+1."""
        return self.noise_seq[j % len(self.noise_seq)]

    def y_cold(self, x0: np.ndarray) -> np.ndarray:
        """Cold-start primal guess (reading G9): x_k = x0 for all k, u_k = u_init."""
        y = np.empty((self.N, self.nv))
        y[:, : self.nx] = x0[None, :]
        y[:, self.nx:] = self.u_init[None, :]
        return y.reshape(-1)

    def lb_full(self) -> np.ndarray:
        return np.tile(self.lb, self.N)

    def ub_full(self) -> np.ndarray:
        return np.tile(self.ub, self.N)


def _vdp(rng) -> OCPConfig:
    N, R = 40, 20
    x0 = rng.uniform(-1.0, 1.0, 2)
    r = rng.uniform(-1.0, 1.0, 2)
    ref = np.tile(r, N)
    noise = rng.normal(0.0, 0.05, (R, 2))
    return OCPConfig(name="C0", title="vdp", model=MODEL_VDP, N=N, nx=2, nu=1, nr=2, dt=0.1,
                     model_params=np.array([10.0, 0.1]),
                     lb=np.array([-3.0, -3.0, -1.0]), ub=np.array([3.0, 3.0, 1.0]),
                     u_init=np.array([0.0]), x0=x0, ref_seq=[ref], noise_seq=noise, R=R,
                     x0_clip=(-2.9, 2.9))


def _distill(rng, name, trays, N, R) -> OCPConfig:
    nx = trays + 2
    feed = trays // 2 + 1                     # 17 for 32 trays (Table 1: N_f = 17), 65 for 128
    u_bar = 2.51459
    params = np.array([1.6, 0.2, 0.4, 0.5, 0.5, 0.25, 1.0, float(feed), u_bar, 0.1])
    x0 = np.linspace(0.9, 0.1, nx)
    refs = []
    for _ in range(R + 1):                    # one setpoint per solve, constant over the horizon
        refs.append(np.full(N, 0.935 + rng.uniform(-0.02, 0.02)))
    noise = np.zeros((1, nx))
    lb = np.concatenate([np.zeros(nx), [0.5]])
    ub = np.concatenate([np.ones(nx), [5.0]])
    return OCPConfig(name=name, title=f"distill-{nx}", model=MODEL_DISTILL, N=N, nx=nx, nu=1, nr=1, dt=1.0,
                     model_params=params, lb=lb, ub=ub, u_init=np.array([u_bar]), x0=x0,
                     ref_seq=refs, noise_seq=noise, R=R, x0_clip=(1e-6, 1.0 - 1e-6))


def _plate(rng, name, g, nseg, N, R, noise_sd) -> OCPConfig:
    nx, nu = g * g, 4 * nseg
    side, alpha, eps, C_A, T_amb, rho_c = 0.1, 1e-4, 0.8, 1215.0, 300.0, 1.0e5
    dx = side / g
    a = alpha / dx ** 2
    kappa_r = 2.0 * SIGMA_SB * eps / C_A
    b = 1.0e4 / (rho_c * dx)
    params = np.array([float(g), a, kappa_r, T_amb, b, float(nseg), 1.0 / (nx * 100.0 ** 2), 1e-4])
    # smooth target field: 300 + 200 * G / max G, G = sum of three Gaussians on the unit square (cell centres)
    amp = rng.uniform(0.5, 1.0, 3)
    ctr = rng.uniform(0.2, 0.8, (3, 2))
    wid = rng.uniform(0.1, 0.25, 3)
    xi = (np.arange(g) + 0.5) / g
    X1, X2 = np.meshgrid(xi, xi, indexing="ij")
    G = np.zeros((g, g))
    for q in range(3):
        G += amp[q] * np.exp(-((X1 - ctr[q, 0]) ** 2 + (X2 - ctr[q, 1]) ** 2) / (2.0 * wid[q] ** 2))
    target = 300.0 + 200.0 * G / G.max()
    ref = np.tile(target.reshape(-1), N)
    noise = rng.normal(0.0, noise_sd, (R, nx)) if noise_sd > 0 else np.zeros((1, nx))
    lb = np.concatenate([np.full(nx, -np.inf), np.zeros(nu)])
    ub = np.concatenate([np.full(nx, 600.0), np.ones(nu)])
    return OCPConfig(name=name, title=f"plate-{g}", model=MODEL_PLATE, N=N, nx=nx, nu=nu, nr=nx, dt=2.0,
                     model_params=params, lb=lb, ub=ub, u_init=np.full(nu, 0.01), x0=np.full(nx, 300.0),
                     ref_seq=[ref], noise_seq=noise, R=R, x0_clip=(-np.inf, 599.0))


def add_path_rows(cfg: OCPConfig, Nc=None, move_limit=None, power_limit=None) -> OCPConfig:
    """Append general linear rows lo <= G y <= hi (module docstring) to `cfg` as CSR data: cfg.g_rows = dict(rowptr, colind,
    val, lo, hi); cfg.m grows by their number.  Pure index bookkeeping: no arithmetic of the method."""
    N, nx, nu, nv = cfg.N, cfg.nx, cfg.nu, cfg.nv
    Nc = N if Nc is None else int(Nc)
    rowptr, colind, val, lo, hi = [0], [], [], [], []

    def row(cols, vals, l, h):
        order = np.argsort(cols)
        colind.extend(int(cols[i]) for i in order); val.extend(float(vals[i]) for i in order)
        rowptr.append(len(colind)); lo.append(l); hi.append(h)

    for k in range(1, N):
        for a in range(nu):
            cols, vals = [(k - 1) * nv + nx + a, k * nv + nx + a], [-1.0, 1.0]
            if k >= Nc:
                row(cols, vals, 0.0, 0.0)
            elif move_limit is not None:
                row(cols, vals, -float(move_limit), float(move_limit))
    if power_limit is not None:
        for k in range(N):
            row([k * nv + nx + a for a in range(nu)], [1.0] * nu, -np.inf, float(power_limit))
    if len(lo) == 0:
        return cfg
    cfg.g_rows = dict(rowptr=np.array(rowptr, dtype=np.int64), colind=np.array(colind, dtype=np.int32),
                      val=np.array(val, dtype=np.float64), lo=np.array(lo, dtype=np.float64), hi=np.array(hi, dtype=np.float64))
    cfg.m = cfg.m_dyn + len(lo)
    cfg.path_rows = dict(Nc=Nc, move_limit=move_limit, power_limit=power_limit)
    return cfg


def make_config(name: str, **override) -> OCPConfig:
    """Return config `name` in {C0..C4}.  `override` may shrink N / g / trays for small test cases
    (the seeded stream is the same; only the sizes change)."""
    idx = CONFIG_NAMES.index(name)
    rng = np.random.default_rng(MASTER_SEED + idx)
    path = {k: override.pop(k) for k in ("Nc", "move_limit", "power_limit") if k in override}
    if name == "C0":
        cfg = _vdp(rng)
    elif name == "C1":
        cfg = _distill(rng, "C1", override.pop("trays", 32), override.pop("N", 100), override.pop("R", 50))
    elif name == "C2":
        cfg = _plate(rng, "C2", override.pop("g", 20), override.pop("nseg", 1), override.pop("N", 50),
                     override.pop("R", 20), 0.0)
    elif name == "C3":
        cfg = _plate(rng, "C3", override.pop("g", 50), override.pop("nseg", 4), override.pop("N", 50),
                     override.pop("R", 10), 2.0)
    elif name == "C4":
        cfg = _distill(rng, "C4", override.pop("trays", 128), override.pop("N", 400), override.pop("R", 50))
    if override:
        raise TypeError(f"unknown overrides {sorted(override)}")
    if path:
        add_path_rows(cfg, **path)
    return cfg


def sigma_sweep_draws(cfg: OCPConfig, count: int = 200, seed_offset: int = 100):
    """C4 refactor sweep (BASELINE.json:configs[4]): per draw Sigma_x (n,), Sigma_s (m,) log-uniform in
    [1e-8, 1e8] and a right-hand side b ~ N(0, I).  Generator -> (sigma_x, sigma_s, b)."""
    rng = np.random.default_rng(MASTER_SEED + seed_offset)
    for _ in range(count):
        sx = 10.0 ** rng.uniform(-8.0, 8.0, cfg.n)
        ss = 10.0 ** rng.uniform(-8.0, 8.0, cfg.m)
        b = rng.normal(0.0, 1.0, cfg.n)
        yield sx, ss, b


def lq_instance(nx: int = 3, nu: int = 2, N: int = 12, dt: float = 0.2, seed: int = 7):
    """Unconstrained linear-quadratic instance for the Riccati pin:
    F(x,u) = A x + B u,  l = x'Qx + u'Ru,  no bounds.  model_params = [A (row-major), B, diag Q, diag R]."""
    rng = np.random.default_rng(MASTER_SEED + 1000 + seed)
    A = rng.normal(0.0, 0.6, (nx, nx)) - 0.5 * np.eye(nx)
    B = rng.normal(0.0, 1.0, (nx, nu))
    q = rng.uniform(0.5, 2.0, nx)
    r = rng.uniform(0.1, 1.0, nu)
    x0 = rng.normal(0.0, 1.0, nx)
    params = np.concatenate([A.reshape(-1), B.reshape(-1), q, r])
    cfg = OCPConfig(name="LQ", title="lq", model=MODEL_LQ, N=N, nx=nx, nu=nu, nr=0, dt=dt, model_params=params,
                    lb=np.full(nx + nu, -np.inf), ub=np.full(nx + nu, np.inf), u_init=np.zeros(nu), x0=x0,
                    ref_seq=[np.zeros(0)], noise_seq=np.zeros((1, nx)), R=0, x0_clip=(-np.inf, np.inf))
    cfg.A, cfg.B, cfg.q, cfg.r = A, B, q, r
    return cfg
