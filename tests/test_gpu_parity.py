"""Parity of the CUDA path (through the C-ABI of include/nmpc.h) against the CPU oracle, element by element on the
same seeded inputs.  Tolerances are north_star's: factor backward error <= 1e-12 (reading G17), normwise solve
residual <= 1e-10 (reading G16), converged primal solution <= 1e-6 relative, IPM iteration counts equal.

Steps covered: a1 parameter update, a2 model/derivative evaluation, a3 condensed assembly,
a4 numeric supernodal Cholesky (+ pivot failure, a4' inertia retry), a5 triangular solves, a6/a7 IPM vector kernels
and the barrier loop (via nmpc_ipm_solve), Algorithm 1 re-solves.
"""
import numpy as np
import pytest
import scipy.sparse as sp
import torch

import paper_2606_04725_b200 as nb
from ocp_inputs import make_config, sigma_sweep_draws
from oracle.ipm import LiftedIPM, nmpc_closed_loop
from oracle.linalg import SparseCholesky
from oracle.nlp import TranscribedOCP
from paper_2606_04725_b200 import binding

from gpu_util import factor_as_sparse, factor_backward_error, normwise_backward_error, values_on_pattern

pytestmark = pytest.mark.gpu

DEV = "cuda:0"
ORDERINGS = [binding.ORDER_NATURAL, binding.ORDER_AMD, binding.ORDER_ND, binding.ORDER_TIME_ND]
# sizes the oracle finishes in seconds that still span several tiles and a ragged tail:
#   C1m: fronts ~40-80 rows (shared-memory kernel, several supernodes per level)
#   C2m: g=9 -> fronts of a few hundred rows -> tiled big-front path with ragged 64-blocks
MID = [("C0", {}), ("C1", dict(trays=18, N=30)), ("C2", dict(g=9, N=7)), ("C3", dict(g=8, nseg=2, N=5)),
       ("C4", dict(trays=40, N=25))]


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).to(DEV)


def kkt_from_oracle(cfg, iters=3):
    """A genuine condensed lifted KKT matrix and right-hand side from a few oracle IPM iterations."""
    ipm = LiftedIPM(cfg, linsolve="blocktri", max_iter=iters)
    ipm.solve()
    ls = ipm.last_step
    K = ls["K0"] if ls["eta"] == 0.0 else (ls["K0"] + ls["eta"] * sp.identity(cfg.n)).tocsc()   # Eq. (13)/(17)
    return K, ls["b"], ipm


@pytest.mark.parametrize("name,ov", MID)
@pytest.mark.parametrize("ordering", ORDERINGS)
def test_factor_and_solve_vs_oracle(name, ov, ordering):
    cfg = make_config(name, **ov)
    K, b, _ = kkt_from_oracle(cfg)
    h = nb.Handle(None, nb.make_ocp(cfg), nb.default_options(ordering=ordering))
    info = h.get_info()
    rp, ci = h.get_kkt_pattern(cfg.n)
    vals = dev(values_on_pattern(K, rp, ci))
    st, _ = h.factor(vals, 0.0)
    assert st == 0
    L = factor_as_sparse(info, h.get_factor())
    assert factor_backward_error(L, K, info["perm"]) <= 1e-12
    x = dev(b)
    h.solve(x)
    xg = x.cpu().numpy()
    assert normwise_backward_error(K, xg, b) <= 1e-10
    xo = SparseCholesky(K, None).factor(K).solve(b)
    # forward error: two backward-stable solves differ by at most ~cond(K) * eps (K unique, x unique)
    cond = np.linalg.cond(K.toarray())
    assert np.abs(xg - xo).max() <= max(1e-10, 50.0 * cond * np.finfo(float).eps) * np.abs(xo).max()
    # nmpc_kkt_multiply reproduces K x
    yv = torch.empty_like(x)
    h.kkt_multiply(x, yv)
    assert np.abs(yv.cpu().numpy() - K @ xg).max() <= 1e-12 * abs(K).sum(axis=1).max() * np.abs(xg).max()
    h.close()


@pytest.mark.parametrize("name,ov", MID)
@pytest.mark.parametrize("ordering", [binding.ORDER_AMD, binding.ORDER_ND])
@pytest.mark.parametrize("bare", [False, True])
def test_rhs_row_fused_forward_solve_vs_oracle(name, ov, ordering, bare):
    """options.fuse_rhs: b rides through the numeric factorization as an extra row, which leaves v = L^-1 P b (Eq. 22) in the
    factor; nmpc_solve_fused then runs Eq. (24)-(25) only.  Checked against the oracle's solve (backward + forward error),
    against the general two-sided nmpc_solve on the same handle for b and for another right-hand side, and the reported
    factor must still be the factor of K alone.  `bare`: a pattern-only handle (no model) with fuse_rhs = 1."""
    cfg = make_config(name, **ov)
    K, b, _ = kkt_from_oracle(cfg)
    if bare:
        Kl = sp.tril(sp.csr_matrix(K), format="csr"); Kl.sort_indices()
        pat = nb.make_pattern(cfg.n, Kl.indptr, Kl.indices)
        h = nb.Handle(pat, None, nb.default_options(ordering=ordering, fuse_rhs=1))
    else:
        h = nb.Handle(None, nb.make_ocp(cfg), nb.default_options(ordering=ordering))
    info = h.get_info()
    assert info["fused_rhs"] == 1 and info["n"] == cfg.n
    rp, ci = h.get_kkt_pattern(cfg.n)
    vals = dev(values_on_pattern(K, rp, ci))
    st, _ = h.factor_rhs(vals, dev(b), 0.0)
    assert st == 0
    L = factor_as_sparse(info, h.get_factor())
    assert factor_backward_error(L, K, info["perm"]) <= 1e-12
    x = torch.full((cfg.n,), np.nan, dtype=torch.float64, device=DEV)      # written only
    h.solve_fused(x)
    xg = x.cpu().numpy()
    assert normwise_backward_error(K, xg, b) <= 1e-10
    xo = SparseCholesky(K, None).factor(K).solve(b)
    cond = np.linalg.cond(K.toarray())
    tol = max(1e-10, 50.0 * cond * np.finfo(float).eps)
    assert np.abs(xg - xo).max() <= tol * np.abs(xo).max()
    x2 = dev(b)
    h.solve(x2)                                                            # the two-sided solve on the same factorization
    assert np.abs(x2.cpu().numpy() - xo).max() <= tol * np.abs(xo).max()
    b3 = np.random.default_rng(5).normal(size=cfg.n)
    x3 = dev(b3)
    h.solve(x3)
    assert normwise_backward_error(K, x3.cpu().numpy(), b3) <= 1e-10
    h.solve_fused(x)                                                       # still b's solution after other solves
    assert np.array_equal(x.cpu().numpy(), xg)
    h.close()


def test_rhs_row_off_and_on_take_the_same_ipm_path():
    """The IPM with the right-hand-side row (default for model handles) and without it (fuse_rhs = 0: forward + backward
    solve kernels) must agree: iteration counts, mu trace, and the converged iterate to solver accuracy."""
    for name, ov in MID[:3]:
        cfg = make_config(name, **ov)
        out = {}
        for fuse in (0, 1):
            h = nb.Handle(None, nb.make_ocp(cfg), nb.default_options(fuse_rhs=fuse))
            assert h.get_info()["fused_rhs"] == fuse
            h.update_params(dev(cfg.x0), dev(cfg.ref_for_solve(0)))
            y = torch.zeros(cfg.n, dtype=torch.float64, device=DEV)
            r = h.ipm_solve(0, y, trace_cap=256)
            out[fuse] = (r, y.cpu().numpy())
            h.close()
        r0, y0 = out[0]; r1, y1 = out[1]
        assert r0["status"] == 0 and r1["status"] == 0
        assert r0["iters"] == r1["iters"], (name, r0["iters"], r1["iters"])
        assert [t["mu"] for t in r0["trace"]] == [t["mu"] for t in r1["trace"]]
        assert np.abs(y0 - y1).max() <= 1e-8 * np.abs(y0).max()


@pytest.mark.timeout(300)
@pytest.mark.parametrize("name,ov", [("C2", dict(g=14, N=12)), ("C3", dict(g=12, nseg=2, N=8))])
def test_tiny_grids_finish_and_agree_bitwise(name, ov):
    """The persistent kernels claim tasks in list order and wait for flags; the backward chain of a tiled supernode even waits
    for helper tasks that come AFTER it in the list.  That must not deadlock for any grid >= 2, and the
    result must not depend on the grid: options.grid_limit = 2, 3, 7 against the full grid, IPM solve and a two-sided solve."""
    cfg = make_config(name, **ov)
    ref = None
    for gl in (0, 2, 3, 7):
        h = nb.Handle(None, nb.make_ocp(cfg), nb.default_options(grid_limit=gl))
        assert h.get_info()["n_large_fronts"] > 0
        h.update_params(dev(cfg.x0), dev(cfg.ref_for_solve(0)))
        y = torch.zeros(cfg.n, dtype=torch.float64, device=DEV)
        r = h.ipm_solve(0, y, check=False)
        b = dev(np.random.default_rng(1).normal(size=cfg.n))
        h.solve(b)
        got = (r["status"], r["iters"], y.cpu().numpy(), b.cpu().numpy())
        if ref is None:
            ref = got
        assert got[0] == 0 and got[1] == ref[1]
        assert np.array_equal(got[2], ref[2]) and np.array_equal(got[3], ref[3]), gl
        h.close()


def _random_interior_point(cfg, nlp, rng):
    lo = np.where(np.isfinite(nlp.lb), nlp.lb, 280.0)
    hi = np.where(np.isfinite(nlp.ub), nlp.ub, 450.0)
    return lo + (hi - lo) * rng.uniform(0.1, 0.9, cfg.n)


@pytest.mark.parametrize("name", ["C1", "C2", "C3", "C4"])
def test_full_size_model_assembly_factor_solve(name):
    """BASELINE.json's full sizes, in the launch configuration bench.py times (default options): a2 and a3 element by
    element against the oracle's model code and SciPy, then a4/a5 on that K through properties that hold at any size:
    no pivot failure, normwise backward error of the solve, and (C1, C2, C4) entries of L L^T sampled on the pattern of K."""
    cfg = make_config(name)
    nlp = TranscribedOCP(cfg)
    rng = np.random.default_rng(23)
    y = _random_interior_point(cfg, nlp, rng)
    lam = rng.normal(size=cfg.m)
    nlp.set_params(cfg.x0, cfg.ref_for_solve(0))
    h = nb.Handle(None, nb.make_ocp(cfg), None)
    h.update_params(dev(cfg.x0), dev(cfg.ref_for_solve(0)))
    jrp, jci = h.get_jac_pattern(cfg.m)
    wrp, wci = h.get_hess_pattern(cfg.n)
    krp, kci = h.get_kkt_pattern(cfg.n)
    c, g = torch.empty(cfg.m, dtype=torch.float64, device=DEV), torch.empty(cfg.n, dtype=torch.float64, device=DEV)
    Jv = torch.empty(int(jrp[-1]), dtype=torch.float64, device=DEV)
    Wv = torch.empty(int(wrp[-1]), dtype=torch.float64, device=DEV)
    h.model_eval(dev(y), dev(lam), c, g, Jv, Wv)
    co, go = nlp.constraints(y), nlp.gradient(y)
    assert np.abs(c.cpu().numpy() - co).max() <= 1e-12 * max(1.0, np.abs(co).max())
    assert np.abs(g.cpu().numpy() - go).max() <= 1e-13 * max(1.0, np.abs(go).max())
    Jo, Wo = nlp.jacobian(y), nlp.hessian(y, lam)
    Jg = sp.csr_matrix((Jv.cpu().numpy(), jci, jrp), shape=(cfg.m, cfg.n))
    assert abs(Jg - Jo).max() <= 1e-13 * abs(Jo).max()
    Wl = sp.csr_matrix((Wv.cpu().numpy(), wci, wrp), shape=(cfg.n, cfg.n))
    assert abs(Wl + sp.tril(Wl, -1).T - Wo).max() <= 1e-12 * max(1e-300, abs(Wo).max())
    # a3 with a late-iteration-like spread of Sigma; W = grad^2 f only (lambda = 0) keeps K positive definite
    h.model_eval(dev(y), dev(np.zeros(cfg.m)), c, g, Jv, Wv)
    W0 = nlp.hessian(y, np.zeros(cfg.m))
    sigx = 10.0 ** rng.uniform(-3, 3, cfg.n)
    q = 10.0 ** rng.uniform(-3, 3, cfg.m)
    Kv = torch.empty(int(krp[-1]), dtype=torch.float64, device=DEV)
    h.assemble(Jv, Wv, dev(sigx), dev(q), 0.0, Kv)
    K = (W0 + sp.diags(sigx) + Jo.T @ sp.diags(q) @ Jo).tocsr()
    scale = values_on_pattern(abs(W0) + sp.diags(sigx) + abs(Jo).T @ sp.diags(q) @ abs(Jo), krp, kci)
    assert np.all(np.abs(Kv.cpu().numpy() - values_on_pattern(K, krp, kci)) <= 1e-13 * scale)
    # a4 + a5
    st, _ = h.factor(Kv, 0.0)
    assert st == 0
    b = rng.normal(size=cfg.n)
    x = dev(b)
    h.solve(x)
    assert normwise_backward_error(K, x.cpu().numpy(), b) <= 1e-10
    if name != "C3":                                         # 1.25 GB of panels: the sampled check is done on the other three
        info = h.get_info()
        L = factor_as_sparse(info, h.get_factor()).tocsr()
        perm = info["perm"]
        KP = K[perm, :][:, perm].tocsr()
        rows = rng.integers(0, cfg.n, 200)
        Knorm = abs(K).max()
        for i in rows:
            cols = KP.indices[KP.indptr[i]:KP.indptr[i + 1]]
            cols = cols[cols <= i]
            li = L.getrow(i)
            for j in cols[:: max(1, len(cols) // 4)]:
                v = (li.multiply(L.getrow(j))).sum()
                assert abs(v - KP[i, j]) <= 1e-12 * Knorm, (i, j)
    h.close()


def _sweep_setup(cfg):
    """Frozen J, grad^2 f at the cold-start point (C4 refactor sweep, BASELINE.json:configs[4]): GPU value arrays + the
    same matrices from the oracle's model code."""
    nlp = TranscribedOCP(cfg)
    nlp.set_params(cfg.x0, cfg.ref_for_solve(0))
    y0 = cfg.y_cold(cfg.x0)
    h = nb.Handle(None, nb.make_ocp(cfg), None)
    h.update_params(dev(cfg.x0), dev(cfg.ref_for_solve(0)))
    jrp, _ = h.get_jac_pattern(cfg.m)
    wrp, _ = h.get_hess_pattern(cfg.n)
    krp, kci = h.get_kkt_pattern(cfg.n)
    c, g = torch.empty(cfg.m, dtype=torch.float64, device=DEV), torch.empty(cfg.n, dtype=torch.float64, device=DEV)
    Jv = torch.empty(int(jrp[-1]), dtype=torch.float64, device=DEV)
    Wv = torch.empty(int(wrp[-1]), dtype=torch.float64, device=DEV)
    h.model_eval(dev(y0), dev(np.zeros(cfg.m)), c, g, Jv, Wv)              # lambda = 0: W = grad^2 f
    Jo, Wo = nlp.jacobian(y0), nlp.hessian(y0, np.zeros(cfg.m))
    return h, Jv, Wv, krp, kci, Jo, Wo


def test_sigma_sweep_midsize_vs_oracle():
    """C4 refactor sweep at a size the oracle factors in seconds: every draw refactors on the fixed structure."""
    cfg = make_config("C4", trays=40, N=25)
    h, Jv, Wv, krp, kci, Jo, Wo = _sweep_setup(cfg)
    info = h.get_info()
    Kv = torch.empty(int(krp[-1]), dtype=torch.float64, device=DEV)
    for k, (sx, ss, b) in enumerate(sigma_sweep_draws(cfg, count=6)):
        h.assemble(Jv, Wv, dev(sx), dev(ss), 0.0, Kv)
        st, _ = h.factor(Kv, 0.0)
        assert st == 0, k
        K = (Wo + sp.diags(sx) + Jo.T @ sp.diags(ss) @ Jo).tocsr()
        L = factor_as_sparse(info, h.get_factor())
        assert factor_backward_error(L, K, info["perm"]) <= 1e-12, k
        x = dev(b)
        h.solve(x)
        xg = x.cpu().numpy()
        assert normwise_backward_error(K, xg, b) <= 1e-10, k
        xo = SparseCholesky(K, None).factor(K).solve(b)
        # cond(K) ~ 1e16 here (Sigma in [1e-8, 1e8]): the two backward-stable solutions agree through K, not entrywise:
        # K (x_gpu - x_oracle) must vanish to the backward-error level of either solve
        Kn = abs(K).sum(axis=1).max()
        assert np.abs(K @ (xg - xo)).max() <= 2e-10 * (Kn * max(np.abs(xg).max(), np.abs(xo).max()) + np.abs(b).max()), k
    h.close()


def test_sigma_sweep_full_size_properties():
    """The sweep at BASELINE's full C4 size (n = 52 400), in the launch configuration bench.py times: properties that hold
    at any size -- no pivot failure, normwise backward error of the solve against K rebuilt by SciPy from the oracle's
    J and grad^2 f, and the same solution from a second refactorization (bitwise)."""
    cfg = make_config("C4")
    h, Jv, Wv, krp, kci, Jo, Wo = _sweep_setup(cfg)
    Kv = torch.empty(int(krp[-1]), dtype=torch.float64, device=DEV)
    for k, (sx, ss, b) in enumerate(sigma_sweep_draws(cfg, count=3)):
        h.assemble(Jv, Wv, dev(sx), dev(ss), 0.0, Kv)
        st, _ = h.factor(Kv, 0.0)
        assert st == 0, k
        x = dev(b)
        h.solve(x)
        xg = x.cpu().numpy()
        K = (Wo + sp.diags(sx) + Jo.T @ sp.diags(ss) @ Jo).tocsr()
        assert normwise_backward_error(K, xg, b) <= 1e-10, k
        st, _ = h.factor(Kv, 0.0)
        x2 = dev(b)
        h.solve(x2)
        assert np.array_equal(x2.cpu().numpy(), xg)
    h.close()


@pytest.mark.parametrize("smem_front_max", [16, 48, 0])
def test_factor_kernel_families_agree(smem_front_max):
    """The shared-memory and the tiled front kernels must give the same factor (to rounding) on the same matrix."""
    cfg = make_config("C2", g=9, N=7)
    K, b, _ = kkt_from_oracle(cfg)
    h = nb.Handle(None, nb.make_ocp(cfg), nb.default_options(smem_front_max=smem_front_max))
    info = h.get_info()
    rp, ci = h.get_kkt_pattern(cfg.n)
    h.factor(dev(values_on_pattern(K, rp, ci)), 0.0)
    L = factor_as_sparse(info, h.get_factor())
    assert factor_backward_error(L, K, info["perm"]) <= 1e-12
    x = dev(b)
    h.solve(x)
    assert normwise_backward_error(K, x.cpu().numpy(), b) <= 1e-10
    h.close()


def test_bare_pattern_handle_multiple_rhs_and_state_errors():
    """nmpc_analyze(pattern) without a model: random SPD matrix on a random sparse pattern, nrhs = 3."""
    rng = np.random.default_rng(5)
    n = 700
    A = sp.random(n, n, density=0.004, random_state=7, format="csr")
    A = A + A.T + sp.identity(n)
    A.data[:] = rng.uniform(-1.0, 1.0, len(A.data))
    A = (A + A.T) * 0.5
    K = (A + sp.diags(np.asarray(abs(A).sum(axis=1)).ravel() + 0.1)).tocsr()
    Kl = sp.tril(K, format="csr")
    Kl.sort_indices()
    pat = nb.make_pattern(n, Kl.indptr, Kl.indices)
    h = nb.Handle(pat, None, None)
    B = rng.normal(size=(3, n))
    X = dev(B)
    with pytest.raises(nb.NmpcError) as ei:
        h.solve(X, 3)
    assert ei.value.status == binding.NMPC_E_STATE
    h.factor(dev(Kl.data), 0.0)
    h.solve(X, 3)
    Xg = X.cpu().numpy()
    for k in range(3):
        assert normwise_backward_error(K, Xg[k], B[k]) <= 1e-10
    with pytest.raises(nb.NmpcError) as ei:
        h.ipm_solve(0)
    assert ei.value.status == binding.NMPC_E_STATE
    h.close()


def test_pivot_failure_and_eta_shift():
    cfg = make_config("C1", trays=6, N=8)
    K, b, _ = kkt_from_oracle(cfg)
    K = sp.lil_matrix(K)
    bad = 17
    K[bad, bad] = -5.0                                      # indefinite: some pivot must fail
    K = sp.csr_matrix(K)
    for ordering in ORDERINGS:
        h = nb.Handle(None, nb.make_ocp(cfg), nb.default_options(ordering=ordering))
        rp, ci = h.get_kkt_pattern(cfg.n)
        vals = dev(values_on_pattern(K, rp, ci))
        st, col = h.factor(vals, 0.0, check=False)
        assert st == binding.NMPC_E_NOT_SPD and 0 <= col < cfg.n
        # oracle on the same permutation fails at the same (original) column
        perm = h.get_info()["perm"]
        from oracle.linalg import NotPositiveDefinite
        with pytest.raises(NotPositiveDefinite) as ei:
            SparseCholesky(K, perm).factor(K)
        assert ei.value.column == col
        # Eq. (13): a large enough eta_y restores positive definiteness; the factor is that of K + eta I
        eta = 1e3
        st, _ = h.factor(vals, eta)
        assert st == 0
        Ke = (K + eta * sp.identity(cfg.n)).tocsr()
        L = factor_as_sparse(h.get_info(), h.get_factor())
        assert factor_backward_error(L, Ke, perm) <= 1e-12
        x = dev(b)
        h.solve(x)
        assert normwise_backward_error(Ke, x.cpu().numpy(), b) <= 1e-10
        h.close()


@pytest.mark.parametrize("name,ov", MID)
def test_model_eval_and_assembly_vs_oracle(name, ov):
    cfg = make_config(name, **ov)
    nlp = TranscribedOCP(cfg)
    rng = np.random.default_rng(11)
    lo = np.where(np.isfinite(nlp.lb), nlp.lb, 280.0)
    hi = np.where(np.isfinite(nlp.ub), nlp.ub, 450.0)
    y = lo + (hi - lo) * rng.uniform(0.1, 0.9, cfg.n)
    lam = rng.normal(size=cfg.m)
    x0 = np.clip(cfg.x0 + 0.01 * rng.normal(size=cfg.nx), *cfg.x0_clip)
    ref = cfg.ref_for_solve(1)
    nlp.set_params(x0, ref)
    h = nb.Handle(None, nb.make_ocp(cfg), None)
    h.update_params(dev(x0), dev(ref))                                         # a1
    jrp, jci = h.get_jac_pattern(cfg.m)
    wrp, wci = h.get_hess_pattern(cfg.n)
    krp, kci = h.get_kkt_pattern(cfg.n)
    c, g = torch.empty(cfg.m, dtype=torch.float64, device=DEV), torch.empty(cfg.n, dtype=torch.float64, device=DEV)
    Jv = torch.empty(int(jrp[-1]), dtype=torch.float64, device=DEV)
    Wv = torch.empty(int(wrp[-1]), dtype=torch.float64, device=DEV)
    h.model_eval(dev(y), dev(lam), c, g, Jv, Wv)                               # a2
    assert np.abs(c.cpu().numpy() - nlp.constraints(y)).max() <= 1e-12 * max(1.0, np.abs(nlp.constraints(y)).max())
    assert np.abs(g.cpu().numpy() - nlp.gradient(y)).max() <= 1e-13 * max(1.0, np.abs(nlp.gradient(y)).max())
    Jg = sp.csr_matrix((Jv.cpu().numpy(), jci, jrp), shape=(cfg.m, cfg.n))
    Jo = nlp.jacobian(y)
    assert abs(Jg - Jo).max() <= 1e-13 * abs(Jo).max()
    Wl = sp.csr_matrix((Wv.cpu().numpy(), wci, wrp), shape=(cfg.n, cfg.n))
    Wg = Wl + sp.tril(Wl, -1).T
    Wo = nlp.hessian(y, lam)
    assert abs(Wg - Wo).max() <= 1e-12 * max(1e-300, abs(Wo).max())
    # a3: K = W + Sigma_x + J^T Q J + eta I on the fixed pattern
    sigx = 10.0 ** rng.uniform(-6, 6, cfg.n)
    q = 10.0 ** rng.uniform(-6, 6, cfg.m)
    eta = 0.37
    Kv = torch.empty(int(krp[-1]), dtype=torch.float64, device=DEV)
    h.assemble(Jv, Wv, dev(sigx), dev(q), eta, Kv)
    Ko = (Wo + sp.diags(sigx + eta) + Jo.T @ sp.diags(q) @ Jo).tocsr()
    Kg = Kv.cpu().numpy()
    Ko_vals = values_on_pattern(Ko, krp, kci)
    # entrywise relative to the magnitude of the terms summed into the entry
    scale = values_on_pattern(abs(Wo) + sp.diags(sigx + eta) + abs(Jo).T @ sp.diags(q) @ abs(Jo), krp, kci)
    assert np.all(np.abs(Kg - Ko_vals) <= 1e-13 * scale)
    assert sp.tril(Ko).nnz <= len(Kg)
    h.close()


def _gpu_ipm(cfg, ordering=binding.ORDER_AUTO, **opts):
    h = nb.Handle(None, nb.make_ocp(cfg), nb.default_options(ordering=ordering, **opts))
    return h


@pytest.mark.parametrize("name,ov", MID + [("C1", {})])
def test_ipm_solve_vs_oracle(name, ov):
    cfg = make_config(name, **ov)
    ref = LiftedIPM(cfg, linsolve="blocktri")
    ro = ref.solve()
    assert ro["status"] == "converged"
    h = _gpu_ipm(cfg)
    h.update_params(dev(cfg.x0), dev(cfg.ref_for_solve(0)))
    y = torch.zeros(cfg.n, dtype=torch.float64, device=DEV)
    rg = h.ipm_solve(0, y, trace_cap=256)
    assert rg["status"] == 0
    assert rg["iters"] == ro["iters"], (rg["iters"], ro["iters"], rg["trace"], ro["trace"])
    yo = ro["state"].y
    assert np.abs(y.cpu().numpy() - yo).max() <= 1e-6 * np.abs(yo).max()
    for tg, to in zip(rg["trace"], ro["trace"]):
        assert tg["mu"] == to["mu"] and tg["eta"] == to["eta"]
        # step lengths are ratios of small quantities: they agree to the conditioning of K, not to rounding
        assert abs(tg["alpha_pr"] - to["alpha_pr"]) <= 1e-3 and abs(tg["alpha_du"] - to["alpha_du"]) <= 1e-3
    # full primal-dual iterate
    m, n = cfg.m, cfg.n
    bufs = [torch.empty(k, dtype=torch.float64, device=DEV) for k in (n, m, m, m, m, n, n)]
    h.get_iterate(*bufs)
    so = ro["state"]
    for g_, o_ in zip(bufs, (so.y, so.sp, so.sm, so.wp, so.wm, so.zL, so.zU)):
        assert np.abs(g_.cpu().numpy() - o_).max() <= 1e-5 * max(1.0, np.abs(o_).max())
    assert rg["objective"] == pytest.approx(ref.nlp.objective(yo), rel=1e-6, abs=1e-9)
    h.close()


@pytest.mark.parametrize("name,ov", [("C2", dict(g=9, N=7)), ("C4", dict(trays=40, N=25)), ("C1", {})])
def test_ipm_solve_vs_oracle_tiled_fronts(name, ov):
    """Same parity bar with the two-CTA-per-SM launch shape and every front above 48 rows forced through the tiled
    (HBM-resident, left-looking 64x64 tile) kernel family -- the path the large workloads take (smem_front_max > 0
    switches the latency mode off)."""
    cfg = make_config(name, **ov)
    ro = LiftedIPM(cfg, linsolve="blocktri" if name != "C1" else "sparse").solve()
    assert ro["status"] == "converged"
    h = _gpu_ipm(cfg, smem_front_max=48)
    assert h.get_info()["n_large_fronts"] > 0
    h.update_params(dev(cfg.x0), dev(cfg.ref_for_solve(0)))
    y = torch.zeros(cfg.n, dtype=torch.float64, device=DEV)
    rg = h.ipm_solve(0, y, trace_cap=256)
    assert rg["status"] == 0
    assert rg["iters"] == ro["iters"], (rg["iters"], ro["iters"])
    yo = ro["state"].y
    assert np.abs(y.cpu().numpy() - yo).max() <= 1e-6 * np.abs(yo).max()
    for tg, to in zip(rg["trace"], ro["trace"]):
        assert tg["mu"] == to["mu"] and tg["eta"] == to["eta"]
    h.close()


@pytest.mark.parametrize("ordering", ORDERINGS)
def test_ipm_result_independent_of_ordering(ordering):
    cfg = make_config("C1", trays=10, N=14)
    ro = LiftedIPM(cfg, linsolve="sparse").solve()
    h = _gpu_ipm(cfg, ordering)
    h.update_params(dev(cfg.x0), dev(cfg.ref_for_solve(0)))
    y = torch.zeros(cfg.n, dtype=torch.float64, device=DEV)
    rg = h.ipm_solve(0, y)
    assert rg["iters"] == ro["iters"]
    assert np.abs(y.cpu().numpy() - ro["state"].y).max() <= 1e-6 * np.abs(ro["state"].y).max()
    h.close()


def test_ipm_inertia_correction_path_matches_oracle():
    """Steps a4' / S7: a VdP solve started (nmpc_set_iterate) from a poor multiplier guess has an indefinite W, so
    the first factorizations fail and eta_y is raised by the schedule of Eq. (13) -- same etas, same counts."""
    cfg = make_config("C0")
    ipm = LiftedIPM(cfg, linsolve="dense")
    st, _ = ipm.cold_start(cfg.y_cold(cfg.x0))
    st.wp[:] = 500.0                                         # lam = w+ - w- strongly positive -> W indefinite
    ipm.state = st.copy()
    ro = ipm.solve(warm=True)
    assert ro["status"] == "converged" and any(t["eta"] > 0 for t in ro["trace"])
    h = _gpu_ipm(cfg)
    h.update_params(dev(cfg.x0), dev(cfg.ref_for_solve(0)))
    h.set_iterate(*[dev(v) for v in (st.y, st.sp, st.sm, st.wp, st.wm, st.zL, st.zU)])
    y = torch.zeros(cfg.n, dtype=torch.float64, device=DEV)
    rg = h.ipm_solve(1, y, trace_cap=256)
    assert rg["iters"] == ro["iters"] and rg["factorizations"] == ro["factorizations"]
    assert rg["eta_retries"] == ro["factorizations"] - ro["iters"] > 0
    assert [t["eta"] for t in rg["trace"]] == [t["eta"] for t in ro["trace"]]
    assert np.abs(y.cpu().numpy() - ro["state"].y).max() <= 1e-6 * np.abs(ro["state"].y).max()
    h.close()


@pytest.mark.parametrize("name,ov,R", [("C0", {}, 20), ("C1", dict(trays=14, N=20), 6), ("C2", dict(g=6, N=5), 3)])
def test_nmpc_resolves_replay_vs_oracle(name, ov, R):
    """Algorithm 1 in replay mode: the GPU run is fed the oracle's recorded x0 / ref sequence;
    every re-solve must take the same number of IPM iterations and reach the same primal solution.  The symbolic
    analysis is done once (nmpc_analyze) and reused by every re-solve."""
    cfg = make_config(name, **ov)
    out, _ = nmpc_closed_loop(cfg, n_resolves=R, linsolve="blocktri")
    h = _gpu_ipm(cfg)
    y = torch.zeros(cfg.n, dtype=torch.float64, device=DEV)
    yh = np.empty(cfg.n)
    for j, o in enumerate(out):
        if j % 2 == 0:
            h.update_params(dev(o["x0"]), dev(o["ref"]))
            rg = h.ipm_solve(int(j > 0), y)
            yg = y.cpu().numpy()
        else:                                                # end-to-end entry with HOST buffers
            rg = h.ipm_solve_host(int(j > 0), o["x0"], np.ascontiguousarray(o["ref"]), yh)
            yg = yh.copy()
        assert rg["status"] == 0
        assert rg["iters"] == o["iters"], (j, rg["iters"], o["iters"])
        assert np.abs(yg - o["y"]).max() <= 1e-6 * np.abs(o["y"]).max()
    # invariant: re-solving the unchanged problem warm takes 0 iterations
    rg = h.ipm_solve(1, y)
    assert rg["iters"] == 0 and rg["status"] == 0
    h.close()


def test_bitwise_reproducible():
    cfg = make_config("C2", g=8, N=6)
    ys = []
    for _ in range(2):
        h = _gpu_ipm(cfg)
        h.update_params(dev(cfg.x0), dev(cfg.ref_for_solve(0)))
        y = torch.zeros(cfg.n, dtype=torch.float64, device=DEV)
        h.ipm_solve(0, y)
        ys.append(y.cpu().numpy().copy())
        h.close()
    assert np.array_equal(ys[0], ys[1])


def test_graph_and_plain_launch_paths_agree():
    cfg = make_config("C1", trays=12, N=16)
    K, b, _ = kkt_from_oracle(cfg)
    xs = []
    for use_graph in (0, 1):
        h = nb.Handle(None, nb.make_ocp(cfg), nb.default_options(use_graph=use_graph))
        rp, ci = h.get_kkt_pattern(cfg.n)
        h.factor(dev(values_on_pattern(K, rp, ci)), 0.0)
        x = dev(b)
        h.solve(x)
        xs.append(x.cpu().numpy())
        assert h.launch_count() > 0
        h.close()
    assert np.array_equal(xs[0], xs[1])
    # the IPM iteration replayed as one CUDA graph (parameters and call numbers read from device memory) must reproduce
    # the plain launch sequence bit for bit, cold and warm
    ys, its = [], []
    for use_graph in (0, 1):
        h = nb.Handle(None, nb.make_ocp(cfg), nb.default_options(use_graph=use_graph))
        y = torch.zeros(cfg.n, dtype=torch.float64, device=DEV)
        h.update_params(dev(cfg.x0), dev(cfg.ref_for_solve(0)))
        r0 = h.ipm_solve(0, y)
        h.update_params(dev(np.clip(cfg.x0 + 0.01, *cfg.x0_clip)), dev(cfg.ref_for_solve(1)))
        r1 = h.ipm_solve(1, y)
        ys.append(y.cpu().numpy().copy()); its.append((r0["iters"], r1["iters"], r0["status"], r1["status"]))
        h.close()
    assert its[0] == its[1] and its[0][2] == 0 and its[0][3] == 0
    assert np.array_equal(ys[0], ys[1])


def test_flag_restart_across_call_number_limit():
    """The completion flags of the persistent kernels are call-number valued and restart from zero before a counter could
    overflow (api.cu: next_epoch).  With the limit forced down to 5 calls (options.epoch_limit, a test hook) a cold solve,
    warm re-solves and bare refactor + solve calls cross the restart many times, on the CUDA-graph path and on the plain
    one; every result must be bitwise what a handle that never restarts gives."""
    cfg = make_config("C1", trays=12, N=16)
    K, b, _ = kkt_from_oracle(cfg)
    outs = []
    for limit, use_graph in ((0, 1), (5, 1), (5, 0), (3, 1)):
        h = nb.Handle(None, nb.make_ocp(cfg), nb.default_options(epoch_limit=limit, use_graph=use_graph))
        y = torch.zeros(cfg.n, dtype=torch.float64, device=DEV)
        h.update_params(dev(cfg.x0), dev(cfg.ref_for_solve(0)))
        res = [h.ipm_solve(0, y)]
        ys = [y.cpu().numpy().copy()]
        for j in range(1, 5):
            h.update_params(dev(np.clip(cfg.x0 + 0.01 * j, *cfg.x0_clip)), dev(cfg.ref_for_solve(j)))
            res.append(h.ipm_solve(1, y))
            ys.append(y.cpu().numpy().copy())
        assert all(r["status"] == 0 for r in res)
        assert sum(r["iters"] for r in res) >= 12            # a restart every 3 factorizations at limit 5
        rp, ci = h.get_kkt_pattern(cfg.n)
        vals = dev(values_on_pattern(K, rp, ci))
        xs = []
        for _ in range(4):                                   # a factorization followed by a run of solves longer than the limit
            h.factor(vals, 0.0)
            for _ in range(7):
                x = dev(b)
                h.solve(x)
                xs.append(x.cpu().numpy())
        assert all(np.array_equal(xs[0], v) for v in xs[1:])
        assert normwise_backward_error(K, xs[0], b) <= 1e-10
        outs.append(([r["iters"] for r in res], ys, xs[0]))
        h.close()
    for o in outs[1:]:
        assert o[0] == outs[0][0]
        assert all(np.array_equal(a, b_) for a, b_ in zip(o[1], outs[0][1]))
        assert np.array_equal(o[2], outs[0][2])


def test_warm_start_after_a_failed_solve_falls_back_to_cold():
    """A solve that ends with a non-finite iterate (NMPC_E_STEP) must not leave that iterate behind as the next warm
    start (include/nmpc.h, nmpc_ipm_solve): the following call with warm = 1 starts cold and converges like a cold solve."""
    cfg = make_config("C0")
    h = _gpu_ipm(cfg)
    h.update_params(dev(cfg.x0), dev(cfg.ref_for_solve(0)))
    y = torch.zeros(cfg.n, dtype=torch.float64, device=DEV)
    r_cold = h.ipm_solve(0, y)
    y_cold = y.cpu().numpy().copy()
    assert r_cold["status"] == 0
    n, m = cfg.n, cfg.m
    bad = [torch.full((k,), 1.0, dtype=torch.float64, device=DEV) for k in (n, m, m, m, m, n, n)]
    bad[1][3] = float("nan")                                # a slack: the warm-start push only repairs y
    h.set_iterate(*bad)
    r_bad = h.ipm_solve(1, y, check=False)
    assert r_bad["status"] == binding.NMPC_E_STEP
    r_next = h.ipm_solve(1, y)                               # warm requested, no usable z*: cold start
    assert r_next["status"] == 0 and r_next["iters"] == r_cold["iters"]
    assert np.array_equal(y.cpu().numpy(), y_cold)
    h.close()


@pytest.mark.parametrize("name,ov", MID)
@pytest.mark.parametrize("steps", [1, 2])
def test_ipm_with_iterative_refinement_vs_oracle(name, ov, steps):
    """options.refine_steps: iterative refinement of the Newton direction on the un-condensed first
    block row of Eq. (10), same steps in the oracle.  With the direction refined the step lengths no longer inherit
    cond(K) * eps from the factorization, so the traces agree far more tightly than without it (1e-5 instead of 1e-3)."""
    cfg = make_config(name, **ov)
    ro = LiftedIPM(cfg, linsolve="blocktri", refine_steps=steps).solve()
    assert ro["status"] == "converged"
    for use_graph in (1, 0):
        h = _gpu_ipm(cfg, refine_steps=steps, use_graph=use_graph)
        h.update_params(dev(cfg.x0), dev(cfg.ref_for_solve(0)))
        y = torch.zeros(cfg.n, dtype=torch.float64, device=DEV)
        rg = h.ipm_solve(0, y, trace_cap=256)
        assert rg["status"] == 0 and rg["iters"] == ro["iters"] and rg["factorizations"] == ro["factorizations"]
        for tg, to in zip(rg["trace"], ro["trace"]):
            assert tg["mu"] == to["mu"] and tg["eta"] == to["eta"]
            assert abs(tg["alpha_pr"] - to["alpha_pr"]) <= 1e-5 and abs(tg["alpha_du"] - to["alpha_du"]) <= 1e-5
        yo = ro["state"].y
        assert np.abs(y.cpu().numpy() - yo).max() <= 1e-8 * np.abs(yo).max()
        h.close()


@pytest.mark.parametrize("name,ov", MID)
def test_ipm_with_filter_line_search_vs_oracle(name, ov):
    """options.globalization = 1: the filter line search of ref. [17] on the primal step, the same
    algorithm step by step in the oracle (globalization="filter").  theta and phi_mu are reduced on the device, the acceptance
    tests are host scalars; iteration counts, the number of halvings in every iteration and the converged point must agree
    (C4's cold solve backtracks, the others accept every full step)."""
    cfg = make_config(name, **ov)
    ro = LiftedIPM(cfg, linsolve="blocktri", globalization="filter").solve()
    assert ro["status"] == "converged"
    h = _gpu_ipm(cfg, globalization=1)
    h.update_params(dev(cfg.x0), dev(cfg.ref_for_solve(0)))
    y = torch.zeros(cfg.n, dtype=torch.float64, device=DEV)
    rg = h.ipm_solve(0, y, trace_cap=256)
    assert rg["status"] == 0
    assert rg["iters"] == ro["iters"], ([t["backtracks"] for t in rg["trace"]], [t["backtracks"] for t in ro["trace"]])
    assert [int(t["backtracks"]) for t in rg["trace"]] == [t["backtracks"] for t in ro["trace"]]
    for tg, to in zip(rg["trace"], ro["trace"]):
        assert tg["mu"] == to["mu"] and tg["eta"] == to["eta"]
        assert abs(tg["alpha_pr"] - to["alpha_pr"]) <= 1e-3 and abs(tg["alpha_du"] - to["alpha_du"]) <= 1e-3
    yo = ro["state"].y
    assert np.abs(y.cpu().numpy() - yo).max() <= 1e-6 * np.abs(yo).max()
    if name == "C4":
        assert sum(t["backtracks"] for t in ro["trace"]) > 0
    # warm re-solve with the filter on: same count as the oracle's
    h.update_params(dev(np.clip(cfg.x0 + cfg.noise_for_solve(0) + 1e-3, *cfg.x0_clip)), dev(cfg.ref_for_solve(1)))
    ipm = LiftedIPM(cfg, linsolve="blocktri", globalization="filter")
    ipm.state = ro["state"].copy()
    ipm.nlp.set_params(np.clip(cfg.x0 + cfg.noise_for_solve(0) + 1e-3, *cfg.x0_clip), cfg.ref_for_solve(1))
    rw = ipm.solve(warm=True)
    rgw = h.ipm_solve(1, y, trace_cap=256)
    assert rgw["status"] == 0 and rgw["iters"] == rw["iters"]
    assert np.abs(y.cpu().numpy() - rw["state"].y).max() <= 1e-6 * np.abs(rw["state"].y).max()
    h.close()


def test_batched_instances_match_single_handle_runs():
    """nmpc_ipm_solve_batch (independent OCP instances, the scenarios of D_xi): six
    handles on six streams with bounded grids, solved concurrently (cold, then two warm re-solves).  Every instance must
    reproduce bit for bit what its own handle computes alone, and instance 0 the oracle."""
    cfg = make_config("C1", trays=14, N=20)
    B = 6
    rng = np.random.default_rng(12)
    x0s = [np.clip(cfg.x0 + (b > 0) * rng.normal(0.0, 0.01, cfg.nx), *cfg.x0_clip) for b in range(B)]
    streams = [torch.cuda.Stream() for _ in range(B)]

    def make(b):
        return nb.Handle(None, nb.make_ocp(cfg), nb.default_options(grid_limit=20), stream=streams[b].cuda_stream)

    def params(h, b, j):
        with torch.cuda.stream(streams[b]):
            h.update_params(dev(np.clip(x0s[b] + 0.002 * j, *cfg.x0_clip)), dev(cfg.ref_for_solve(j)))
        streams[b].synchronize()

    hs = [make(b) for b in range(B)]
    ys = [torch.zeros(cfg.n, dtype=torch.float64, device=DEV) for _ in range(B)]
    got = []
    for j in range(3):
        for b in range(B):
            params(hs[b], b, j)
        stats = nb.ipm_solve_batch(hs, [int(j > 0)] * B, ys)
        torch.cuda.synchronize()
        assert all(s["status"] == 0 for s in stats)
        got.append(([s["iters"] for s in stats], [y.cpu().numpy().copy() for y in ys]))
    for h in hs:
        h.close()
    for b in range(B):                                       # the same instance on its own
        h = make(b)
        y = torch.zeros(cfg.n, dtype=torch.float64, device=DEV)
        for j in range(3):
            params(h, b, j)
            r = h.ipm_solve(int(j > 0), y)
            torch.cuda.synchronize()
            assert r["iters"] == got[j][0][b]
            assert np.array_equal(y.cpu().numpy(), got[j][1][b])
        h.close()
    ro = LiftedIPM(cfg, linsolve="sparse").solve()
    assert got[0][0][0] == ro["iters"]
    assert np.abs(got[0][1][0] - ro["state"].y).max() <= 1e-6 * np.abs(ro["state"].y).max()
    with pytest.raises(nb.NmpcError):                        # a handle twice / a shared stream is refused
        h1 = make(0)
        try:
            nb.ipm_solve_batch([h1, h1], [0, 0], None)
        finally:
            h1.close()
