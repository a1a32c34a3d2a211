"""Pins for oracle/linalg.py + oracle/chol.c (CPU only).

Each test pins the oracle to something other than itself: brute force, LAPACK, the defining identity
K = L L^T, or a structural property the paper states (Eq. 18-25).
"""
import os

import numpy as np
import pytest
import scipy.linalg as sla
import scipy.sparse as sp

from ocp_inputs import make_config
from oracle.ipm import LiftedIPM
from oracle.linalg import BlockTridiagCholesky, DenseCholesky, NotPositiveDefinite, SparseCholesky

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def tiny_kkt(name="C1", **ov):
    """A genuine condensed lifted KKT matrix K_c^l (Eq. 17) from two IPM iterations of a shrunken config."""
    cfg = make_config(name, **ov)
    ipm = LiftedIPM(cfg, linsolve="dense", max_iter=2)
    ipm.solve()
    return cfg, ipm.last_step["K0"], ipm.last_step["b"]


def rel_backward(L, K):
    K = K.toarray() if sp.issparse(K) else K
    return np.linalg.norm(L @ L.T - K) / np.linalg.norm(K)


def test_dense_cholesky_eq21_bruteforce_and_lapack():
    cfg, K, b = tiny_kkt("C1", trays=4, N=6)            # n = 6*7 = 42
    Kd = K.toarray()
    ch = DenseCholesky(cfg.n).factor(K)
    assert rel_backward(ch.L, Kd) <= 1e-13               # north_star: ||LL^T-K||/||K|| <= 1e-13
    L_lapack = sla.cholesky(Kd, lower=True)
    assert np.allclose(ch.L, L_lapack, rtol=1e-10, atol=1e-10 * np.abs(L_lapack).max())
    x = ch.solve(b)
    assert np.allclose(x, np.linalg.solve(Kd, b), rtol=1e-8, atol=1e-12)


@pytest.mark.parametrize("name,ov", [("C0", {}), ("C1", dict(trays=6, N=8)), ("C2", dict(g=4, N=4))])
@pytest.mark.parametrize("perm_kind", ["natural", "random", "reverse"])
def test_sparse_cholesky_vs_dense(name, ov, perm_kind):
    cfg, K, b = tiny_kkt(name, **ov)
    n = cfg.n
    rng = np.random.default_rng(3)
    perm = {"natural": None, "random": rng.permutation(n), "reverse": np.arange(n)[::-1].copy()}[perm_kind]
    ch = SparseCholesky(K, perm).factor(K)
    p = ch.perm
    KP = K.toarray()[p][:, p]                            # Eq. (19)
    L = ch.L_matrix().toarray()
    assert rel_backward(L, KP) <= 1e-13
    # L is THE Cholesky factor of K_P (unique): compare with LAPACK entry by entry
    Lref = sla.cholesky(KP, lower=True)
    assert np.allclose(L, Lref, rtol=1e-9, atol=1e-10 * np.abs(Lref).max())
    # Eq. (22)-(25)
    x = ch.solve(b)
    xref = np.linalg.solve(K.toarray(), b)
    assert np.linalg.norm(K @ x - b, np.inf) <= 1e-14 * (abs(K).sum(axis=1).max() * np.abs(x).max() + np.abs(b).max()) * n
    assert np.allclose(x, xref, rtol=1e-7, atol=1e-12)


def test_symbolic_structure_matches_dense_factor_pattern():
    """S_L (Eq. 18) = non-zero pattern of the dense factor of a random-valued SPD matrix on the same pattern;
    parent[j] = min{i>j : L_ij != 0}; sum of column counts = nnz(L)."""
    cfg, K, _ = tiny_kkt("C2", g=4, N=3)
    n = cfg.n
    rng = np.random.default_rng(11)
    perm = rng.permutation(n)
    pat = sp.csr_matrix(K)
    pat.data[:] = 1.0
    ch = SparseCholesky(pat, perm)
    # random values on the pattern, strictly diagonally dominant -> SPD, no accidental cancellation
    R = sp.tril(pat, -1).tocsr()
    R.data = rng.uniform(0.5, 1.5, R.nnz)
    A = (R + R.T).toarray()
    A += np.diag(np.abs(A).sum(axis=1) + 1.0)
    Ld = np.linalg.cholesky(A[perm][:, perm])
    dense_pat = np.abs(Ld) > 1e-14
    S_L = np.zeros((n, n), dtype=bool)
    for j in range(n):
        S_L[ch.lrow[ch.lcolptr[j]:ch.lcolptr[j + 1]], j] = True
    assert np.array_equal(S_L, dense_pat)
    for j in range(n):
        below = np.nonzero(dense_pat[j + 1:, j])[0]
        assert ch.parent[j] == (j + 1 + below[0] if len(below) else -1)
    assert ch.nnzL == int(dense_pat.sum()) == int(np.sum(np.diff(ch.lcolptr)))


def test_fig1_children_property_golden():
    """'columns 1 and 2 are children of column 3' (fixture tests/golden/fig1_etree_property.txt)."""
    tok = {}
    for line in open(os.path.join(GOLDEN, "fig1_etree_property.txt")):
        if line.startswith("#") or not line.strip():
            continue
        key, *vals = line.split()
        tok[key] = [int(v) for v in vals]
    n = tok["n"][0]
    e = np.array(tok["entries"]).reshape(-1, 2) - 1
    pat = sp.coo_matrix((np.ones(len(e)), (e[:, 0], e[:, 1])), shape=(n, n))
    pat = (pat + pat.T + sp.identity(n)).tocsc()
    ch = SparseCholesky(pat)
    assert (ch.parent + 1).tolist() == tok["parent"]


def test_block_tridiagonal_cholesky_vs_dense():
    cfg, K, b = tiny_kkt("C2", g=5, N=5)
    ch = BlockTridiagCholesky(cfg.N, cfg.nv).factor(K)
    Kd = K.toarray()
    L = np.zeros_like(Kd)
    nv = cfg.nv
    for k in range(cfg.N):
        L[k * nv:(k + 1) * nv, k * nv:(k + 1) * nv] = ch.Ld[k]
        if k + 1 < cfg.N:
            L[(k + 1) * nv:(k + 2) * nv, k * nv:(k + 1) * nv] = ch.Lo[k]
    assert rel_backward(L, Kd) <= 1e-13
    assert np.allclose(L, sla.cholesky(Kd, lower=True), rtol=1e-9, atol=1e-10 * np.abs(Kd).max())
    x = ch.solve(b)
    assert np.allclose(x, np.linalg.solve(Kd, b), rtol=1e-7, atol=1e-12)


def test_pivot_failure_is_reported():
    """Reading G11: failure <=> pivot <= 0 or non-finite.  An indefinite matrix must raise, for all three."""
    n, nv = 12, 3
    rng = np.random.default_rng(5)
    T = sp.diags([np.full(n - 1, -1.0), np.full(n, 2.5), np.full(n - 1, -1.0)], [-1, 0, 1]).tolil()
    T[7, 7] = -1.0                                        # makes the matrix indefinite
    T = T.tocsc()
    assert np.linalg.eigvalsh(T.toarray()).min() < 0
    for ch in (DenseCholesky(n), SparseCholesky(T), BlockTridiagCholesky(n // nv, nv)):
        with pytest.raises(NotPositiveDefinite):
            ch.factor(T)


def test_solution_independent_of_ordering():
    """G14/G18: dy = K^-1 b is unique; orderings only change L."""
    cfg, K, b = tiny_kkt("C1", trays=8, N=10)
    rng = np.random.default_rng(9)
    xs = [SparseCholesky(K, p).factor(K).solve(b) for p in (None, rng.permutation(cfg.n), rng.permutation(cfg.n))]
    for x in xs[1:]:
        assert np.linalg.norm(x - xs[0], np.inf) <= 1e-9 * np.linalg.norm(xs[0], np.inf)
