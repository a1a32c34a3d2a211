"""oracle/linalg.py -- TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).

Sparse Cholesky of the condensed lifted KKT matrix, following PAPER.md §3.2.3:

  SymCholesky (Eq. 18)  : P, S_L from the pattern of K              -> SparseCholesky.__init__
  reordering  (Eq. 19)  : K_P = P K P^T                             -> SparseCholesky._permuted_lower
  NumCholesky (Eq. 20-21): values of L_P on S_L                      -> SparseCholesky.factor
  solves      (Eq. 22-25): L_P v = P b ; L_P^T Omega = v ; dy = P^T Omega -> SparseCholesky.solve

Three interchangeable solvers (all pinned against brute force in tests/test_oracle_linalg.py):
  O0  DenseCholesky          Eq. (21) triple loop on the densified matrix (tiny systems only)
  O1  SparseCholesky         scalar column Cholesky on S_L (plain C, oracle/chol.c), any permutation
  O2  BlockTridiagCholesky   Eq. (21) written block-wise for the stage-block-tridiagonal K of an OCP, with
                             LAPACK (scipy.linalg) dense Cholesky / triangular solves as the library steps.
                             Used where O1 would need minutes per factorization (plate configs).
`perm[i]` is the ORIGINAL index of the variable placed at position i, i.e. K_P[i,j] = K[perm[i], perm[j]].
"""
from __future__ import annotations

import ctypes

import numpy as np
import scipy.linalg as sla
import scipy.sparse as sp
from threadpoolctl import threadpool_limits

from . import _build

_lib = None


def _c():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(_build.build())
        i64, pd, pi = ctypes.c_int64, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int64)
        _lib.orc_dense_cholesky.restype = i64
        _lib.orc_dense_cholesky.argtypes = [i64, pd]
        _lib.orc_sparse_symbolic.restype = i64
        _lib.orc_sparse_symbolic.argtypes = [i64, pi, pi, pi, pi, pi]
        _lib.orc_sparse_numeric.restype = i64
        _lib.orc_sparse_numeric.argtypes = [i64, pi, pi, pd, pi, pi, pd]
        _lib.orc_lower_solve.restype = None
        _lib.orc_lower_solve.argtypes = [i64, pi, pi, pd, pd]
        _lib.orc_upper_solve.restype = None
        _lib.orc_upper_solve.argtypes = [i64, pi, pi, pd, pd]
    return _lib


def _pd(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _pi(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int64))


class NotPositiveDefinite(Exception):
    """Raised when a pivot is <= 0 or not finite (reading G11).  .column is the failing column."""

    def __init__(self, column):
        super().__init__(f"pivot <= 0 or non-finite at column {column}")
        self.column = column


# ------------------------------------------------------------------------------------------------------
class DenseCholesky:
    """O0: Eq. (21) as printed, on the dense matrix.  PAPER.md:251."""

    def __init__(self, n):
        self.n = n
        self.L = None

    def factor(self, K):
        A = np.ascontiguousarray(K.toarray() if sp.issparse(K) else np.array(K, dtype=np.float64))
        fail = _c().orc_dense_cholesky(self.n, _pd(A))
        if fail:
            raise NotPositiveDefinite(fail - 1)
        self.L = A
        return self

    def solve(self, b):
        v = sla.solve_triangular(self.L, b, lower=True)              # Eq. (23)
        return sla.solve_triangular(self.L.T, v, lower=False)        # Eq. (24)


# ------------------------------------------------------------------------------------------------------
class SparseCholesky:
    """O1: symbolic analysis once (Eq. 18), numeric factorization on the fixed structure (Eq. 20-21)."""

    def __init__(self, K_pattern, perm=None):
        K_pattern = sp.csc_matrix(K_pattern)
        n = K_pattern.shape[0]
        self.n = n
        self.perm = np.arange(n, dtype=np.int64) if perm is None else np.asarray(perm, dtype=np.int64)
        assert sorted(self.perm.tolist()) == list(range(n)), "perm is not a permutation"
        KP = self._permuted_lower(K_pattern)
        self.colptr = KP.indptr.astype(np.int64)
        self.rowind = KP.indices.astype(np.int64)
        # every column must carry its diagonal (first after sorting)
        assert np.all(self.rowind[self.colptr[:-1]] == np.arange(n)), "missing diagonal entry"
        self._keys = np.repeat(np.arange(n, dtype=np.int64), np.diff(self.colptr)) * n + self.rowind
        self.parent = np.empty(n, dtype=np.int64)
        self.lcolptr = np.empty(n + 1, dtype=np.int64)
        nnzL = _c().orc_sparse_symbolic(n, _pi(self.colptr), _pi(self.rowind), _pi(self.parent),
                                        _pi(self.lcolptr), None)
        self.lrow = np.empty(nnzL, dtype=np.int64)
        _c().orc_sparse_symbolic(n, _pi(self.colptr), _pi(self.rowind), _pi(self.parent), _pi(self.lcolptr),
                                 _pi(self.lrow))
        self.nnzL = int(nnzL)
        self.lval = np.zeros(nnzL)
        self.flops = float(np.sum(np.diff(self.lcolptr).astype(np.float64) ** 2))

    def _permuted_lower(self, K):
        """Eq. (19): K_P = P K P^T, returned as sorted lower-triangular CSC."""
        p = self.perm
        KP = sp.csc_matrix(K)[p, :][:, p]
        KP = sp.tril(KP, format="csc")
        KP.sort_indices()
        return KP

    def factor(self, K):
        KP = self._permuted_lower(sp.csc_matrix(K))
        # align the values with the analysed pattern (K may omit structural entries that are exactly zero)
        n = self.n
        colK = np.repeat(np.arange(n, dtype=np.int64), np.diff(KP.indptr))
        keyK = colK * n + KP.indices.astype(np.int64)
        idx = np.searchsorted(self._keys, keyK)
        assert np.all(idx < len(self._keys)) and np.array_equal(self._keys[idx], keyK), \
            "K has entries outside the analysed pattern"
        kfull = np.zeros(len(self.rowind))
        kfull[idx] = KP.data
        kval = np.ascontiguousarray(kfull, dtype=np.float64)
        fail = _c().orc_sparse_numeric(self.n, _pi(self.colptr), _pi(self.rowind), _pd(kval),
                                       _pi(self.lcolptr), _pi(self.lrow), _pd(self.lval))
        if fail:
            raise NotPositiveDefinite(int(self.perm[fail - 1]))
        return self

    def solve(self, b):
        x = np.ascontiguousarray(np.asarray(b, dtype=np.float64)[self.perm])      # P b          (Eq. 22)
        _c().orc_lower_solve(self.n, _pi(self.lcolptr), _pi(self.lrow), _pd(self.lval), _pd(x))   # Eq. 23
        _c().orc_upper_solve(self.n, _pi(self.lcolptr), _pi(self.lrow), _pd(self.lval), _pd(x))   # Eq. 24
        out = np.empty(self.n)
        out[self.perm] = x                                                         # P^T Omega    (Eq. 25)
        return out

    def L_matrix(self):
        """L_P as a SciPy CSC matrix (for the tests)."""
        return sp.csc_matrix((self.lval.copy(), self.lrow, self.lcolptr), shape=(self.n, self.n))


# ------------------------------------------------------------------------------------------------------
class BlockTridiagCholesky:
    """O2: Eq. (21) in block form for K = blocktridiag(D_k, E_k) with N blocks of size nv (stage order):
         L_kk L_kk^T = D_k - L_{k,k-1} L_{k,k-1}^T ,   L_{k+1,k} = E_k L_kk^{-T}
    """

    def __init__(self, N, nv):
        self.N, self.nv, self.n = N, nv, N * nv
        self.Ld = [None] * N
        self.Lo = [None] * (N - 1)
        self.threads = 1 if nv <= 1024 else 4

    def factor(self, K):
        # BLAS thread count: small blocks run fastest (and most reproducibly) single-threaded
        with threadpool_limits(limits=self.threads, user_api="blas"):
            return self._factor(K)

    def _factor(self, K):
        K = sp.csr_matrix(K)
        N, nv = self.N, self.nv
        S = None
        for k in range(N):
            D = K[k * nv:(k + 1) * nv, k * nv:(k + 1) * nv].toarray()
            if k > 0:
                D = D - S
            try:
                Lkk = sla.cholesky(D, lower=True, check_finite=True)
            except (sla.LinAlgError, ValueError):
                raise NotPositiveDefinite(k * nv)
            self.Ld[k] = Lkk
            if k + 1 < N:
                E = K[(k + 1) * nv:(k + 2) * nv, k * nv:(k + 1) * nv].toarray()
                Lo = sla.solve_triangular(Lkk, E.T, lower=True).T          # E L_kk^{-T}
                self.Lo[k] = Lo
                S = Lo @ Lo.T
        return self

    def solve(self, b):
        with threadpool_limits(limits=self.threads, user_api="blas"):
            return self._solve(b)

    def _solve(self, b):
        N, nv = self.N, self.nv
        v = np.array(b, dtype=np.float64).reshape(N, nv)
        for k in range(N):                                                   # Eq. (23)
            if k > 0:
                v[k] -= self.Lo[k - 1] @ v[k - 1]
            v[k] = sla.solve_triangular(self.Ld[k], v[k], lower=True)
        for k in range(N - 1, -1, -1):                                       # Eq. (24)
            if k + 1 < N:
                v[k] -= self.Lo[k].T @ v[k + 1]
            v[k] = sla.solve_triangular(self.Ld[k].T, v[k], lower=False)
        return v.reshape(-1)
