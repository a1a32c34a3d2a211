"""Helpers shared by the `-m gpu` parity tests (argument marshalling and error measures only)."""
import numpy as np
import scipy.sparse as sp


def lower_csr(A):
    L = sp.tril(sp.csr_matrix(A), format="csr")
    L.sort_indices()
    return L.indptr.astype(np.int64), L.indices.astype(np.int32), L.data.astype(np.float64)


def values_on_pattern(K, rp, ci):
    """Values of the symmetric matrix K at the entries of a lower-CSR pattern (structural zeros -> 0.0)."""
    K = sp.csr_matrix(K)
    n = K.shape[0]
    rows = np.repeat(np.arange(n), np.diff(rp))
    return np.asarray(K[rows, ci]).reshape(-1).astype(np.float64)


def factor_as_sparse(info, panels):
    """L_P (CSC) from the supernodal panels returned by nmpc_get_factor (column-major r x w per supernode)."""
    n = info["n"]
    rows_all, cols_all, vals_all = [], [], []
    off = 0
    for s in range(info["nsuper"]):
        c0, c1 = int(info["super_start"][s]), int(info["super_start"][s + 1])
        rows = info["rows"][info["rows_ptr"][s]:info["rows_ptr"][s + 1]].astype(np.int64)
        r, w = len(rows), c1 - c0
        ld = (r + 1) & ~1                                    # panel leading dimension: r rounded up to even (include/nmpc.h)
        P = panels[off:off + ld * w].reshape(w, ld).T[:r]    # P[i, j]
        off += ld * w
        for j in range(w):
            rows_all.append(rows[j:])
            cols_all.append(np.full(r - j, c0 + j, dtype=np.int64))
            vals_all.append(P[j:, j])
    return sp.csc_matrix((np.concatenate(vals_all), (np.concatenate(rows_all), np.concatenate(cols_all))), shape=(n, n))


def factor_backward_error(L, K, perm):
    """||L L^T - P K P^T||_F / ||K||_F (reading G17), evaluated sparsely."""
    K = sp.csr_matrix(K)
    KP = K[perm, :][:, perm]
    D = (L @ L.T - KP).tocsr()
    return float(np.sqrt((D.data ** 2).sum()) / np.sqrt((K.data ** 2).sum()))


def normwise_backward_error(K, x, b):
    """||b - K x||_inf / (||K||_inf ||x||_inf + ||b||_inf)   (reading G16)."""
    K = sp.csr_matrix(K)
    r = b - K @ x
    return float(np.abs(r).max() / (abs(K).sum(axis=1).max() * np.abs(x).max() + np.abs(b).max()))
