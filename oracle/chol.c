/* oracle/chol.c -- TEST INFRASTRUCTURE ONLY (CPU oracle; see oracle/__init__.py).
 *
 * Plain, slow, obviously-correct Cholesky routines written from the paper's own statement of the
 * factorization.  Nothing here is shared with, included by, or derived from the CUDA path.
 *
 *   orc_dense_cholesky   Eq. (21), written out as the triple loop it is.
 *   orc_sparse_symbolic  SymCholesky, Eq. (18) + PAPER.md:236-242: elimination tree (parent of column j is
 *                        the first sub-diagonal non-zero row of L_j) and the structure S_L obtained by
 *                        "combining the lower triangular sparsity structures of its children with that of
 *                        the corresponding column" of K.
 *   orc_sparse_numeric   NumCholesky, Eq. (20)-(21), restricted to S_L (left-looking column form: column j
 *                        minus the sum over sigma<j of L_{j,sigma} * L_{:,sigma}, then the square root / divide).
 *   orc_lower_solve      Eq. (23)  L v = b          (forward substitution)
 *   orc_upper_solve      Eq. (24)  L^T Omega = v    (backward substitution)
 *
 * The permutation P of Eq. (19) is applied by the Python caller (oracle/linalg.py); these routines see
 * K_P = P K P^T in compressed-sparse-column form, lower triangle, row indices sorted, diagonal first.
 * Return convention of the factorizations: 0 on success, j+1 if the pivot of column j is <= 0 or not finite.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef int64_t i64;

/* ---- Eq. (21) on a dense row-major n x n array; only the lower triangle is read and written ---------- */
i64 orc_dense_cholesky(i64 n, double *A)
{
    for (i64 j = 0; j < n; ++j) {
        double d = A[j * n + j];
        for (i64 s = 0; s < j; ++s) d -= A[j * n + s] * A[j * n + s];
        if (!(d > 0.0) || !isfinite(d)) return j + 1;
        d = sqrt(d);
        A[j * n + j] = d;
        for (i64 i = j + 1; i < n; ++i) {
            double v = A[i * n + j];
            for (i64 s = 0; s < j; ++s) v -= A[i * n + s] * A[j * n + s];
            A[i * n + j] = v / d;
        }
    }
    for (i64 i = 0; i < n; ++i)
        for (i64 j = i + 1; j < n; ++j) A[i * n + j] = 0.0;
    return 0;
}

/* ---- SymCholesky: pass 1 (lrow == NULL) returns nnz(L) and fills parent[], lcolptr[]; pass 2 fills lrow[] -- */
i64 orc_sparse_symbolic(i64 n, const i64 *colptr, const i64 *rowind, i64 *parent, i64 *lcolptr, i64 *lrow)
{
    /* children lists of the elimination tree, built as columns complete */
    i64 *first_child = (i64 *)malloc(sizeof(i64) * n), *next_sib = (i64 *)malloc(sizeof(i64) * n);
    i64 *mark = (i64 *)malloc(sizeof(i64) * n);
    i64 **cols = (i64 **)calloc(n, sizeof(i64 *));     /* structure of each L column (sorted) */
    i64 *cnt = (i64 *)malloc(sizeof(i64) * n);
    i64 *buf = (i64 *)malloc(sizeof(i64) * n);
    for (i64 j = 0; j < n; ++j) { first_child[j] = -1; next_sib[j] = -1; mark[j] = -1; parent[j] = -1; }
    i64 total = 0;
    for (i64 j = 0; j < n; ++j) {
        i64 len = 0;
        mark[j] = j; buf[len++] = j;
        for (i64 p = colptr[j]; p < colptr[j + 1]; ++p) {          /* column j of K (lower part) */
            i64 i = rowind[p];
            if (i > j && mark[i] != j) { mark[i] = j; buf[len++] = i; }
        }
        for (i64 c = first_child[j]; c != -1; c = next_sib[c])      /* union with children, minus {c} */
            for (i64 q = 0; q < cnt[c]; ++q) {
                i64 i = cols[c][q];
                if (i > j && mark[i] != j) { mark[i] = j; buf[len++] = i; }
            }
        /* sort (insertion sort is fine for the oracle's sizes; use qsort for long columns) */
        if (len > 64) {
            /* simple shell sort */
            for (i64 gap = len / 2; gap > 0; gap /= 2)
                for (i64 a = gap; a < len; ++a) {
                    i64 t = buf[a], b = a;
                    while (b >= gap && buf[b - gap] > t) { buf[b] = buf[b - gap]; b -= gap; }
                    buf[b] = t;
                }
        } else {
            for (i64 a = 1; a < len; ++a) {
                i64 t = buf[a], b = a;
                while (b > 0 && buf[b - 1] > t) { buf[b] = buf[b - 1]; --b; }
                buf[b] = t;
            }
        }
        cols[j] = (i64 *)malloc(sizeof(i64) * len);
        memcpy(cols[j], buf, sizeof(i64) * len);
        cnt[j] = len;
        lcolptr[j] = total;
        total += len;
        if (len > 1) {                                              /* parent = first sub-diagonal row */
            i64 pj = buf[1];
            parent[j] = pj;
            next_sib[j] = first_child[pj];
            first_child[pj] = j;
        }
        /* children of j are no longer needed */
        for (i64 c = first_child[j]; c != -1; c = next_sib[c]) {
            if (lrow) memcpy(lrow + lcolptr[c], cols[c], sizeof(i64) * cnt[c]);
            free(cols[c]); cols[c] = NULL;
        }
    }
    lcolptr[n] = total;
    for (i64 j = 0; j < n; ++j)
        if (cols[j]) { if (lrow) memcpy(lrow + lcolptr[j], cols[j], sizeof(i64) * cnt[j]); free(cols[j]); }
    free(first_child); free(next_sib); free(mark); free(cols); free(cnt); free(buf);
    return total;
}

/* ---- NumCholesky on the fixed structure (lcolptr, lrow); kval are the values of K_P on (colptr,rowind) ---- */
i64 orc_sparse_numeric(i64 n, const i64 *colptr, const i64 *rowind, const double *kval,
                       const i64 *lcolptr, const i64 *lrow, double *lval)
{
    double *x = (double *)calloc(n, sizeof(double));     /* dense accumulator for the current column      */
    i64 *head = (i64 *)malloc(sizeof(i64) * n);          /* head[j]: list of columns sigma with L_{j,sigma} != 0 */
    i64 *next = (i64 *)malloc(sizeof(i64) * n);
    i64 *pos = (i64 *)malloc(sizeof(i64) * n);           /* pos[sigma]: index in column sigma of its next row   */
    for (i64 j = 0; j < n; ++j) head[j] = -1;
    i64 fail = 0;
    for (i64 j = 0; j < n && !fail; ++j) {
        for (i64 p = colptr[j]; p < colptr[j + 1]; ++p) x[rowind[p]] = kval[p];        /* K_{P,ij}, i >= j */
        i64 s = head[j];
        while (s != -1) {                                 /* subtract L_{j,sigma} * L_{i,sigma}, i >= j */
            i64 snext = next[s];
            i64 p0 = pos[s];
            double ljs = lval[p0];
            for (i64 p = p0; p < lcolptr[s + 1]; ++p) x[lrow[p]] -= lval[p] * ljs;
            if (p0 + 1 < lcolptr[s + 1]) {                /* re-file sigma under its next row */
                pos[s] = p0 + 1;
                i64 r = lrow[p0 + 1];
                next[s] = head[r]; head[r] = s;
            }
            s = snext;
        }
        double d = x[j];
        if (!(d > 0.0) || !isfinite(d)) { fail = j + 1; break; }
        d = sqrt(d);
        i64 q0 = lcolptr[j];
        lval[q0] = d; x[j] = 0.0;
        for (i64 q = q0 + 1; q < lcolptr[j + 1]; ++q) { lval[q] = x[lrow[q]] / d; x[lrow[q]] = 0.0; }
        if (q0 + 1 < lcolptr[j + 1]) {
            pos[j] = q0 + 1;
            i64 r = lrow[q0 + 1];
            next[j] = head[r]; head[r] = j;
        }
    }
    free(x); free(head); free(next); free(pos);
    return fail;
}

/* ---- Eq. (23): L v = b, in place ---- */
void orc_lower_solve(i64 n, const i64 *lcolptr, const i64 *lrow, const double *lval, double *b)
{
    for (i64 j = 0; j < n; ++j) {
        double v = b[j] / lval[lcolptr[j]];
        b[j] = v;
        for (i64 q = lcolptr[j] + 1; q < lcolptr[j + 1]; ++q) b[lrow[q]] -= lval[q] * v;
    }
}

/* ---- Eq. (24): L^T Omega = v, in place ---- */
void orc_upper_solve(i64 n, const i64 *lcolptr, const i64 *lrow, const double *lval, double *b)
{
    for (i64 j = n - 1; j >= 0; --j) {
        double v = b[j];
        for (i64 q = lcolptr[j] + 1; q < lcolptr[j + 1]; ++q) v -= lval[q] * b[lrow[q]];
        b[j] = v / lval[lcolptr[j]];
    }
}
