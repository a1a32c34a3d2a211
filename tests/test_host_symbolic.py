"""Host-side checks of the C-ABI library (CPU only, no compute calls):

  * libnmpc_b200.so loads and exports every symbol include/nmpc.h declares
  * step a0 (SymCholesky, Eq. 18-19): permutation, elimination tree, column structure,
    supernode partition and the K -> panel scatter map, each pinned to brute force on small patterns
    (non-zero pattern of a dense Cholesky factor of a random-valued SPD matrix on the permuted pattern;
    parent[j] = min{i > j : L_ij != 0}, the Figure 1 property of PAPER.md:236)
  * the model's J / W / K patterns against the oracle's densely computed ones
  * pattern validation (NMPC_E_PATTERN) and the "no CPU fallback" rule (nmpc_analyze -> NMPC_E_CUDA without a GPU)
"""
import os
import re

import numpy as np
import pytest
import scipy.sparse as sp

import paper_2606_04725_b200 as nb
from ocp_inputs import make_config
from oracle.nlp import TranscribedOCP
from paper_2606_04725_b200 import _build, binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")

SMALL = [("C0", {}), ("C1", dict(trays=6, N=8)), ("C2", dict(g=5, N=4)), ("C3", dict(g=6, nseg=2, N=3)),
         ("C4", dict(trays=9, N=12))]
ORDERINGS = [nb.binding.ORDER_NATURAL, nb.binding.ORDER_AMD, nb.binding.ORDER_ND, nb.binding.ORDER_TIME_ND]


@pytest.fixture(scope="session", autouse=True)
def _built():
    _build.build()


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "nmpc.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(nmpc_[a-z_0-9]+)\s*\(", hdr))
    assert {"nmpc_analyze", "nmpc_update_params", "nmpc_factor", "nmpc_solve", "nmpc_ipm_solve"} <= declared
    lib = nb.load_library()
    for name in sorted(declared):
        assert hasattr(lib, name), f"{name} declared in include/nmpc.h but not exported"
    assert declared == set(binding.SIGNATURES), "binding.SIGNATURES out of step with include/nmpc.h"


def test_measurement_aids_live_in_their_own_library():
    """include/nmpc_aids.h (fp64 peak microbenchmarks, per-task timestamps) is exported by libnmpc_b200_aids.so only:
    the product library carries neither symbol."""
    hdr = open(os.path.join(ROOT, "include", "nmpc_aids.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(nmpc_[a-z_0-9]+)\s*\(", hdr))
    assert declared == set(binding.AIDS_SIGNATURES)
    aids, prod = binding.load_aids_library(), nb.load_library()
    for name in sorted(declared | set(binding.SIGNATURES)):
        assert hasattr(aids, name), name
    for name in sorted(declared):
        assert not hasattr(prod, name), f"{name} must not be in the product library"


def _lower_csr(A):
    L = sp.tril(sp.csr_matrix(A), format="csr")
    L.sort_indices()
    return L.indptr.astype(np.int64), L.indices.astype(np.int32)


def _dense_factor_pattern(n, rp, ci, perm, seed=0):
    """Non-zero pattern of the Cholesky factor of P K P^T by brute-force boolean elimination (Eq. 21 on
    booleans: eliminating column j joins all its below-diagonal rows pairwise), cross-checked on small n
    against the numeric factor of a random-valued diagonally dominant matrix (no accidental cancellation)."""
    A = np.zeros((n, n), dtype=bool)
    for i in range(n):
        A[i, ci[rp[i]:rp[i + 1]]] = True
    A = A | A.T
    AP = A[perm][:, perm]
    Lb = np.tril(AP)
    for j in range(n):
        rows = np.nonzero(Lb[j + 1:, j])[0] + j + 1
        Lb[np.ix_(rows, rows)] |= True
    Lb = np.tril(Lb)
    if n <= 60:
        rng = np.random.default_rng(seed)
        V = np.where(AP, rng.uniform(0.5, 1.5, (n, n)), 0.0)
        V = np.tril(V) + np.tril(V, -1).T
        V[np.arange(n), np.arange(n)] = np.abs(V).sum(axis=1) + 1.0
        assert np.array_equal(np.abs(np.linalg.cholesky(V)) > 1e-13, Lb)
    return Lb


def _struct_from_info(info):
    """Boolean n x n structure of the supernodal L (panel entries on or below the diagonal)."""
    n = info["n"]
    S = np.zeros((n, n), dtype=bool)
    for s in range(info["nsuper"]):
        c0, c1 = info["super_start"][s], info["super_start"][s + 1]
        rows = info["rows"][info["rows_ptr"][s]:info["rows_ptr"][s + 1]]
        assert np.array_equal(rows[: c1 - c0], np.arange(c0, c1))
        assert np.all(np.diff(rows) > 0)
        for j in range(c1 - c0):
            S[rows[j:], c0 + j] = True
    return S


@pytest.mark.parametrize("name,ov", SMALL)
@pytest.mark.parametrize("ordering", ORDERINGS)
def test_symbolic_structure_vs_dense_factor(name, ov, ordering):
    cfg = make_config(name, **ov)
    # exact (un-amalgamated) structure: relaxation off
    sym = nb.Symbolic(None, nb.make_ocp(cfg), nb.default_options(ordering=ordering, relax_small=0, relax_zeros=0.0))
    info = sym.info()
    n = info["n"]
    assert n == cfg.n
    perm = info["perm"]
    assert sorted(perm.tolist()) == list(range(n))
    rp, ci = sym.pattern()
    Lpat = _dense_factor_pattern(n, rp, ci, perm)
    S = _struct_from_info(info)
    assert np.array_equal(S, Lpat), "supernodal structure differs from the dense factor's non-zero pattern"
    assert info["nnz_L"] == int(Lpat.sum())
    cc = Lpat.sum(axis=0).astype(np.float64)
    assert info["flops"] == pytest.approx(float((cc ** 2).sum()), rel=1e-12)
    # Figure 1 property: parent[j] = min{ i > j : L_ij != 0 }
    for j in range(n):
        below = np.nonzero(Lpat[j + 1:, j])[0]
        assert info["etree_parent"][j] == (j + 1 + below[0] if len(below) else -1)
    # supernodal tree: parent = supernode of the first below-diagonal row; levels strictly increase to the root
    for s in range(info["nsuper"]):
        w = info["super_start"][s + 1] - info["super_start"][s]
        rows = info["rows"][info["rows_ptr"][s]:info["rows_ptr"][s + 1]]
        p = info["super_parent"][s]
        if len(rows) > w:
            assert info["super_start"][p] <= rows[w] < info["super_start"][p + 1]
            assert info["super_level"][p] > info["super_level"][s]
            prow = set(info["rows"][info["rows_ptr"][p]:info["rows_ptr"][p + 1]].tolist())
            assert set(rows[w:].tolist()) <= prow, "child rows not nested in the parent front"
        else:
            assert p == -1
    sym.close()


@pytest.mark.parametrize("name,ov", SMALL[:3])
def test_relaxed_supernodes_contain_exact_structure_and_kmap_scatters_K(name, ov):
    cfg = make_config(name, **ov)
    for ordering in ORDERINGS:
        sym = nb.Symbolic(None, nb.make_ocp(cfg), nb.default_options(ordering=ordering))
        info = sym.info()
        n = info["n"]
        rp, ci = sym.pattern()
        Lpat = _dense_factor_pattern(n, rp, ci, info["perm"])
        S = _struct_from_info(info)
        assert np.all(S[Lpat]), "amalgamated structure lost an entry of L"
        assert info["nnz_L"] == int(S.sum())
        # scatter map: writing value e at (supernode, offset) must land on (P K P^T)[i, j] of that entry
        sn, off = sym.kmap()
        iperm = np.empty(n, np.int64)
        iperm[info["perm"]] = np.arange(n)
        ld = (np.diff(info["rows_ptr"]) + 1) & ~1            # panel leading dimension: r rounded up to even
        panel_ptr = np.concatenate([[0], np.cumsum(ld * np.diff(info["super_start"]))])
        e = 0
        for i in range(n):
            for p in range(rp[i], rp[i + 1]):
                a, b = iperm[i], iperm[ci[p]]
                r_, c_ = max(a, b), min(a, b)
                s = sn[p]
                c0 = info["super_start"][s]
                rows = info["rows"][info["rows_ptr"][s]:info["rows_ptr"][s + 1]]
                local = off[p] - panel_ptr[s]
                assert c0 <= c_ < info["super_start"][s + 1]
                assert local // ld[s] == c_ - c0 and rows[local % ld[s]] == r_
                e += 1
        assert e == info["nnz_K"]
        sym.close()


@pytest.mark.parametrize("name,ov", SMALL)
def test_rhs_row_leaves_the_reported_structure_that_of_K(name, ov):
    """options.fuse_rhs analyses [K b; b^T 0] with the extra variable ordered last (the factorization then carries
    v = L^-1 P b of Eq. 22 as the last row of L).  What the C-ABI reports must still be the factor structure of K alone:
    exact dense-factor pattern without relaxation, the scatter map lands on the right entries, the roots of K's
    elimination forest point to n."""
    cfg = make_config(name, **ov)
    for ordering in ORDERINGS:
        sym = nb.Symbolic(None, nb.make_ocp(cfg), nb.default_options(ordering=ordering, relax_small=0, relax_zeros=0.0, fuse_rhs=1))
        info = sym.info()
        n = info["n"]
        assert n == cfg.n and info["fused_rhs"] == 1
        perm = info["perm"]
        assert sorted(perm.tolist()) == list(range(n))
        rp, ci = sym.pattern()
        assert rp[-1] == info["nnz_K"]
        Lpat = _dense_factor_pattern(n, rp, ci, perm)
        S = _struct_from_info(info)
        assert np.array_equal(S, Lpat)
        assert info["nnz_L"] == int(Lpat.sum())
        cc = Lpat.sum(axis=0).astype(np.float64)
        assert info["flops"] == pytest.approx(float((cc ** 2).sum()), rel=1e-12)
        for j in range(n):
            below = np.nonzero(Lpat[j + 1:, j])[0]
            assert info["etree_parent"][j] == (j + 1 + below[0] if len(below) else n)
        sn, off = sym.kmap()
        iperm = np.empty(n, np.int64)
        iperm[perm] = np.arange(n)
        ld = (np.diff(info["rows_ptr"]) + 1) & ~1
        panel_ptr = np.concatenate([[0], np.cumsum(ld * np.diff(info["super_start"]))])
        assert panel_ptr[-1] == info["panel_doubles"]
        for i in range(n):
            for p in range(rp[i], rp[i + 1]):
                a, b = iperm[i], iperm[ci[p]]
                r_, c_ = max(a, b), min(a, b)
                s_ = sn[p]
                rows = info["rows"][info["rows_ptr"][s_]:info["rows_ptr"][s_ + 1]]
                local = off[p] - panel_ptr[s_]
                assert local // ld[s_] == c_ - info["super_start"][s_] and rows[local % ld[s_]] == r_
        sym.close()


def test_fig1_children_property_golden_through_the_library():
    txt = [l for l in open(os.path.join(GOLDEN, "fig1_etree_property.txt")) if not l.startswith("#")]
    n = int(txt[0].split()[1])
    ent = list(map(int, txt[1].split()[1:]))
    parent = list(map(int, txt[2].split()[1:]))
    A = sp.identity(n, format="lil")
    for r, c in zip(ent[0::2], ent[1::2]):
        A[r - 1, c - 1] = 1.0
    rp, ci = _lower_csr(A)
    sym = nb.Symbolic(nb.make_pattern(n, rp, ci), None, nb.default_options(ordering=nb.binding.ORDER_NATURAL))
    info = sym.info()
    assert np.array_equal(info["perm"], np.arange(n))
    assert [p + 1 for p in info["etree_parent"]] == parent


# general linear rows below the dynamics rows (include/nmpc.h: nmpc_ocp.n_g; reading G22): hold, move limits, input-sum limit
WITH_ROWS = [("C0", dict(Nc=25, move_limit=0.3)), ("C1", dict(trays=6, N=8, Nc=5, move_limit=0.2)), ("C2", dict(g=5, N=4, power_limit=1.2, Nc=3)),
             ("C3", dict(g=6, nseg=2, N=3, power_limit=2.0))]


@pytest.mark.parametrize("name,ov", SMALL + WITH_ROWS)
def test_model_K_pattern_matches_oracle(name, ov):
    cfg = make_config(name, **ov)
    sym = nb.Symbolic(None, nb.make_ocp(cfg), None)
    rp, ci = sym.pattern()
    rp_o, ci_o = _lower_csr(TranscribedOCP(cfg).K_pattern())
    assert np.array_equal(rp, rp_o) and np.array_equal(ci, ci_o)


def test_bad_patterns_are_rejected():
    lib = nb.load_library()

    def status(n, rp, ci):
        try:
            nb.Symbolic(nb.make_pattern(n, np.array(rp), np.array(ci)), None, None)
        except nb.NmpcError as e:
            return e.status
        return 0

    assert status(2, [0, 1, 3], [0, 0, 1]) == 0
    assert status(2, [0, 1, 2], [0, 0]) == binding.NMPC_E_PATTERN            # missing diagonal in row 1
    assert status(2, [0, 2, 3], [0, 1, 1]) == binding.NMPC_E_PATTERN         # entry above the diagonal
    assert status(3, [0, 1, 2, 5], [0, 1, 1, 0, 2]) == binding.NMPC_E_PATTERN  # unsorted row
    assert status(3, [0, 1, 2, 5], [0, 1, 0, 0, 2]) == binding.NMPC_E_PATTERN  # duplicate
    assert lib is not None


def test_full_size_symbolic_sizes():
    """C1 and C4 at full size: invariants that hold at any size (sum of panel entries, level sets cover all
    supernodes, permutation valid) and the variable counts BASELINE.json names (~3.5k, ~52k)."""
    for name, nvars in (("C1", 3500), ("C4", 52400)):
        cfg = make_config(name)
        info = nb.Symbolic(None, nb.make_ocp(cfg), None).info()
        assert info["n"] == nvars
        assert np.array_equal(np.sort(info["perm"]), np.arange(nvars))
        r = np.diff(info["rows_ptr"])
        w = np.diff(info["super_start"])
        assert info["nnz_L"] == int((r * w - w * (w - 1) // 2).sum())
        assert info["super_level"].max() + 1 == info["nlevels"]
        assert np.all(w >= 1) and np.all(r >= w)


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    cfg = make_config("C0")
    with pytest.raises(nb.NmpcError) as ei:
        nb.Handle(None, nb.make_ocp(cfg), None)
    assert ei.value.status == binding.NMPC_E_CUDA
