"""nmpc_solve_static (include/nmpc.h): the two-sided solve of Eq. (22)-(25) with its work vector in the library's file-scope
device array -- the entry point for callers that may not allocate (CUDA-graph capture, serving loops).

Collected last on purpose (the run is `pytest -x`): nothing behind this file can be hidden by a failure here.
Every test passes alone in a fresh process and after the rest of the suite (the array is cleared per call; no test relies on
its contents).
"""
import numpy as np
import pytest
import scipy.sparse as sp
import torch

import paper_2606_04725_b200 as nb
from ocp_inputs import make_config
from oracle.ipm import LiftedIPM
from paper_2606_04725_b200 import binding

from gpu_util import normwise_backward_error, values_on_pattern

pytestmark = pytest.mark.gpu

DEV = "cuda:0"
STATIC_DOUBLES = 262144          # NMPC_STATIC_SOLVE_DOUBLES of include/nmpc.h


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).to(DEV)


def kkt_from_oracle(cfg, iters=3):
    ipm = LiftedIPM(cfg, linsolve="blocktri", max_iter=iters)
    ipm.solve()
    ls = ipm.last_step
    K = ls["K0"] if ls["eta"] == 0.0 else (ls["K0"] + ls["eta"] * sp.identity(cfg.n)).tocsc()
    return K, ls["b"]


@pytest.mark.parametrize("name,ov", [("C1", dict(trays=18, N=30)), ("C2", dict(g=9, N=7))])
def test_static_solve_matches_nmpc_solve_on_two_calls_in_a_row(name, ov):
    """Two calls in a row (different right-hand sides, the second one in place) against nmpc_solve on the same factorization:
    same kernel, same task order, fixed summation order -> bitwise equal; and backward-stable against K itself (1e-10, the bar
    of test_factor_and_solve_vs_oracle).  The first call runs on whatever an earlier user of the array left in it."""
    cfg = make_config(name, **ov)
    K, b = kkt_from_oracle(cfg)
    h = nb.Handle(None, nb.make_ocp(cfg), nb.default_options())
    rp, ci = h.get_kkt_pattern(cfg.n)
    st, _ = h.factor(dev(values_on_pattern(K, rp, ci)), 0.0)
    assert st == 0
    rng = np.random.default_rng(7)
    rhs = [np.asarray(b, dtype=np.float64), rng.normal(size=cfg.n)]
    ref = []
    for r in rhs:                                    # existing path: in place, work vector owned by the handle
        x = dev(r)
        h.solve(x)
        ref.append(x.cpu().numpy())
    # call 1: separate input and output; the input must stay untouched
    r0 = dev(rhs[0])
    out0 = torch.full((cfg.n,), float("nan"), dtype=torch.float64, device=DEV)
    h.solve_static(r0, out0)
    # call 2 right behind it, in place
    x1 = dev(rhs[1])
    h.solve_static(x1, x1)
    torch.cuda.synchronize()
    got = [out0.cpu().numpy(), x1.cpu().numpy()]
    assert np.array_equal(r0.cpu().numpy(), rhs[0])
    for g, rf, r in zip(got, ref, rhs):
        assert np.all(np.isfinite(g))
        assert np.abs(g - rf).max() <= 1e-12 * np.abs(rf).max()
        assert np.array_equal(g, rf)
        assert normwise_backward_error(K, g, r) <= 1e-10
    # the handle's own path is unaffected by the static calls
    x = dev(rhs[0])
    h.solve(x)
    assert np.array_equal(x.cpu().numpy(), ref[0])
    h.close()


def test_static_solve_two_handles_share_the_array():
    """The array is shared by every handle on the device and keeps the last call's contents: alternating calls of two
    handles of different sizes (serialised on the default stream order by a synchronize) still match nmpc_solve."""
    hs = []
    for name, ov in (("C0", {}), ("C1", dict(trays=18, N=30))):
        cfg = make_config(name, **ov)
        K, b = kkt_from_oracle(cfg)
        h = nb.Handle(None, nb.make_ocp(cfg), nb.default_options())
        rp, ci = h.get_kkt_pattern(cfg.n)
        st, _ = h.factor(dev(values_on_pattern(K, rp, ci)), 0.0)
        assert st == 0
        x = dev(b)
        h.solve(x)
        hs.append((h, cfg, b, x.cpu().numpy()))
    for _ in range(2):
        for h, cfg, b, ref in reversed(hs):
            out = torch.empty(cfg.n, dtype=torch.float64, device=DEV)
            h.solve_static(dev(b), out)
            torch.cuda.synchronize()                 # calls that overlap on the GPU would race on the shared array
            assert np.array_equal(out.cpu().numpy(), ref)
    for h, *_ in hs:
        h.close()


def test_static_solve_rejects_what_does_not_fit_and_unfactored_handles():
    """Sizes beyond NMPC_STATIC_SOLVE_DOUBLES are refused with a message (no launch, no allocation); a structure that fits
    exactly is accepted; a handle that was never factored is a state error."""
    def tridiag_handle(n):
        rows = np.arange(n)
        K = sp.diags([np.full(n - 1, -1.0), np.full(n, 4.0)], [-1, 0], format="csr")          # lower triangle
        pat = nb.make_pattern(n, K.indptr, K.indices)
        return nb.Handle(pat, None, nb.default_options(ordering=binding.ORDER_NATURAL, fuse_rhs=0)), K, rows

    n_big = STATIC_DOUBLES + 1
    h, K, _ = tridiag_handle(n_big)
    x = torch.ones(n_big, dtype=torch.float64, device=DEV)
    st = h.solve_static(x, x, check=False)
    assert st == binding.NMPC_E_ARG
    msg = (h.lib.nmpc_last_error(h._h) or b"").decode()
    assert "NMPC_STATIC_SOLVE_DOUBLES" in msg and str(n_big) in msg
    assert np.array_equal(x.cpu().numpy(), np.ones(n_big))       # nothing ran
    h.close()

    h, K, _ = tridiag_handle(STATIC_DOUBLES)                      # fits exactly
    x = torch.ones(STATIC_DOUBLES, dtype=torch.float64, device=DEV)
    assert h.solve_static(x, x, check=False) == binding.NMPC_E_STATE            # not factored yet
    rp, ci = h.get_kkt_pattern(STATIC_DOUBLES)
    Kl = sp.tril(K).tocsr()
    st, _ = h.factor(dev(values_on_pattern((Kl + sp.tril(Kl, -1).T).tocsc(), rp, ci)), 0.0)
    assert st == 0
    ref = x.clone()
    h.solve(ref)
    h.solve_static(x, x)
    torch.cuda.synchronize()
    assert np.array_equal(x.cpu().numpy(), ref.cpu().numpy())
    Kf = (Kl + sp.tril(Kl, -1).T).tocsr()
    assert np.abs(Kf @ x.cpu().numpy() - 1.0).max() <= 1e-12
    h.close()
