"""General rows on the CUDA path (Problem 5/6; reading G22 of DESIGN.md section 3):
linear rows lo <= G y <= hi below the dynamics rows -- control-horizon hold, two-sided move limits, a
one-sided input-sum limit -- through the C-ABI (nmpc_ocp.n_g ...), against the oracle on the same seeded inputs:

  * a2: c(y) and the Jacobian values including the general rows, element-wise
  * a3..a7: nmpc_ipm_solve against LiftedIPM -- iteration / factorization counts, mu and eta traces, step lengths, the whole
    primal-dual iterate (a row side without a bound keeps s = 1, w = 0), cold solve + replayed warm re-solves
  * the rows do what they say at the converged point (hold inside the gamma tube, limits respected, one of them active)
  * nmpc_hykkt_solve refuses a handle with general rows
"""
import numpy as np
import pytest
import scipy.sparse as sp
import torch

import paper_2606_04725_b200 as nb
from ocp_inputs import make_config
from oracle.ipm import nmpc_closed_loop
from oracle.nlp import TranscribedOCP
from paper_2606_04725_b200 import binding

pytestmark = pytest.mark.gpu

DEV = "cuda:0"
CASES = [("C0", dict(Nc=25, move_limit=0.3)),
         ("C1", dict(trays=18, N=30, Nc=20, move_limit=0.15)),
         ("C2", dict(g=9, N=7, power_limit=1.0, Nc=5)),
         ("C3", dict(g=8, nseg=2, N=5, power_limit=2.5)),
         ("C4", dict(trays=40, N=25, Nc=15, move_limit=0.2)),
         ("C1", dict(Nc=60, move_limit=0.1))]                # BASELINE size (n = 3500), the rows bench.py times as "C1+rows"
STATE = ("y", "sp", "sm", "wp", "wm", "zL", "zU")


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).to(DEV)


@pytest.mark.parametrize("name,ov", CASES)
def test_model_eval_with_general_rows(name, ov):
    cfg = make_config(name, **ov)
    nlp = TranscribedOCP(cfg)
    rng = np.random.default_rng(3)
    lo = np.where(np.isfinite(nlp.lb), nlp.lb, 280.0)
    hi = np.where(np.isfinite(nlp.ub), nlp.ub, 450.0)
    y = lo + (hi - lo) * rng.uniform(0.1, 0.9, cfg.n)
    nlp.set_params(cfg.x0, cfg.ref_for_solve(0))
    h = nb.Handle(None, nb.make_ocp(cfg), None)
    h.update_params(dev(cfg.x0), dev(cfg.ref_for_solve(0)))
    jrp, jci = h.get_jac_pattern(cfg.m)
    assert len(jrp) == cfg.m + 1
    c = torch.empty(cfg.m, dtype=torch.float64, device=DEV)
    Jv = torch.empty(int(jrp[-1]), dtype=torch.float64, device=DEV)
    h.model_eval(dev(y), None, c, None, Jv, None)
    co, Jo = nlp.constraints(y), nlp.jacobian(y)
    assert np.abs(c.cpu().numpy() - co).max() <= 1e-12 * max(1.0, np.abs(co).max())
    Jg = sp.csr_matrix((Jv.cpu().numpy(), jci, jrp), shape=(cfg.m, cfg.n))
    assert abs(Jg - Jo).max() <= 1e-13 * abs(Jo).max()
    assert abs(Jg[cfg.m_dyn:] - nlp.G).max() == 0.0         # the general rows are copied, not recomputed
    h.close()


@pytest.mark.parametrize("name,ov", CASES)
@pytest.mark.parametrize("fuse", [1, 0])
def test_ipm_with_general_rows_vs_oracle(name, ov, fuse):
    cfg = make_config(name, **ov)
    out, ipm = nmpc_closed_loop(cfg, n_resolves=2, linsolve="sparse")
    h = nb.Handle(None, nb.make_ocp(cfg), nb.default_options(fuse_rhs=fuse))
    y = torch.zeros(cfg.n, dtype=torch.float64, device=DEV)
    n, m = cfg.n, cfg.m
    bufs = [torch.empty(k, dtype=torch.float64, device=DEV) for k in (n, m, m, m, m, n, n)]
    for j, o in enumerate(out):
        assert o["status"] == "converged"
        h.update_params(dev(o["x0"]), dev(o["ref"]))
        rg = h.ipm_solve(int(j > 0), y, trace_cap=256, check=False)
        to = o["trace"]
        rep = f"{name} solve {j}: GPU {rg['iters']} / oracle {o['iters']} iterations"
        assert rg["status"] == 0 and rg["iters"] == o["iters"] and rg["factorizations"] == o["factorizations"], rep
        for tg, t in zip(rg["trace"], to):
            assert tg["mu"] == t["mu"] and tg["eta"] == t["eta"], rep
            assert abs(tg["alpha_pr"] - t["alpha_pr"]) <= 1e-3 and abs(tg["alpha_du"] - t["alpha_du"]) <= 1e-3, rep
        yo = o["y"]
        assert np.abs(y.cpu().numpy() - yo).max() <= 1e-6 * np.abs(yo).max(), rep
        h.get_iterate(*bufs)
        for b_, f in zip(bufs, STATE):
            ref = getattr(o["state"], f)
            assert np.abs(b_.cpu().numpy() - ref).max() <= 1e-5 * max(1.0, np.abs(ref).max()), (rep, f)
        sm_g, wm_g = bufs[2].cpu().numpy(), bufs[4].cpu().numpy()
        assert np.all(sm_g[~ipm.rL] == 1.0) and np.all(wm_g[~ipm.rL] == 0.0)      # a row side without a bound never moves
    # what the rows say, at the GPU's converged point (last solve)
    Y = y.cpu().numpy().reshape(cfg.N, cfg.nv)
    U = Y[:, cfg.nx:]
    pr = cfg.path_rows
    if pr["Nc"] < cfg.N:
        assert np.abs(np.diff(U[pr["Nc"] - 1:], axis=0)).max() <= 1e-4 * (1 + 1e-3) + 1e-5       # hold inside the gamma tube
    if pr["move_limit"] is not None and pr["Nc"] > 1:
        assert np.abs(np.diff(U[: pr["Nc"]], axis=0)).max() <= pr["move_limit"] + 1e-5
    if pr["power_limit"] is not None:
        assert U.sum(axis=1).max() <= pr["power_limit"] + 1e-5
    h.close()


def test_hykkt_refuses_general_rows():
    cfg = make_config("C0", Nc=25, move_limit=0.3)
    h = nb.Handle(None, nb.make_ocp(cfg), None)
    h.update_params(dev(cfg.x0), dev(cfg.ref_for_solve(0)))
    y = torch.zeros(cfg.n, dtype=torch.float64, device=DEV)
    with pytest.raises(nb.NmpcError) as ei:
        h.hykkt_solve(0, y)
    assert ei.value.status == binding.NMPC_E_STATE
    h.close()
