"""Parity of nmpc_hykkt_solve (the HyKKT variant of Algorithm 2; reading G21 of DESIGN.md section 3) against
oracle/hykkt.py on the same seeded inputs: iteration counts, mu / eta traces, conjugate-gradient iteration counts, the
primal-dual iterate (y, lam, zL, zU), closed-loop re-solves in replay mode.
"""
import numpy as np
import pytest
import torch

import paper_2606_04725_b200 as nb
from ocp_inputs import make_config
from oracle.hykkt import HyKKTIPM, hykkt_closed_loop

pytestmark = pytest.mark.gpu

DEV = "cuda:0"
MID = [("C0", {}), ("C1", dict(trays=18, N=30)), ("C2", dict(g=9, N=7)), ("C3", dict(g=8, nseg=2, N=5)),
       ("C4", dict(trays=40, N=25))]


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).to(DEV)


def _handle(cfg, **opt):
    return nb.Handle(None, nb.make_ocp(cfg), nb.default_options(**opt))


def _compare(cfg, rg, ro, h, y):
    assert rg["status"] == 0
    assert rg["iters"] == ro["iters"], (rg["iters"], ro["iters"], rg["trace"], ro["trace"])
    assert rg["factorizations"] == ro["factorizations"]
    yo = ro["state"].y
    assert np.abs(y.cpu().numpy() - yo).max() <= 1e-6 * np.abs(yo).max()
    for tg, to in zip(rg["trace"], ro["trace"]):
        assert tg["mu"] == to["mu"] and tg["eta"] == to["eta"]
        assert abs(tg["alpha_pr"] - to["alpha_pr"]) <= 1e-3 and abs(tg["alpha_du"] - to["alpha_du"]) <= 1e-3
        # CG stops on a relative residual: one iteration more or less when the last residual sits at the threshold
        assert abs(int(tg["backtracks"]) - to["cg"]) <= 1, (tg, to)
    m, n = cfg.m, cfg.n
    bufs = [torch.empty(k, dtype=torch.float64, device=DEV) for k in (n, m, m, m, m, n, n)]
    h.get_iterate(*bufs)
    so = ro["state"]
    for g_, o_ in ((bufs[0], so.y), (bufs[3], so.lam), (bufs[5], so.zL), (bufs[6], so.zU)):
        assert np.abs(g_.cpu().numpy() - o_).max() <= 1e-5 * max(1.0, np.abs(o_).max())
    assert float(bufs[4].abs().max()) == 0.0


@pytest.mark.parametrize("name,ov", MID + [("C1", {})])
def test_hykkt_solve_vs_oracle(name, ov):
    cfg = make_config(name, **ov)
    ref = HyKKTIPM(cfg, linsolve="blocktri")
    ro = ref.solve()
    assert ro["status"] == "converged"
    h = _handle(cfg)
    h.update_params(dev(cfg.x0), dev(cfg.ref_for_solve(0)))
    y = torch.zeros(cfg.n, dtype=torch.float64, device=DEV)
    rg = h.hykkt_solve(0, y, trace_cap=256)
    _compare(cfg, rg, ro, h, y)
    # the equalities themselves hold at the solution (no gamma tube): |c|_inf <= eps_outer, from the oracle's model code
    ref.nlp.set_params(cfg.x0, cfg.ref_for_solve(0))
    assert np.abs(ref.nlp.constraints(y.cpu().numpy())).max() <= 1e-5
    h.close()


@pytest.mark.parametrize("name,ov,R", [("C0", {}, 10), ("C1", dict(trays=14, N=20), 6), ("C2", dict(g=6, N=5), 3)])
def test_hykkt_resolves_replay_vs_oracle(name, ov, R):
    cfg = make_config(name, **ov)
    out, _ = hykkt_closed_loop(cfg, n_resolves=R, linsolve="blocktri")
    h = _handle(cfg)
    y = torch.zeros(cfg.n, dtype=torch.float64, device=DEV)
    for j, o in enumerate(out):
        h.update_params(dev(o["x0"]), dev(o["ref"]))
        rg = h.hykkt_solve(int(j > 0), y)
        assert rg["status"] == 0
        assert rg["iters"] == o["iters"], (j, rg["iters"], o["iters"])
        assert np.abs(y.cpu().numpy() - o["y"]).max() <= 1e-6 * np.abs(o["y"]).max()
    rg = h.hykkt_solve(1, y)
    assert rg["iters"] == 0 and rg["status"] == 0
    h.close()


def test_hykkt_and_lifted_agree_at_headline_size():
    """C1 at BASELINE size: both variants converge to the same control sequence up to the gamma tube."""
    cfg = make_config("C1")
    h = _handle(cfg)
    h.update_params(dev(cfg.x0), dev(cfg.ref_for_solve(0)))
    yl = torch.zeros(cfg.n, dtype=torch.float64, device=DEV)
    yh = torch.zeros(cfg.n, dtype=torch.float64, device=DEV)
    rl = h.ipm_solve(0, yl)
    rh = h.hykkt_solve(0, yh)
    assert rl["status"] == 0 and rh["status"] == 0
    assert float((yl - yh).abs().max() / yh.abs().max()) <= 5e-3
    h.close()
