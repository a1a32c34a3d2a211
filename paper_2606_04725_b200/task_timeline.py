"""Per-task timeline of the persistent factorization / solve kernels (measurement utility, not on the product path).

    python -m paper_2606_04725_b200.task_timeline --workload C3 [--resolves 2] > profiles/<name>.md

Runs a cold solve and a few warm re-solves of the closed loop on a handle of the MEASUREMENT build
(libnmpc_b200_aids.so, include/nmpc_aids.h: the kernels record globaltimer stamps per task and the time thread 0 of the
CTA spends waiting on completion flags), then summarises the LAST factorization and the LAST solve as markdown:

  * span of the kernel, CTA-time inside tasks, and how that time splits into assembly / tile GEMM / POTRF-TRSM / stores and
    into flag waits (idle CTA time: a persistent CTA is always inside a task, so idle time shows up as waiting);
  * the critical chain: for the largest tiled fronts the time per block column (POTRF(J) -> TRSM(J+1,J) -> GEMM tail ->
    POTRF(J+1)), and the chain of fronts from the last-finished root down the tree;
  * executed vs algorithmic flops of the tile GEMMs (tile padding + amalgamation zeros).

Timestamps perturb the kernels a little (one globaltimer read + store per phase and per wait of thread 0); the numbers
are for where the time goes, not for the bench line.
"""
from __future__ import annotations

import argparse
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

TILE = 64


def tile_bounds(w, r):
    """Block boundaries of a tiled front (csrc/device.h: tile_bound)."""
    nbp = (w + TILE - 1) // TILE
    b = [k * TILE for k in range(nbp)] + [w]
    if r > w:
        v = w + TILE - (w & 1)
        while v < r:
            b.append(v); v += TILE
        b.append(r)
    return nbp, b


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="C3")
    ap.add_argument("--resolves", type=int, default=2)
    ap.add_argument("--top", type=int, default=6, help="how many of the largest tiled fronts to list")
    a = ap.parse_args()

    import torch

    import paper_2606_04725_b200 as nb
    from ocp_inputs import make_config

    cfg = make_config(a.workload)
    dev = "cuda:0"
    td = lambda v: torch.as_tensor(np.ascontiguousarray(v), dtype=torch.float64).to(dev)   # noqa: E731
    h = nb.Handle(None, nb.make_ocp(cfg), None, aids=True)
    y = torch.zeros(cfg.n, dtype=torch.float64, device=dev)
    x0 = np.array(cfg.x0)
    for j in range(1 + a.resolves):
        h.update_params(td(x0), td(cfg.ref_for_solve(j)))
        r = h.ipm_solve(int(j > 0), y, check=False)
        x0 = np.clip(y[: cfg.nx].cpu().numpy() + cfg.noise_for_solve(j), *cfg.x0_clip)
    torch.cuda.synchronize()
    info = h.get_info()
    ss, rp, par = info["super_start"], info["rows_ptr"], info["super_parent"]
    W = lambda s: int(ss[s + 1] - ss[s])                  # noqa: E731
    R = lambda s: int(rp[s + 1] - rp[s])                  # noqa: E731
    out = []
    P = out.append
    P(f"# Task timeline, {cfg.name} {cfg.title} (n = {cfg.n}), last factorization / solve of warm re-solve {a.resolves}")
    P("")
    P(f"Command: `python -m paper_2606_04725_b200.task_timeline --workload {a.workload} --resolves {a.resolves}` "
      f"(measurement build libnmpc_b200_aids.so; last re-solve: {r['iters']} IPM iterations, status {r['status']}).")
    P(f"Structure: {info['nsuper']} supernodes, {info['nlevels']} levels, largest front {info['max_front']} rows, "
      f"{info['n_large_fronts']} tiled fronts, stored nnz(L) {info['nnz_L']:.3e}, algorithmic flops sum cc^2 = {info['flops']:.4e}.")
    P("")

    # ------------------------------------------------------------------ factorization
    tasks, st = h.get_task_trace(0)
    st = st.astype(np.int64)
    is_last = np.ones(len(tasks), dtype=np.int64)         # every tile is one task
    t0, t1 = st[:, 0].min(), st[:, 4].max()
    span = (t1 - t0) / 1e3
    dur = (st[:, 4] - st[:, 0]) / 1e3
    wait = st[:, 6] / 1e3
    sms = np.unique(st[:, 5])
    # CTAs: every (sm, overlapping) ... the grid is known from the number of distinct concurrently running tasks; use busy time
    tile = tasks[:, 0] == 1
    P("## Factorization (`factor_dag_kernel`)")
    P("")
    P(f"* kernel span (first claim to last task done): **{span:.0f} us**; {len(tasks)} tasks ({int(tile.sum())} tile tasks of "
      f"{int((tile & (is_last == 1)).sum())} tiles, {int((~tile).sum())} shared-memory fronts) on {len(sms)} SMs")
    busy = dur.sum()
    P(f"* CTA-time inside tasks: {busy / 1e3:.1f} CTA-ms = {busy / span:.0f} CTAs busy on average; of it **{wait.sum() / busy * 100:.1f} % is "
      f"thread 0 waiting on completion flags** (idle CTA time), {100 - wait.sum() / busy * 100:.1f} % is work")
    ph = [(st[:, k + 1] - st[:, k]) / 1e3 for k in range(4)]
    for nm, m, lab in (("tile tasks", tile, ("assemble tile (K entries, children)", "left-looking GEMM incl. flag waits", "POTRF / TRSM / (update tiles: none)", "store + publish")),
                       ("shared-memory fronts", ~tile, ("wait for children", "assemble (K entries, extend-add)", "partial Cholesky", "store update matrix + publish"))):
        if m.any():
            tot = [p[m].sum() for p in ph]
            P(f"* {nm}: CTA-ms per phase: " + "; ".join(f"{l} {t / 1e3:.2f}" for l, t in zip(lab, tot)) +
              f"; flag waits {wait[m].sum() / 1e3:.2f}")
    # executed vs algorithmic flops of the tile GEMMs
    exec_flops = 0.0
    big = [s for s in range(info["nsuper"]) if (tasks[(tasks[:, 1] == s), 0] == 1).any()] if tile.any() else []
    fl = {}
    for s in big:
        w, r = W(s), R(s)
        nbp, b = tile_bounds(w, r)
        nbt = len(b) - 1
        f = 0.0
        for J in range(nbt):
            kend = b[J] if J < nbp else w
            f += 2.0 * TILE * TILE * (-(-kend // 16) * 16) * (nbt - J)
        fl[s] = f
        exec_flops += f
    if big:
        alg_big = 0.0
        for s in big:
            w, r = W(s), R(s)
            alg_big += sum((r - j) ** 2 for j in range(w))
        P(f"* tile GEMMs: executed {exec_flops:.4e} flops (64x64 tiles, K rounded to 16) for {alg_big:.4e} flops of the stored (amalgamated) "
          f"tiled fronts = {exec_flops / alg_big:.3f}x (tile padding + the triangle of the diagonal tiles computed in full); "
          f"stored-structure flops of all fronts vs the elimination tree's sum cc^2: "
          f"{sum(sum((R(s) - j) ** 2 for j in range(W(s))) for s in range(info['nsuper'])) / info['flops']:.3f}x (amalgamation zeros)")
    P("")
    # critical chain of the largest tiled fronts
    if big:
        P("### Block-column chain of the largest tiled fronts")
        P("")
        P("| front | level | w | r | block cols | first claim us | done us | chain step us (median POTRF(J) done -> POTRF(J+1) done) | of it: POTRF->TRSM(J+1,J) done | ->diag GEMM done | ->POTRF done | bulk-bound estimate us (front flops / 296 CTAs at 100 GFLOP/s) |")
        P("|---|---|---|---|---|---|---|---|---|---|---|---|")
        idx = {(int(t[1]), int(t[2]), int(t[3])): k for k, t in enumerate(tasks) if t[0] == 1 and is_last[k]}
        for s in sorted(big, key=lambda q: -fl[q])[: a.top]:
            w, r = W(s), R(s)
            nbp, b = tile_bounds(w, r)
            m = tile & (tasks[:, 1] == s)
            steps, a1, a2, a3 = [], [], [], []
            for J in range(nbp - 1):
                d0, d1, sd = idx.get((s, J, J)), idx.get((s, J + 1, J + 1)), idx.get((s, J + 1, J))
                if d0 is None or d1 is None or sd is None:
                    continue
                steps.append((st[d1, 3] - st[d0, 3]) / 1e3)
                a1.append((st[sd, 4] - st[d0, 3]) / 1e3)
                a2.append((st[d1, 2] - st[sd, 4]) / 1e3)
                a3.append((st[d1, 3] - st[d1, 2]) / 1e3)
            med = lambda v: float(np.median(v)) if v else float("nan")   # noqa: E731
            P(f"| {s} | {info['super_level'][s]} | {w} | {r} | {nbp} | {(st[m, 0].min() - t0) / 1e3:.0f} | {(st[m, 4].max() - t0) / 1e3:.0f} | "
              f"{med(steps):.1f} | {med(a1):.1f} | {med(a2):.1f} | {med(a3):.1f} | {fl[s] / 296 / 100e3:.0f} |")
        P("")
        # tile tasks by kind: where the CTA time of the panel tiles goes (the wait for the diagonal tile's POTRF)
        P("### Tile tasks by kind (CTA-ms; mean us per task in brackets)")
        P("")
        T, Ss = tasks[tile], st[tile]
        nbp_t = np.zeros(len(T), dtype=np.int64); w_t = np.zeros(len(T), dtype=np.int64)
        for s in big:
            ms = T[:, 1] == s
            nbp_t[ms] = tile_bounds(W(s), R(s))[0]; w_t[ms] = W(s)
        Ti, Tj = T[:, 2], T[:, 3]
        kind = np.where(Tj >= nbp_t, 2, np.where(Ti == Tj, 0, 1))
        Kt = np.where(Tj < nbp_t, Tj * TILE, w_t)
        pht = [(Ss[:, k + 1] - Ss[:, k]) / 1e3 for k in range(4)]
        ideal = 2.0 * TILE * TILE * Kt / 100e9 * 1e6
        P("| kind | tasks | assemble | product (its flops at 100 GFLOP/s per CTA) | POTRF / TRSM | store + publish |")
        P("|---|---|---|---|---|---|")
        for k, nm in enumerate(("diagonal panel tile (POTRF)", "panel tile below the diagonal (TRSM)", "update tile")):
            mk = kind == k
            if mk.any():
                P(f"| {nm} | {int(mk.sum())} | {pht[0][mk].sum() / 1e3:.1f} ({pht[0][mk].mean():.1f}) | {pht[1][mk].sum() / 1e3:.1f} ({pht[1][mk].mean():.1f}; "
                  f"{ideal[mk].sum() / 1e3:.1f}) | {pht[2][mk].sum() / 1e3:.1f} ({pht[2][mk].mean():.1f}) | {pht[3][mk].sum() / 1e3:.1f} ({pht[3][mk].mean():.1f}) |")
        mk = kind == 1
        if mk.any():
            pdone = {(int(a), int(c)): t for a, b, c, t in zip(T[:, 1], Ti, Tj, Ss[:, 3]) if b == c}
            pd_ = np.array([pdone[(int(a), int(c))] for a, c in zip(T[mk, 1], Tj[mk])])
            g_, e_ = Ss[mk, 2], Ss[mk, 3]
            waitp = np.maximum(0, pd_ - g_) / 1e3
            after = (e_ - np.maximum(pd_, g_)) / 1e3
            P("")
            P(f"Panel tiles below the diagonal: {100 * (g_ < pd_).mean():.1f} % finish their product BEFORE the POTRF of their block column's diagonal "
              f"tile has ended; they wait {waitp.sum() / 1e3:.1f} CTA-ms for it (mean {waitp.mean():.1f} us per tile, "
              f"{100 * waitp.sum() / (dur.sum()):.1f} % of all CTA time) and need {after.mean():.1f} us after it "
              f"(tiles that arrive later: {after[g_ >= pd_].mean() if (g_ >= pd_).any() else float('nan'):.1f} us).")
        P("")
        # chain of fronts from the last finished root
        P("### Chain of fronts from the last-finished root down the tree (each: the child that finished last)")
        P("")
        P("| front | type | w | r | start us (first claim) | children done us | done us | span us | block cols x median step |")
        P("|---|---|---|---|---|---|---|---|---|")
        done_s = np.zeros(info["nsuper"]); first_s = np.full(info["nsuper"], 1e30)
        for k, t in enumerate(tasks):
            s = int(t[1])
            done_s[s] = max(done_s[s], (st[k, 4] - t0) / 1e3); first_s[s] = min(first_s[s], (st[k, 0] - t0) / 1e3)
        children = [[] for _ in range(info["nsuper"])]
        for s in range(info["nsuper"]):
            if par[s] >= 0:
                children[par[s]].append(s)
        s = int(np.argmax(done_s))
        total_chain = 0.0
        while True:
            cd = max([done_s[c] for c in children[s]], default=0.0)
            is_tile = s in fl
            nbp = (W(s) + TILE - 1) // TILE
            P(f"| {s} | {'tiled' if is_tile else 'smem'} | {W(s)} | {R(s)} | {first_s[s]:.0f} | {cd:.0f} | {done_s[s]:.0f} | {done_s[s] - cd:.0f} | "
              f"{nbp if is_tile else '-'} |")
            total_chain += done_s[s] - cd
            if not children[s]:
                break
            s = max(children[s], key=lambda c: done_s[c])
        P("")
        P(f"Sum of (done - children done) along this chain: {total_chain:.0f} us of the {span:.0f} us span: the time the factorization "
          f"cannot hide behind other work if nothing else changes.")
        P("")

    # ------------------------------------------------------------------ solves
    tasks, st = h.get_task_trace(1)
    st = st.astype(np.int64)
    ran = st[:, 0] > 0                                    # a fused solve (options.fuse_rhs) runs the backward tasks only
    if ran.any():
        t0 = st[ran, 0].min()
        fwd = (tasks[:, 3] == 0) & ran
        bwd = (tasks[:, 3] == 1) & ran
        P("## Solves (`solve_dag_kernel`)" + ("" if fwd.any() else " -- fused: v = L^-1 P b came out of the factorization, backward tasks only"))
        P("")
        for nm, m in (("forward (L v = P b)", fwd), ("backward (L^T x = v)", bwd)):
            if m.any():
                P(f"* {nm}: {int(m.sum())} tasks, first claim {(st[m, 0].min() - t0) / 1e3:.0f} us, last done {(st[m, 4].max() - t0) / 1e3:.0f} us, "
                  f"median task {np.median(st[m, 4] - st[m, 0]) / 1e3:.1f} us, CTA-time {((st[m, 4] - st[m, 0]).sum()) / 1e6:.1f} CTA-ms")
        tl = tasks[:, 0] == 1
        for nm, m in (("forward block rows of tiled supernodes", fwd & tl), ("backward block columns of tiled supernodes", bwd & tl)):
            if m.any():
                # hop time along the pivot blocks of the largest tiled supernode
                s = int(np.bincount(tasks[m, 1]).argmax())
                mm = m & (tasks[:, 1] == s)
                nbp = (W(s) + TILE - 1) // TILE
                order = np.argsort(tasks[mm, 2])
                ends = st[mm, 4][order][:nbp] if nm.startswith("forward") else st[mm, 4][order][::-1]
                hops = np.diff(np.sort(ends)) / 1e3
                P(f"* {nm}: supernode {s} (w = {W(s)}, r = {R(s)}): median hop between consecutive pivot blocks {np.median(hops):.2f} us "
                  f"over {len(hops)} hops = {hops.sum():.0f} us")
        if bwd.any():
            # chain of the backward solve: from the supernode that finished last up to the root
            ns = info["nsuper"]
            done_b = np.zeros(ns); first_b = np.full(ns, 1e30); cnt_b = np.zeros(ns, dtype=np.int64)
            for k in np.nonzero(bwd)[0]:
                q = int(tasks[k, 1])
                done_b[q] = max(done_b[q], (st[k, 4] - t0) / 1e3); first_b[q] = min(first_b[q], (st[k, 0] - t0) / 1e3); cnt_b[q] += 1
            P("")
            P("### Backward chain: from the supernode that finished last up to the root (each starts when its parent is done)")
            P("")
            P("| supernode | type | w | r | block cols | parent done us | done us | span us | span / block col us |")
            P("|---|---|---|---|---|---|---|---|---|")
            q = int(np.argmax(done_b))
            rows_out = []
            while q >= 0:
                pd = done_b[par[q]] if par[q] >= 0 else 0.0
                nbp = (W(q) + TILE - 1) // TILE
                tiled = cnt_b[q] > 1 or R(q) > 240
                rows_out.append(f"| {q} | {'tiled' if tiled else 'smem'} | {W(q)} | {R(q)} | {nbp if tiled else '-'} | {pd:.0f} | {done_b[q]:.0f} | {done_b[q] - pd:.0f} | "
                                f"{(done_b[q] - pd) / nbp if tiled else float('nan'):.1f} |")
                q = int(par[q])
            for ln in rows_out[::-1]:
                P(ln)
    h.close()
    print("\n".join(out))


if __name__ == "__main__":
    main()
