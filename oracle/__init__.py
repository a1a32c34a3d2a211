"""CPU oracle for the parametric interior-point NMPC hot path of arxiv/paper_2606_04725.

TEST INFRASTRUCTURE ONLY.  This package is a plain, slow, obviously-correct CPU restatement (NumPy / SciPy
fp64 + a few lines of plain C in `chol.c`) of what the CUDA path computes.  It exists so that the CUDA path
can be checked against something written independently from the paper.  Only `tests/`,
`__graft_entry__.smoke()` and the `cpu_baseline` / `--impl reference` legs of `bench.py` may import it.
The product (`paper_2606_04725_b200/`) never imports, links or executes anything in here, and nothing in
here imports the product.  The only shared code is the seeded input generator `ocp_inputs.py`, which holds
none of the method's arithmetic.

Contents
  models.py   stage models F(x,u), their first and second derivatives, stage costs
  nlp.py      the transcribed OCP (5)/(6): f, grad f, c = h(y;p), J, W as SciPy sparse
  linalg.py   Cholesky / triangular solves, Eq. (18)-(25)
  chol.c      the plain-C loops behind linalg.py
  ipm.py      Algorithm 2 (LiftedIPM) step by step + Algorithm 1 (NMPC loop)

Pins (tests/test_oracle_*.py, `-m "not gpu"`):
  * dense / sparse / block-tridiagonal Cholesky vs brute force  ||LL^T-K||_F/||K||_F <= 1e-13, vs LAPACK
  * symbolic structure vs the non-zero pattern of a dense factor; parent[j] = min{i>j: L_ij != 0}
  * derivatives vs central finite differences
  * condensation algebra Eq. (10)->(14)->(17) vs a dense solve of the un-condensed Newton system
  * inertia relation Eq. (15) on tiny systems
  * Riccati closed form on an unconstrained LQ instance
  * KKT conditions (8) recomputed from raw model functions at the converged point
  * distillation steady state vs Table 1 (sanity, tol 1e-3)
Parity unpinned: the IPM constants and iteration counts (the paper prints neither; readings in DESIGN.md §3).
"""
