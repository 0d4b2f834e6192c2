"""CPU oracle for the nodal finite-difference LLG right-hand side (arxiv 2411.11725).

TEST INFRASTRUCTURE, NOT PRODUCT.  Only `tests/`, `__graft_entry__.smoke()` and the
`cpu_baseline` / `--impl reference` legs of `bench.py` may import this package.  The CUDA
library under `paper_2411_11725_b200/` shares no code with it and never imports it.

Everything here is plain fp64 numpy (plus one plain-C file evaluated in `__float128`,
`newell_quad.c`, for the demagnetisation tensor whose closed form cancels catastrophically
in fp64).  Each function cites the passage of /root/reference/PAPER.md (or the SURVEY.md
§8(c) reading, C1..C8) that it follows; no blocking, fusion or reordering beyond what the
passage states.

Array conventions (the paper's multi-indices, Eqs. 8-10):
  nodal vector field   m[j, n1, n2, n3]   shape (3, N1+1, N2+1, N3+1)
  nodal scalar field   L[n1, n2, n3]      shape (N1+1, N2+1, N3+1)
  cell scalar field    Ms[c1, c2, c3]     shape (N1, N2, N3)
  cell vector field    M[j, c1, c2, c3]   shape (3, N1, N2, N3)

Reduced bases for films and rods (Eqs. 23-24): oracle/lowdim.py; nodal arrays keep
three spatial axes, the reduced ones of extent 1 (Problem.basis = 2 or 1).

Parity unpinned: none (every function below is pinned by tests/test_oracle_*.py).
"""
