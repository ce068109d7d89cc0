"""ORACLE — test infrastructure, not product code.

A plain, slow, fp64 CPU implementation (numpy) of the nodal-DG + HABC time step of arXiv 1610.05023,
written from the paper (`/root/reference/PAPER.md`, cited as PAPER.md:L<line>) with the readings listed
in DESIGN.md §3.  It shares no code with `paper_1610_05023_b200/` (the CUDA library) and neither imports
the other; only `workloads/` (seeded inputs, no method arithmetic) is common.

Who may use it: `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs.  The product path never calls into this package.

Parity status of each part (pins live in tests/test_oracle_*.py):
  refelem   pinned: exact differentiation of monomials, D·1=0, mass/area/SBP identities (P4)
  habc      pinned: Padé closed forms, J=1 matrices, block structure, plane-wave identities (P1,P2,P15)
  mesh      pinned: hierarchy counts incl. the paper's Table 3 totals, brute-force node matching (P3)
  solver    pinned: h-convergence ~N+1 (P5), energy non-increase / spectrum for J=0 and walls (P6),
            J=0 == characteristic ABC (P7), reflection decreasing with J (P9), dt inside the LSRK
            stability region (P10), LSRK order conditions (P11), edge/corner role symmetry (P13).
  Readings R8/R9 (how 1+c_i enters the discrete 2D/1D operators; heterogeneous coefficients on the
  boundary levels) are pinned only indirectly through P9: the paper prints no number that would
  distinguish alternative readings.
"""
