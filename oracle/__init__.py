"""ORACLE — test infrastructure, not product code.

A plain, slow, fp64 CPU implementation (numpy) of the nodal-DG + HABC time step of arXiv 1610.05023,
written from the paper (`/root/reference/PAPER.md`, cited as PAPER.md:L<line>) with the readings listed
in DESIGN.md §3.  It shares no code with `paper_1610_05023_b200/` (the CUDA library) and neither imports
the other; only `workloads/` (seeded inputs, no method arithmetic) is common.

Who may use it: `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs.  The product path never calls into this package.

Parity status of each part (pins live in tests/test_oracle_*.py; DESIGN.md §2 has the table):
  refelem   pinned: exact differentiation of monomials, D·1=0, mass/area/SBP identities (P4)
  habc      pinned: Padé closed forms, J=1 matrices, block structure, plane-wave identities (P1,P2,P15)
  mesh      pinned: hierarchy counts incl. the paper's Table 3 totals, brute-force node matching (P3);
            material inheritance of triangles / lines (reading R9) checked by brute force (test_oracle_heterogeneous)
  solver    pinned: h-convergence ~N+1 in 3D (P5) and, calling dg_rhs on the surface and line meshes alone, in 2D
            and 1D (L1); energy non-increase / spectrum for J=0 and walls, uniform and random media (P6, H2);
            interior flux with rho*c jumping across faces against the Riemann invariants and against the two-layer
            reflection / transmission amplitudes (H1, H3); J=0 == characteristic ABC (P7); truncation error of F
            on an exact solution of the continuous HABC problem converging at rate N on every level and for every
            auxiliary set (L2: pins (29)-(35), the 1/(1+c_i), 1/(1+c_i+c_j) row scales of reading R8 and the i/j
            conventions); reflection decreasing with J (P9); dt inside the LSRK stability region (P10); LSRK order
            conditions (P11); edge/corner role symmetry (P13); analytic spherical wave of the point source (P14).
  staged    oracle/staged.py is the Algorithm 1-5 organisation (qb/q0 carried); P12 pins it to solver.py at 1e-13.
  Reading R9 is a reading, not a result: the paper is silent on materials of the boundary levels (L41, L857); the
  tests pin that the code does what the reading says, nothing in the paper can pin the reading itself.
"""
