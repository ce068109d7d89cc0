"""Pin P12: the oracle organised as the paper's Algorithms 1-5 — physical p_i00, p_ij0 stored,
qb / q0 arrays carried between stages and refreshed in the kernel order of PAPER.md:L627 (oracle/staged.py) — must
give the same fields as the recompute-from-state oracle (oracle/solver.py) to round-off.  Guards reading R5 and the
claim that every qb / q0 array is an algebraic function of the state."""
import numpy as np
import pytest

from oracle.solver import OracleSolver
from oracle.staged import StagedOracleSolver
from workloads import make_workload


@pytest.mark.parametrize("name,kw,nsteps", [("cfg1", {}, 50), ("cfg5", dict(n=2, N=2, J=3), 30)])
def test_staged_algorithms_match_method_of_lines_oracle(name, kw, nsteps):
    w = make_workload(name, **kw)
    o = OracleSolver(w.verts, w.tets, w.N, w.J, w.c, w.rho)
    x = o.nodes()
    cn = np.repeat(w.c[:, None], x.shape[1], axis=1)
    q0 = np.stack(w.fields(x[..., 0] + (0.4 if name == "cfg1" else 0.0), x[..., 1] + 0.3 * (name == "cfg1"), x[..., 2], cn, 1.0))
    o.set_initial(q0)
    s = StagedOracleSolver(w.verts, w.tets, w.N, w.J, w.c, w.rho, dt=o.dt)
    s.set_initial(q0)
    o.step(nsteps)
    s.step(nsteps)
    ref, got = o.get_fields(), s.get_fields()
    for name_, a, b in zip(("q", "face_aux", "edge_aux"), got, ref):
        assert np.linalg.norm(b) > 1e-3 * np.linalg.norm(ref[0][0]), name_          # P16: the level carries data
        assert np.abs(a - b).max() < 1e-13 * max(1.0, np.abs(b).max()), (name_, np.abs(a - b).max())
