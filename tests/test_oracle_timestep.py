"""Pins P17, P18: the two time-related lines of the oracle that no other pin fixes.

P17 -- eq (46), reading R7: dt = min_k 1 / (c_k (N+1)^2 Fscale_k), "F_scale,k is the maximum ratio
of surface to volume Jacobian of the k-th mesh cell".  The oracle takes Fscale from its metric terms (|grad of the
face's level-set coordinate|, oracle/mesh.py::_geometry).  Here the same number comes from elementary geometry that the
oracle does not use: with the reference tetrahedron of volume 4/3 and reference faces of area 2, J_k = 3 V_k / 4 and
sJ_f = area_f / 2, so Fscale_kf = 2 area_f / (3 V_k), with area_f from a cross product and V_k from a determinant of
the vertex coordinates.  On Kuhn cubes this is the closed form dt = h / (2 sqrt 2 c_max (N+1)^2).
The meshes are chosen so that every ingredient matters: per-cell speeds make min_k differ from "the fastest cell on
the smallest cell", anisotropic and perturbed cells make max_f differ from min_f and from the mean.

P18 -- PAPER.md:L531-540 with L776-786: the source term S(t) of the pressure equation is evaluated at the LSRK stage
times t + c_n dt.  With the stage times right the scheme is fourth order in dt for this non-autonomous system; with
S frozen at t, or with shifted c_n, it drops to first order.  The test measures the order by time refinement on one
fixed mesh (the spatial error cancels)."""
import numpy as np
import pytest

from oracle.solver import OracleSolver
from workloads.configs import box_mesh, cube_mesh


def geometric_dt(verts, tets, c, N, face_pick=np.max, cell_pick=np.min):
    """eq (46) from vertex coordinates only"""
    V4 = verts[tets]                                                        # [K,4,3]
    vol = np.abs(np.linalg.det(V4[:, 1:] - V4[:, :1])) / 6.0
    area = np.empty((len(tets), 4))
    for f, (a, b, d) in enumerate(((0, 1, 2), (0, 1, 3), (1, 2, 3), (0, 2, 3))):
        area[:, f] = 0.5 * np.linalg.norm(np.cross(V4[:, b] - V4[:, a], V4[:, d] - V4[:, a]), axis=1)
    fscale = face_pick(2.0 * area / (3.0 * vol[:, None]), axis=1)
    return float(cell_pick(1.0 / (c * (N + 1) ** 2 * fscale)))


@pytest.mark.parametrize("n,N", [(1, 1), (2, 3), (3, 5)])
def test_dt_closed_form_on_kuhn_cubes(n, N):
    """h = 2/n on [-1,1]^3; the largest face of a Kuhn tetrahedron is h^2 sqrt(2) / 2, its volume h^3 / 6."""
    v, t = cube_mesh(n)
    rng = np.random.default_rng(5)
    c = rng.uniform(1.0, 3.0, size=len(t))
    o = OracleSolver(v, t, N, 0, c, np.ones(len(t)))
    h = 2.0 / n
    assert o.dt == pytest.approx(h / (2.0 * np.sqrt(2.0) * c.max() * (N + 1) ** 2), rel=1e-13)
    assert OracleSolver(v, t, N, 0, c, np.ones(len(t)), cfl=0.5).dt == pytest.approx(0.5 * o.dt, rel=1e-15)


@pytest.mark.parametrize("shape,box,perturb", [
    ((3, 3, 3), ((-1.0, 1.0),) * 3, 0.25),                                  # configs[2]'s recipe: perturbed interior
    ((4, 3, 2), ((0.0, 35.0), (0.0, 40.0), (0.0, 15.0)), 0.2),              # SEAM aspect, anisotropic
])
def test_dt_from_cross_products_on_general_meshes(shape, box, perturb):
    rng = np.random.default_rng(11)
    v, t = box_mesh(shape, box, perturb, rng)
    K = len(t)
    # speeds anti-correlated with cell size, so that neither the fastest nor the smallest cell alone decides
    V4 = v[t]
    vol = np.abs(np.linalg.det(V4[:, 1:] - V4[:, :1])) / 6.0
    c = 1.5 + 2.5 * (vol / vol.max()) * rng.uniform(0.5, 1.0, size=K)
    N = 3
    o = OracleSolver(v, t, N, 0, c, np.ones(K))
    want = geometric_dt(v, t, c, N)
    assert o.dt == pytest.approx(want, rel=1e-12)
    # the test discriminates: each plausible misreading of (46) gives a clearly different number on this mesh
    for wrong in (geometric_dt(v, t, c, N, face_pick=np.min),               # "minimum ratio"
                  geometric_dt(v, t, c, N, face_pick=np.mean),
                  geometric_dt(v, t, c, N, cell_pick=np.max),               # the printed "max_k" (reading R7)
                  geometric_dt(v, t, np.full(K, c.max()), N),               # global c_max on the worst cell
                  geometric_dt(v, t, c, N + 1), geometric_dt(v, t, c, N) * (N + 1)):
        assert abs(wrong / want - 1.0) > 0.02


def _run_source(dt, tf, N=2):
    v, t = box_mesh((2, 2, 2), ((-0.5, 0.5),) * 3)
    K = len(t)
    o = OracleSolver(v, t, N, 1, np.ones(K), np.ones(K), dt=dt)
    o.set_source(np.array([0.03, 0.02, 0.01]), 2.5, 0.5)
    nst = int(round(tf / dt))
    assert abs(nst * dt - tf) < 1e-12
    o.step(nst)
    return o.q.copy(), o


def test_source_is_evaluated_at_the_lsrk_stage_times():
    """Errors against a run with dt/8 at t = 0.64 (the wavelet S(t) peaks near t_s = 0.5): halving dt must divide the
    error by about 2^4.  Measured order 4.0; a source frozen at the start of the step gives 1.0."""
    v, t = box_mesh((2, 2, 2), ((-0.5, 0.5),) * 3)
    dt0 = OracleSolver(v, t, 2, 1, np.ones(len(t)), np.ones(len(t))).dt
    tf = 0.64
    n0 = int(np.ceil(tf / dt0))
    dt = tf / n0                                                            # <= the stable step of eq (46)
    q1, o1 = _run_source(dt, tf)
    q2, _ = _run_source(dt / 2, tf)
    qr, _ = _run_source(dt / 8, tf)
    assert np.linalg.norm(qr[0]) > 1e-3                                     # the source has acted
    e1, e2 = np.linalg.norm(q1 - qr), np.linalg.norm(q2 - qr)
    order = np.log2(e1 / e2)
    assert e2 > 1e-12 * np.linalg.norm(qr)                                  # above round-off: the order is meaningful
    assert order > 3.5, (order, e1, e2)
    assert abs(o1.t - tf) < 1e-12
