"""Pins of the oracle's interior flux where the impedance rho*c jumps across a cell face (the
"exact Riemann solver"; configs 3 and 5 and the SEAM-shaped workload all exercise it) and of reading R9 (materials
of the boundary levels).  Nothing here retypes the oracle's flux formula:

  H1  Riemann invariants.  For cell-wise CONSTANT data the volume term vanishes and the cell integral of F is the
      flux through the cell's faces, so  int_D rhs_p = -rho c^2 sum_f |f| ((n.u)* - n.u^int)  and
      int_D rhs_u = -(1/rho) sum_f |f| (p* - p^int) n_f.  The star state of the acoustic Riemann problem is fixed
      by the two characteristic invariants that reach the interface (textbook: LeVeque, FVM for hyperbolic
      problems, §9.9):  p* + Z^int (n.u)* = p^int + Z^int n.u^int  and  p* - Z^ext (n.u)* = p^ext - Z^ext n.u^ext;
      the test solves that 2x2 system per face (numpy.linalg.solve), with neighbours, areas and normals recomputed
      here from the vertex coordinates.  Walls enter through mirror states (rigid: p, -n.u; p = 0: -p, n.u,
      L516-518) and the basic ABC through a zero incoming invariant (L514).
  H2  Energy.  With rho, c random per cell the energy of (47) (L802) is non-increasing under the exact Riemann
      flux and walls, and the dense operator has no eigenvalue in the right half plane.
  H3  Two-layer transmission at normal incidence: reflected / transmitted pressure amplitudes
      (Z2-Z1)/(Z2+Z1) and 2 Z2/(Z2+Z1).
"""
import itertools

import numpy as np
import pytest

from oracle.mesh import build_hierarchy
from oracle.solver import OracleSolver, dg_rhs
from workloads import cube_mesh
from workloads.configs import box_mesh


def _random_media(K, seed):
    rng = np.random.default_rng(seed)
    return rng.uniform(1.0, 3.0, K), rng.uniform(0.5, 2.0, K)


# ----------------------------------------------------------------------------- H1
@pytest.mark.parametrize("N,kinds", [(1, ("rigid", "dirichlet", "habc")), (3, ("habc", "rigid", "dirichlet"))])
def test_riemann_invariants_fix_the_interface_state(N, kinds):
    verts, tets = cube_mesh(2)
    K = len(tets)
    c, rho = _random_media(K, 11)
    Z = rho * c
    bc = {(a, s): kinds[a] for a in range(3) for s in (-1, 1)}
    H = build_hierarchy(verts, tets, N, c, rho, bc)
    rng = np.random.default_rng(5)
    state = rng.normal(size=(4, K))                                    # p, u, v, w constant per cell
    Np = H.tet.ref.Np
    q = np.repeat(state[:, :, None], Np, axis=2)
    nslots = max(1, (H.tri.K if H.tri is not None else 0) * H.tet.ref.Nfp)
    rp, rU = dg_rhs(H.tet, q[0][None], q[1:4][None], np.zeros((1, nslots)))  # J = 0: r^- = 0
    Mref = H.tet.ref.M
    one = np.ones(Np)
    # the test's own geometry: volumes, face areas, outward normals, neighbours by shared vertex triples
    X = verts[tets]                                                    # [K,4,3]
    vol = np.abs(np.linalg.det(X[:, 1:] - X[:, :1])) / 6.0
    cen = X.mean(axis=1)
    owner = {}
    for k in range(K):
        for f in itertools.combinations(range(4), 3):
            owner.setdefault(tuple(sorted(tets[k, list(f)])), []).append(k)
    exp_p = np.zeros(K)
    exp_u = np.zeros((3, K))
    for k in range(K):
        for f in itertools.combinations(range(4), 3):
            P = X[k, list(f)]
            nvec = np.cross(P[1] - P[0], P[2] - P[0])
            area = 0.5 * np.linalg.norm(nvec)
            n = nvec / (2.0 * area)
            if np.dot(n, P.mean(axis=0) - cen[k]) < 0:
                n = -n
            pM, unM, ZM = state[0, k], float(n @ state[1:, k]), Z[k]
            nb = [j for j in owner[tuple(sorted(tets[k, list(f)]))] if j != k]
            if nb:
                j = nb[0]
                pP, unP, ZP = state[0, j], float(n @ state[1:, j]), Z[j]
                incoming = pP - ZP * unP
            else:
                axis = int(np.argmax(np.abs(n)))
                kind, ZP = kinds[axis], ZM
                if kind == "rigid":
                    incoming = pM - ZP * (-unM)
                elif kind == "dirichlet":
                    incoming = -pM - ZP * unM
                else:
                    incoming = 0.0
            pst, unst = np.linalg.solve(np.array([[1.0, ZM], [1.0, -ZP]]), np.array([pM + ZM * unM, incoming]))
            exp_p[k] += -rho[k] * c[k] ** 2 * area * (unst - unM)
            exp_u[:, k] += -(1.0 / rho[k]) * area * (pst - pM) * n
    # int_D f dx = |J| 1^T M f with 1^T M 1 = 4/3 and |D| = (4/3)|J|
    detJ = vol / (4.0 / 3.0)
    got_p = detJ * (rp[0] @ Mref @ one)
    got_u = detJ[None, :] * np.einsum("dkn,nm,m->dk", rU[0], Mref, one)
    scale = np.abs(exp_p).max()
    assert np.abs(got_p - exp_p).max() < 1e-12 * scale
    assert np.abs(got_u - exp_u).max() < 1e-12 * np.abs(exp_u).max()
    # the impedances really differ across faces, so a flux that mixes up Z^int and Z^ext cannot pass
    assert (Z.max() / Z.min()) > 3.0


# ----------------------------------------------------------------------------- H2
@pytest.mark.parametrize("kind", ["rigid", "dirichlet", "habc"])
def test_energy_nonincreasing_in_random_media(kind):
    verts, tets = cube_mesh(2)
    K = len(tets)
    c, rho = _random_media(K, 23)
    bc = {(a, s): kind for a in range(3) for s in (-1, 1)}
    o = OracleSolver(verts, tets, 2, 0, c, rho, face_bc=bc)
    x = o.nodes()
    p = np.exp(-((x - np.array([0.1, -0.2, 0.15])) ** 2).sum(-1) / (2 * 0.35 ** 2))
    rng = np.random.default_rng(3)
    q0 = np.stack([p, 0.3 * p, -0.2 * p, 0.1 * p]) + 0.05 * rng.normal(size=(4,) + p.shape)   # with inter-cell jumps
    o.set_initial(q0)
    e = [o.energy()]
    for _ in range(25):
        o.step(4)
        e.append(o.energy())
    e = np.array(e)
    assert np.all(np.diff(e) <= 1e-14 * e[0]), kind
    assert e[-1] < 0.9 * e[0]                       # upwind dissipation of the jumps is visible


@pytest.mark.parametrize("kind", ["rigid", "dirichlet", "habc"])
def test_dense_spectrum_in_random_media(kind):
    verts, tets = cube_mesh(1)
    K = len(tets)
    c, rho = _random_media(K, 31)
    bc = {(a, s): kind for a in range(3) for s in (-1, 1)}
    o = OracleSolver(verts, tets, 2, 0, c, rho, face_bc=bc)
    ev = np.linalg.eigvals(o.dense_operator())
    assert ev.real.max() <= 1e-11 * np.abs(ev).max()
    assert np.abs(ev.imag).max() * o.dt < 3.34 and np.abs(ev.real).max() * o.dt < 4.66


# ----------------------------------------------------------------------------- H3
def test_two_layer_reflection_and_transmission():
    """x-only data in a bar [-2,2] x [0,.25]^2 with rigid side walls and the basic ABC at both ends (exact at
    normal incidence): medium 1 (x < 0) rho = 1, c = 1; medium 2 rho = 1.5, c = 2.  A right-going pulse of unit
    amplitude splits into a reflected pulse of amplitude (Z2-Z1)/(Z2+Z1) = 1/2 and a transmitted one of
    amplitude 2 Z2/(Z2+Z1) = 3/2, stretched by c2/c1."""
    verts, tets = box_mesh((16, 1, 1), ((-2.0, 2.0), (0.0, 0.25), (0.0, 0.25)))
    K = len(tets)
    xc = verts[tets].mean(axis=1)[:, 0]
    rho = np.where(xc < 0, 1.0, 1.5)
    c = np.where(xc < 0, 1.0, 2.0)
    Z1, Z2 = 1.0, 3.0
    bc = {(a, s): "rigid" for a in (1, 2) for s in (-1, 1)}
    o = OracleSolver(verts, tets, 5, 0, c, rho, face_bc=bc)
    x = o.nodes()[..., 0]
    p0 = np.exp(-((x + 1.0) / 0.25) ** 2)
    o.set_initial(np.stack([p0, p0 / Z1, 0 * p0, 0 * p0]))          # right-going: p = Z1 u
    e0 = o.energy()
    t_end = 1.6
    ns = int(np.ceil(t_end / o.dt))
    o.dt = t_end / ns
    o.step(ns)
    p, u = o.q[0], o.q[1]
    left, right = x < -1e-9, x > 1e-9
    # reflected pulse: centred at x = -0.6, left-going (p = -Z1 u); transmitted: centred at 1.2, right-going
    assert abs(p[left].max() - (Z2 - Z1) / (Z2 + Z1)) < 5e-3
    assert abs(p[right].max() - 2 * Z2 / (Z2 + Z1)) < 5e-3
    assert abs(x[left][np.argmax(p[left])] + 0.6) < 0.03 and abs(x[right][np.argmax(p[right])] - 1.2) < 0.05
    assert np.abs(p[left] + Z1 * u[left]).max() < 5e-3 and np.abs(p[right] - Z2 * u[right]).max() < 5e-3
    # energy is conserved by the interface (R^2 + (Z1/Z2) T^2 = 1) up to the scheme's dissipation
    assert 0.995 < o.energy() / e0 <= 1.0 + 1e-14
    assert np.abs(o.q[2:]).max() < 2e-3                              # stays 1D up to discretisation (tets break y,z symmetry)


# ----------------------------------------------------------------------------- R9 bookkeeping
def test_boundary_levels_inherit_materials_as_reading_R9_states():
    """Reading R9 (the paper is silent, L41/L857): a boundary triangle carries rho, c of the tetrahedron
    it is a face of; a line cell those of its parent triangle on the face with the lower normal axis.  Checked by
    brute force: the parent is found here from coordinates alone (the only tet that has all three triangle
    vertices / the only triangle on that face with both line vertices)."""
    verts, tets = cube_mesh(3)
    K = len(tets)
    c, rho = _random_media(K, 47)
    H = build_hierarchy(verts, tets, 2, c, rho)
    X = verts[tets]

    def has_points(cell_pts, pts):
        return all(np.abs(cell_pts - q).max(axis=1).min() < 1e-12 for q in pts)

    r2, r1 = H.tri.ref, H.lin.ref
    corners2 = [int(np.argmin(np.abs(r2.rst - np.array(v)).sum(axis=1))) for v in ((-1, -1), (1, -1), (-1, 1))]
    for t in range(H.tri.K):
        pts = H.tri.x[t, corners2]
        parents = [k for k in range(K) if has_points(X[k], pts)]
        assert len(parents) == 1
        assert H.tri.c[t] == c[parents[0]] and H.tri.rho[t] == rho[parents[0]]
    ends = [int(np.argmin(r1.rst[:, 0])), int(np.argmax(r1.rst[:, 0]))]
    for e in range(H.lin.K):
        pts = H.lin.x[e, ends]
        tang = int(np.argmax(np.abs(pts[1] - pts[0])))
        a = min(d for d in range(3) if d != tang)                       # lower normal axis of the two faces
        plane = pts[0, a]
        cands = [t for t in range(H.tri.K)
                 if np.abs(H.tri.x[t][:, a] - plane).max() < 1e-12 and has_points(H.tri.x[t], pts)]
        assert len(cands) == 1
        assert H.lin.c[e] == H.tri.c[cands[0]] and H.lin.rho[e] == H.tri.rho[cands[0]]


def test_edge_outgoing_characteristic_uses_the_impedance_of_its_own_face():
    """H5 (reading R9 inside the edge closure, eq (33)): the outgoing characteristic that a face's 2D
    field sends across a domain edge is r^+ = (p + Z n.u)/2 with Z = rho c of THAT face's triangle.  With q = 0 and only
    the tangential velocities of the triangle on side 0 of one line non-zero, every p_i00 vanishes, the edge system is
    linear in r^+, and its solution must scale with that triangle's impedance and ignore the other side's.  (A closure
    that takes Z from the triangle across the edge passes every other pin: found by mutation in round 3.)"""
    from oracle.solver import OracleSolver
    from workloads import cube_mesh
    v, t = cube_mesh(2)
    K, N, J = len(t), 2, 2
    base = OracleSolver(v, t, N, J, np.ones(K), np.ones(K))
    H = base.H
    parent = H.tri_tetnode[:, 0] // H.tet.ref.Np
    line = next(l for l in range(base.E) if parent[H.lin_tri[l, 0]] != parent[H.lin_tri[l, 1]])
    rng = np.random.default_rng(3)
    vel = rng.normal(size=(J, 2, H.tet.ref.Nfp))

    def incoming(heavy_side):
        rho = np.ones(K)
        if heavy_side is not None:
            rho[parent[H.lin_tri[line, heavy_side]]] = 3.0
        o = OracleSolver(v, t, N, J, np.ones(K), rho)
        assert np.array_equal(o.H.lin_tri, H.lin_tri)
        q, fa, ea = np.zeros_like(o.q), np.zeros_like(o.fa), np.zeros_like(o.ea)
        fa[:, 1:3, H.lin_tri[line, 0]] = vel
        return o.closures((q, fa, ea))["rm_tri"]

    r1, r_own, r_other = incoming(None), incoming(0), incoming(1)
    assert np.linalg.norm(r1) > 1e-3
    assert np.allclose(r_own, 3.0 * r1, rtol=1e-12, atol=1e-14)
    assert np.allclose(r_other, r1, rtol=1e-12, atol=1e-14)
