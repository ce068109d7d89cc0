"""Pins P1, P2, P4, P11, P15 of DESIGN.md §3: the oracle's reference elements, Padé algebra, compatibility
systems and LSRK coefficients against closed forms and identities fixed by the paper / the mathematics."""
import itertools

import numpy as np
import pytest

from oracle import habc
from oracle.refelem import lgl_nodes, make_refelem
from oracle.solver import RK4A, RK4B, RK4C


# ----------------------------------------------------------------------------- P4 reference elements
@pytest.mark.parametrize("N", [1, 2, 3, 4, 5, 6, 8])
def test_tet_differentiates_monomials_exactly(N):
    """BASELINE north_star: exact differentiation of degree <= N polynomials."""
    e = make_refelem(3, N)
    r, s, t = e.rst.T
    assert e.Np == (N + 1) * (N + 2) * (N + 3) // 6 and e.Nfp == (N + 1) * (N + 2) // 2
    for a, b, c in itertools.product(range(N + 1), repeat=3):
        if a + b + c > N:
            continue
        f = r ** a * s ** b * t ** c
        dr = a * r ** max(a - 1, 0) * s ** b * t ** c if a else 0 * r
        ds = b * r ** a * s ** max(b - 1, 0) * t ** c if b else 0 * r
        dt = c * r ** a * s ** b * t ** max(c - 1, 0) if c else 0 * r
        tol = 2e-13 * (N + 1) ** 2
        assert np.abs(e.D[0] @ f - dr).max() < tol
        assert np.abs(e.D[1] @ f - ds).max() < tol
        assert np.abs(e.D[2] @ f - dt).max() < tol


@pytest.mark.parametrize("dim,N", [(1, 1), (1, 4), (2, 1), (2, 3), (2, 5), (3, 1), (3, 2), (3, 4), (3, 5), (3, 7)])
def test_mass_sbp_lift_identities(dim, N):
    e = make_refelem(dim, N)
    one = np.ones(e.Np)
    vol = {1: 2.0, 2: 2.0, 3: 4.0 / 3.0}[dim]
    assert abs(one @ e.M @ one - vol) < 1e-13                       # measure of the reference simplex
    for D in e.D:
        assert np.abs(D @ one).max() < 1e-12                        # D 1 = 0
    # mass matrix integrates products exactly: int r^2 over the simplex (degree 2 <= 2N)
    r = e.rst[:, 0]
    exact = {1: 2.0 / 3.0, 2: 2.0 / 3.0, 3: 8.0 / 15.0}[dim]      # closed forms (Dirichlet integrals of barycentrics)
    assert abs(r @ e.M @ r - exact) < 1e-13
    # M LIFT = E, face mass matrices have total measure 2 (3D faces: parametric area 2; 2D edges: length 2)
    assert np.abs(e.M @ e.LIFT - e.Emat).max() < 1e-13
    for f in range(e.Nfaces):
        cols = slice(f * e.Nfp, (f + 1) * e.Nfp)
        assert abs(e.Emat[:, cols].sum() - (2.0 if dim > 1 else 1.0)) < 1e-13
    # summation by parts: M D_a + (M D_a)^T = sum_f nhat_a^f E_f (scattered face mass)
    for a in range(dim):
        lhs = e.M @ e.D[a] + (e.M @ e.D[a]).T
        rhs = np.zeros_like(lhs)
        for f in range(e.Nfaces):
            rhs[:, e.Fmask[f]] += e.nhat[f, a] * e.Emat[:, f * e.Nfp:(f + 1) * e.Nfp]
        assert np.abs(lhs - rhs).max() < 1e-12


def test_lgl_and_face_nodes_match():
    """triangle/line nodes = the tet's face/edge nodes; edges carry LGL points."""
    x = lgl_nodes(4).astype(float)
    assert np.allclose(x, [-1, -np.sqrt(3 / 7), 0, np.sqrt(3 / 7), 1], atol=1e-15)      # textbook values
    x = lgl_nodes(3).astype(float)
    assert np.allclose(x, [-1, -np.sqrt(1 / 5), np.sqrt(1 / 5), 1], atol=1e-15)
    for N in (2, 5):
        e3, e2, e1 = make_refelem(3, N), make_refelem(2, N), make_refelem(1, N)
        for f, ch in enumerate(((0, 1), (0, 2), (1, 2), (1, 2))):
            assert np.abs(e3.rst[e3.Fmask[f]][:, ch] - e2.rst).max() < 1e-14
        assert np.abs(e2.rst[e2.Fmask[0], 0] - e1.rst[:, 0]).max() < 1e-14
        # symmetric node set: permuting barycentric coordinates maps the set onto itself
        lam = np.stack([-(1 + e3.rst.sum(1)) / 2] + [(1 + e3.rst[:, d]) / 2 for d in range(3)], axis=1)
        for perm in itertools.permutations(range(4)):
            d = np.abs(lam[:, None, :] - lam[None, :, list(perm)]).max(axis=2).min(axis=1)
            assert d.max() < 1e-13


# ----------------------------------------------------------------------------- P1 Padé
@pytest.mark.parametrize("J", [1, 2, 3, 4, 8, 12])
def test_pade_closed_forms(J):
    M, c = habc.pade_coefficients(J)
    X = np.linspace(-0.95, 2.0, 60)
    assert np.abs(habc.f_pade5(J, X) - habc.f_pade6(J, X)).max() < 1e-13       # (5) == (6)
    assert abs(c.sum() - J * M) < 1e-9 * J * M
    # reflection coefficient of a plane wave at incidence theta: -((1-cos)/(1+cos))^M
    th = np.linspace(0.05, 1.4, 20)
    cs = np.cos(th)
    f = habc.f_pade6(J, -np.sin(th) ** 2)
    assert np.abs((cs - f) / (cs + f) + ((1 - cs) / (1 + cs)) ** M).max() < 1e-12
    # Padé order: f_J - sqrt(1+X) = O(X^(2J+1))
    if J <= 3:
        e1 = abs(habc.f_pade6(J, 0.1) - np.sqrt(1.1))
        e2 = abs(habc.f_pade6(J, 0.05) - np.sqrt(1.05))
        assert abs(np.log2(e1 / e2) - (2 * J + 1)) < 0.5


def test_pade_J1_rational():
    X = np.linspace(-0.9, 3, 17)
    assert np.abs(habc.f_pade6(1, X) - (4 + 3 * X) / (4 + X)).max() < 1e-14


# ----------------------------------------------------------------------------- P2, P13 edge / corner systems
def test_edge_corner_J1_values():
    L, T, Ba, Bb = habc.edge_system(1)
    assert np.allclose(L * 7, [[30, -12], [-12, 30]], atol=1e-12)
    assert np.allclose(T * 7, [[-9, 12], [12, -9]], atol=1e-12)
    assert np.allclose(Ba, [[3.0]]) and np.allclose(Bb, [[3.0]])
    Lc, Tc = habc.corner_system(1)
    assert np.allclose(Lc, 4.8 * np.eye(3) - 1.2 * (np.ones((3, 3)) - np.eye(3)), atol=1e-12)
    assert np.allclose(np.linalg.solve(Lc, Tc @ np.ones(3)), 0.25, atol=1e-13)


@pytest.mark.parametrize("J", [2, 3, 4, 8])
def test_edge_corner_block_structure(J):
    """the inverse edge matrix has 2 independent JxJ blocks, the inverse corner matrix 3
    independent J^2xJ^2 blocks; role symmetry (P13); contraction r+ -> r- with radius J/(J+1)."""
    L, T, Ba, Bb = habc.edge_system(J)
    Li = np.linalg.inv(L)
    assert np.abs(Li[:J, :J] - Li[J:, J:]).max() < 1e-13 and np.abs(Li[:J, J:] - Li[J:, :J]).max() < 1e-13
    assert np.linalg.cond(L) < 16
    assert abs(np.abs(np.linalg.eigvals(Li @ T)).max() - J / (J + 1.0)) < 1e-10
    # swapping the roles of the two faces (i<->j, a<->b) is the same system
    P = np.block([[np.zeros((J, J)), np.eye(J)], [np.eye(J), np.zeros((J, J))]])
    assert np.abs(P @ L @ P - L).max() < 1e-13
    Lc, Tc = habc.corner_system(J)
    n = J * J
    Lci = np.linalg.inv(Lc)
    B = [[Lci[a * n:(a + 1) * n, b * n:(b + 1) * n] for b in range(3)] for a in range(3)]
    # cyclic relabelling x->y->z->x: X[j,k] -> Y'[..]; with the cyclic unknown ordering X(j,k), Y(k,i), Z(i,j)
    tr = np.arange(n).reshape(J, J).T.reshape(-1)                  # transposes the two set indices
    Pc = np.zeros((3 * n, 3 * n))
    Pc[np.arange(n), np.arange(n)] = 1                              # X(j,k)
    Pc[n + np.arange(n), n + tr] = 1                                # Y stored (i,k) -> (k,i)
    Pc[2 * n + np.arange(n), 2 * n + np.arange(n)] = 1              # Z(i,j)
    Lcyc = np.linalg.inv(Pc @ Lc @ Pc.T)
    Bc = [[Lcyc[a * n:(a + 1) * n, b * n:(b + 1) * n] for b in range(3)] for a in range(3)]
    for s in range(3):                                              # block-circulant: 3 distinct blocks
        for a in range(3):
            assert np.abs(Bc[a][(a + s) % 3] - Bc[0][s]).max() < 1e-12
    assert np.linalg.cond(Lc) < 16
    assert abs(np.abs(np.linalg.eigvals(Lci @ Tc)).max() - J / (J + 1.0)) < 1e-9
    assert len(B) == 3


# ----------------------------------------------------------------------------- P15 plane-wave identities
def test_plane_wave_symbols_satisfy_closures():
    """For p = exp(i(k.x - w t)), w^2 = c^2 |k|^2, the symbol of M^x_i is m = (1+c_i)w^2/((1+c_i)w^2 - c^2 k_perp^2)
    (eq (8)).  Feeding these exact values to the oracle's closures: (30)/(23) on a face (as an
    approximation of the exact ABC, checked through f_J), (33) on an edge and (35) at a corner hold exactly."""
    rng = np.random.default_rng(7)
    J = 3
    M, c = habc.pade_coefficients(J)
    cs = 1.3
    k = rng.normal(size=3)
    w2 = cs * cs * (k @ k)
    sym = lambda ci, kp2: (1 + ci) * w2 / ((1 + ci) * w2 - cs * cs * kp2)      # noqa: E731
    mx = np.array([sym(ci, k[1] ** 2 + k[2] ** 2) for ci in c])
    my = np.array([sym(ci, k[0] ** 2 + k[2] ** 2) for ci in c])
    mz = np.array([sym(ci, k[0] ** 2 + k[1] ** 2) for ci in c])
    # corner (35): with S^x_jk = p_0jk = my_j mz_k etc. and r^-x_0jk = (1/M) sum_i c_i (p_ijk - p_0jk) (19a / 27a
    # time-integrated), p_ijk = mx_i my_j mz_k: the oracle's T must reproduce M r^- = T S
    Lc, Tc = habc.corner_system(J)
    SX = np.outer(my, mz)
    SY = np.outer(mx, mz)
    SZ = np.outer(mx, my)
    S = np.concatenate([SX.ravel(), SY.ravel(), SZ.ravel()])
    rX = np.array([[sum(c[i] * (mx[i] - 1) for i in range(J)) * my[j] * mz[kk] for kk in range(J)] for j in range(J)]) / M
    rY = np.array([[sum(c[j] * (my[j] - 1) for j in range(J)) * mx[i] * mz[kk] for kk in range(J)] for i in range(J)]) / M
    rZ = np.array([[sum(c[kk] * (mz[kk] - 1) for kk in range(J)) * mx[i] * my[j] for j in range(J)] for i in range(J)]) / M
    r = np.concatenate([rX.ravel(), rY.ravel(), rZ.ravel()])
    assert np.abs(Tc @ S / M - r).max() < 1e-12 * np.abs(r).max()
    # edge (33) with k_z = 0: p_ij0 = C_ij p_0j0 + C_ji p_i00 exactly (time-integrated (18a)), so p*_ij = 0
    k[2] = 0.0
    w2 = cs * cs * (k @ k)
    mx = np.array([sym(ci, k[1] ** 2) for ci in c])
    my = np.array([sym(ci, k[0] ** 2) for ci in c])
    for i in range(J):
        for j in range(J):
            assert abs(mx[i] * my[j] - habc.C2(c, i, j) * my[j] - habc.C2(c, j, i) * mx[i]) < 1e-12
    L, T, Ba, Bb = habc.edge_system(J)
    Sv = np.concatenate([my, mx])                       # S^a_j = p_0j0 = my_j ; S^b_i = p_i00 = mx_i
    ra = np.array([sum(c[i] * (mx[i] * my[j] - my[j]) for i in range(J)) for j in range(J)]) / M   # (25a)
    rb = np.array([sum(c[j] * (mx[i] * my[j] - mx[i]) for j in range(J)) for i in range(J)]) / M   # (25b)
    assert np.abs(T @ Sv / M - np.concatenate([ra, rb])).max() < 1e-12


# ----------------------------------------------------------------------------- P11 LSRK
def test_lsrk_order_conditions():
    """2N-storage form -> Butcher tableau; 4th-order conditions; stability polynomial; c consistency."""
    s = 5
    A = np.zeros((s, s))
    b = np.zeros(s)
    # propagate: S_n = a_n S_{n-1} + dt F_n ; y += b_n S_n  => weights of F_m in y after stage n
    wS = np.zeros(s)
    wy = np.zeros(s)
    for n in range(s):
        A[n] = wy
        wS = RK4A[n] * wS
        wS[n] += 1.0
        wy = wy + RK4B[n] * wS
    b = wy
    cc = A.sum(axis=1)
    assert np.abs(cc - RK4C).max() < 1e-13
    assert abs(b.sum() - 1) < 1e-14
    assert abs(b @ cc - 1 / 2) < 1e-14
    assert abs(b @ cc ** 2 - 1 / 3) < 1e-14 and abs(b @ A @ cc - 1 / 6) < 1e-14
    assert abs(b @ cc ** 3 - 1 / 4) < 1e-13 and abs((b * cc) @ A @ cc - 1 / 8) < 1e-13
    assert abs(b @ A @ cc ** 2 - 1 / 12) < 1e-13 and abs(b @ A @ A @ cc - 1 / 24) < 1e-13
    assert abs(b @ A @ A @ A @ cc - 1 / 200) < 1e-4      # z^5 coefficient of the stability polynomial (O7)
