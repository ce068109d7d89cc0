"""Direct pins of the oracle's 2D (face) and 1D (edge) levels ("the same numerical scheme";
eq (31a-c), (34a-b) L439-441) and of the whole closure chain against an exact solution.

  L1  `dg_rhs` on the surface mesh and on the line mesh alone, with p = 0 walls (L516-518): the standing modes
      cos(pi x/2) cos(pi y/2) cos(w t), w = c pi/sqrt(2), and cos(pi x/2) cos(w t), w = c pi/2, converge at
      rate ~ N+1 under h-refinement (pins the in-plane geometric factors, normals, LIFT2D/LIFT1D, Fscale, and
      where rho and c enter, since rho, c != 1 here).
  L2  Truncation error of F at EVERY level on an exact solution of the continuous HABC problem.  For a time-harmonic
      plane wave exp(i(k.x - w t)), w = c|k|, the operator M^x_i of eq (8) (L87) is the number
      m^x_i = (1+c_i) w^2 / ((1+c_i) w^2 - c^2 (k_y^2 + k_z^2)), the same for the wave reflected by the face
      x = L, whose amplitude follows from (9) (L92): R_x = exp(2 i k_x L) (cos t - f_J)/(cos t + f_J),
      cos t = c k_x / w, f_J = 1 - (2/M) sum_n c_n (m^x_n - 1).  The product of the three 1D patterns
      (exp(i k_a x_a) + R_a exp(-i k_a x_a)) therefore satisfies the HABC on the faces x, y, z = +L exactly,
      with auxiliary fields p_ijk = m^x_i m^y_j m^z_k p, u_ijk likewise (eq (11), (22) L296-298) and
      p*_i00 = p_i00 - p (29), p*_ij0 = p_ij0 - C_ji p_i00 - C_ij p_0j0 (32).  Interpolated at the nodes, every
      flux jump of the scheme vanishes on it (interior faces: continuity; HABC faces, edges, the corner: (30), (33),
      (35) return the exact incoming characteristics), so F(I y) - I(dy/dt) is pure interpolation error: it shrinks
      like h^N for the 3D fields AND for every auxiliary set.  A wrong constant anywhere in (29)-(35), in the
      1/(1+c_i) and 1/(1+c_i+c_j) row scales of (31a)/(34a) (reading R8), or in the i/j conventions leaves an O(1)
      residual that does not converge.  Only cells away from the three "-" faces are looked at (the wave does not
      satisfy the HABC there).
"""
import numpy as np
import pytest

from oracle.mesh import build_hierarchy
from oracle.solver import RK4A, RK4B, OracleSolver, dg_rhs
from workloads import cube_mesh

C0, RHO0 = 2.0, 1.5


def _level_mode_error(dim, n, N):
    verts, tets = cube_mesh(n)
    K = len(tets)
    bc = {(a, s): "dirichlet" for a in range(3) for s in (-1, 1)}
    bc[(2, 1)] = "habc"
    if dim == 1:
        bc[(1, 1)] = "habc"
    H = build_hierarchy(verts, tets, N, np.full(K, C0), np.full(K, RHO0), bc)
    L = H.tri if dim == 2 else H.lin
    assert L.K == (2 * n * n if dim == 2 else n)
    x = L.x
    if dim == 2:
        p0 = np.cos(np.pi * x[..., 0] / 2) * np.cos(np.pi * x[..., 1] / 2)
        w = C0 * np.pi / np.sqrt(2.0)
    else:
        p0 = np.cos(np.pi * x[..., 0] / 2)
        w = C0 * np.pi / 2
    t_end = 2.4 / w                                                   # cos(w t_end) = -0.74
    p = p0[None].copy()
    U = np.zeros((1, dim) + p0.shape)
    dt = 0.5 / (C0 * (N + 1) ** 2 * L.Fs.max())
    ns = int(np.ceil(t_end / dt))
    dt = t_end / ns
    sp, sU = np.zeros_like(p), np.zeros_like(U)
    none = np.zeros((1, 1))
    for _ in range(ns):
        for s in range(5):
            rp, rU = dg_rhs(L, p, U, none)
            sp = RK4A[s] * sp + dt * rp
            sU = RK4A[s] * sU + dt * rU
            p = p + RK4B[s] * sp
            U = U + RK4B[s] * sU
    e = p[0] - p0 * np.cos(w * t_end)
    return np.sqrt(np.sum(L.detJ * np.einsum("kn,nm,km->k", e, L.ref.M, e)))


@pytest.mark.parametrize("dim,N", [(2, 1), (2, 2), (2, 3), (1, 1), (1, 2), (1, 3)])
def test_face_and_edge_level_h_convergence(dim, N):
    e1, e2 = _level_mode_error(dim, 2, N), _level_mode_error(dim, 4, N)
    rate = np.log2(e1 / e2)
    assert N + 0.7 < rate < N + 1.8, (dim, N, e1, e2, rate)


# ----------------------------------------------------------------------------- L2
def _exact_habc_state(o, J, kvec, c, rho, L=1.0):
    """Complex amplitudes at t = 0 of the exact solution described in the module docstring, laid out as the
    oracle's state (q [4,K,Np], fa [J,3,T,Nfp], ea [J,J,2,E,N1]); returns (state, omega)."""
    M = 2 * J + 1
    cn = np.tan(np.arange(1, J + 1) * np.pi / M) ** 2                      # eq (6)
    kvec = np.asarray(kvec, dtype=np.float64)
    w = c * np.linalg.norm(kvec)
    m = np.empty((3, J))
    R = np.empty(3, dtype=complex)
    for a in range(3):
        kperp2 = kvec @ kvec - kvec[a] ** 2
        m[a] = (1 + cn) * w * w / ((1 + cn) * w * w - c * c * kperp2)      # symbol of eq (8)
        fJ = 1.0 - (2.0 / M) * np.sum(cn * (m[a] - 1.0))                   # eq (6)/(9)
        cost = c * kvec[a] / w
        R[a] = np.exp(2j * kvec[a] * L) * (cost - fJ) / (cost + fJ)

    def fields(x):
        """p and u (3 components) at points x [..., 3]"""
        p = np.zeros(x.shape[:-1], dtype=complex)
        u = np.zeros((3,) + x.shape[:-1], dtype=complex)
        for sx in (1, -1):
            for sy in (1, -1):
                for sz in (1, -1):
                    sg = np.array([sx, sy, sz])
                    amp = np.prod([1.0 if sg[a] > 0 else R[a] for a in range(3)])
                    kap = sg * kvec
                    comp = amp * np.exp(1j * (x @ kap))
                    p += comp
                    for d in range(3):
                        u[d] += kap[d] / (rho * w) * comp                   # rho du/dt = -grad p  (1b)
        return p, u

    H = o.H
    p3, u3 = fields(H.tet.x)
    q = np.stack([p3, u3[0], u3[1], u3[2]])
    T, E = H.tri.K, H.lin.K
    fa = np.zeros((J, 3, T, H.tet.ref.Nfp), dtype=complex)
    pt, ut = fields(H.tri.x)
    for t in range(T):
        a = H.tri_axis[t]
        for i in range(J):
            fa[i, 0, t] = (m[a, i] - 1.0) * pt[t]                           # (29): p* = p_i00 - (r^- + r^+) = p_i00 - p
            for d in range(2):
                fa[i, 1 + d, t] = m[a, i] * ut[H.tri.axes[t, d], t]
    ea = np.zeros((J, J, 2, E, o.N + 1), dtype=complex)
    pe, ue = fields(H.lin.x)
    for e in range(E):
        a, b = H.lin_ab[e]
        for i in range(J):
            for j in range(J):
                Cij = (1 + cn[i]) / (1 + cn[i] + cn[j])                     # L404
                Cji = (1 + cn[j]) / (1 + cn[i] + cn[j])
                ea[i, j, 0, e] = (m[a, i] * m[b, j] - Cji * m[a, i] - Cij * m[b, j]) * pe[e]    # (32)
                ea[i, j, 1, e] = m[a, i] * m[b, j] * ue[H.lin_axis[e], e]
    return (q, fa, ea), w


def _truncation_errors(n, N, J):
    verts, tets = cube_mesh(n)
    K = len(tets)
    c, rho = 1.3, 0.8
    o = OracleSolver(verts, tets, N, J, np.full(K, c), np.full(K, rho))
    y, w = _exact_habc_state(o, J, (1.1, 0.8, 1.4), c, rho)
    F = o.rhs(tuple(np.ascontiguousarray(a.real) for a in y))
    exact = [(-1j * w * a).real for a in y]
    h = 2.0 / n
    keep = [np.all(L.x.mean(axis=1) > -1.0 + h, axis=1) for L in (o.H.tet, o.H.tri, o.H.lin)]
    assert keep[1].sum() >= 3 * 2 * (n - 1) ** 2 and keep[2].sum() >= 3 * (n - 1)
    out = {}

    def rel(got, ref, mask):
        return float(np.linalg.norm((got - ref)[..., mask, :]) / np.linalg.norm(ref[..., mask, :]))

    out["p"] = rel(F[0][0], exact[0][0], keep[0])
    out["u"] = rel(F[0][1:], exact[0][1:], keep[0])
    for i in range(J):
        out[f"face_p{i}"] = rel(F[1][i, 0], exact[1][i, 0], keep[1])
        out[f"face_u{i}"] = rel(F[1][i, 1:], exact[1][i, 1:], keep[1])
        for j in range(J):
            out[f"edge_p{i}{j}"] = rel(F[2][i, j, 0], exact[2][i, j, 0], keep[2])
            out[f"edge_w{i}{j}"] = rel(F[2][i, j, 1], exact[2][i, j, 1], keep[2])
    return out


@pytest.mark.parametrize("N,J", [(3, 2), (4, 3)])
def test_plane_wave_truncation_error_converges_on_every_level(N, J):
    e1, e2 = _truncation_errors(4, N, J), _truncation_errors(8, N, J)
    for key in e1:
        rate = np.log2(e1[key] / e2[key])
        assert rate > N - 0.5, (key, e1[key], e2[key], rate)          # observed: N-0.25 .. N+0.15
        assert e2[key] < (5e-3 if N == 3 else 3e-4), (key, e2[key])   # observed: 3.3e-3, 1.7e-4 (a wrong constant: O(1))
