"""ORACLE (test infrastructure) — reference elements of the nodal DG scheme in 1D, 2D, 3D.

PAPER.md:L489 (§3.2): Warp & Blend nodes on the tetrahedron [68]; triangle / line nodes are the tet's
face / edge nodes.  PAPER.md:L529: differentiation and lifting matrices "defined in [42]" (Hesthaven &
Warburton): with an orthonormal basis psi_m and V_nm = psi_m(r_n):  D_r = V_r V^-1,  M = (V V^T)^-1,
LIFT = M^-1 E with E the face mass matrices scattered to the face nodes.

Everything is evaluated in x87 extended precision (np.longdouble) and rounded once to float64, so that an
independent implementation doing the same agrees to about one ulp (reading R13/§7 hard part 5).
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

LD = np.longdouble

# Warp & Blend blending parameter per degree N (3D table of [68]/[42]; data, reading R13).
ALPHA_TET = {1: 0.0, 2: 0.0, 3: 0.0, 4: 0.1002, 5: 1.1332, 6: 1.5608, 7: 1.3413, 8: 1.2577}


# ----------------------------------------------------------------------------- Jacobi polynomials
def jacobi_p(x, alpha: int, beta: int, n: int):
    """Orthonormal Jacobi polynomial P_n^{(alpha,beta)}(x), integer alpha,beta >= 0 (three-term recurrence)."""
    x = np.asarray(x, dtype=LD)
    a, b = alpha, beta
    # gamma0 = 2^(a+b+1)/(a+b+1) * a! b! / (a+b)!   (exact integer arithmetic, then one rounding)
    g0 = LD(2 ** (a + b + 1) * math.factorial(a) * math.factorial(b)) / LD((a + b + 1) * math.factorial(a + b))
    p_prev = np.ones_like(x) / np.sqrt(g0)
    if n == 0:
        return p_prev
    g1 = LD((a + 1) * (b + 1)) / LD(a + b + 3) * g0
    p = (LD(a + b + 2) * x / 2 + LD(a - b) / 2) / np.sqrt(g1)
    if n == 1:
        return p
    a_old = LD(2) / LD(2 + a + b) * np.sqrt(LD((a + 1) * (b + 1)) / LD(a + b + 3))
    for i in range(1, n):
        h1 = 2 * i + a + b
        a_new = LD(2) / LD(h1 + 2) * np.sqrt(LD((i + 1) * (i + 1 + a + b) * (i + 1 + a) * (i + 1 + b))
                                             / LD((h1 + 1) * (h1 + 3)))
        b_new = -LD(a * a - b * b) / LD(h1 * (h1 + 2))
        p_next = (-a_old * p_prev + (x - b_new) * p) / a_new
        p_prev, p, a_old = p, p_next, a_new
    return p


def grad_jacobi_p(x, alpha: int, beta: int, n: int):
    """d/dx P_n^{(a,b)} = sqrt(n (n+a+b+1)) P_{n-1}^{(a+1,b+1)}."""
    x = np.asarray(x, dtype=LD)
    if n == 0:
        return np.zeros_like(x)
    return np.sqrt(LD(n * (n + alpha + beta + 1))) * jacobi_p(x, alpha + 1, beta + 1, n - 1)


def lgl_nodes(N: int):
    """Legendre-Gauss-Lobatto points on [-1,1]: the end points and the zeros of P_N'(x) (Newton, long double)."""
    if N == 1:
        return np.array([-1, 1], dtype=LD)
    # interior: zeros of P^{(1,1)}_{N-1}; start from the Golub-Welsch eigenvalues in double
    n = N - 1
    k = np.arange(1, n)
    off = 2.0 / (2 * k + 2) * np.sqrt(k * (k + 2) * (k + 1) * (k + 1) / ((2 * k + 1) * (2 * k + 3.0)))
    x = np.sort(np.linalg.eigvalsh(np.diag(off, 1) + np.diag(off, -1))) if n > 1 else np.array([0.0])
    x = x.astype(LD)
    for _ in range(6):
        f = jacobi_p(x, 1, 1, n)
        df = grad_jacobi_p(x, 1, 1, n)
        x = x - f / df
    x = (x - x[::-1]) / 2          # enforce exact symmetry
    return np.concatenate([[LD(-1)], x, [LD(1)]]).astype(LD)


# ----------------------------------------------------------------------------- Warp & Blend nodes
def _edge_warp(N: int, x):
    """w(x) = sum_i (x_i^LGL - x_i^eq) l_i^eq(x): displacement interpolated on the equispaced nodes [68]."""
    x = np.asarray(x, dtype=LD)
    req = np.array([LD(-1) + LD(2 * i) / LD(N) for i in range(N + 1)], dtype=LD)
    rgl = lgl_nodes(N)
    w = np.zeros_like(x)
    for i in range(N + 1):
        li = np.ones_like(x)
        for j in range(N + 1):
            if j != i:
                li = li * (x - req[j]) / (req[i] - req[j])
        w = w + (rgl[i] - req[i]) * li
    return w


def _scaled_edge_warp(N: int, x):
    """w(x)/(1-x^2), set to 0 at |x|=1 (there the blend factor vanishes as well)."""
    x = np.asarray(x, dtype=LD)
    w = _edge_warp(N, x)
    den = 1 - x * x
    ok = np.abs(den) > LD(1e-12)
    out = np.zeros_like(x)
    out[ok] = w[ok] / den[ok]
    return out


def tet_equispaced_barycentric(N: int):
    """Barycentric coordinates of the equispaced lattice, ordered t-major, then s, then r fastest."""
    lam = []
    for n in range(N + 1):               # t index
        for m in range(N + 1 - n):       # s index
            for q in range(N + 1 - n - m):   # r index
                # lambda_k belongs to vertex k: v1=(-1,-1,-1), v2=(1,-1,-1), v3=(-1,1,-1), v4=(-1,-1,1)
                lam.append([N - n - m - q, q, m, n])
    return np.array(lam, dtype=LD) / LD(N)


def nodes_tet(N: int, alpha: float | None = None):
    """Warp & Blend interpolation nodes on the reference tet {r,s,t>=-1, r+s+t<=-1} (explicit
    construction of [68]): equispaced lattice on the equilateral tet, displaced by the blended face
    warps; a face warp is the sum over the face's three edges of the 1D LGL warp along the edge."""
    if alpha is None:
        alpha = ALPHA_TET[N]
    alpha = LD(alpha)
    lam = tet_equispaced_barycentric(N)                       # [Np,4]
    s3, s6 = np.sqrt(LD(3)), np.sqrt(LD(6))
    VT = np.array([[-1, -1 / s3, -1 / s6], [1, -1 / s3, -1 / s6], [0, 2 / s3, -1 / s6], [0, 0, 3 / s6]], dtype=LD)
    X = lam @ VT
    tol = LD(1e-10)
    nz = lam > tol
    nnz = nz.sum(axis=1)
    shift = np.zeros_like(X)

    def face_warp(b, c, d, a_weight):
        """2D warp vector of the face with vertices (b,c,d); a_weight(o) gives (1+(alpha*lam_o)^2)."""
        wv = np.zeros_like(X)
        for (m, n, o) in ((b, c, d), (c, d, b), (d, b, c)):
            wf = _scaled_edge_warp(N, lam[:, n] - lam[:, m])
            amp = 4 * lam[:, m] * lam[:, n] * wf * (1 + (alpha * lam[:, o]) ** 2)
            wv = wv + amp[:, None] * ((VT[n] - VT[m]) / 2)[None, :]
        return wv

    gen = nnz >= 3                                            # face-interior and volume-interior nodes
    for a in range(4):
        b, c, d = [k for k in range(4) if k != a]
        wv = face_warp(b, c, d, None)
        la = lam[:, a]
        num = lam[:, b] * lam[:, c] * lam[:, d]
        den = (lam[:, b] + la / 2) * (lam[:, c] + la / 2) * (lam[:, d] + la / 2)
        blend = np.zeros_like(la)
        blend[gen] = (1 + (alpha * la[gen]) ** 2) * num[gen] / den[gen]
        shift = shift + blend[:, None] * wv
    # tet-edge nodes (exactly two non-zero barycentrics): the pure 1D warp along that edge
    for i in np.nonzero(nnz == 2)[0]:
        m, n = np.nonzero(nz[i])[0]
        wf = _scaled_edge_warp(N, np.array([lam[i, n] - lam[i, m]], dtype=LD))[0]
        shift[i] = 4 * lam[i, m] * lam[i, n] * wf * (VT[n] - VT[m]) / 2
    X = X + shift
    # back to (r,s,t): X = v1 + (1+r)/2 (v2-v1) + (1+s)/2 (v3-v1) + (1+t)/2 (v4-v1)
    A = np.stack([(VT[1] - VT[0]) / 2, (VT[2] - VT[0]) / 2, (VT[3] - VT[0]) / 2], axis=1)
    rst = (_inv_ld(A) @ (X - VT[0]).T).T - 1
    # snap lattice-exact coordinates (faces, edges, vertices) and keep the result symmetric
    for k in range(3):
        lk = lam[:, k + 1]
        rst[lk < tol, k] = LD(-1)
    on3 = lam[:, 0] < tol                                     # face r+s+t=-1: fix t from r,s
    rst[on3, 2] = -1 - rst[on3, 0] - rst[on3, 1]
    return rst[:, 0].copy(), rst[:, 1].copy(), rst[:, 2].copy()


# ----------------------------------------------------------------------------- small dense helpers
def _inv_ld(A):
    """Gauss-Jordan inverse with partial pivoting in long double (numpy.linalg has no long double)."""
    A = np.array(A, dtype=LD)
    n = A.shape[0]
    M = np.concatenate([A, np.eye(n, dtype=LD)], axis=1)
    for c in range(n):
        p = c + int(np.argmax(np.abs(M[c:, c])))
        if p != c:
            M[[c, p]] = M[[p, c]]
        M[c] = M[c] / M[c, c]
        for r in range(n):
            if r != c and M[r, c] != 0:
                M[r] = M[r] - M[r, c] * M[c]
    return M[:, n:]


# ----------------------------------------------------------------------------- orthonormal simplex bases
def basis_1d(r, i):
    return jacobi_p(r, 0, 0, i)


def grad_basis_1d(r, i):
    return grad_jacobi_p(r, 0, 0, i)


def _collapse_2d(r, s):
    r = np.asarray(r, dtype=LD)
    s = np.asarray(s, dtype=LD)
    a = -np.ones_like(r)
    ok = np.abs(1 - s) > LD(1e-14)
    a[ok] = 2 * (1 + r[ok]) / (1 - s[ok]) - 1
    return a, s.copy()


def _pw(x, e):
    """x**e with the convention that a negative exponent only ever multiplies a zero factor."""
    return np.zeros_like(x) if e < 0 else x ** e


def basis_2d(r, s, i, j):
    a, b = _collapse_2d(r, s)
    return np.sqrt(LD(2)) * jacobi_p(a, 0, 0, i) * jacobi_p(b, 2 * i + 1, 0, j) * _pw(1 - b, i)


def grad_basis_2d(r, s, i, j):
    """Chain rule through a = 2(1+r)/(1-s)-1, b = s (da/dr = 2/(1-b), da/ds = (1+a)/(1-b))."""
    a, b = _collapse_2d(r, s)
    A, dA = jacobi_p(a, 0, 0, i), grad_jacobi_p(a, 0, 0, i)
    B, dB = jacobi_p(b, 2 * i + 1, 0, j), grad_jacobi_p(b, 2 * i + 1, 0, j)
    rt2 = np.sqrt(LD(2))
    dr = rt2 * 2 * dA * B * _pw(1 - b, i - 1)
    ds = rt2 * (dA * (1 + a) * B * _pw(1 - b, i - 1) + A * (dB * _pw(1 - b, i) - i * B * _pw(1 - b, i - 1)))
    return dr, ds


def _collapse_3d(r, s, t):
    r = np.asarray(r, dtype=LD)
    s = np.asarray(s, dtype=LD)
    t = np.asarray(t, dtype=LD)
    a = -np.ones_like(r)
    b = -np.ones_like(r)
    ok = np.abs(s + t) > LD(1e-14)
    a[ok] = -2 * (1 + r[ok]) / (s[ok] + t[ok]) - 1
    ok = np.abs(1 - t) > LD(1e-14)
    b[ok] = 2 * (1 + s[ok]) / (1 - t[ok]) - 1
    return a, b, t.copy()


def basis_3d(r, s, t, i, j, k):
    a, b, c = _collapse_3d(r, s, t)
    return (2 * np.sqrt(LD(2)) * jacobi_p(a, 0, 0, i) * jacobi_p(b, 2 * i + 1, 0, j) * _pw(1 - b, i)
            * jacobi_p(c, 2 * (i + j) + 2, 0, k) * _pw(1 - c, i + j))


def grad_basis_3d(r, s, t, i, j, k):
    """Chain rule with  da/dr = 4/((1-b)(1-c)), da/ds = da/dt = 2(1+a)/((1-b)(1-c)),
    db/ds = 2/(1-c), db/dt = (1+b)/(1-c), dc/dt = 1."""
    a, b, c = _collapse_3d(r, s, t)
    A, dA = jacobi_p(a, 0, 0, i), grad_jacobi_p(a, 0, 0, i)
    B, dB = jacobi_p(b, 2 * i + 1, 0, j), grad_jacobi_p(b, 2 * i + 1, 0, j)
    C, dC = jacobi_p(c, 2 * (i + j) + 2, 0, k), grad_jacobi_p(c, 2 * (i + j) + 2, 0, k)
    ob, oc = 1 - b, 1 - c
    e = i + j
    common = dA * B * _pw(ob, i - 1) * C * _pw(oc, e - 1)
    Gb = dB * _pw(ob, i) - i * B * _pw(ob, i - 1)              # d/db [B (1-b)^i]
    Gc = dC * _pw(oc, e) - e * C * _pw(oc, e - 1)              # d/dc [C (1-c)^(i+j)]
    dr = 4 * common
    ds = 2 * (1 + a) * common + 2 * A * Gb * C * _pw(oc, e - 1)
    dt = 2 * (1 + a) * common + A * Gb * (1 + b) * C * _pw(oc, e - 1) + A * B * _pw(ob, i) * Gc
    f = 2 * np.sqrt(LD(2))
    return f * dr, f * ds, f * dt


def vandermonde(dim: int, N: int, *coords):
    """V[n,m] = psi_m(x_n) and the list of its reference-coordinate derivatives (long double)."""
    if dim == 1:
        (r,) = coords
        V = np.stack([basis_1d(r, i) for i in range(N + 1)], axis=1)
        G = [np.stack([grad_basis_1d(r, i) for i in range(N + 1)], axis=1)]
    elif dim == 2:
        r, s = coords
        idx = [(i, j) for i in range(N + 1) for j in range(N + 1 - i)]
        V = np.stack([basis_2d(r, s, i, j) for (i, j) in idx], axis=1)
        g = [grad_basis_2d(r, s, i, j) for (i, j) in idx]
        G = [np.stack([x[d] for x in g], axis=1) for d in range(2)]
    else:
        r, s, t = coords
        idx = [(i, j, k) for i in range(N + 1) for j in range(N + 1 - i) for k in range(N + 1 - i - j)]
        V = np.stack([basis_3d(r, s, t, i, j, k) for (i, j, k) in idx], axis=1)
        g = [grad_basis_3d(r, s, t, i, j, k) for (i, j, k) in idx]
        G = [np.stack([x[d] for x in g], axis=1) for d in range(3)]
    return V, G


# ----------------------------------------------------------------------------- the reference element
@dataclasses.dataclass
class RefElem:
    dim: int
    N: int
    Np: int
    Nfp: int
    Nfaces: int
    rst: np.ndarray        # [Np, dim] float64 nodes
    D: list                # dim matrices [Np,Np] float64
    M: np.ndarray          # mass [Np,Np]
    LIFT: np.ndarray       # [Np, Nfaces*Nfp]
    Fmask: np.ndarray      # [Nfaces, Nfp] node indices of each face (increasing node index)
    nhat: np.ndarray       # [Nfaces, dim] unnormalised reference outward normals (gradient of the face's level set)
    V: np.ndarray          # Vandermonde (float64), for interpolation / tests
    Emat: np.ndarray       # [Np, Nfaces*Nfp] face-mass scatter matrix (M @ LIFT), for tests
    rst_ld: np.ndarray     # long double nodes


def _face_param(dim, rst, f):
    """(dim-1)-dimensional reference coordinates of the nodes of face f (any affine chart of the face
    onto the (dim-1)-simplex gives the same face mass matrix)."""
    if dim == 3:
        r, s, t = rst[:, 0], rst[:, 1], rst[:, 2]
        return [(r, s), (r, t), (s, t), (s, t)][f]
    if dim == 2:
        r, s = rst[:, 0], rst[:, 1]
        return [(r,), (s,), (s,)][f]
    return ()


def make_refelem(dim: int, N: int) -> RefElem:
    tol = LD(1e-10)
    if dim == 3:
        r, s, t = nodes_tet(N)
        rst = np.stack([r, s, t], axis=1)
        masks = [np.abs(1 + t) < tol, np.abs(1 + s) < tol, np.abs(1 + r + s + t) < tol, np.abs(1 + r) < tol]
        nhat = np.array([[0, 0, -1], [0, -1, 0], [1, 1, 1], [-1, 0, 0]], dtype=np.float64)
    elif dim == 2:
        # triangle nodes = nodes of a tet face (face t=-1, coordinates (r,s))
        r3, s3, t3 = nodes_tet(N)
        on = np.abs(1 + t3) < tol
        r, s = r3[on], s3[on]
        rst = np.stack([r, s], axis=1)
        masks = [np.abs(1 + s) < tol, np.abs(r + s) < tol, np.abs(1 + r) < tol]
        nhat = np.array([[0, -1], [1, 1], [-1, 0]], dtype=np.float64)
    else:
        r = lgl_nodes(N)                     # = the tet's edge nodes
        rst = r[:, None]
        masks = [np.abs(1 + r) < tol, np.abs(1 - r) < tol]
        nhat = np.array([[-1.0], [1.0]])
    Np = rst.shape[0]
    Fmask = np.array([np.nonzero(m)[0] for m in masks])
    Nfaces, Nfp = Fmask.shape
    V, G = vandermonde(dim, N, *[rst[:, d] for d in range(dim)])
    Vinv = _inv_ld(V)
    D = [g @ Vinv for g in G]
    Minv = V @ V.T
    M = Vinv.T @ Vinv
    E = np.zeros((Np, Nfaces * Nfp), dtype=LD)
    for f in range(Nfaces):
        if dim == 1:
            E[Fmask[f, 0], f] = 1
            continue
        fc = _face_param(dim, rst[Fmask[f]], f)
        Vf, _ = vandermonde(dim - 1, N, *fc)
        Mf = _inv_ld(Vf @ Vf.T)
        E[np.ix_(Fmask[f], np.arange(f * Nfp, (f + 1) * Nfp))] = Mf
    LIFT = Minv @ E
    f64 = np.float64
    return RefElem(dim=dim, N=N, Np=Np, Nfp=Nfp, Nfaces=Nfaces, rst=rst.astype(f64), D=[d.astype(f64) for d in D],
                   M=M.astype(f64), LIFT=LIFT.astype(f64), Fmask=Fmask, nhat=nhat, V=V.astype(f64),
                   Emat=E.astype(f64), rst_ld=rst)
