"""ORACLE (test infrastructure) — the algebra of the Padé HABC and its edge / corner compatibility systems.

Notation follows BASELINE.json / DESIGN.md: J = number of auxiliary fields per face (the paper's N),
M = 2J+1.  Citations are PAPER.md lines.

  pade_coefficients   eq (6):  c_n = tan^2(n pi / M)
  f_pade5 / f_pade6   eq (5) and (6), L67-71: two printed forms of the Padé approximant of sqrt(1+X)
  edge_system         eq (33a-b), L406-408 (reading R4: the sum in (33a) runs over j)
  corner_system       eq (35a-c)
Both systems are assembled literally from the printed equations in the form
        M r^- = b + T (r^- + r^+)      ==>      (M I - T) r^- = b + T r^+ ,
so the returned pair is (L, T) with L = M I - T.  The oracle solves them densely (numpy.linalg.solve)
at every node; no block structure is exploited here.
"""
from __future__ import annotations

import numpy as np


def pade_coefficients(J: int):
    """(M, c[1..J]) of eq (6)."""
    M = 2 * J + 1
    n = np.arange(1, J + 1, dtype=np.float64)
    return M, np.tan(n * np.pi / M) ** 2


def f_pade5(J: int, X):
    """eq (5): 1 + (2/M) sum a_n X / (1 + b_n X), a_n = sin^2, b_n = cos^2."""
    M = 2 * J + 1
    X = np.asarray(X, dtype=np.float64)
    out = np.ones_like(X)
    for n in range(1, J + 1):
        a, b = np.sin(n * np.pi / M) ** 2, np.cos(n * np.pi / M) ** 2
        out = out + (2.0 / M) * a * X / (1.0 + b * X)
    return out


def f_pade6(J: int, X):
    """eq (6): 1 + (2/M) sum c_n (1 - (1+c_n)/(1+c_n+X))."""
    M, c = pade_coefficients(J)
    X = np.asarray(X, dtype=np.float64)
    out = np.ones_like(X)
    for n in range(J):
        out = out + (2.0 / M) * c[n] * (1.0 - (1.0 + c[n]) / (1.0 + c[n] + X))
    return out


def C2(c, i, j):
    """C_ij = (1+c_i)/(1+c_i+c_j), PAPER.md:L404 (0-based i,j)."""
    return (1.0 + c[i]) / (1.0 + c[i] + c[j])


def C3(c, i, j, k):
    """C_ijk = (1+c_i)/(1+c_i+c_j+c_k), PAPER.md:L343 (0-based)."""
    return (1.0 + c[i]) / (1.0 + c[i] + c[j] + c[k])


def edge_system(J: int):
    """Edge between face A (operator index i, first subscript) and face B (index j, second subscript).

    Unknown ordering: [ r^{-a}_j , j=0..J-1 ;  r^{-b}_i , i=0..J-1 ]  where
      r^{-a}_j : incoming characteristic along axis a of face B's field p_0j0   (paper: r^{-x}_{0j0})
      r^{-b}_i : incoming characteristic along axis b of face A's field p_i00   (paper: r^{-y}_{i00})
    eq (33b): M r^{-a}_j = sum_i c_i ( p*_ij + C_ji S^b_i + (C_ij - 1) S^a_j )
    eq (33a): M r^{-b}_i = sum_j c_j ( p*_ij + (C_ji - 1) S^b_i + C_ij S^a_j )
    with S = r^- + r^+.  Returns (L, T, Ba, Bb): L = M I - T, and the two [J, J*J] matrices mapping the
    flattened p*_ij (index i*J+j) to b^a_j = sum_i c_i p*_ij and b^b_i = sum_j c_j p*_ij.
    """
    M, c = pade_coefficients(J)
    T = np.zeros((2 * J, 2 * J))
    Ba = np.zeros((J, J * J))
    Bb = np.zeros((J, J * J))
    ia = lambda j: j            # noqa: E731  position of r^{-a}_j
    ib = lambda i: J + i        # noqa: E731  position of r^{-b}_i
    for j in range(J):
        for i in range(J):
            T[ia(j), ib(i)] += c[i] * C2(c, j, i)
            T[ia(j), ia(j)] += c[i] * (C2(c, i, j) - 1.0)
            Ba[j, i * J + j] += c[i]
    for i in range(J):
        for j in range(J):
            T[ib(i), ib(i)] += c[j] * (C2(c, j, i) - 1.0)
            T[ib(i), ia(j)] += c[j] * C2(c, i, j)
            Bb[i, i * J + j] += c[j]
    L = M * np.eye(2 * J) - T
    return L, T, Ba, Bb


def corner_system(J: int):
    """Corner where the edges along x, y, z meet.  Unknown ordering (each block J*J, row-major):
        X[j,k] = r^{-x}_{0jk}   (edge along x; j <-> y-face operator, k <-> z-face operator)
        Y[i,k] = r^{-y}_{i0k}   (edge along y)
        Z[i,j] = r^{-z}_{ij0}   (edge along z)
    eq (35a-c), assembled literally as  M r^- = T (r^- + r^+).
    Returns (L, T) with L = M I - T."""
    M, c = pade_coefficients(J)
    n = J * J
    ix = lambda j, k: j * J + k             # noqa: E731
    iy = lambda i, k: n + i * J + k         # noqa: E731
    iz = lambda i, j: 2 * n + i * J + j     # noqa: E731
    T = np.zeros((3 * n, 3 * n))
    for i in range(J):
        for j in range(J):
            for k in range(J):
                # (35a): row X[j,k], sum over i
                T[ix(j, k), ix(j, k)] += c[i] * (C3(c, i, j, k) - 1.0)
                T[ix(j, k), iy(i, k)] += c[i] * C3(c, j, k, i)
                T[ix(j, k), iz(i, j)] += c[i] * C3(c, k, i, j)
                # (35b): row Y[i,k], sum over j
                T[iy(i, k), ix(j, k)] += c[j] * C3(c, i, j, k)
                T[iy(i, k), iy(i, k)] += c[j] * (C3(c, j, k, i) - 1.0)
                T[iy(i, k), iz(i, j)] += c[j] * C3(c, k, i, j)
                # (35c): row Z[i,j], sum over k
                T[iz(i, j), ix(j, k)] += c[k] * C3(c, i, j, k)
                T[iz(i, j), iy(i, k)] += c[k] * C3(c, j, k, i)
                T[iz(i, j), iz(i, j)] += c[k] * (C3(c, k, i, j) - 1.0)
    L = M * np.eye(3 * n) - T
    return L, T
