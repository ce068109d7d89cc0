"""ORACLE (test infrastructure) — the same time step organised as the paper's Algorithms 1-5 (PAPER.md:L410-435,
L585-750): the boundary levels store the PHYSICAL pressures p_i00, p_ij0 in q^tri, q^lin, and the arrays
    qb^tet (incoming characteristic r^-_000 per boundary face node),   q0^tet (the sum r^- + r^+, L754),
    qb^tri / q0^tri (the 2J incoming characteristics per edge node and the sums S^a_j, S^b_i),   qb^lin
are CARRIED from stage to stage and refreshed by the update "kernels" in the order of L627: per LSRK stage first
the right-hand sides of all three levels from stage-(n-1) data, then the updates 3D -> 2D -> 1D -> 0D, each one
recovering p* = p - (previous sum) before the Runge-Kutta update and re-adding the new sum after it (Alg. 3
L646-659, Alg. 4).

`oracle/solver.py` keeps none of these arrays and recomputes the closure chain from the state at every stage
(SURVEY.md §8(c)).  Pin P12 (tests/test_oracle_staged.py) demands that the two agree to round-off: it guards
reading R5 (zero auxiliary ODE state, cached arrays initialised by one pass of the closures) and the kernel order.
Written separately from `OracleSolver.closures` on purpose; it shares only `dg_rhs`, the hierarchy and the
assembled systems of `oracle/habc.py`.
"""
from __future__ import annotations

import numpy as np

from . import habc
from .mesh import build_hierarchy
from .solver import RK4A, RK4B, dg_rhs


class StagedOracleSolver:
    def __init__(self, verts, tets, N: int, J: int, c, rho, dt: float, face_bc=None):
        assert J > 0
        self.N, self.J, self.dt = N, J, float(dt)
        self.H = H = build_hierarchy(verts, tets, N, c, rho, face_bc)
        assert H.tri is not None and H.lin is not None and H.cor_vertex.size > 0, "written for the full hierarchy"
        self.M, self.cn = habc.pade_coefficients(J)
        self.Le, self.Te, self.Ba, self.Bb = habc.edge_system(J)
        self.Lc, self.Tc = habc.corner_system(J)
        self.T, self.E, self.C = H.tri.K, H.lin.K, H.cor_vertex.size

    # ---- outgoing characteristics (28a-c) with reading R1: r^+ = (p + Z n.u)/2
    def _rplus_tet(self):
        H = self.H
        ids = H.tri_tetnode
        un = np.empty(ids.shape)
        for t in range(self.T):
            un[t] = self.q[1 + H.tri_axis[t]].reshape(-1)[ids[t]] * H.tri_sign[t]
        Z = (H.tri.rho * H.tri.c)[:, None]
        return 0.5 * (self.q[0].reshape(-1)[ids] + Z * un)                   # [T,Nfp]

    def _rplus_tri(self):
        """per line: r^{+b}_i from face A's fields (side 0) and r^{+a}_j from face B's (side 1), each [J,E,N1]"""
        H, J = self.H, self.J
        out = []
        for side in range(2):
            r = np.empty((J, self.E, self.N + 1))
            for e in range(self.E):
                t = H.lin_tri[e, side]
                nodes = H.lin_trinode[e, side] - t * H.tet.ref.Nfp           # local node ids on triangle t
                axis_n, sgn = H.lin_ab[e, 1 - side], H.lin_sign[e, 1 - side]  # normal of the OTHER face
                slot = list(H.tri.axes[t]).index(axis_n)
                Z = H.tri.rho[t] * H.tri.c[t]
                r[:, e] = 0.5 * (self.qtri[:, 0, t][:, nodes] + Z * sgn * self.qtri[:, 1 + slot, t][:, nodes])
            out.append(r)
        return out[1], out[0]                                                # (r^{+a}_j, r^{+b}_i)

    def _rplus_lin(self):
        H, J = self.H, self.J
        r = np.empty((3, J, J, self.C))
        for cidx in range(self.C):
            for d in range(3):
                ell, end, s = H.cor_line[cidx, d], H.cor_end[cidx, d], H.cor_sign[cidx, d]
                node = 0 if end == 0 else self.N
                Z = H.lin.rho[ell] * H.lin.c[ell]
                r[d, :, :, cidx] = 0.5 * (self.qlin[:, :, 0, ell, node] + Z * s * self.qlin[:, :, 1, ell, node])
        return r

    # ---- the closure halves of the update kernels (Alg. 3, Alg. 4, Alg. 5)
    def _close_face(self, pstar):
        charOut = self._rplus_tet()
        charIn = np.tensordot(self.cn, pstar, axes=(0, 0)) / self.M           # (30)
        self.qb_tet = charIn.copy()
        self.q0_tet = charOut + charIn
        self.qtri[:, 0] = pstar + self.q0_tet[None]                           # (29)

    def _edge_sum(self, Sa, Sb):
        J, cn = self.J, self.cn
        out = np.empty((J, J, self.E, self.N + 1))
        for i in range(J):
            for j in range(J):
                out[i, j] = habc.C2(cn, j, i) * Sb[i] + habc.C2(cn, i, j) * Sa[j]     # (32)
        return out

    def _close_edge(self, pstar):
        J, E, N1 = self.J, self.E, self.N + 1
        rpa, rpb = self._rplus_tri()
        ps = pstar.reshape(J * J, E * N1)
        rhs = np.concatenate([self.Ba @ ps, self.Bb @ ps], axis=0) \
            + self.Te @ np.concatenate([rpa.reshape(J, -1), rpb.reshape(J, -1)], axis=0)
        sol = np.linalg.solve(self.Le, rhs)                                   # (33a-b)
        rma, rmb = sol[:J].reshape(J, E, N1), sol[J:].reshape(J, E, N1)
        self.qb_tri = np.stack([rmb, rma], axis=2).reshape(J, -1)             # slot (line, side, node); side A <- r^{-b}_i
        self.q0_tri = (rma + rpa, rmb + rpb)
        self.qlin[:, :, 0] = pstar + self._edge_sum(*self.q0_tri)

    def _close_corner(self):
        J = self.J
        rp = self._rplus_lin().reshape(3 * J * J, self.C)
        rm = np.linalg.solve(self.Lc, self.Tc @ rp).reshape(3, J * J, self.C)  # (35a-c)
        self.qb_lin = np.transpose(rm, (1, 2, 0)).reshape(J * J, self.C * 3)  # slot = corner*3 + axis

    # ---- boundary
    def set_initial(self, q):
        """3D data given; auxiliary ODE state zero (p* = 0, velocities 0; L130, L355, reading R5); the carried
        arrays are initialised by one pass of the closures."""
        H, J = self.H, self.J
        self.q = np.array(q, dtype=np.float64).reshape(4, H.tet.K, H.tet.ref.Np)
        self.qtri = np.zeros((J, 3, self.T, H.tet.ref.Nfp))
        self.qlin = np.zeros((J, J, 2, self.E, self.N + 1))
        self._close_face(np.zeros((J, self.T, H.tet.ref.Nfp)))
        self._close_edge(np.zeros((J, J, self.E, self.N + 1)))
        self._close_corner()
        self.res3 = np.zeros_like(self.q)
        self.res2 = np.zeros_like(self.qtri)
        self.res1 = np.zeros_like(self.qlin)

    def step(self, nsteps: int = 1):
        H, J, cn, dt = self.H, self.J, self.cn, self.dt
        E, N1 = self.E, self.N + 1
        for _ in range(nsteps):
            for n in range(5):
                # volume + surface kernels of the three levels, all on stage-(n-1) data (L627)
                rp3, rU3 = dg_rhs(H.tet, self.q[0][None], self.q[1:4][None], self.qb_tet.reshape(1, -1))
                rp2, rU2 = dg_rhs(H.tri, self.qtri[:, 0], self.qtri[:, 1:3], self.qb_tri)
                rp1, rU1 = dg_rhs(H.lin, self.qlin[:, :, 0].reshape(J * J, E, N1),
                                  self.qlin[:, :, 1].reshape(J * J, 1, E, N1), self.qb_lin)
                a, b = RK4A[n], RK4B[n]
                # 3D update kernel (Alg. 2)
                self.res3 = a * self.res3 + dt * np.concatenate([rp3, rU3[0]], axis=0)
                self.q = self.q + b * self.res3
                # 2D update kernel (Alg. 3)
                self.res2[:, 0] = a * self.res2[:, 0] + dt * rp2 / (1.0 + cn)[:, None, None]        # (31a)
                self.res2[:, 1:3] = a * self.res2[:, 1:3] + dt * rU2
                pstar = self.qtri[:, 0] - self.q0_tet[None]                   # previous p* from the previous sum
                pstar = pstar + b * self.res2[:, 0]
                self.qtri[:, 1:3] = self.qtri[:, 1:3] + b * self.res2[:, 1:3]
                self._close_face(pstar)
                # 1D update kernel (Alg. 4)
                scale = (1.0 + cn[:, None] + cn[None, :])[:, :, None, None]
                self.res1[:, :, 0] = a * self.res1[:, :, 0] + dt * rp1.reshape(J, J, E, N1) / scale   # (34a)
                self.res1[:, :, 1] = a * self.res1[:, :, 1] + dt * rU1[:, 0].reshape(J, J, E, N1)
                pstar = self.qlin[:, :, 0] - self._edge_sum(*self.q0_tri)
                pstar = pstar + b * self.res1[:, :, 0]
                self.qlin[:, :, 1] = self.qlin[:, :, 1] + b * self.res1[:, :, 1]
                self._close_edge(pstar)
                # 0D update kernel (Alg. 5)
                self._close_corner()

    def get_fields(self):
        """same layout as OracleSolver.get_fields"""
        J = self.J
        face_aux = np.transpose(self.qtri, (2, 0, 1, 3)).copy()
        edge_aux = np.transpose(self.qlin.reshape(J * J, 2, self.E, self.N + 1), (2, 0, 1, 3)).copy()
        return self.q.copy(), face_aux, edge_aux
