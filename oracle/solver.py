"""ORACLE (test infrastructure) — the DG + HABC time step of arXiv 1610.05023 as a method-of-lines ODE
y' = F(y) integrated by LSRK4(5), in float64 numpy.  Plain and slow on purpose; see oracle/__init__.py.

State y = (q, fa, ea)   (DESIGN.md §3 O4; Table 1: Nfields = 4/3/2, Nsets = 1/J/J^2)
    q  [4, K, Np]            p, u, v, w of the volume solver
    fa [J, 3, T, Nfp]        p*_i00 and the two tangential velocities (in-plane axes in increasing order)
    ea [J, J, 2, E, N+1]     p*_ij0 and the tangential velocity; first index <-> face A (lower normal axis)
F(y) = closure chain (eq (28)-(30), (32)-(33), (35); Algorithm 1) followed by the same nodal-DG
right-hand side on every level (eq (37)-(41) L493-529, (31a-c) L392-396, (34a-b) L439-441).
Readings R1..R16 of DESIGN.md §3 apply; in particular r^± = (p ± rho c n.u)/2 (R1).
"""
from __future__ import annotations

import numpy as np

from . import habc
from .mesh import BC_DIRICHLET, BC_HABC, BC_INT, BC_RIGID, Hierarchy, Level, build_hierarchy

# LSRK4(5) of Carpenter & Kennedy, ref. [10] of the paper (coefficients not printed there,
# pinned by the order conditions in tests/test_oracle_refelem_habc.py::test_lsrk_order_conditions)
RK4A = np.array([0.0,
                 -567301805773.0 / 1357537059087.0,
                 -2404267990393.0 / 2016746695238.0,
                 -3550918686646.0 / 2091501179385.0,
                 -1275806237668.0 / 842570457699.0])
RK4B = np.array([1432997174477.0 / 9575080441755.0,
                 5161836677717.0 / 13612068292357.0,
                 1720146321549.0 / 2090206949498.0,
                 3134564353537.0 / 4481467310338.0,
                 2277821191437.0 / 14882151754819.0])
RK4C = np.array([0.0,
                 1432997174477.0 / 9575080441755.0,
                 2526269341429.0 / 6820363962896.0,
                 2006345519317.0 / 3224310063776.0,
                 2802321613138.0 / 2924317926251.0])


def dg_rhs(L: Level, p, U, rminus):
    """Nodal DG right-hand side of the pressure-velocity system on one level, strong form of (37),(38).

    p [S, K, Np], U [S, dim, K, Np] (velocity components along L.axes), rminus [S, nslots] incoming
    characteristics for the BC_HABC faces.  Returns (rhs_p, rhs_U) of the same shapes:
        rhs_p = -rho c^2 div U   - LIFT[ Fs (rho c^2)^int ((n.u)* - n.u^int) ]
        rhs_U = -(1/rho) grad p  - LIFT[ Fs (1/rho^int) (p* - p^int) n ]
    with the upwind fluxes of L499-518.
    """
    ref = L.ref
    S = p.shape[0]
    dim, K, Np = L.dim, L.K, ref.Np
    nfn = ref.Nfaces * ref.Nfp
    rho, c = L.rho, L.c
    Z = rho * c
    # ---- volume term: physical derivatives d/dx_d = sum_a G[k,a,d] D_a
    Dp = [np.einsum("nm,skm->skn", ref.D[a], p) for a in range(dim)]
    grad = [sum(L.G[None, :, a, d, None] * Dp[a] for a in range(dim)) for d in range(dim)]
    div = np.zeros_like(p)
    for d in range(dim):
        for a in range(dim):
            div += L.G[None, :, a, d, None] * np.einsum("nm,skm->skn", ref.D[a], U[:, d])
    # ---- traces
    pf = p.reshape(S, K * Np)
    Uf = U.reshape(S, dim, K * Np)
    pM, pP = pf[:, L.vmapM], pf[:, L.vmapP]                          # [S,K,nfn]
    nrm = np.repeat(L.n, ref.Nfp, axis=1)                            # [K,nfn,dim]
    unM = sum(nrm[None, :, :, d] * Uf[:, d][:, L.vmapM] for d in range(dim))
    unP = sum(nrm[None, :, :, d] * Uf[:, d][:, L.vmapP] for d in range(dim))
    ZM = Z[:, None] * np.ones((1, nfn))
    ZP = np.repeat(Z[L.EToE], ref.Nfp, axis=1)
    bc = np.repeat(L.bc, ref.Nfp, axis=1)                            # [K,nfn]
    # interior: exact Riemann solver, L499-502 ({X} = (X+ + X-)/2, [[X]] = (X+ - X-)/2)
    avg_p_over_Z = 0.5 * (pP / ZP + pM / ZM)
    avg_inv_Z = 0.5 * (1.0 / ZP + 1.0 / ZM)
    jump_un = 0.5 * (unP - unM)
    pstar = (avg_p_over_Z - jump_un) / avg_inv_Z
    avg_Zun = 0.5 * (ZP * unP + ZM * unM)
    jump_p = 0.5 * (pP - pM)
    avg_Z = 0.5 * (ZP + ZM)
    unstar = (avg_Zun - jump_p) / avg_Z
    # characteristic boundary, (39),(40) with r^+ from the interior trace and r^- supplied, L504-514
    m = bc == BC_HABC
    if m.any():
        rp = 0.5 * (pM + ZM * unM)
        rm = np.zeros_like(pM)
        rm[:, m] = rminus[:, L.bslot[m]]
        pstar = np.where(m, rp + rm, pstar)
        unstar = np.where(m, (rp - rm) / ZM, unstar)
    m = bc == BC_DIRICHLET                                           # L516-518
    if m.any():
        pstar = np.where(m, 0.0, pstar)
        unstar = np.where(m, unM + pM / ZM, unstar)
    m = bc == BC_RIGID                                               # mirror state: p+ = p-, n.u+ = -n.u-
    if m.any():
        pstar = np.where(m, pM + ZM * unM, pstar)
        unstar = np.where(m, 0.0, unstar)
    Fs = np.repeat(L.Fs, ref.Nfp, axis=1)                            # [K,nfn]
    flux_p = Fs * (rho * c * c)[:, None] * (unstar - unM)
    flux_pu = Fs * (1.0 / rho)[:, None] * (pstar - pM)
    rhs_p = -(rho * c * c)[None, :, None] * div - np.einsum("nj,skj->skn", ref.LIFT, flux_p)
    rhs_U = np.empty_like(U)
    for d in range(dim):
        rhs_U[:, d] = -(1.0 / rho)[None, :, None] * grad[d] \
            - np.einsum("nj,skj->skn", ref.LIFT, flux_pu * nrm[None, :, :, d])
    return rhs_p, rhs_U


class OracleSolver:
    """dg_create / dg_set_initial / dg_step / dg_get_fields of the boundary, computed the slow way."""

    def __init__(self, verts, tets, N: int, J: int, c, rho, cfl: float = 1.0, dt: float | None = None,
                 face_bc=None):
        self.N, self.J = N, J
        self.H: Hierarchy = build_hierarchy(verts, tets, N, c, rho, face_bc)
        H = self.H
        self.M, self.cn = habc.pade_coefficients(J)
        self.T = H.tri.K if (H.tri is not None and J > 0) else 0
        self.E = H.lin.K if (H.lin is not None and J > 0) else 0
        self.C = H.cor_vertex.size if J > 0 else 0
        if J > 0:
            self.Le, self.Te, self.Ba, self.Bb = habc.edge_system(J)
            self.Lc, self.Tc = habc.corner_system(J)
        # eq (46), reading R7: dt = cfl * min_k 1 / (c_k (N+1)^2 Fscale_k), Fscale_k = max_f sJ_f/J_k
        self.dt = float(dt) if dt else cfl * float(np.min(1.0 / (H.tet.c * (N + 1) ** 2 * H.tet.Fs.max(axis=1))))
        self._verts, self._tets = np.asarray(verts, dtype=np.float64), np.asarray(tets)
        self.source = None
        self.set_initial(np.zeros((4, H.tet.K, H.tet.ref.Np)))

    # ------------------------------------------------------------------ state
    def nodes(self):
        return self.H.tet.x

    def set_initial(self, q):
        """q [4,K,Np]; all auxiliary ODE state is zero (reading R5)."""
        H, J = self.H, self.J
        self.q = np.array(q, dtype=np.float64).reshape(4, H.tet.K, H.tet.ref.Np)
        self.fa = np.zeros((J, 3, self.T, H.tet.ref.Nfp))
        self.ea = np.zeros((J, J, 2, self.E, self.N + 1))
        self.res = None
        self.t = 0.0

    # ------------------------------------------------------------------ point source (eq (44))
    def set_source(self, xs, f_peak: float, t_s: float, amplitude: float = 1.0):
        """Dirac source delta(x - xs) * amplitude * S(t) in the pressure equation (L780), S(t) = (t - t_s)
        exp(-pi^2 f_peak^2 (t - t_s)^2) the integral of the Ricker wavelet (44) (L784).  Galerkin projection onto
        the cell that contains xs (the first one in the caller's order whose barycentric coordinates are all
        >= -1e-12):  M J dp/dt = ... + l(xs) S  =>  dp_n/dt += S (M^-1 l(r_s))_n / J,  M^-1 l(r) = V psi(r)."""
        xs = np.asarray(xs, dtype=np.float64)
        V4 = self._verts[self._tets]                                     # [K,4,3]
        A = np.transpose(V4[:, 1:] - V4[:, :1], (0, 2, 1))               # columns = edge vectors
        lam = np.linalg.solve(A, np.broadcast_to(xs - V4[:, 0], (len(V4), 3))[..., None])[..., 0]
        bary = np.concatenate([1.0 - lam.sum(axis=1, keepdims=True), lam], axis=1)
        inside = np.nonzero(bary.min(axis=1) >= -1e-12)[0]
        if inside.size == 0:
            raise ValueError("the source point is outside the mesh")
        k = int(inside[0])
        r, s_, t_ = (-1.0 + 2.0 * bary[k, 1 + a] for a in range(3))
        from .refelem import vandermonde
        LD = np.longdouble
        psi, _ = vandermonde(3, self.N, np.array([r], dtype=LD), np.array([s_], dtype=LD), np.array([t_], dtype=LD))
        w = (self.H.tet.ref.V @ np.asarray(psi[0], dtype=np.float64)) / self.H.tet.detJ[k]
        self.source = dict(k=k, w=w, f=float(f_peak), ts=float(t_s), amp=float(amplitude))

    def source_S(self, t):
        src = self.source
        tau = t - src["ts"]
        return src["amp"] * tau * np.exp(-(np.pi * src["f"] * tau) ** 2)

    def state(self):
        return (self.q, self.fa, self.ea)

    # ------------------------------------------------------------------ closure chain (DESIGN.md §3 O5)
    def closures(self, y):
        q, fa, ea = y
        H, J, M, cn = self.H, self.J, self.M, self.cn
        if H.tri is None:
            return {"rm_tet": np.zeros((1, 1))}
        Ttot = H.tri.K
        out = {"rm_tet": np.zeros((1, Ttot * H.tet.ref.Nfp))}
        # 1. face: r^+ from the 3D trace, r^- by (30), S = r^- + r^+, p_i00 = p*_i00 + S  (29)
        ids = H.tri_tetnode
        pt = q[0].reshape(-1)[ids]
        un = np.zeros_like(pt)
        for a in range(3):
            m = H.tri_axis == a
            un[m] = q[1 + a].reshape(-1)[ids[m]] * H.tri_sign[m, None]
        Zt = (H.tri.rho * H.tri.c)[:, None]
        rp = 0.5 * (pt + Zt * un)
        if J == 0:
            return out                                    # r^- = 0: the basic ABC (L514)
        rm = np.tensordot(cn, fa[:, 0], axes=(0, 0)) / M                  # (30)
        Sf = rp + rm
        p_face = fa[:, 0] + Sf[None]
        out.update(rm_tet=rm.reshape(1, -1), S_face=Sf, p_face=p_face)
        out["rm_tri"] = np.zeros((J, max(self.E, 1) * 2 * (self.N + 1)))
        if H.lin is None:
            return out
        E, N1 = self.E, self.N + 1
        # 2. edge: outgoing characteristics of both faces' 2D fields across the edge
        vel = fa[:, 1:3].reshape(J, 2, Ttot * H.tet.ref.Nfp)
        rplus = []
        for side in range(2):
            ids = H.lin_trinode[:, side]                                   # [E,N1] flattened triangle nodes
            t = H.lin_tri[:, side]
            oth_axis, oth_sign = H.lin_ab[:, 1 - side], H.lin_sign[:, 1 - side]
            slot = np.array([list(H.tri.axes[t[e]]).index(oth_axis[e]) for e in range(E)])
            ps = p_face.reshape(J, -1)[:, ids]                             # [J,E,N1]
            us = np.where((slot == 0)[None, :, None], vel[:, 0][:, ids], vel[:, 1][:, ids]) * oth_sign[None, :, None]
            Zs = (H.tri.rho * H.tri.c)[t][None, :, None]
            rplus.append(0.5 * (ps + Zs * us))
        rpb, rpa = rplus                                                   # face A gives r^{+b}_i, face B r^{+a}_j
        pst = ea[:, :, 0].reshape(J * J, E * N1)
        rpl = np.concatenate([rpa.reshape(J, -1), rpb.reshape(J, -1)], axis=0)     # ordering of habc.edge_system
        bvec = np.concatenate([self.Ba @ pst, self.Bb @ pst], axis=0)
        sol = np.linalg.solve(self.Le, bvec + self.Te @ rpl)               # (33a-b)
        rma, rmb = sol[:J].reshape(J, E, N1), sol[J:].reshape(J, E, N1)
        Sa, Sb = rma + rpa, rmb + rpb                                      # S^a_j, S^b_i
        p_edge = np.empty((J, J, E, N1))
        for i in range(J):
            for j in range(J):
                p_edge[i, j] = ea[i, j, 0] + habc.C2(cn, j, i) * Sb[i] + habc.C2(cn, i, j) * Sa[j]    # (32)
        rm_tri = np.stack([rmb, rma], axis=2)                              # [J,E,side,N1]: side A <- r^{-b}_i
        out.update(rm_tri=rm_tri.reshape(J, -1), S_a=Sa, S_b=Sb, p_edge=p_edge)
        out["rm_lin"] = np.zeros((J * J, max(self.C, 1) * 3))
        if self.C == 0:
            return out
        # 3. corner: outgoing characteristics of the three edges' 1D fields, 3J^2 system (35a-c)
        C = self.C
        rp3 = np.empty((3, J, J, C))
        for d in range(3):
            ell, e, s = H.cor_line[:, d], H.cor_end[:, d], H.cor_sign[:, d]
            node = np.where(e == 0, 0, N1 - 1)
            pe = p_edge[:, :, ell, node]
            we = ea[:, :, 1, ell, node]
            Zl = (H.lin.rho * H.lin.c)[ell]
            rp3[d] = 0.5 * (pe + Zl * s * we)
        solc = np.linalg.solve(self.Lc, self.Tc @ rp3.reshape(3 * J * J, C))
        rm3 = solc.reshape(3, J * J, C)
        out["rm_lin"] = np.transpose(rm3, (1, 2, 0)).reshape(J * J, C * 3)     # slot = corner*3 + axis
        out["rp_cor"] = rp3
        return out

    # ------------------------------------------------------------------ F(y)
    def rhs(self, y, t=None):
        """F(y) (autonomous), plus the point source evaluated at time t when one is set."""
        q, fa, ea = y
        H, J, cn = self.H, self.J, self.cn
        cl = self.closures(y)
        rp, rU = dg_rhs(H.tet, q[0][None], q[1:4][None], cl["rm_tet"])
        dq = np.concatenate([rp, rU[0]], axis=0)
        if self.source is not None and t is not None:
            dq[0, self.source["k"]] += self.source_S(t) * self.source["w"]
        dfa, dea = np.zeros_like(fa), np.zeros_like(ea)
        if self.T and J:
            rp, rU = dg_rhs(H.tri, cl["p_face"], fa[:, 1:3], cl["rm_tri"])
            dfa[:, 0] = rp / (1.0 + cn)[:, None, None]                      # (31a)
            dfa[:, 1:3] = rU                                               # (31b-c)
        if self.E and J:
            E, N1 = self.E, self.N + 1
            rp, rU = dg_rhs(H.lin, cl["p_edge"].reshape(J * J, E, N1), ea[:, :, 1].reshape(J * J, 1, E, N1),
                            cl["rm_lin"])
            scale = (1.0 + cn[:, None] + cn[None, :]).reshape(J * J, 1, 1)
            dea[:, :, 0] = (rp / scale).reshape(J, J, E, N1)               # (34a)
            dea[:, :, 1] = rU[:, 0].reshape(J, J, E, N1)                   # (34b)
        return (dq, dfa, dea)

    # ------------------------------------------------------------------ LSRK4(5), DESIGN.md §3 O7
    def step(self, nsteps: int = 1):
        y = [self.q, self.fa, self.ea]
        s = [np.zeros_like(a) for a in y]
        for _ in range(nsteps):
            for n in range(5):
                F = self.rhs(tuple(y), self.t + RK4C[n] * self.dt)
                for a in range(3):
                    s[a] = RK4A[n] * s[a] + self.dt * F[a]
                    y[a] = y[a] + RK4B[n] * s[a]
            self.t += self.dt
        self.q, self.fa, self.ea = y

    # ------------------------------------------------------------------ outputs (DESIGN.md §3 O8)
    def get_fields(self):
        """(q [4,K,Np], face_aux [T,J,3,Nfp] physical p_i00 + 2 tangential velocities,
            edge_aux [E,J*J,2,N+1] physical p_ij0 + tangential velocity)."""
        cl = self.closures(self.state())
        J = self.J
        face_aux = np.zeros((self.T, J, 3, self.H.tet.ref.Nfp))
        edge_aux = np.zeros((self.E, J * J, 2, self.N + 1))
        if self.T and J:
            face_aux[:, :, 0] = np.transpose(cl["p_face"], (1, 0, 2))
            face_aux[:, :, 1:3] = np.transpose(self.fa[:, 1:3], (2, 0, 1, 3))
        if self.E and J:
            edge_aux[:, :, 0] = np.transpose(cl["p_edge"].reshape(J * J, self.E, -1), (1, 0, 2))
            edge_aux[:, :, 1] = np.transpose(self.ea[:, :, 1].reshape(J * J, self.E, -1), (1, 0, 2))
        return self.q.copy(), face_aux, edge_aux

    def energy(self, q=None):
        """Discrete acoustic energy, the integrand of (47)."""
        q = self.q if q is None else q
        t = self.H.tet
        Mm = t.ref.M
        ep = np.einsum("kn,nm,km->k", q[0], Mm, q[0]) / (t.rho * t.c ** 2)
        eu = sum(np.einsum("kn,nm,km->k", q[d], Mm, q[d]) for d in (1, 2, 3)) * t.rho
        return 0.5 * float(np.sum(t.detJ * (ep + eu)))

    # ------------------------------------------------------------------ dense F for tiny meshes (pins P6, P10)
    def pack(self, y):
        return np.concatenate([a.reshape(-1) for a in y])

    def unpack(self, v):
        out, o = [], 0
        for a in (self.q, self.fa, self.ea):
            out.append(v[o:o + a.size].reshape(a.shape))
            o += a.size
        return tuple(out)

    def dense_operator(self):
        n = self.q.size + self.fa.size + self.ea.size
        A = np.empty((n, n))
        for j in range(n):
            e = np.zeros(n)
            e[j] = 1.0
            A[:, j] = self.pack(self.rhs(self.unpack(e)))
        return A
