"""ORACLE (test infrastructure) — mesh hierarchy of the multidimensional solver (§3.2):

  volume mesh  K^tet tetrahedra,
  surface mesh K^tri = the cell faces lying on domain faces that carry the HABC,
  line mesh    K^lin = the cell edges lying on domain edges where two HABC faces cross,
  K^pnt corners where three HABC faces cross,

with F_bnd^tet = K^tri, F_bnd^tri = 2 K^lin, F_bnd^lin = 3 K^pnt (L487).  Everything here is geometry and
bookkeeping: faces are matched by sorted vertex ids, nodes are matched by brute-force coordinate
comparison (DESIGN.md §3 O3).  Geometric factors for affine simplices follow [42].

Boundary-condition codes (per domain face; 'habc' is the product's only mode, the others are oracle test
hooks used by the pins P5/P6/P8):
    BC_INT = 0 interior, BC_HABC = 1 incoming characteristic supplied by the level below,
    BC_DIRICHLET = 2 (p = 0, L516-518), BC_RIGID = 3 (n.u = 0, mirror state).
"""
from __future__ import annotations

import dataclasses

import numpy as np

from .refelem import RefElem, make_refelem

BC_INT, BC_HABC, BC_DIRICHLET, BC_RIGID = 0, 1, 2, 3
_BC_CODE = {"habc": BC_HABC, "dirichlet": BC_DIRICHLET, "rigid": BC_RIGID}

# local vertex lists of the faces of the reference tet / triangle / line, in the order of RefElem.Fmask
TET_FACE_VERTS = ((0, 1, 2), (0, 1, 3), (1, 2, 3), (0, 2, 3))
TRI_FACE_VERTS = ((0, 1), (1, 2), (0, 2))


@dataclasses.dataclass
class Level:
    """One DG level (dim = 3, 2 or 1) with everything `solver.dg_rhs` needs."""
    dim: int
    ref: RefElem
    K: int
    x: np.ndarray          # [K, Np, 3] physical node coordinates
    axes: np.ndarray       # [K, dim] Cartesian axes spanned by the element (3D: 0,1,2)
    G: np.ndarray          # [K, dim_ref, dim] G[k,a,d] = d(ref coordinate a)/d(x_axes[k,d])
    detJ: np.ndarray       # [K] |det| of the affine map
    n: np.ndarray          # [K, Nfaces, dim] outward unit normals (components along `axes`)
    Fs: np.ndarray         # [K, Nfaces] surface Jacobian / volume Jacobian
    vmapM: np.ndarray      # [K, Nfaces*Nfp] flattened own node index k*Np + n
    vmapP: np.ndarray      # [K, Nfaces*Nfp] flattened neighbour node index (own index on a boundary)
    EToE: np.ndarray       # [K, Nfaces] neighbour element (own on a boundary)
    bc: np.ndarray         # [K, Nfaces] BC_* code
    bslot: np.ndarray      # [K, Nfaces*Nfp] slot in the level's incoming-characteristic array (-1 if none)
    rho: np.ndarray        # [K]
    c: np.ndarray          # [K]


@dataclasses.dataclass
class Hierarchy:
    N: int
    tet: Level
    tri: Level | None
    lin: Level | None
    # surface mesh
    tri_tet: np.ndarray      # [T] parent tetrahedron
    tri_face: np.ndarray     # [T] local face of the parent
    tri_axis: np.ndarray     # [T] axis of the domain face normal
    tri_sign: np.ndarray     # [T] +-1 outward sign
    tri_tetnode: np.ndarray  # [T, Nfp] flattened tet node index of each triangle node
    # line mesh
    lin_axis: np.ndarray     # [E] tangent axis
    lin_ab: np.ndarray       # [E, 2] normal axes (a < b) of the two faces A, B
    lin_sign: np.ndarray     # [E, 2] outward signs of faces A, B
    lin_tri: np.ndarray      # [E, 2] parent triangles on faces A and B
    lin_trinode: np.ndarray  # [E, 2, N+1] flattened triangle node index of each line node (faces A, B)
    # corners
    cor_vertex: np.ndarray   # [C] vertex id
    cor_line: np.ndarray     # [C, 3] line along x, y, z meeting at the corner
    cor_end: np.ndarray      # [C, 3] which end (0: r=-1, 1: r=+1) of that line
    cor_sign: np.ndarray     # [C, 3] outward sign along x, y, z


def _affine_nodes(ref: RefElem, V):
    """x = sum_k lambda_k(r) V_k for simplex vertices V [K, dim+1, 3]; lambda from the reference coords."""
    rst = ref.rst
    lam0 = -(np.sum(rst, axis=1) + (ref.dim - 2)) / 2.0          # 1D: (1-r)/2; 2D: -(r+s)/2; 3D: -(1+r+s+t)/2
    lams = [lam0] + [(1.0 + rst[:, d]) / 2.0 for d in range(ref.dim)]
    lam = np.stack(lams, axis=1)                                   # [Np, dim+1]
    return np.einsum("nv,kvd->knd", lam, V)


def _geometry(ref: RefElem, Vin):
    """Vin [K, dim+1, dim] in-plane vertex coordinates.  Returns G, |detJ|, normals, Fscale ([42] ch. 3/6/10)."""
    dim = ref.dim
    # Jm[k, d, a] = d x_d / d ref_a = (V_{a+1} - V_0)_d / 2
    Jm = np.stack([(Vin[:, a + 1, :] - Vin[:, 0, :]) / 2.0 for a in range(dim)], axis=2)
    det = np.linalg.det(Jm)
    G = np.linalg.inv(Jm)                                          # G[k, a, d] = d ref_a / d x_d
    nvec = np.einsum("fa,kad->kfd", ref.nhat, G)                   # grad of the face's level set
    mag = np.linalg.norm(nvec, axis=2)
    return G, np.abs(det), nvec / mag[:, :, None], mag            # Fscale = sJ/|J| = |nvec|


def _match_nodes(xa, xb, tol):
    """For each row of xa [F, n, 3] the index in xb [F, n, 3] of the coincident point (brute force)."""
    out = np.empty(xa.shape[:2], dtype=np.int64)
    step = max(1, 4_000_000 // (xa.shape[1] ** 2))
    for s in range(0, xa.shape[0], step):
        d = np.abs(xa[s:s + step, :, None, :] - xb[s:s + step, None, :, :]).max(axis=3)
        idx = np.argmin(d, axis=2)
        assert np.all(np.take_along_axis(d, idx[:, :, None], axis=2) < tol), "node matching failed"
        out[s:s + step] = idx
    return out


def _pair_faces(keys):
    """keys [F, m] sorted vertex ids (+ optional group id).  Returns partner[F] (own index if unmatched)."""
    F = keys.shape[0]
    order = np.lexsort(keys.T[::-1])
    ks = keys[order]
    same = np.all(ks[1:] == ks[:-1], axis=1)
    partner = np.arange(F)
    a, b = order[:-1][same], order[1:][same]
    partner[a], partner[b] = b, a
    # a key may appear at most twice
    if same.size > 1:
        assert not np.any(same[1:] & same[:-1]), "non-manifold mesh"
    return partner


def build_hierarchy(verts, tets, N: int, c, rho, face_bc=None) -> Hierarchy:
    """verts [nv,3], tets [K,4] positively oriented, c/rho [K].  face_bc: {(axis, sign): 'habc'|'dirichlet'|
    'rigid'} for the six domain faces (default: 'habc' everywhere)."""
    verts = np.asarray(verts, dtype=np.float64)
    tets = np.asarray(tets, dtype=np.int64)
    c = np.asarray(c, dtype=np.float64)
    rho = np.asarray(rho, dtype=np.float64)
    K = tets.shape[0]
    lo, hi = verts.min(axis=0), verts.max(axis=0)
    size = float((hi - lo).max())
    tol = 1e-9 * size
    bc_of = {(a, s): "habc" for a in range(3) for s in (-1, 1)}
    if face_bc:
        bc_of.update(face_bc)

    def on_plane(xyz):
        """[..., 3] -> (axis mask for the low planes, for the high planes)"""
        return np.abs(xyz - lo) < tol, np.abs(xyz - hi) < tol

    # ------------------------------------------------------------------ 3D level
    r3 = make_refelem(3, N)
    Np, Nfp = r3.Np, r3.Nfp
    V = verts[tets]                                                # [K,4,3]
    x3 = _affine_nodes(r3, V)
    G3, det3, n3, Fs3 = _geometry(r3, V)
    assert np.all(np.linalg.det(np.stack([(V[:, a + 1] - V[:, 0]) / 2 for a in range(3)], axis=2)) > 0)
    fv = np.stack([tets[:, list(f)] for f in TET_FACE_VERTS], axis=1)   # [K,4,3]
    partner = _pair_faces(np.sort(fv.reshape(-1, 3), axis=1))
    kk, ff = np.divmod(np.arange(4 * K), 4)
    nodeid = (kk[:, None] * Np + r3.Fmask[ff]).reshape(K, 4 * Nfp)     # vmapM
    xf = x3.reshape(-1, 3)[nodeid.reshape(4 * K, Nfp)]                  # [4K, Nfp, 3]
    perm = _match_nodes(xf, xf[partner], tol)
    vmapP3 = np.take_along_axis(nodeid.reshape(4 * K, Nfp)[partner], perm, axis=1).reshape(K, 4 * Nfp)
    EToE3 = (partner // 4).reshape(K, 4)
    isb = (partner == np.arange(4 * K))
    bc3 = np.zeros(4 * K, dtype=np.int64)
    b_idx = np.nonzero(isb)[0]
    # domain face of every boundary cell face
    fx = verts[fv.reshape(-1, 3)[b_idx]]                                # [B,3,3]
    lo_m, hi_m = on_plane(fx)
    b_axis = np.full(b_idx.size, -1)
    b_sign = np.zeros(b_idx.size, dtype=np.int64)
    for a in range(3):
        m = lo_m[:, :, a].all(axis=1)
        b_axis[m], b_sign[m] = a, -1
        m = hi_m[:, :, a].all(axis=1)
        b_axis[m], b_sign[m] = a, 1
    assert np.all(b_axis >= 0), "boundary cell face not on a plane of the bounding box (non-cuboid domain)"
    for q, (a, s) in enumerate(zip(b_axis, b_sign)):
        bc3[b_idx[q]] = _BC_CODE[bc_of[(int(a), int(s))]]
    habc = bc3[b_idx] == BC_HABC
    t_idx = b_idx[habc]                                                 # flattened (k,f) of each triangle
    T = t_idx.size
    bslot3 = np.full((4 * K, Nfp), -1, dtype=np.int64)
    bslot3[t_idx] = np.arange(T)[:, None] * Nfp + np.arange(Nfp)[None, :]
    tet = Level(dim=3, ref=r3, K=K, x=x3, axes=np.tile(np.arange(3), (K, 1)), G=G3, detJ=det3, n=n3, Fs=Fs3,
                vmapM=nodeid, vmapP=vmapP3, EToE=EToE3, bc=bc3.reshape(K, 4), bslot=bslot3.reshape(K, 4 * Nfp),
                rho=rho, c=c)
    tri_tet, tri_face = t_idx // 4, t_idx % 4
    tri_axis, tri_sign = b_axis[habc], b_sign[habc]
    tri_tetnode = nodeid.reshape(4 * K, Nfp)[t_idx]
    empty = np.zeros((0,), dtype=np.int64)
    if T == 0:
        return Hierarchy(N=N, tet=tet, tri=None, lin=None, tri_tet=tri_tet, tri_face=tri_face, tri_axis=tri_axis,
                         tri_sign=tri_sign, tri_tetnode=tri_tetnode, lin_axis=empty, lin_ab=np.zeros((0, 2), int),
                         lin_sign=np.zeros((0, 2), int), lin_tri=np.zeros((0, 2), int),
                         lin_trinode=np.zeros((0, 2, N + 1), int), cor_vertex=empty, cor_line=np.zeros((0, 3), int),
                         cor_end=np.zeros((0, 3), int), cor_sign=np.zeros((0, 3), int))

    # ------------------------------------------------------------------ 2D level (surface mesh)
    r2 = make_refelem(2, N)
    N1 = N + 1
    tv = fv.reshape(-1, 3)[t_idx]                                       # [T,3] vertex ids, tet-face order
    axes2 = np.array([[d for d in range(3) if d != a] for a in tri_axis])   # in-plane axes, increasing
    Vt = verts[tv]                                                      # [T,3,3]
    Vin2 = np.take_along_axis(Vt, axes2[:, None, :], axis=2)            # [T,3,2]
    x2 = _affine_nodes(r2, Vt)
    assert np.abs(x2 - x3.reshape(-1, 3)[tri_tetnode]).max() < tol      # triangle nodes = tet face nodes (L489)
    G2, det2, n2, Fs2 = _geometry(r2, Vin2)
    ev = np.stack([tv[:, list(e)] for e in TRI_FACE_VERTS], axis=1)     # [T,3,2]
    dface = (tri_axis * 2 + (tri_sign > 0)).astype(np.int64)           # domain face id 0..5
    key2 = np.concatenate([np.sort(ev.reshape(-1, 2), axis=1), np.repeat(dface, 3)[:, None]], axis=1)
    partner2 = _pair_faces(key2)
    tt, ee = np.divmod(np.arange(3 * T), 3)
    nodeid2 = (tt[:, None] * Nfp + r2.Fmask[ee]).reshape(T, 3 * N1)
    xe = x2.reshape(-1, 3)[nodeid2.reshape(3 * T, N1)]
    perm2 = _match_nodes(xe, xe[partner2], tol)
    vmapP2 = np.take_along_axis(nodeid2.reshape(3 * T, N1)[partner2], perm2, axis=1).reshape(T, 3 * N1)
    isb2 = partner2 == np.arange(3 * T)
    bc2 = np.zeros(3 * T, dtype=np.int64)
    bslot2 = np.full((3 * T, N1), -1, dtype=np.int64)
    # every unmatched triangle edge lies on a domain edge: find the other domain face it belongs to
    e_idx = np.nonzero(isb2)[0]
    ex = verts[ev.reshape(-1, 2)[e_idx]]                                # [B2,2,3]
    lo_e, hi_e = on_plane(ex)
    other = []                                                          # (axis, sign) of the other face
    for q, g in enumerate(e_idx):
        a_own = tri_axis[g // 3]
        cand = [(a, -1) for a in range(3) if a != a_own and lo_e[q, :, a].all()] + \
               [(a, 1) for a in range(3) if a != a_own and hi_e[q, :, a].all()]
        assert len(cand) == 1, "triangle edge without neighbour is not on a domain edge"
        other.append(cand[0])
        bc2[g] = _BC_CODE[bc_of[cand[0]]]
    # ------------------------------------------------------------------ 1D level (line mesh)
    lines = {}                                                          # sorted vertex pair -> line id
    lin_v, lin_ab, lin_sign, lin_tri, lin_te = [], [], [], [], []
    for q, g in enumerate(e_idx):
        if bc2[g] != BC_HABC:
            continue
        t = g // 3
        own, oth = (int(tri_axis[t]), int(tri_sign[t])), other[q]
        key = tuple(sorted(ev.reshape(-1, 2)[g]))
        side = 0 if own[0] < oth[0] else 1                              # face A has the lower normal axis
        if key not in lines:
            lines[key] = len(lin_v)
            tang = 3 - own[0] - oth[0]
            v0, v1 = key if verts[key[0], tang] < verts[key[1], tang] else key[::-1]
            lin_v.append((v0, v1))
            A, B = (own, oth) if side == 0 else (oth, own)
            lin_ab.append((A[0], B[0]))
            lin_sign.append((A[1], B[1]))
            lin_tri.append([-1, -1])
            lin_te.append([-1, -1])
        ell = lines[key]
        lin_tri[ell][side] = t
        lin_te[ell][side] = g
    E = len(lin_v)
    tri = Level(dim=2, ref=r2, K=T, x=x2, axes=axes2, G=G2, detJ=det2, n=n2, Fs=Fs2, vmapM=nodeid2, vmapP=vmapP2,
                EToE=(partner2 // 3).reshape(T, 3), bc=bc2.reshape(T, 3), bslot=bslot2.reshape(T, 3 * N1),
                rho=rho[tri_tet], c=c[tri_tet])
    if E == 0:
        return Hierarchy(N=N, tet=tet, tri=tri, lin=None, tri_tet=tri_tet, tri_face=tri_face, tri_axis=tri_axis,
                         tri_sign=tri_sign, tri_tetnode=tri_tetnode, lin_axis=empty, lin_ab=np.zeros((0, 2), int),
                         lin_sign=np.zeros((0, 2), int), lin_tri=np.zeros((0, 2), int),
                         lin_trinode=np.zeros((0, 2, N1), int), cor_vertex=empty, cor_line=np.zeros((0, 3), int),
                         cor_end=np.zeros((0, 3), int), cor_sign=np.zeros((0, 3), int))
    r1 = make_refelem(1, N)
    lin_v = np.array(lin_v)
    lin_ab = np.array(lin_ab)
    lin_sign = np.array(lin_sign)
    lin_tri = np.array(lin_tri)
    lin_te = np.array(lin_te)
    assert np.all(lin_tri >= 0), "a line cell must have one parent triangle on each of its two faces (L487)"
    lin_axis = 3 - lin_ab[:, 0] - lin_ab[:, 1]
    Vl = verts[lin_v]                                                   # [E,2,3]
    x1 = _affine_nodes(r1, Vl)
    Vin1 = np.take_along_axis(Vl, lin_axis[:, None, None], axis=2)      # [E,2,1]
    G1, det1, n1, Fs1 = _geometry(r1, Vin1)
    # line node <-> triangle node maps, and the triangles' boundary slots: r^- array of the tri level is
    # indexed [line, side, node]  (slot = (ell*2 + side)*N1 + m)
    lin_trinode = np.empty((E, 2, N1), dtype=np.int64)
    for side in range(2):
        g = lin_te[:, side]
        ids = nodeid2.reshape(3 * T, N1)[g]                             # triangle-edge nodes, flattened ids
        pm = _match_nodes(x1, x2.reshape(-1, 3)[ids], tol)              # line node m -> position on the edge
        lin_trinode[:, side] = np.take_along_axis(ids, pm, axis=1)
        inv = _match_nodes(x2.reshape(-1, 3)[ids], x1, tol)             # triangle-edge node -> line node
        bslot2[g] = (np.arange(E)[:, None] * 2 + side) * N1 + inv
    tri.bslot = bslot2.reshape(T, 3 * N1)
    # line connectivity along each domain edge
    dedge = lin_ab[:, 0] * 16 + lin_ab[:, 1] * 4 + (lin_sign[:, 0] > 0) * 2 + (lin_sign[:, 1] > 0)
    key1 = np.stack([lin_v.reshape(-1), np.repeat(dedge, 2)], axis=1)   # end e of line ell -> row 2*ell+e
    partner1 = _pair_faces(key1)
    nodeid1 = (np.arange(E)[:, None] * N1 + r1.Fmask[:, 0][None, :])    # [E,2]
    vmapP1 = nodeid1.reshape(-1)[partner1].reshape(E, 2)
    isb1 = partner1 == np.arange(2 * E)
    bc1 = np.zeros(2 * E, dtype=np.int64)
    bslot1 = np.full(2 * E, -1, dtype=np.int64)
    corners = {}
    cor_vertex, cor_line, cor_end, cor_sign = [], [], [], []
    for g in np.nonzero(isb1)[0]:
        ell, e = divmod(int(g), 2)
        v = int(lin_v[ell, e])
        tang = int(lin_axis[ell])
        s = -1 if abs(verts[v, tang] - lo[tang]) < tol else 1
        assert abs(verts[v, tang] - (lo[tang] if s < 0 else hi[tang])) < tol, "line end is not at a corner"
        kind = bc_of[(tang, s)]
        bc1[g] = _BC_CODE[kind]
        if kind != "habc":
            continue
        if v not in corners:
            corners[v] = len(cor_vertex)
            cor_vertex.append(v)
            cor_line.append([-1, -1, -1])
            cor_end.append([-1, -1, -1])
            cor_sign.append([0, 0, 0])
        cid = corners[v]
        cor_line[cid][tang], cor_end[cid][tang], cor_sign[cid][tang] = ell, e, s
        bslot1[g] = cid * 3 + tang              # r^- array of the line level is indexed [corner, axis] (per set)
    lin = Level(dim=1, ref=r1, K=E, x=x1, axes=lin_axis[:, None], G=G1, detJ=det1, n=n1, Fs=Fs1, vmapM=nodeid1,
                vmapP=vmapP1, EToE=(partner1 // 2).reshape(E, 2), bc=bc1.reshape(E, 2), bslot=bslot1.reshape(E, 2),
                rho=tri.rho[lin_tri[:, 0]], c=tri.c[lin_tri[:, 0]])
    cor_line = np.array(cor_line).reshape(-1, 3)
    assert np.all(cor_line >= 0), "a corner must be the end of three line cells (L487)"
    return Hierarchy(N=N, tet=tet, tri=tri, lin=lin, tri_tet=tri_tet, tri_face=tri_face, tri_axis=tri_axis,
                     tri_sign=tri_sign, tri_tetnode=tri_tetnode, lin_axis=lin_axis, lin_ab=lin_ab, lin_sign=lin_sign,
                     lin_tri=lin_tri, lin_trinode=lin_trinode, cor_vertex=np.array(cor_vertex, dtype=np.int64),
                     cor_line=cor_line, cor_end=np.array(cor_end).reshape(-1, 3),
                     cor_sign=np.array(cor_sign).reshape(-1, 3))


def count_unknowns(K, T, E, N: int, J: int) -> int:
    """Total number of discrete unknowns, Table 1: Nfields = 4/3/2 and Nsets = 1/J/J^2 for
    the volume / surface / line meshes, Np = (N+1)(N+2)(N+3)/6, (N+1)(N+2)/2, N+1 nodes per cell."""
    Np3, Np2, Np1 = (N + 1) * (N + 2) * (N + 3) // 6, (N + 1) * (N + 2) // 2, N + 1
    return K * 4 * Np3 + T * 3 * J * Np2 + E * 2 * J * J * Np1
