"""Synthetic cuboid workloads shaped like the paper's runs (BASELINE.json `configs`).

Recipe (also stated in DESIGN.md §4):
  * mesh: cube [-1,1]^3 cut into n^3 hexahedra, each split into 6 tetrahedra around the hex diagonal
    (0,0,0)-(1,1,1) (Kuhn/Freudenthal split; the same orientation in every hex makes it conforming),
    every tetrahedron positively oriented; optional seeded perturbation U[-a*h, a*h]^3 of strictly
    interior vertices (boundary vertices stay on their planes).
  * materials: rho = 1; c constant, or piecewise constant per horizontal layer of hexahedra
    (layer index from the hex z-index), speeds drawn from U[lo,hi] with the config's seed.
  * initial data: Gaussian pressure pulse exp(-|x-x0|^2 / (2 w^2)), w = 0.2, seeded centre; optionally a
    superposed plane wave p = A cos(2 pi k.x), u = k p / (rho c) with a seeded unit direction k.
  * "seam": a cuboid with the aspect of the paper's SEAM Phase I run (35 x 40 x 15 km -> 3.5 x 4.0 x 1.5):
    70 x 80 x 30 hexahedra = 1,008,000 tetrahedra (the paper's mesh: 1,179,989), N = 3, J = 3, free surface (p = 0) on
    the top face and HABC on the other five, strongly heterogeneous c and rho (depth gradient 1.5 -> 3.5, a fast
    4.5 inclusion, seeded +-3 % cell-to-cell variation; rho = 1 + (c - 1.5) / 4).  The SEAM model itself is not available.
  * seeds: 1610_05023 + config index, numpy PCG64.
The paper's own meshes (70,895-tet cube, SEAM Phase I model) are not available; these stand in for them.
"""
from __future__ import annotations

import dataclasses
import itertools

import numpy as np

SEED0 = 161005023


@dataclasses.dataclass
class Workload:
    """One fully specified problem instance (inputs only)."""
    name: str
    n: int                      # hexes per side
    N: int                      # polynomial degree (paper's P)
    J: int                      # HABC order (paper's N)
    nsteps: int
    precisions: tuple
    verts: np.ndarray           # [nverts,3] float64
    tets: np.ndarray            # [ntets,4] int32, positively oriented
    c: np.ndarray               # [ntets] float64
    rho: np.ndarray             # [ntets] float64
    pulse_centre: np.ndarray    # [3]
    pulse_width: float
    plane_dir: np.ndarray | None
    plane_amp: float
    seed: int
    shape: tuple = None         # hexes per axis (n, n, n for the cube configs)
    face_bc: dict = None        # {(axis, sign): "dirichlet" | "rigid"} for domain faces without HABC (None: HABC everywhere)

    @property
    def K(self) -> int:
        return int(self.tets.shape[0])

    def fields(self, x, y, z, c_node, rho_node):
        return initial_fields(self, x, y, z, c_node, rho_node)


def cube_mesh(n: int, perturb: float = 0.0, rng: np.random.Generator | None = None):
    """Kuhn 6-tet split of an n^3 hex grid on [-1,1]^3 (see box_mesh)."""
    return box_mesh((n, n, n), ((-1.0, 1.0),) * 3, perturb, rng)


def box_mesh(shape, box, perturb: float = 0.0, rng: np.random.Generator | None = None):
    """Kuhn 6-tet split of an nx x ny x nz hex grid on the cuboid `box` = ((x0,x1),(y0,y1),(z0,z1)).  Element order:
    hex-major (x fastest), the six tets of a hex consecutive.  Returns (verts[nv,3] f64, tets[K,4] i32), all tets
    positively oriented."""
    nx, ny, nz = shape
    gx, gy, gz = (np.linspace(b[0], b[1], m + 1) for b, m in zip(box, shape))
    X, Y, Z = np.meshgrid(gx, gy, gz, indexing="ij")
    verts = np.stack([X.ravel(), Y.ravel(), Z.ravel()], axis=1).astype(np.float64)

    def vid(i, j, k):
        return (i * (ny + 1) + j) * (nz + 1) + k

    if perturb > 0.0:
        assert rng is not None
        h = np.array([(b[1] - b[0]) / m for b, m in zip(box, shape)])
        I, Jx, Kx = np.meshgrid(np.arange(nx + 1), np.arange(ny + 1), np.arange(nz + 1), indexing="ij")
        interior = ((I > 0) & (I < nx) & (Jx > 0) & (Jx < ny) & (Kx > 0) & (Kx < nz)).ravel()
        d = rng.uniform(-perturb, perturb, size=verts.shape) * h
        verts[interior] += d[interior]

    # the six monotone lattice paths (0,0,0)->(1,1,1): one tet per permutation of the axes
    corner_paths = []
    for perm in itertools.permutations(range(3)):
        p = np.zeros(3, dtype=np.int64)
        path = [p.copy()]
        for ax in perm:
            p[ax] += 1
            path.append(p.copy())
        corner_paths.append(np.array(path))            # [4,3]
    corner_paths = np.array(corner_paths)              # [6,4,3]

    kk, jj, ii = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")  # x fastest
    hexes = np.stack([ii.ravel(), jj.ravel(), kk.ravel()], axis=1)                        # [n^3,3]
    cidx = hexes[:, None, None, :] + corner_paths[None, :, :, :]                          # [hexes,6,4,3]
    tets = vid(cidx[..., 0], cidx[..., 1], cidx[..., 2]).reshape(-1, 4)
    # orient positively
    a = verts[tets[:, 1]] - verts[tets[:, 0]]
    b = verts[tets[:, 2]] - verts[tets[:, 0]]
    cvec = verts[tets[:, 3]] - verts[tets[:, 0]]
    det = np.einsum("ij,ij->i", np.cross(a, b), cvec)
    neg = det < 0
    tets[neg, 2], tets[neg, 3] = tets[neg, 3].copy(), tets[neg, 2].copy()
    return verts, tets.astype(np.int32)


def layered_speed(n: int, nlayers: int, lo: float, hi: float, rng: np.random.Generator):
    """c per tetrahedron: `nlayers` horizontal layers of hexahedra (by hex z-index), speeds ~ U[lo,hi]."""
    speeds = rng.uniform(lo, hi, size=nlayers)
    kz = np.repeat(np.arange(n), n * n)                # hex z index for hex-major (x fastest) ordering
    layer = np.minimum((kz * nlayers) // n, nlayers - 1)
    return np.repeat(speeds[layer], 6).astype(np.float64)


def initial_fields(w: Workload, x, y, z, c_node, rho_node):
    """Closed-form initial data at arbitrary points.  c_node/rho_node broadcast against x."""
    x = np.asarray(x, dtype=np.float64)
    x0 = w.pulse_centre
    r2 = (x - x0[0]) ** 2 + (np.asarray(y) - x0[1]) ** 2 + (np.asarray(z) - x0[2]) ** 2
    p = np.exp(-r2 / (2.0 * w.pulse_width ** 2))
    u = np.zeros_like(p)
    v = np.zeros_like(p)
    ww = np.zeros_like(p)
    if w.plane_dir is not None:
        k = w.plane_dir
        pw = w.plane_amp * np.cos(2.0 * np.pi * (k[0] * x + k[1] * y + k[2] * z))
        p = p + pw
        s = pw / (rho_node * c_node)
        u = u + k[0] * s
        v = v + k[1] * s
        ww = ww + k[2] * s
    return p, u, v, ww


SEAM_BOX = ((0.0, 3.5), (0.0, 4.0), (0.0, 1.5))


def seam_shape(n: int):
    """hexes per axis of the SEAM-shaped cuboid with n hexes along x (70 -> 70 x 80 x 30)"""
    return (n, max(1, round(n * 8 / 7)), max(1, round(n * 3 / 7)))


def seam_materials(shape, box, rng: np.random.Generator):
    """(c, rho) per tetrahedron of the SEAM-shaped stand-in: depth gradient + fast inclusion + seeded variation."""
    nx, ny, nz = shape
    cen = [b[0] + (np.arange(m) + 0.5) * (b[1] - b[0]) / m for b, m in zip(box, shape)]
    Zc, Yc, Xc = np.meshgrid(cen[2], cen[1], cen[0], indexing="ij")           # hex-major, x fastest
    L = [b[1] - b[0] for b in box]
    depth = (box[2][1] - Zc) / L[2]
    c = 1.5 + 2.0 * depth
    inside = ((Xc - 0.55 * L[0]) / (0.2 * L[0])) ** 2 + ((Yc - 0.5 * L[1]) / (0.25 * L[1])) ** 2 \
        + ((Zc - 0.45 * L[2]) / (0.25 * L[2])) ** 2 < 1.0
    c = np.where(inside, 4.5, c)
    c = c * (1.0 + 0.03 * rng.uniform(-1.0, 1.0, size=c.shape))
    rho = 1.0 + (c - 1.5) / 4.0
    return np.repeat(c.ravel(), 6).astype(np.float64), np.repeat(rho.ravel(), 6).astype(np.float64)


# name -> static description (BASELINE.json configs[0..4]); config 4 is a sweep, see `sweep`.
CONFIGS = {
    "cfg1": dict(index=1, n=2, N=3, J=2, nsteps=100, precisions=("f64",), c=("const", 1.0),
                 pulse="centre", plane=False, perturb=0.0),
    "cfg2": dict(index=2, n=8, N=4, J=4, nsteps=500, precisions=("f64", "f32"), c=("const", 1.0),
                 pulse="centre", plane=True, perturb=0.0),
    "cfg3": dict(index=3, n=32, N=4, J=6, nsteps=200, precisions=("f64",), c=("layers", 4, 1.0, 3.0),
                 pulse="corner", plane=False, perturb=0.1),
    "cfg4": dict(index=4, n=24, N=4, J=4, nsteps=100, precisions=("f64", "f32"), c=("const", 1.0),
                 pulse="corner", plane=False, perturb=0.0,
                 sweep=dict(N=tuple(range(1, 9)), J=(0, 4, 8))),
    "cfg5": dict(index=5, n=64, N=5, J=8, nsteps=100, precisions=("f64", "f32"),
                 c=("layers", 4, 1.5, 4.5), pulse="corner", plane=False, perturb=0.0),
    # SEAM-shaped workload (not one of BASELINE's five configs; see the module docstring)
    "seam": dict(index=6, n=70, N=3, J=3, nsteps=100, precisions=("f32", "f64"), c=("seam",), pulse="seam",
                 plane=False, perturb=0.0, face_bc={(2, 1): "dirichlet"}),
}


def make_workload(name: str, *, n: int | None = None, N: int | None = None, J: int | None = None,
                  nsteps: int | None = None) -> Workload:
    """Build the named configuration; n/N/J/nsteps override the table (used by the degree sweep of
    cfg4 and by reduced-size variants that keep every other rule of the recipe)."""
    d = CONFIGS[name]
    n = d["n"] if n is None else n
    N = d["N"] if N is None else N
    J = d["J"] if J is None else J
    nsteps = d["nsteps"] if nsteps is None else nsteps
    rng = np.random.default_rng(SEED0 + d["index"])
    if name == "seam":
        shape, box = seam_shape(n), SEAM_BOX
    else:
        shape, box = (n, n, n), ((-1.0, 1.0),) * 3
    verts, tets = box_mesh(shape, box, d["perturb"], rng)
    K = tets.shape[0]
    rho = np.ones(K, dtype=np.float64)
    if d["c"][0] == "const":
        c = np.full(K, d["c"][1], dtype=np.float64)
    elif d["c"][0] == "seam":
        c, rho = seam_materials(shape, box, rng)
    else:
        _, nl, lo, hi = d["c"]
        c = layered_speed(n, nl, lo, hi, rng)
    jitter = rng.uniform(-1.0, 1.0, size=3)
    if d["pulse"] == "centre":
        centre = 0.3 * jitter / max(1.0, np.linalg.norm(jitter))        # |x0| < 0.3
    elif d["pulse"] == "seam":
        # near the bottom (+x, +y, -z) corner: three HABC faces, their edges and a corner carry data from t = 0
        centre = np.array([box[0][1] - 0.3, box[1][1] - 0.3, box[2][0] + 0.3]) + 0.03 * jitter
    else:
        # near the (+,+,+) corner so that faces, edges and one corner carry O(0.1) data at t=0
        # (the stated step counts cover too little time for a central pulse to arrive)
        centre = np.array([0.75, 0.75, 0.75]) + 0.05 * jitter
    plane_dir = None
    if d["plane"]:
        k = rng.normal(size=3)
        plane_dir = k / np.linalg.norm(k)
    return Workload(name=name, n=n, N=N, J=J, nsteps=nsteps, precisions=d["precisions"], verts=verts,
                    tets=tets, c=c, rho=rho, pulse_centre=centre, pulse_width=0.2, plane_dir=plane_dir,
                    plane_amp=0.5, seed=SEED0 + d["index"], shape=shape, face_bc=d.get("face_bc"))


def scaled_workload(name: str, n: int, nsteps: int) -> Workload:
    """The named config on a coarser (or finer) hex grid: same N, J, materials rule, pulse and seed."""
    return make_workload(name, n=n, nsteps=nsteps)
