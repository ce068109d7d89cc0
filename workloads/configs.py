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

    @property
    def K(self) -> int:
        return int(self.tets.shape[0])

    def fields(self, x, y, z, c_node, rho_node):
        return initial_fields(self, x, y, z, c_node, rho_node)


def cube_mesh(n: int, perturb: float = 0.0, rng: np.random.Generator | None = None):
    """Kuhn 6-tet split of an n^3 hex grid on [-1,1]^3.  Element order: hex-major (x fastest), the six
    tets of a hex consecutive.  Returns (verts[nv,3] f64, tets[K,4] i32), all tets positively oriented."""
    g = np.linspace(-1.0, 1.0, n + 1)
    X, Y, Z = np.meshgrid(g, g, g, indexing="ij")
    verts = np.stack([X.ravel(), Y.ravel(), Z.ravel()], axis=1).astype(np.float64)

    def vid(i, j, k):
        return (i * (n + 1) + j) * (n + 1) + k

    if perturb > 0.0:
        assert rng is not None
        h = 2.0 / n
        I, Jx, Kx = np.meshgrid(np.arange(n + 1), np.arange(n + 1), np.arange(n + 1), indexing="ij")
        interior = ((I > 0) & (I < n) & (Jx > 0) & (Jx < n) & (Kx > 0) & (Kx < n)).ravel()
        d = rng.uniform(-perturb * h, perturb * h, size=verts.shape)
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

    kk, jj, ii = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")  # x fastest
    hexes = np.stack([ii.ravel(), jj.ravel(), kk.ravel()], axis=1)                        # [n^3,3]
    cidx = hexes[:, None, None, :] + corner_paths[None, :, :, :]                          # [n^3,6,4,3]
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
    verts, tets = cube_mesh(n, d["perturb"], rng)
    K = tets.shape[0]
    if d["c"][0] == "const":
        c = np.full(K, d["c"][1], dtype=np.float64)
    else:
        _, nl, lo, hi = d["c"]
        c = layered_speed(n, nl, lo, hi, rng)
    rho = np.ones(K, dtype=np.float64)
    jitter = rng.uniform(-1.0, 1.0, size=3)
    if d["pulse"] == "centre":
        centre = 0.3 * jitter / max(1.0, np.linalg.norm(jitter))        # |x0| < 0.3
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
                    plane_amp=0.5, seed=SEED0 + d["index"])


def scaled_workload(name: str, n: int, nsteps: int) -> Workload:
    """The named config on a coarser (or finer) hex grid: same N, J, materials rule, pulse and seed."""
    return make_workload(name, n=n, nsteps=nsteps)
