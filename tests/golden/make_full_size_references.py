"""Writes tests/golden/full_size_<case>.npz: the ORACLE's result at BASELINE.json's FULL size after the STATED number
of steps (north_star: "match the oracle ... after the stated step counts"), for the configurations where one CPU can
afford it once, offline:

    cfg3        configs[2] whole: 196,608 tets, perturbed mesh, 4 layers of c, N = 4, J = 6, 200 steps   (about 1 h)
    cfg4_N1_J8  configs[3] at the low end of the sweep: 82,944 tets, N = 1, J = 8, 100 steps             (minutes)
    cfg4_N4_J4  configs[3] at its base degree: 82,944 tets, N = 4, J = 4, 100 steps                       (about 15 min)

configs[4] whole (1.57 M tets, 8.8 G node-updates: about 6.5 h and 30 GB with this numpy oracle) is out of reach; it
stays on the rule + corner-block + kernel-vs-kernel evidence of tests/test_gpu_full_configs.py.

Calls only `oracle/` and `workloads/`.  Stored (float64): the time step, and SAMPLES of the final state -- for a seeded
choice of tetrahedra (every cell of the 2^3 hexes at the (+,+,+) corner, 500 cells of the 10^3-hex block around the
pulse, 100 cells anywhere) their caller-order index, node coordinates and p, u, v, w; for a seeded choice of boundary
triangles (all of the 6 x 6-hex patches of the three faces at that corner, 150 anywhere on the six faces) node
coordinates and every auxiliary set (p_i00 and both tangential velocities); the same for boundary lines (the 10 nearest
the corner on each of its three edges, 40 anywhere).  tests/test_gpu_full_size_golden.py runs the CUDA library at full
size for the same number of steps and compares these samples per field and per set.

    python tests/golden/make_full_size_references.py cfg3 | cfg4_N1_J8 | cfg4_N4_J4
"""
import os
import sys
import time

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
from oracle.solver import OracleSolver  # noqa: E402
from workloads import make_workload  # noqa: E402

CASES = {"cfg3": ("cfg3", {}), "cfg4_N1_J8": ("cfg4", dict(N=1, J=8)), "cfg4_N4_J4": ("cfg4", dict(N=4, J=4))}
HERE = os.path.dirname(os.path.abspath(__file__))


def sample_indices(w, o, rng):
    """seeded choice of tetrahedra (caller order), triangles and lines (oracle order)"""
    n, h = w.n, 2.0 / w.n
    cen = o.nodes().mean(axis=1)
    corner2 = np.nonzero((cen > 1.0 - 2 * h).all(axis=1))[0]
    block10 = np.nonzero((cen > 1.0 - 10 * h).all(axis=1))[0]
    tets = np.unique(np.concatenate([corner2, rng.choice(block10, 500, replace=False),
                                     rng.choice(w.K, 100, replace=False)]))
    xf = o.H.tri.x.mean(axis=1)
    on_corner_faces = (xf > 1.0 - 1e-9).any(axis=1) & (xf > 1.0 - 6 * h).all(axis=1)
    tris = np.unique(np.concatenate([np.nonzero(on_corner_faces)[0], rng.choice(o.T, 150, replace=False)]))
    xe = o.H.lin.x.mean(axis=1)
    on_corner_edges = ((xe > 1.0 - 1e-9).sum(axis=1) == 2) & (xe > 1.0 - 10 * h).all(axis=1)
    lins = np.unique(np.concatenate([np.nonzero(on_corner_edges)[0], rng.choice(o.E, 40, replace=False)]))
    return tets, tris, lins


def main(case):
    name, over = CASES[case]
    w = make_workload(name, **over)
    t0 = time.time()
    o = OracleSolver(w.verts, w.tets, w.N, w.J, w.c, w.rho)
    x = o.nodes()
    cn = np.repeat(w.c[:, None], x.shape[1], axis=1)
    rn = np.repeat(w.rho[:, None], x.shape[1], axis=1)
    o.set_initial(np.stack(w.fields(x[..., 0], x[..., 1], x[..., 2], cn, rn)))
    print(f"{case}: K={w.K} N={w.N} J={w.J} T={o.T} E={o.E} dt={o.dt!r} setup {time.time() - t0:.0f}s", flush=True)
    for s in range(w.nsteps):
        o.step(1)
        if (s + 1) % 10 == 0:
            print(f"  step {s + 1}/{w.nsteps}  {time.time() - t0:.0f}s", flush=True)
    q, fa, ea = o.get_fields()
    tets, tris, lins = sample_indices(w, o, np.random.default_rng(w.seed + 77))
    out = os.path.join(HERE, f"full_size_{case}.npz")
    np.savez_compressed(out, dt=o.dt, nsteps=w.nsteps, K=w.K, N=w.N, J=w.J, T=o.T, E=o.E,
                        tet_index=tets, x=x[tets], q=q[:, tets],
                        xf=o.H.tri.x[tris], fa=fa[tris], xe=o.H.lin.x[lins], ea=ea[lins],
                        norm_p_all=np.linalg.norm(q[0]), norm_fa_all=np.linalg.norm(fa), norm_ea_all=np.linalg.norm(ea))
    print("wrote", out, os.path.getsize(out), "bytes", f"{time.time() - t0:.0f}s")


if __name__ == "__main__":
    main(sys.argv[1])
