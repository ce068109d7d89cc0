"""Writes tests/golden/reflection_reference.npz — the pin P9 reference: a Gaussian pulse
propagated by the ORACLE in the large domain [-3,3]^3 (reflections cannot return before t_final), sampled on
the elements inside [-1,1]^3.  Calls only `oracle/` and the seeded mesh generator.  ~3 min on 8 cores.

    python tests/golden/make_reflection_reference.py
"""
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
from oracle.solver import OracleSolver  # noqa: E402
from workloads import cube_mesh  # noqa: E402

N, n, T_END = 3, 4, 2.4
X0, WIDTH = np.array([0.2, 0.1, -0.15]), 0.3


def initial(o):
    x = o.nodes()
    p = np.exp(-((x - X0) ** 2).sum(-1) / (2 * WIDTH * WIDTH))
    return np.stack([p, 0 * p, 0 * p, 0 * p])


if __name__ == "__main__":
    vb, tb = cube_mesh(3 * n)
    vb = vb * 3.0
    ob = OracleSolver(vb, tb, N, 0, np.ones(len(tb)), np.ones(len(tb)))
    ns = int(np.ceil(T_END / ob.dt))
    ob.dt = T_END / ns
    ob.set_initial(initial(ob))
    ob.step(ns)
    cb = ob.nodes().mean(1)
    idx = np.nonzero(np.all(np.abs(cb) < 1, axis=1))[0]
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "reflection_reference.npz")
    np.savez_compressed(out, centroid=cb[idx], p=ob.q[0][idx], x=ob.nodes()[idx], dt=ob.dt, nsteps=ns)
    print("wrote", out, "nsteps", ns, "dt", ob.dt)
