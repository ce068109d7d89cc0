"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (-m gpu).

configs[1] (3,072 tets, 500 steps) is small enough for the oracle to run whole.  For configs[2..4] (up to 1.57 M
tets) the oracle cannot: there the full-size GPU run is compared on SAMPLED outputs that the oracle can compute
exactly.  One time step = 5 LSRK stages, and one stage moves information across one cell face (3D), one triangle
edge (2D) or one line end (1D), i.e. by at most one hexahedron; so after s steps the solution in the two hex layers
around the (+,+,+) corner -- where the seeded pulse sits and where three HABC faces, three edges and a corner are
active -- depends only on the data inside the corner block of (2 + 5 s + 1)^3 hexes.  The oracle is run on that
block as a mesh of its own (same vertices, materials, dt and initial data; its three cut planes become artificial
boundaries 5 s + 1 hexes away from everything that is compared) and must agree with the full-size GPU run there,
element by element, on p, u and every face and edge auxiliary set: 3 steps on an 18^3 block where the oracle
manages that in about a minute (N <= 5), 2 steps on a 13^3 block at N = 6, 8.  The stated step counts against the
oracle are run on smaller grids by tests/test_gpu_stated_steps.py; here properties that hold at any size cover
them at full size: finite fields, fp32 against fp64, and the scalar-FMA kernel against the tensor-pipe kernel.
"""
import numpy as np
import pytest

import parity
from workloads import make_workload

pytestmark = pytest.mark.gpu
TOL = {64: 1e-11, 32: 1e-4}
KEEP = 2                    # compared: the 2^3 hexes nearest the corner


def block_for(nsteps):
    """hexes per side of the oracle's corner block for nsteps steps (domain of dependence + one spare layer)"""
    return KEEP + 5 * nsteps + 1


def corner_block(w, m):
    """The m^3 hexes of workload w nearest the (+,+,+) corner as a workload of its own (vertex positions, c, rho and
    initial data unchanged; vertices of the three cut planes snapped onto them so that the block is a cuboid)."""
    import copy
    n = w.n
    hexid = np.arange(n ** 3)
    i, j, k = hexid % n, (hexid // n) % n, hexid // (n * n)            # hex-major, x fastest (workloads/configs.py)
    sel_hex = (i >= n - m) & (j >= n - m) & (k >= n - m)
    sel = np.repeat(sel_hex, 6)
    tets = w.tets[sel]
    used = np.unique(tets)
    remap = -np.ones(w.verts.shape[0], dtype=np.int64)
    remap[used] = np.arange(used.size)
    verts = w.verts[used].copy()
    cut = 1.0 - m * (2.0 / n)
    # lattice index of every used vertex from its position in the unperturbed grid numbering
    vi = used // ((n + 1) * (n + 1)), (used // (n + 1)) % (n + 1), used % (n + 1)
    for ax in range(3):
        verts[vi[ax] == n - m, ax] = cut
    sub = copy.copy(w)
    sub.n, sub.verts, sub.tets = m, verts, remap[tets].astype(np.int32)
    sub.c, sub.rho = w.c[sel], w.rho[sel]
    return sub


def near_corner(x, h, keep=KEEP):
    """cells (first axis of x [cells, nodes, 3]) whose centroid lies in the `keep` hex layers at the corner"""
    return (x.mean(axis=1) > 1.0 - keep * h).all(axis=1)


def compare_corner(lib, ora, h):
    out = {}
    ml, mo = near_corner(lib["x"], h), near_corner(ora["x"], h)
    assert ml.sum() == mo.sum() == 6 * KEEP ** 3
    sub_l = dict(lib, x=lib["x"][ml], q=lib["q"][:, ml])
    sub_o = dict(ora, x=ora["x"][mo], q=ora["q"][:, mo])
    for key, xs, arr in (("face", "xf", "fa"), ("edge", "xe", "ea")):
        if lib[arr].size == 0:                                   # J = 0: no auxiliary fields
            sub_o[arr] = np.zeros(0)
            continue
        a, b = near_corner(lib[xs], h), near_corner(ora[xs], h)
        assert a.sum() == b.sum() > 0
        sub_l[xs], sub_l[arr] = lib[xs][a], lib[arr][a]
        sub_o[xs], sub_o[arr] = ora[xs][b], ora[arr][b]
    sub_o["T"], sub_o["E"] = 1, 1
    out = parity.compare(sub_l, sub_o)
    return out


def check(err, prec, aux=True):
    parity.check(err, TOL[prec], aux)


# ------------------------------------------------------------------------------------------ configs[1], whole
@pytest.fixture(scope="module")
def cfg2_oracle():
    w = make_workload("cfg2")
    return w, parity.run_oracle(w)


@pytest.mark.parametrize("prec", [64, 32])
def test_cfg2_full_500_steps(cfg2_oracle, prec):
    """BASELINE configs[1]: 3,072 tets, N=4, J=4, Gaussian + plane wave, all 500 steps, fp64 and fp32."""
    w, ora = cfg2_oracle
    lib = parity.run_library(w, precision=prec)
    check(parity.compare(lib, ora), prec)


# ------------------------------------------------------------------------------------------ configs[2..4], sampled
_block_oracle = {}


def steps_corner(name, prec, nsteps, **over):
    w = make_workload(name, nsteps=nsteps, **over)
    lib = parity.run_library(w, precision=prec)
    key = (name, nsteps, tuple(sorted(over.items())))
    if key not in _block_oracle:                       # one oracle run serves both precisions
        _block_oracle.clear()                          # (and only the latest one is kept: they are large)
        _block_oracle[key] = parity.run_oracle(corner_block(w, block_for(nsteps)), dt=lib["dt"])
    ora = _block_oracle[key]
    assert abs(ora["dt"] - lib["dt"]) <= 1e-15 * lib["dt"]
    return compare_corner(lib, ora, 2.0 / w.n), lib


def test_cfg3_full_size_corner_block():
    """configs[2]: 196,608 tets, perturbed mesh, layered c, N=4, J=6; 3 steps."""
    err, lib = steps_corner("cfg3", 64, 3)
    assert lib["info"]["K"] == 196608
    check(err, 64)


@pytest.mark.parametrize("N,J,prec,nsteps", [(1, 8, 64, 3), (6, 8, 64, 2), (6, 8, 32, 2), (8, 4, 64, 2), (8, 4, 32, 2),
                                             (8, 0, 64, 1), (8, 0, 32, 1)])
def test_cfg4_full_size_corner_block(N, J, prec, nsteps):
    """configs[3]: the 82,944-tet mesh at both ends of the degree sweep, default kernels (N >= 6: k_vol3d_mmag in fp64,
    k_vol3d_tf32g in fp32)."""
    err, lib = steps_corner("cfg4", prec, nsteps, N=N, J=J)
    assert lib["info"]["K"] == 82944
    check(err, prec, aux=J > 0)


@pytest.mark.parametrize("prec", [64, 32])
def test_cfg5_full_size_corner_block(prec):
    """configs[4], the bench workload: 1,572,864 tets, N=5, J=8, in the configuration bench.py times; 3 steps."""
    err, lib = steps_corner("cfg5", prec, 3)
    assert lib["info"]["K"] == 1572864 and lib["info"]["launches_per_step"] == 30
    check(err, prec)


def test_cfg5_full_size_stated_steps_properties():
    """configs[4] for its 100 steps: finite, fp32 against fp64 within the fp32 tolerance, and the scalar-FMA 3D kernel
    against the tensor-pipe kernel within the fp64 tolerance -- two independent index paths over 1.57 M tets."""
    from paper_1610_05023_b200 import Solver
    w = make_workload("cfg5")

    def run(prec, kernel, nsteps):
        s = Solver(w.verts, w.tets, w.N, w.J, w.c, w.rho, precision=prec, kernel=kernel)
        x, y, z = s.get_nodes()
        cn = np.repeat(w.c[:, None], s.Np, axis=1)
        s.set_initial(*w.fields(x, y, z, cn, 1.0))
        del x, y, z, cn
        s.step(nsteps)
        out = s.get_fields()
        s.close()
        assert all(np.isfinite(a).all() for a in out)
        return out

    for (pa, ka, pb, kb, nsteps, tol) in ((32, 0, 64, 0, 100, 1e-4), (64, 1, 64, 0, 100, 1e-11)):
        ref = dict(zip(("q", "fa", "ea"), run(pb, kb, nsteps)))
        got = dict(zip(("q", "fa", "ea"), run(pa, ka, nsteps)))
        parity.check(parity.compare_same_order(got, ref), tol)       # per field and per auxiliary set, not pooled
        del ref, got


def test_cfg3_full_size_stated_steps_properties():
    """configs[2] for its 200 steps at full size (196,608 tets, perturbed mesh): finite, and the scalar-FMA kernel
    against the tensor-pipe kernel within the fp64 tolerance on p, u and all auxiliary fields."""
    w = make_workload("cfg3")
    a = parity.run_library(w, kernel=0)
    b = parity.run_library(w, kernel=1)
    assert a["info"]["K"] == 196608
    for key in ("q", "fa", "ea"):
        assert np.isfinite(a[key]).all()
    parity.check(parity.compare_same_order(b, a), 1e-11)             # per field and per auxiliary set, not pooled
