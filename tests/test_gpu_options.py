"""The dg_options paths that the parity tests do not take by default (-m gpu): dg_options.cfl, workspace_dev = NULL
(the library's own cudaMalloc), stream = NULL (legacy default stream, plain launches), and a point source switched on
after some steps (the host clock that dg_set_source uploads)."""
import numpy as np
import pytest

import parity
from workloads import make_workload

pytestmark = pytest.mark.gpu


def _run(w, nsteps, **kw):
    from paper_1610_05023_b200 import Solver
    s = Solver(w.verts, w.tets, w.N, w.J, w.c, w.rho, **kw)
    x, y, z = s.get_nodes()
    s.set_initial(*parity.initial_on(w, x, y, z, w.c, w.rho))
    s.step(nsteps)
    q, fa, ea = s.get_fields()
    _, _, _, _, xf = s.get_face_map()
    _, _, _, xe = s.get_edge_map()
    out = dict(dt=s.dt, x=np.stack([x, y, z], axis=-1), q=q, fa=fa, ea=ea, xf=xf, xe=xe, T=s.T, E=s.E, C=s.C, info=s.info)
    s.close()
    return out


def test_cfl_scales_the_time_step_of_eq_46():
    """dg_options.cfl multiplies eq (46); the oracle takes the same factor."""
    from oracle.solver import OracleSolver
    w = make_workload("cfg3", n=3, nsteps=20)
    base = _run(w, 0)
    lib = _run(w, 20, cfl=0.6)
    assert lib["dt"] == pytest.approx(0.6 * base["dt"], rel=1e-15)
    o = OracleSolver(w.verts, w.tets, w.N, w.J, w.c, w.rho, cfl=0.6)
    assert lib["dt"] == pytest.approx(o.dt, rel=1e-13)
    x = o.nodes()
    o.set_initial(np.stack(parity.initial_on(w, x[..., 0], x[..., 1], x[..., 2], w.c, w.rho)))
    o.step(20)
    q, fa, ea = o.get_fields()
    ora = dict(x=x, q=q, fa=fa, ea=ea, xf=o.H.tri.x, xe=o.H.lin.x, T=o.T, E=o.E)
    parity.check(parity.compare(lib, ora), 1e-11)


@pytest.mark.parametrize("prec", [64, 32])
def test_library_allocated_workspace_and_default_stream(prec):
    """workspace_dev = NULL (cudaMalloc inside dg_create, cudaFree in dg_destroy) and stream = NULL (no graph) compute
    the same numbers, bit for bit, as the torch-workspace / torch-stream / CUDA-graph path the other tests use."""
    w = make_workload("cfg5", n=3, nsteps=12)
    ref = _run(w, 12, precision=prec)
    own = _run(w, 12, precision=prec, torch_workspace=False)
    dflt = _run(w, 12, precision=prec, default_stream=True)
    both = _run(w, 12, precision=prec, torch_workspace=False, default_stream=True, use_graph=False)
    assert np.linalg.norm(ref["fa"]) > 0 and np.linalg.norm(ref["ea"]) > 0
    for other in (own, dflt, both):
        for key in ("q", "fa", "ea"):
            assert np.array_equal(other[key], ref[key]), key


@pytest.mark.parametrize("prec,use_graph", [(64, True), (64, False), (32, True)])
def test_source_switched_on_after_some_steps(prec, use_graph):
    """dg_set_source after n1 steps: the wavelet must be evaluated on the clock that started at dg_set_initial
    (PAPER.md:L776-786), i.e. the host clock uploaded by dg_set_source has to equal n1 dt.  The oracle does the same
    (OracleSolver.t runs from set_initial)."""
    from oracle.solver import OracleSolver
    from paper_1610_05023_b200 import Solver
    w = make_workload("cfg1")
    xs, f, ts = np.array([0.11, -0.07, 0.05]), 1.5, 0.35
    n1, n2 = 7, 25
    s = Solver(w.verts, w.tets, w.N, w.J, w.c, w.rho, precision=prec, use_graph=use_graph)
    x, y, z = s.get_nodes()
    s.set_initial(*parity.initial_on(w, x, y, z, w.c, w.rho))
    s.step(3)
    s.step(n1 - 3)                                  # two calls: the clock adds up over calls
    s.set_source(xs, f, ts, 2.0)
    s.step(n2)
    q, fa, ea = s.get_fields()
    _, _, _, _, xf = s.get_face_map()
    _, _, _, xe = s.get_edge_map()
    lib = dict(x=np.stack([x, y, z], axis=-1), q=q, fa=fa, ea=ea, xf=xf, xe=xe)
    s.close()
    o = OracleSolver(w.verts, w.tets, w.N, w.J, w.c, w.rho)
    xo = o.nodes()
    o.set_initial(np.stack(parity.initial_on(w, xo[..., 0], xo[..., 1], xo[..., 2], w.c, w.rho)))
    o.step(n1)
    o.set_source(xs, f, ts, 2.0)
    o.step(n2)
    assert abs(o.source_S(o.t)) > 1e-3              # the wavelet is on at these times: a shifted clock would show
    qo, fo, eo = o.get_fields()
    ora = dict(x=xo, q=qo, fa=fo, ea=eo, xf=o.H.tri.x, xe=o.H.lin.x, T=o.T, E=o.E)
    parity.check(parity.compare(lib, ora), {64: 1e-11, 32: 1e-4}[prec])
    # and a clock that had restarted at dg_set_source would be seen: the oracle with that mistake differs by far more
    o2 = OracleSolver(w.verts, w.tets, w.N, w.J, w.c, w.rho)
    o2.set_initial(np.stack(parity.initial_on(w, xo[..., 0], xo[..., 1], xo[..., 2], w.c, w.rho)))
    o2.step(n1)
    o2.t = 0.0
    o2.set_source(xs, f, ts, 2.0)
    o2.step(n2)
    assert parity.rel_l2(o2.q[0], qo[0]) > 1e-3


def test_time_kernels_switched_on_an_existing_solver():
    """dg_set_time_kernels: off -> on -> off on one solver (what bench.py does between its headline run and its kernel
    timing).  The events exist only while the option is on, and the state advances exactly as without them."""
    from paper_1610_05023_b200 import DgError, Solver
    w = make_workload("cfg5", n=4, nsteps=1)
    out = []
    for switch in (False, True):
        s = Solver(w.verts, w.tets, w.N, w.J, w.c, w.rho)
        x, y, z = s.get_nodes()
        s.set_initial(*parity.initial_on(w, x, y, z, w.c, w.rho))
        s.step(3)
        if switch:
            with pytest.raises(DgError):
                s.last_step_kernel_ms()
            s.set_time_kernels(True)
            with pytest.raises(DgError):
                s.last_step_kernel_ms()                      # no step since the switch
            s.step(2)
            ms = s.last_step_kernel_ms()
            assert ms.shape == (5,) and (ms > 0).all()
            s.set_time_kernels(False)
            s.step(2)
            with pytest.raises(DgError):
                s.last_step_kernel_ms()
        else:
            s.step(4)
        out.append(s.get_fields())
        s.close()
    for a, b in zip(*out):
        assert np.array_equal(a, b)


@pytest.mark.parametrize("prec", [64, 32])
def test_random_per_cell_media_on_every_level(prec):
    """c and rho drawn per TETRAHEDRON (not per layer or per hex as in the BASELINE recipes): neighbouring cells,
    the two boundary triangles that meet at a domain edge, and consecutive lines then all differ in impedance, so the
    heterogeneous flux of every level and the impedances inside the face / edge / corner closures (reading R9; oracle
    pins H1-H5) are all exercised against the oracle."""
    w = make_workload("cfg3", n=3, N=3, J=3, nsteps=25)
    rng = np.random.default_rng(2025)
    w.c = rng.uniform(1.0, 3.0, size=w.K)
    w.rho = rng.uniform(0.5, 2.0, size=w.K)
    lib, ora = parity.run_library(w, precision=prec), parity.run_oracle(w)
    assert lib["dt"] == pytest.approx(ora["dt"], rel=1e-13)
    parity.check(parity.compare(lib, ora), {64: 1e-11, 32: 1e-4}[prec])
