"""Parity tests proper (-m gpu): the CUDA path through the C ABI against the oracle, element by element, on the
same seeded inputs.  Tolerances are BASELINE.json north_star's: relative L2 <= 1e-11 (fp64), <= 1e-4 (fp32) on
p, u and every auxiliary field."""
import numpy as np
import pytest

import parity
from workloads import make_workload

pytestmark = pytest.mark.gpu
TOL = {64: 1e-11, 32: 1e-4}


def _check(err, prec, aux=True):
    parity.check(err, TOL[prec], aux)


def test_cfg1_full_fp64():
    """BASELINE configs[0]: 48 tets, N=3, J=2, 100 steps."""
    w = make_workload("cfg1")
    lib, ora = parity.run_library(w), parity.run_oracle(w)
    assert lib["dt"] == pytest.approx(ora["dt"], rel=1e-14)
    assert (lib["T"], lib["E"], lib["C"]) == (48, 24, 8)
    _check(parity.compare(lib, ora), 64)


@pytest.mark.parametrize("prec", [64, 32])
def test_cfg2_reduced_steps(prec):
    """BASELINE configs[1] (3,072 tets, N=4, J=4, Gaussian + plane wave) for 60 of its 500 steps (the full count
    is run by tests/test_gpu_full_configs.py)."""
    w = make_workload("cfg2")
    lib, ora = parity.run_library(w, precision=prec, nsteps=60), parity.run_oracle(w, nsteps=60)
    _check(parity.compare(lib, ora), prec)


def test_cfg3_shape_perturbed_layered():
    """configs[2] recipe (perturbed interior vertices, 4 layers of c in U[1,3], N=4, J=6) on a 6^3 hex grid:
    several batches of the persistent kernel plus a ragged tail (1296 tets = 40 batches of 32 + 16)."""
    w = make_workload("cfg3", n=6, nsteps=40)
    assert np.unique(w.c).size == 4
    lib, ora = parity.run_library(w), parity.run_oracle(w)
    _check(parity.compare(lib, ora), 64)


@pytest.mark.parametrize("prec", [64, 32])
def test_cfg5_shape(prec):
    """configs[4] recipe (N=5, J=8, layered c in U[1.5,4.5]) on a 5^3 hex grid (750 tets: ragged tail of 14)."""
    w = make_workload("cfg5", n=5, nsteps=30)
    lib, ora = parity.run_library(w, precision=prec), parity.run_oracle(w)
    _check(parity.compare(lib, ora), prec)


@pytest.mark.parametrize("N", [1, 2, 3, 4, 5, 6, 7, 8])
@pytest.mark.parametrize("J", [0, 4])
def test_cfg4_degree_sweep(N, J):
    """configs[3]: every degree N=1..8 with J in {0,4} (J=8 in test_J8_degree below) on a 3^3 hex grid."""
    w = make_workload("cfg4", n=3, N=N, J=J, nsteps=10)
    lib, ora = parity.run_library(w), parity.run_oracle(w)
    _check(parity.compare(lib, ora), 64, aux=J > 0)


@pytest.mark.parametrize("N", [2, 6])
def test_J8_degree(N):
    w = make_workload("cfg4", n=2, N=N, J=8, nsteps=10)
    for prec in (64, 32):
        lib, ora = parity.run_library(w, precision=prec), parity.run_oracle(w)
        _check(parity.compare(lib, ora), prec)


@pytest.mark.parametrize("N,J", [(2, 1), (3, 3), (5, 5), (4, 7), (5, 6), (3, 9)])
@pytest.mark.parametrize("prec", [64, 32])
def test_partial_set_groups(N, J, prec):
    """The 2D solvers work on groups of four auxiliary sets: J that is not a multiple of four leaves a partial last
    group (1, 2 or 3 sets), J > 8 three groups per triangle.  fp64 runs k_face2d_mma, fp32 k_face2d."""
    w = make_workload("cfg3", n=3, N=N, J=J, nsteps=15)
    lib, ora = parity.run_library(w, precision=prec), parity.run_oracle(w)
    _check(parity.compare(lib, ora), prec)


@pytest.mark.parametrize("N,kernel", [(4, 1), (4, 2), (4, 3), (5, 1), (5, 2), (5, 3), (1, 2), (2, 2), (1, 3), (2, 3), (3, 3), (3, 2), (6, 1), (6, 5), (7, 1), (7, 5), (8, 5)])
def test_3d_kernel_variants(N, kernel):
    """dg_options.kernel (DG_KERNEL_*): 1 scalar FMA, 2 batch-synchronous DMMA, 3 warp-specialised DMMA, 5 tensor pipe
    with the operators read through L1/L2 (N >= 6) -- the same numbers.
    5^3 hexes = 750 tets: 93 batches of 8 + a ragged tail of 6, several batches per persistent CTA."""
    w = make_workload("cfg5", n=5, N=N, J=3, nsteps=12)
    lib, ora = parity.run_library(w, kernel=kernel), parity.run_oracle(w)
    _check(parity.compare(lib, ora), 64)


@pytest.mark.parametrize("N,kernel", [(3, 4), (4, 4), (5, 4), (1, 1), (2, 1), (1, 6), (2, 6), (3, 1), (5, 1), (5, 0), (6, 5), (7, 5), (8, 5), (6, 1)])
def test_3d_kernel_variants_fp32(N, kernel):
    """fp32: 1 scalar FMA, 6 one thread per element (N = 1, 2), 4 / 5 tensor cores with 3xTF32 error compensation
    (N = 3..5 / N = 6..8) -- all inside the
    fp32 tolerance, and the compensated tensor-core result no worse than 4x the FMA kernel's error.
    750 tets = 46 batches of 16 + a ragged tail of 14."""
    w = make_workload("cfg5", n=5, N=N, J=3, nsteps=12)
    ora = parity.run_oracle(w)
    err = parity.compare(parity.run_library(w, precision=32, kernel=kernel), ora)
    _check(err, 32)
    if kernel in (4, 5):
        ref = parity.compare(parity.run_library(w, precision=32, kernel=1), ora)
        assert err["p"] <= 4 * ref["p"] + 1e-7 and err["u"] <= 4 * ref["u"] + 1e-7, (err, ref)


def test_kernel_choice_is_validated():
    """a kernel that does not cover (precision, N) is refused with DG_EINVAL, not silently replaced"""
    from paper_1610_05023_b200 import DgError, Solver
    w = make_workload("cfg1")
    for N, prec, kernel in ((6, 64, 2), (6, 64, 3), (5, 64, 4), (2, 32, 4), (5, 32, 5), (3, 32, 6), (2, 64, 6), (3, 64, 7), (3, 64, -1)):
        with pytest.raises(DgError):
            Solver(w.verts, w.tets, N, 2, w.c, w.rho, precision=prec, kernel=kernel)


FREE_SURFACE = {(2, -1): "dirichlet"}
BC_CASES = {
    "free_surface": FREE_SURFACE,                                          # 5 HABC faces, 8 edges, 4 corners
    "habc_x_rigid_yz": {(1, -1): "rigid", (1, 1): "rigid", (2, -1): "rigid", (2, 1): "rigid"},   # faces only, no edges
    "mixed": {(0, -1): "dirichlet", (0, 1): "rigid", (1, 1): "dirichlet"},  # HABC on -y, -z, +z: 2 edges, no corner
    "all_walls": {(a, sg): ("dirichlet" if a else "rigid") for a in range(3) for sg in (-1, 1)},
}


@pytest.mark.parametrize("case", sorted(BC_CASES))
@pytest.mark.parametrize("N,prec,kernel", [(3, 64, 0), (5, 64, 0), (4, 64, 1), (5, 32, 0), (6, 32, 0)])
def test_mixed_boundary_conditions(case, N, prec, kernel):
    """dg_options.face_bc: p = 0 and rigid walls on some domain faces, HABC on the others, auxiliary
    fields only where HABC faces meet -- against the oracle's per-face boundary flags, through every 3D kernel."""
    face_bc = BC_CASES[case]
    w = make_workload("cfg1", n=3, N=N, J=3, nsteps=60)
    lib = parity.run_library(w, precision=prec, kernel=kernel, face_bc=face_bc)
    ora = parity.run_oracle(w, face_bc=face_bc)
    assert (lib["T"], lib["E"], lib["C"]) == (ora["T"], ora["E"], ora["C"])
    err = parity.compare(lib, ora)
    for k in ("p", "u", "face", "edge"):
        if k in err:
            assert err[k] <= TOL[prec], (k, err)
    assert ("face" in err) == (ora["T"] > 0) and ("edge" in err) == (ora["E"] > 0)
    if case == "free_surface":
        assert (lib["T"], lib["E"], lib["C"]) == (5 * 18, 8 * 3, 4)
        assert err["norm_face"] > 1e-3 * err["norm_p"] and err["norm_edge"] > 1e-5 * err["norm_p"], err


@pytest.mark.parametrize("prec", [64, 32])
def test_seam_shaped_workload(prec):
    """the SEAM-shaped stand-in (cuboid 3.5 x 4 x 1.5, free surface on top, HABC on the other five faces,
    strongly heterogeneous c AND rho varying from cell to cell, N = 3, J = 3) on a 7 x 8 x 3 hex grid."""
    w = make_workload("seam", n=7, nsteps=80)
    assert w.shape == (7, 8, 3) and w.face_bc == {(2, 1): "dirichlet"} and np.unique(w.rho).size > 100
    lib, ora = parity.run_library(w, precision=prec), parity.run_oracle(w)
    assert (lib["T"], lib["E"], lib["C"]) == (ora["T"], ora["E"], ora["C"]) == (2 * (7 * 8 + 2 * 7 * 3 + 2 * 8 * 3), 4 * 3 + 2 * 7 + 2 * 8, 4)
    _check(parity.compare(lib, ora), prec)


@pytest.mark.parametrize("N,prec,kernel,graph", [(3, 64, 0, True), (5, 64, 0, True), (4, 64, 1, False), (5, 32, 0, True), (2, 32, 0, True)])
def test_point_source(N, prec, kernel, graph):
    """Ricker point source in the pressure equation on top of the seeded pulse, against
    the oracle; the source cell is strictly inside the mesh and the stage times t + c_n dt matter (S changes sign)."""
    w = make_workload("cfg1", n=3, N=N, J=2, nsteps=40)
    src = ([0.11, -0.07, 0.05], 2.5, 0.05, 3.0)
    lib = parity.run_library(w, precision=prec, kernel=kernel, use_graph=graph, source=src)
    ora = parity.run_oracle(w, source=src)
    nosrc = parity.run_oracle(w)
    assert parity.rel_l2(ora["q"], nosrc["q"]) > 0.05                # the source really contributes
    _check(parity.compare(lib, ora), prec)
    assert lib["info"]["launches_per_step"] == 35


def test_point_source_spherical_wave_and_reset():
    """The CUDA path against the analytic spherical wave (45a-b) at a resolution the oracle would need minutes for
    (12^3 x 6 tets, N = 4), and dg_set_initial restarting the clock / amplitude 0 switching the source off."""
    from paper_1610_05023_b200 import Solver
    from workloads.configs import box_mesh
    v, t = box_mesh((12, 12, 12), ((-0.5, 0.5),) * 3)
    K = len(t)
    xs, f, ts = np.array([0.03, 0.02, 0.01]), 2.5, 0.5
    s = Solver(v, t, 4, 4, np.ones(K), np.ones(K))
    x, y, z = s.get_nodes()
    zero = np.zeros_like(x)

    def solve(amplitude):
        s.set_initial(zero, zero, zero, zero)
        s.set_source(xs, f, ts, amplitude)
        nst = int(round(0.9 / s.dt))
        s.step(nst)
        return s.get_fields(aux=False)[0], nst * s.dt

    q, tf = solve(1.0)
    d = np.stack([x, y, z], axis=-1) - xs
    r = np.linalg.norm(d, axis=-1)
    a = (np.pi * f * (tf - r - ts)) ** 2
    pref = (1.0 - 2.0 * a) * np.exp(-a) / (4.0 * np.pi * r)
    m = r > 0.15
    err = np.linalg.norm((q[0] - pref)[m]) / np.linalg.norm(pref[m])
    assert err < 0.02, err
    q2, _ = solve(1.0)                                               # same answer after a restart: the clock was reset
    assert np.abs(q2 - q).max() <= 1e-13 * np.abs(q).max()
    q0, _ = solve(0.0)
    assert not q0.any()
    s.close()


def test_edge_cases():
    """Smallest mesh (one hex, 6 tets: every tet touches the boundary), J=1, J=12 (maximum), graph off,
    negatively oriented input cells, zero initial data, nsteps=0."""
    w = make_workload("cfg1", n=1, N=2, J=1, nsteps=15)
    _check(parity.compare(parity.run_library(w), parity.run_oracle(w)), 64)
    w = make_workload("cfg1", n=1, N=1, J=12, nsteps=15)
    _check(parity.compare(parity.run_library(w, use_graph=False), parity.run_oracle(w)), 64)
    # flipped vertex order in half the cells: same solution
    w = make_workload("cfg1", nsteps=10)
    ora = parity.run_oracle(w)
    w.tets = w.tets.copy()
    w.tets[::2] = w.tets[::2][:, [0, 1, 3, 2]]
    _check(parity.compare(parity.run_library(w), ora), 64)
    # nsteps = 0 returns the initial data; zero data stays zero
    lib = parity.run_library(w, nsteps=0)
    x = lib["x"]
    p0 = w.fields(x[..., 0], x[..., 1], x[..., 2], 1.0, 1.0)[0]
    assert np.abs(lib["q"][0] - p0).max() == 0.0
    from paper_1610_05023_b200 import Solver
    s = Solver(w.verts, w.tets, 3, 2, w.c, w.rho)
    s.step(3)
    q, fa, ea = s.get_fields()
    assert not q.any() and not fa.any() and not ea.any()
    s.close()


@pytest.mark.parametrize("prec", [64, 32])
def test_device_view_matches_get_fields(prec):
    """dg_get_device_ptrs (optional): the raw device state read through the exported pointers and the
    documented layouts is what dg_get_fields returns (p_i00 = p*_i + S, eq (29))."""
    import torch
    from cuda.bindings import runtime as cudart
    from paper_1610_05023_b200 import Solver
    w = make_workload("cfg1", n=2, N=3, J=2, nsteps=7)
    s = Solver(w.verts, w.tets, w.N, w.J, w.c, w.rho, precision=prec)
    x, y, z = s.get_nodes()
    s.set_initial(*parity.initial_on(w, x, y, z, w.c, w.rho))
    s.step(7)
    q, fa, ea = s.get_fields()
    v = s.device_view()
    assert v["elem_bytes"] == prec // 8
    dt = torch.float64 if prec == 64 else torch.float32

    def view(ptr, n):
        t = torch.empty(n, dtype=dt, device="cuda")
        s.stream.synchronize()
        err, = cudart.cudaMemcpy(t.data_ptr(), ptr, n * v["elem_bytes"], cudart.cudaMemcpyKind.cudaMemcpyDeviceToDevice)
        assert int(err) == 0
        return t.cpu().double().numpy()

    qd = view(v["q"], s.K * s.Np * 4).reshape(s.K, s.Np, 4)
    assert np.array_equal(qd.transpose(2, 0, 1), q)
    fd = view(v["face_aux"], s.T * s.J * 3 * s.Nfp).reshape(s.T, s.J, 3, s.Nfp)
    S = view(v["face_S"], s.T * s.Nfp).reshape(s.T, 1, s.Nfp)
    assert np.array_equal(fd[:, :, 1:], fa[:, :, 1:])
    assert np.abs(fd[:, :, 0] + S - fa[:, :, 0]).max() <= 4 * np.finfo(np.float64 if prec == 64 else np.float32).eps * np.abs(fa[:, :, 0]).max()
    ed = view(v["edge_aux"], s.E * s.J * s.J * 2 * (s.N + 1)).reshape(s.E, s.J * s.J, 2, s.N + 1)
    assert np.array_equal(ed[:, :, 1], ea[:, :, 1])
    s.close()


def test_in_step_kernel_timing():
    """dg_options.time_kernels: events inside the (graph-replayed) step give the 3D kernel's time per stage; the numbers
    are positive, below the whole step's time, and the option does not change the result."""
    import time
    import torch
    from paper_1610_05023_b200 import DgError, Solver
    w = make_workload("cfg5", n=6, nsteps=5)
    out = []
    for timed in (False, True):
        s = Solver(w.verts, w.tets, w.N, w.J, w.c, w.rho, time_kernels=timed)
        x, y, z = s.get_nodes()
        s.set_initial(*parity.initial_on(w, x, y, z, w.c, w.rho))
        if timed:
            with pytest.raises(DgError):
                s.last_step_kernel_ms()                      # no step yet
        s.step(4)
        s.stream.synchronize()
        t0 = time.perf_counter()
        s.step(1)
        s.stream.synchronize()
        step_ms = 1e3 * (time.perf_counter() - t0)
        if timed:
            ms = s.last_step_kernel_ms()
            assert ms.shape == (5,) and (ms > 0).all() and ms.sum() < step_ms, (ms, step_ms)
        else:
            with pytest.raises(DgError):
                s.last_step_kernel_ms()
        out.append(s.get_fields()[0])
        s.close()
    assert np.array_equal(out[0], out[1])


def test_missing_device_is_loud(monkeypatch):
    import torch
    from paper_1610_05023_b200 import DgError, Solver
    monkeypatch.setattr(torch.cuda, "is_available", lambda: False)
    w = make_workload("cfg1")
    with pytest.raises(DgError):
        Solver(w.verts, w.tets, 3, 2, w.c, w.rho)
