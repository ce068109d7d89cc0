"""CPU tests of the CUDA library's host side: the C-ABI library loads and exports every symbol of
include/dg_habc.h; its reference operators and mesh hierarchy (written independently of the oracle) agree
with the oracle's; error codes."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_1610_05023_b200 as pkg
from oracle.mesh import build_hierarchy
from oracle.refelem import make_refelem
from workloads import cube_mesh, make_workload


def test_library_exports_every_declared_symbol(repo_root):
    header = open(os.path.join(repo_root, "include", "dg_habc.h")).read()
    declared = set(re.findall(r"^(?:int|void|const char\*)\s+(dg_[a-z_]+)\s*\(", header, flags=re.M))
    assert {"dg_create", "dg_set_initial", "dg_step", "dg_get_fields", "dg_destroy"} <= declared
    lib = pkg.lib()
    for name in declared:
        assert hasattr(lib, name), name
    assert set(pkg.binding.EXPORTS) == declared


@pytest.mark.parametrize("dim,N", [(d, n) for d in (1, 2, 3) for n in range(1, 9)])
def test_reference_operators_match_oracle(dim, N):
    rst, D, LIFT, Fm = pkg.dg_reference_element(dim, N)
    e = make_refelem(dim, N)
    assert np.abs(rst - e.rst).max() < 1e-15
    for a in range(dim):
        assert np.abs(D[a] - e.D[a]).max() <= 4e-16 * np.abs(e.D[a]).max()
    assert np.abs(LIFT - e.LIFT).max() <= 4e-16 * np.abs(e.LIFT).max()
    assert (Fm == e.Fmask).all()


@pytest.mark.parametrize("n", [1, 2, 5])
def test_mesh_counts_match_oracle(n):
    v, t = cube_mesh(n)
    K = len(t)
    H = build_hierarchy(v, t, 1, np.ones(K), np.ones(K))
    assert pkg.dg_mesh_counts(v, t) == (K, H.tri.K, H.lin.K, H.cor_vertex.size) == (6 * n ** 3, 12 * n * n, 12 * n, 8)
    w = make_workload("cfg3", n=4)                                   # perturbed interior, planar boundary
    assert pkg.dg_mesh_counts(w.verts, w.tets) == (384, 192, 48, 8)
    # any vertex order inside a tet is accepted
    t2 = t.copy()
    t2[::2] = t2[::2][:, [1, 0, 2, 3]]
    assert pkg.dg_mesh_counts(v, t2)[0] == K


@pytest.mark.parametrize("face_bc", [
    {(2, -1): "dirichlet"},                                              # free surface: 5 HABC faces, 8 edges, 4 corners
    {(1, -1): "rigid", (1, 1): "rigid", (2, -1): "rigid", (2, 1): "rigid"},  # HABC on the two x faces only
    {(0, -1): "dirichlet", (0, 1): "rigid", (1, 1): "dirichlet"},
    {(a, s): "dirichlet" for a in range(3) for s in (-1, 1)},             # no auxiliary level at all
])
def test_mixed_boundary_hierarchy_matches_oracle(face_bc):
    """dg_options.face_bc: triangles only on HABC faces, lines between two of
    them, corners where three meet -- the same counts as the oracle's hierarchy builder."""
    n = 3
    v, t = cube_mesh(n)
    K = len(t)
    H = build_hierarchy(v, t, 1, np.ones(K), np.ones(K), face_bc)
    nh = 6 - len(face_bc)
    got = pkg.dg_mesh_counts(v, t, face_bc)
    size = lambda level: 0 if level is None else level.K
    ncor = 0 if getattr(H, "cor_vertex", None) is None else H.cor_vertex.size
    assert got == (K, size(H.tri), size(H.lin), ncor)
    assert got[1] == 2 * n * n * nh
    if face_bc == {(2, -1): "dirichlet"}:
        assert got[2:] == (8 * n, 4)                                      # the paper's K^pnt = 4 configuration


def test_error_codes():
    lib = pkg.lib()
    v, t = cube_mesh(2)
    with pytest.raises(pkg.DgError, match=r"\[-2\]"):                 # a duplicated tet: face shared by 3 cells
        pkg.dg_mesh_counts(v, np.concatenate([t, t[:1]]))
    with pytest.raises(pkg.DgError, match=r"\[-1\]"):                 # non-cuboid: remove a corner hex
        pkg.dg_mesh_counts(v, t[6:])
    with pytest.raises(pkg.DgError, match=r"\[-2\]"):
        pkg.dg_mesh_counts(v, np.array([[0, 0, 1, 2]], dtype=np.int32))
    assert lib.dg_reference_element(3, 9, None, None, None, None, None) == -1
    assert b"N in 1..8" in lib.dg_last_error()
    nbytes = ctypes.c_uint64(0)
    m, keep = pkg.binding._mesh(v, t)
    assert lib.dg_workspace_bytes(ctypes.byref(m), 3, 2, 64, ctypes.byref(nbytes)) == 0 and nbytes.value > 48 * 20 * 4 * 8 * 3
    assert lib.dg_workspace_bytes(ctypes.byref(m), 3, 13, 64, ctypes.byref(nbytes)) == -1
    assert lib.dg_workspace_bytes(ctypes.byref(m), 3, 2, 16, ctypes.byref(nbytes)) == -1
    bad = np.array([0, 0, 3, 0, 0, 0], dtype=np.int32)
    out = np.zeros(4, dtype=np.int32)
    assert lib.dg_mesh_counts(ctypes.byref(m), pkg.binding._ip(bad), pkg.binding._ip(out)) == -1
