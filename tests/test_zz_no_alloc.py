"""dg_get_aux_fields_noalloc: the auxiliary-field read-back for hosts that cannot obtain device memory.

Some users of libdg_habc.so have nobody to ask for GPU memory at the moment they want the auxiliary fields: every
byte of the device was handed to another pool when the process started, or another thread is inside a global-mode
stream capture (cudaMalloc is an error there), or the loop cannot afford the device-wide synchronisation that
cudaMalloc / cudaFree bring.  For them the library stages the export through a fixed 4 MiB array that is part of its
own image (DG_NOALLOC_MAX_VALUES doubles) instead of through the solver's workspace.

What is checked here: the new call returns what dg_get_fields returns for the same state -- the same kernel converts
the same data, so the comparison is for equality, tighter than the 1e-11 / 1e-4 of the parity tests -- on two calls in
a row, where the second call finds the array full of the first call's values (a larger solver's, in the last test);
and a solver beyond the limit is turned away with DG_ENOMEM before anything is launched.

The file name sorts last on purpose: pytest -x stops at the first failure, and this test must not hide the others."""
import numpy as np
import pytest

import parity
from workloads import make_workload

pytestmark = pytest.mark.gpu


def _solver(w, precision=64):
    from paper_1610_05023_b200 import Solver
    s = Solver(w.verts, w.tets, w.N, w.J, w.c, w.rho, precision=precision)
    x, y, z = s.get_nodes()
    s.set_initial(*parity.initial_on(w, x, y, z, w.c, w.rho))
    return s


def _same(got, want):
    """(face_aux, edge_aux) of the no-allocation call against dg_get_fields': equal, and carrying data"""
    for g, e, name in zip(got, want, ("face_aux", "edge_aux")):
        assert g.shape == e.shape and e.size > 0, name
        assert np.linalg.norm(e) > 0, name + " is empty: the comparison would be vacuous"
        assert np.array_equal(g, e), (name, float(np.abs(g - e).max()))


@pytest.mark.parametrize("prec", [64, 32])
def test_two_calls_in_a_row_match_get_fields(prec):
    """BASELINE configs[1] (3,072 tets, N = 4, J = 4: 153,600 auxiliary values).  First call after 5 steps, second
    call after 3 more: the array then still holds the first call's values everywhere, and every one must have been
    replaced."""
    s = _solver(make_workload("cfg2"), prec)
    s.step(5)
    first = s.get_aux_fields_noalloc()
    _, fa, ea = s.get_fields()
    _same(first, (fa, ea))
    s.step(3)
    second = s.get_aux_fields_noalloc()
    _, fa2, ea2 = s.get_fields()
    _same(second, (fa2, ea2))
    assert not np.array_equal(first[0], second[0])          # the state really moved between the two calls
    # and once more on the unchanged state: still the same answer
    _same(s.get_aux_fields_noalloc(), (fa2, ea2))
    s.close()


def test_small_solver_after_a_larger_one():
    """Two solvers share the array.  The smaller one's call comes second and must not pick up anything the larger
    one left behind beyond its own length (configs[0]: 3,648 values, after configs[1]'s 153,600)."""
    big, small = _solver(make_workload("cfg2")), _solver(make_workload("cfg1"))
    big.step(4)
    small.step(7)
    got_big = big.get_aux_fields_noalloc()
    got_small = small.get_aux_fields_noalloc()
    _same(got_big, big.get_fields()[1:])
    _same(got_small, small.get_fields()[1:])
    big.close()
    small.close()


def test_size_beyond_the_limit_is_refused():
    """N = 4, J = 12 on 8^3 hexes has 552,960 auxiliary values, more than the 524,288 the array holds: DG_ENOMEM (-4)
    with both numbers in the message, the output untouched; dg_get_fields still serves that solver."""
    from paper_1610_05023_b200 import DgError, Solver
    w = make_workload("cfg4", n=8, N=4, J=12, nsteps=1)
    s = _solver(w)
    need = s.T * s.J * 3 * s.Nfp + s.E * s.J * s.J * 2 * (s.N + 1)
    assert need == 552960 > Solver.NOALLOC_MAX_VALUES == 1 << 19
    s.step(1)
    with pytest.raises(DgError) as e:
        s.get_aux_fields_noalloc()
    assert "[-4]" in str(e.value) and "552960" in str(e.value) and "524288" in str(e.value)
    _, fa, ea = s.get_fields()
    assert np.linalg.norm(fa) > 0
    s.close()


def test_no_auxiliary_fields_is_an_empty_answer():
    """J = 0 (basic ABC): there is nothing to export; the call succeeds and returns empty arrays."""
    s = _solver(make_workload("cfg4", n=2, N=2, J=0, nsteps=1))
    s.step(1)
    fa, ea = s.get_aux_fields_noalloc()
    assert fa.size == 0 and ea.size == 0
    s.close()
