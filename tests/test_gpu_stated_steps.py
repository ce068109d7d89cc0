"""Parity with the ORACLE after the STATED step counts of BASELINE.json's configs[2..4] (-m gpu).

north_star: "match the oracle ... on p, u and all auxiliary fields after the stated step counts"; SURVEY.md §8(d):
"the parity run itself must cover the full stated step count at least once per precision".  The oracle cannot run
196,608 .. 1,572,864 tets for 100-200 steps, so each config's RULE (mesh recipe, materials, N, J, pulse, seed,
step count, precisions) is run on a hex grid the oracle finishes in about a minute: 8^3 hexes (3,072 tets: 384
batches of 8, several per persistent CTA) for configs[2] and configs[4], 3^3 hexes for the degree sweep of
configs[3].  Every field and every auxiliary set is compared on its own (tests/parity.py).  The full-size meshes
are covered by tests/test_gpu_full_configs.py (oracle on a corner block for the first steps)."""
import numpy as np
import pytest

import parity
from workloads import make_workload

pytestmark = pytest.mark.gpu
TOL = {64: 1e-11, 32: 1e-4}


@pytest.fixture(scope="module")
def cfg5_rule():
    w = make_workload("cfg5", n=8)
    assert (w.N, w.J, w.nsteps) == (5, 8, 100) and np.unique(w.c).size == 4
    return w, parity.run_oracle(w)


@pytest.mark.parametrize("prec", [64, 32])
def test_cfg5_rule_all_100_steps(cfg5_rule, prec):
    """configs[4] (N=5, J=8, layered c in U[1.5,4.5], pulse at the corner), 100 steps, fp64 and fp32, default kernels
    (k_vol3d_ws<5> / k_vol3d_tf32<5>, the ones bench.py times)."""
    w, ora = cfg5_rule
    lib = parity.run_library(w, precision=prec)
    assert lib["dt"] == pytest.approx(ora["dt"], rel=1e-14)
    parity.check(parity.compare(lib, ora), TOL[prec])


def test_cfg3_rule_all_200_steps():
    """configs[2] (perturbed interior vertices, 4 layers of c in U[1,3], N=4, J=6), 200 steps, fp64."""
    w = make_workload("cfg3", n=8)
    assert (w.N, w.J, w.nsteps) == (4, 6, 200)
    lib, ora = parity.run_library(w), parity.run_oracle(w)
    parity.check(parity.compare(lib, ora), TOL[64])


_cfg4_oracle = {}


def _cfg4(N, J):
    if (N, J) not in _cfg4_oracle:
        w = make_workload("cfg4", n=3, N=N, J=J)
        assert w.nsteps == 100
        _cfg4_oracle[(N, J)] = (w, parity.run_oracle(w))
    return _cfg4_oracle[(N, J)]


@pytest.mark.parametrize("J", [0, 4, 8])
@pytest.mark.parametrize("N,prec", [(1, 64), (4, 64), (6, 64), (8, 64), (2, 32), (6, 32), (8, 32)])
def test_cfg4_rule_all_100_steps(N, J, prec):
    """configs[3]: the degree sweep's ends and middle, every J of the sweep, 100 steps, default kernel of each
    (precision, N): k_vol3d_mma / k_vol3d_mmag in fp64, k_vol3d / k_vol3d_tf32g in fp32."""
    w, ora = _cfg4(N, J)
    lib = parity.run_library(w, precision=prec)
    parity.check(parity.compare(lib, ora), TOL[prec], aux=J > 0)
