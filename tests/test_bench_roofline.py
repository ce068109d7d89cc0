"""CPU checks of bench.py's roofline numerators and of its JSON plumbing (no GPU, no library calls): the algorithmic
bytes / flops per element are the figures DESIGN.md §7 states, and both arms print the same workload `config`."""
import importlib.util
import os

import pytest


@pytest.fixture(scope="module")
def bench(repo_root):
    spec = importlib.util.spec_from_file_location("bench", os.path.join(repo_root, "bench.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


def test_algorithmic_work_per_element_matches_design(bench):
    # B(N, prec) = (prec / 8) (16 Np + 16 Nfp + 24) + 20;  F(N) = Np (12 Np + 24 + 8 Nfp + 40) + 4 Nfp 14
    assert bench.algorithmic_bytes_per_element(5, 64) == 10068
    assert bench.algorithmic_bytes_per_element(5, 32) == 5044
    assert bench.algorithmic_flops_per_element(5) == 51800
    for N in range(1, 9):
        Np, Nfp = (N + 1) * (N + 2) * (N + 3) // 6, (N + 1) * (N + 2) // 2
        # q and res in and out are 16 Np values: never less than that, and the traces add at most the 4 faces' nodes
        assert 16 * Np * 8 < bench.algorithmic_bytes_per_element(N, 64) <= (16 * Np + 16 * Nfp + 24) * 8 + 20
        # six matvec rows per node (12 Np flop) dominate from N = 3 on
        assert bench.algorithmic_flops_per_element(N) > 12 * Np * Np


def test_both_arms_name_the_same_workload(bench):
    from workloads import make_workload
    w = make_workload("cfg1")
    c = bench.workload_config("cfg1", w)
    assert c == {"workload": "cfg1", "n_hex": 2, "hex_grid": [2, 2, 2], "N": 3, "J": 2, "K": 48, "nodes": 960}


def test_traffic_table_names_the_default_kernels(repo_root):
    rows = [ln.split(",", 3) for ln in open(os.path.join(repo_root, "profiles", "traffic.csv")).read().splitlines()[1:]]
    assert {r[0]: r[2] for r in rows} == {"cfg5_f64": "k_vol3d_ws<5>", "cfg5_f32": "k_vol3d_tf32<5>"}
    for r in rows:
        assert os.path.exists(os.path.join(repo_root, r[3].split(" ")[0])), r[3]
        assert 0.5 < float(r[1]) / 1572864 / (10068 if r[0].endswith("f64") else 5044) < 1.0   # below the algorithmic count
