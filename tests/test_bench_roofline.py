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


def test_workload_config_names_what_is_run(bench):
    from workloads import make_workload
    w = make_workload("cfg1")
    c = bench.workload_config("cfg1", w)
    assert c == {"workload": "cfg1", "n_hex": 2, "hex_grid": [2, 2, 2], "N": 3, "J": 2, "K": 48, "nodes": 960}


def test_habc_numerators(bench):
    """DESIGN.md §7, HABC levels, at configs[3]'s J = 4, N = 4 in fp64 (T = 6,912, E = 288, C = 8), retyped here."""
    T, E, C, J, Nfp, N1 = 6912, 288, 8, 4, 15, 5
    work = bench.habc_work_per_launch(4, J, T, E, C, 64)
    assert work["face2d"] == (T * (J * (12 * 15 + 45) * 8 + (15 + 15 + 23) * 8 + 72), T * J * (15 * (120 + 30 + 30) + 210))
    assert work["edge1d"] == (E * (16 * 46 * 8 + 48 * 8 + 8), E * 16 * (5 * 36 + 28))
    assert work["close_face"] == (T * (15 * 14 * 8 + 16), T * 15 * 20)
    assert work["close_edge"] == (E * 5 * 56 * 8 + 128 * 8, E * 5 * (224 + 48))
    assert work["close_corner"] == (C * 144 * 8 + 9 * 256 * 8, C * (18 * 256 + 192))
    # the state traffic dominates every count, and fp32 moves about half the bytes
    assert work["face2d"][0] > T * J * 12 * Nfp * 8
    half = bench.habc_work_per_launch(4, J, T, E, C, 32)
    assert 0.5 <= half["face2d"][0] / work["face2d"][0] < 0.55 and half["face2d"][1] == work["face2d"][1]
    assert bench.habc_work_per_launch(3, 0, T, E, C, 64)["close_edge"] == (0, 0)


def test_reference_arm_names_the_sample_it_times(bench, monkeypatch, capsys):
    """--impl reference times the oracle on the config's rule on an 8^3 grid: its `config` says so (K = 3,072 of the
    sample, not cfg5's 1,572,864) and names the full configuration in `sample_of`."""
    import argparse
    import json
    seen = {}

    def fake_sample(workload, precision, budget_s=20.0):
        seen["n"] = min(bench.CONFIGS[workload]["n"], 8)
        return 1.0e5, "stub", 1, 0.5, 8
    monkeypatch.setattr(bench, "oracle_sample", fake_sample)
    bench.run_reference(argparse.Namespace(workload="cfg5", steps=1, warmup=0, gpus=1, n=None, N=None, J=None))
    line = json.loads(capsys.readouterr().out)
    assert line["impl"] == "reference" and line["config"]["sample_of"] == "cfg5"
    assert (line["config"]["n_hex"], line["config"]["K"], line["config"]["N"], line["config"]["J"]) == (seen["n"], 3072, 5, 8)
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["cpu_baseline"]["kind"] == "oracle"


def test_traffic_table_names_the_default_kernels(repo_root):
    rows = [ln.split(",", 3) for ln in open(os.path.join(repo_root, "profiles", "traffic.csv")).read().splitlines()[1:]]
    assert {r[0]: r[2] for r in rows} == {"cfg5_f64": "k_vol3d_ws<5>", "cfg5_f32": "k_vol3d_tf32<5>"}
    for r in rows:
        assert os.path.exists(os.path.join(repo_root, r[3].split(" ")[0])), r[3]
        assert 0.5 < float(r[1]) / 1572864 / (10068 if r[0].endswith("f64") else 5044) < 1.0   # below the algorithmic count
