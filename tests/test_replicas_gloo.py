"""The N > 1 path of bench.py on CPU: world_size 2 over gloo ("replicas only").  Covers the host logic
only -- rank/env handling, barrier, max-over-ranks timing, whole-job aggregation, rank-0 reporting; the kernels
themselves are single-GPU and covered by the -m gpu parity tests."""
import json
import os
import socket
import subprocess
import sys
import textwrap


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


WORKER = textwrap.dedent("""
    import json, sys
    sys.path.insert(0, {root!r})
    from paper_1610_05023_b200.replicas import Replicas
    rep = Replicas.from_env("gloo")
    rep.barrier()
    seconds = 0.5 + 0.25 * rep.rank                       # rank 1 is the slow one
    out = dict(rank=rep.rank, world=rep.world, local=rep.local, root=rep.is_root,
               tmax=rep.max_over_ranks(seconds), rate=rep.aggregate_rate(1000.0, seconds),
               all_true=rep.all_true(True), one_false=rep.all_true(rep.rank != 1))
    rep.barrier()
    rep.close()
    print("RESULT " + json.dumps(out), flush=True)
""")


def test_world_size_2_gloo(repo_root, tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=repo_root))
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), GLOO_SOCKET_IFNAME="lo")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    results = {}
    for p in procs:
        out, err = p.communicate(timeout=240)
        assert p.returncode == 0, err[-2000:]
        line = [ln for ln in out.splitlines() if ln.startswith("RESULT ")][0]
        r = json.loads(line[len("RESULT "):])
        results[r["rank"]] = r
    assert set(results) == {0, 1}
    for rank, r in results.items():
        assert r["world"] == 2 and r["local"] == rank and r["root"] == (rank == 0)
        assert r["tmax"] == 0.75                               # the slowest rank's time, on every rank
        assert abs(r["rate"] - 2 * 1000.0 / 0.75) < 1e-9       # whole-job units over the slowest rank's time
        assert r["all_true"] is True and r["one_false"] is False


def test_single_process_needs_no_process_group(monkeypatch):
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK"):
        monkeypatch.delenv(k, raising=False)
    from paper_1610_05023_b200.replicas import Replicas
    rep = Replicas.from_env("gloo")
    assert (rep.rank, rep.world, rep.local, rep.backend) == (0, 1, 0, None)
    assert rep.max_over_ranks(1.5) == 1.5 and rep.aggregate_rate(10.0, 2.0) == 5.0 and rep.is_root
    rep.close()


def test_reference_arm_runs_on_rank0_only(repo_root):
    """bench.py --impl reference under torchrun: ranks != 0 exit 0 without work or output."""
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT="1")
    r = subprocess.run([sys.executable, os.path.join(repo_root, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=240)
    assert r.returncode == 0 and r.stdout.strip() == ""
