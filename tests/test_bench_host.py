"""Host logic of bench.py that needs no GPU: the byte/flop model against DESIGN.md's figures, the
replica aggregation, and the N>1 plumbing (barrier + max over ranks) on a world-size-2 gloo group."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import bench  # noqa: E402
import workloads as W  # noqa: E402


def test_byte_model_matches_survey_totals():
    """190 B (fp64, 8 ppc, sort every 4), 98.5 B (fp32, 8 ppc), 325 B (fp64, 2 ppc)."""
    assert bench.model(W.CONFIGS["C2"])["step_bytes"] == pytest.approx(104 + 45 + 41, abs=0.01)
    assert bench.model(W.CONFIGS["C3"])["step_bytes"] == pytest.approx(52 + 22.5 + 24, abs=0.01)
    c4 = W.scaled(W.CONFIGS["C4"], W.CONFIGS["C4"].n_cells, z_first=0)     # 2 ppc everywhere
    assert bench.model(c4)["step_bytes"] == pytest.approx(104 + 180 + 41, abs=0.01)


def test_aggregate_is_all_ranks_over_slowest():
    assert bench.aggregate(1000, 4, 10, 2.0) == pytest.approx(1000 * 4 * 10 / 2e-3)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


_WORKER = r"""
import json, os, sys
sys.path.insert(0, %(root)r)
import bench
dist = bench.init_dist("gloo")
rank, _, world = bench.dist_env()
bench.barrier(dist)
ms = bench.max_over_ranks(dist, 10.0 + 5.0 * rank)      # rank 1 is the slow one
val = bench.aggregate(1000, world, 4, ms)
bench.barrier(dist)
print(json.dumps({"rank": rank, "ms": ms, "value": val}))
"""


def test_world_size_two_gloo_max_over_ranks(tmp_path):
    port = _free_port()
    script = tmp_path / "worker.py"
    script.write_text(_WORKER % {"root": ROOT})
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=240)
        assert p.returncode == 0, e
        outs.append(json.loads(o.strip().splitlines()[-1]))
    for o in outs:
        assert o["ms"] == 15.0                                   # the max, on every rank
        assert o["value"] == pytest.approx(1000 * 2 * 4 / 15e-3)


def test_reference_arm_other_ranks_exit_without_work():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=240)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_reference_arm_prints_contract_line():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "C1",
                        "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "particle-steps/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["value"] == line["value"]
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
