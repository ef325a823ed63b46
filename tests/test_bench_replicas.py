"""The N > 1 path of bench.py on CPU (gloo, world_size 2): replicas only, so the only
collectives are the MAX of the per-rank times and the SUM of the per-rank units
(DESIGN.md section 7).  Also the reference arm under torchrun: rank 0 alone prints the line."""
import json
import os
import subprocess
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent

WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank = dist.get_rank()
times, counts = bench.aggregate_replicas([10.0 + 5.0 * rank, 1.0 + rank], [3.0 + rank, 7.0], dist, "cpu")
if rank == 0:
    print(json.dumps({{"times": times, "counts": counts, "world": dist.get_world_size()}}))
dist.destroy_process_group()
"""


def _torchrun(args, port):
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="2")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(port)] + args
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)


def test_replica_aggregation_gloo_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=str(ROOT)))
    r = _torchrun([str(script)], 29611)
    assert r.returncode == 0, r.stderr[-2000:]
    line = [l for l in r.stdout.splitlines() if l.startswith("{")][-1]
    out = json.loads(line)
    assert out["world"] == 2
    assert out["times"] == [15.0, 2.0]          # max over ranks
    assert out["counts"] == [7.0, 14.0]         # sum over ranks


def test_reference_arm_under_torchrun_prints_one_line():
    r = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "1",
                   "--workload", "config1"], 29612)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    out = json.loads(lines[0])
    assert out["impl"] == "reference" and out["n_gpus"] == 2
    assert out["cpu_baseline"]["kind"] == "oracle" and out["e2e"]["h2d_bytes_per_step"] == 0
    assert out["value"] > 0 and out["gpu_launches"] == 0


STUB_WORKER = r"""
import os, sys, json, argparse
sys.path.insert(0, {root!r})
import bench
from workloads import make_workload

def fake_measure(args, w, wname, rank, local, dist):
    # rank-dependent numbers: rank 1 is the slower replica
    return {{"t_ms": 100.0 + 50.0 * rank, "t_e2e_ms": 300.0 + 100.0 * rank, "cycles_total": 10 + rank,
            "e2e_cycles": 4, "e2e_steps": 2, "launches": 123, "status": 0, "cycles": 5, "relres": 1e-9,
            "levels": 4, "t_solve_ms": 20.0, "t_setrho_ms": 1.0, "t_vc_ms": 2.0, "launches_per_vcycle": 30,
            "kernels": {{}}, "clocks": {{"sm_mhz": None, "reasons": []}}, "proj": None, "seq": None}}

args = argparse.Namespace(gpus=2, steps=2, warmup=3, no_cpu_baseline=True)
w = make_workload(1, None)
bench.run_cuda(args, w, "config1 stub", measure=fake_measure, backend="gloo")
"""


def test_run_cuda_control_flow_world2_with_stubbed_solver(tmp_path):
    """bench.run_cuda at world size 2 (gloo): every rank measures, rank 0 alone prints ONE line whose
    value is the summed units over the MAX time."""
    script = tmp_path / "stub_worker.py"
    script.write_text(STUB_WORKER.format(root=str(ROOT)))
    r = _torchrun([str(script)], 29613)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    out = json.loads(lines[0])
    assert out["n_gpus"] == 2 and out["scaling"] == "weak" and out["gpu_launches"] == 123
    n_cells, upd = 32 ** 3, 4
    assert out["value"] == pytest.approx(n_cells * upd * (10 + 11) / 0.150 / 1e9)      # max over ranks: 150 ms
    assert out["ms_per_step"] == pytest.approx(75.0)
    assert out["e2e"]["value"] == pytest.approx(n_cells * upd * 8 / 0.400 / 1e9)
    assert "cpu_baseline" not in out and out["time_to_rtol_best"] is None and out["time_to_rtol_ms"] == 20.0


def test_gpus_flag_spawns_ranks_when_no_launcher_did():
    import argparse
    import bench

    a = argparse.Namespace(gpus=4)
    cmd = bench.spawn_command(a, ["--gpus", "4", "--steps", "2"], {})
    assert cmd[1:4] == ["-m", "torch.distributed.run", "--nnodes=1"] and "--nproc-per-node=4" in cmd
    assert cmd[-4:] == ["--gpus", "4", "--steps", "2"] and cmd[-5].endswith("bench.py")
    assert "127.0.0.1" in cmd
    assert bench.spawn_command(a, [], {"WORLD_SIZE": "4"}) is None          # already under a launcher
    assert bench.spawn_command(argparse.Namespace(gpus=1), [], {}) is None


def test_both_arms_name_the_workload_with_the_same_config_keys():
    import bench
    from workloads import make_workload

    w = make_workload(1, None)
    c = bench.workload_config(w, "x")
    assert set(c) == {"workload", "cells", "bc", "cycle", "rtol", "step", "parallelism"}
