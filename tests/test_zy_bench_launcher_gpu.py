"""bench.py --gpus N started WITHOUT torchrun must start its N ranks itself (it used to run one rank and print
n_gpus = 1).  Run here as a functional check on one GPU: `--dist-backend gloo` lets the two ranks share the device (every
collective is a host-level call, no kernel waits for another rank's).  Collected late (file name) so that a failure here
cannot hide the parity tests under `pytest -x`."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
pytestmark = pytest.mark.gpu


def run_bench(*extra, env=None):
    e = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    e.update(env or {})
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--workload", "C0", "--steps", "2", "--warmup", "3",
                           "--no-e2e", "--no-cpu-baseline", *extra], capture_output=True, text=True, cwd=ROOT, timeout=600, env=e)


def test_gpus_2_without_torchrun_starts_two_ranks():
    out = run_bench("--gpus", "2", "--dist-backend", "gloo")
    assert out.returncode == 0, out.stderr[-3000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1                                   # rank 0 alone prints
    line = json.loads(lines[0])
    assert line["n_gpus"] == 2 and line["config"]["parallelism"] == "energy-parallel x2"
    one = json.loads([ln for ln in run_bench().stdout.splitlines() if ln.startswith("{")][0])
    assert one["n_gpus"] == 1
    # weak scaling: twice the energy points in the job; rank 0 of the 2-rank run owns energies 0, 2, 4, 6 of an 8-point grid,
    # so the grids differ and only the closed-form invariant is compared: 0 <= T <= bs
    assert 0.0 <= line["T_first_energy"] <= 16.0 and 0.0 <= one["T_first_energy"] <= 16.0


def test_gpus_must_agree_with_world_size():
    out = run_bench("--gpus", "1", env={"WORLD_SIZE": "2", "RANK": "0", "LOCAL_RANK": "0"})
    assert out.returncode != 0 and "must agree" in (out.stderr + out.stdout)


def test_more_gpus_than_devices_fails_loudly():
    import torch
    n = torch.cuda.device_count() + 1
    out = run_bench("--gpus", str(n))
    assert out.returncode != 0 and "visible" in (out.stderr + out.stdout)
