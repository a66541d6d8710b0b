"""CPU checks of bench.py's contract: the reference arm (the oracle timed on the host cores) prints one JSON line with the
keys the driver reads, flags its extrapolation, reports the time it actually ran, and spells `config` exactly like the
CUDA arm does (both go through bench.config_dict)."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "C0", "--steps", "2",
                          "--warmup", "1"], capture_output=True, text=True, cwd=ROOT, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1
    line = json.loads(lines[0])
    for k in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e"):
        assert k in line, k
    assert line["impl"] == "reference" and line["metric"] == "energy_point_solves_per_s" and line["higher_is_better"] is True
    cb = line["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and "sample" in cb
    assert cb["extrapolated"] is True and cb["scale"] == 2.0            # C0: nb = 8 truncated to 4 blocks
    # the line's time is the time that elapsed, the value is that time extrapolated by `scale`
    assert abs(line["value"] * (line["ms_per_step"] * 1e-3) * cb["scale"] - 1.0) < 1e-9
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0


def test_reference_arm_config_is_config_dict_of_the_workload():
    """Both arms build `config` with bench.config_dict (the driver compares the two lines): the reference arm's printed
    config must be exactly that function's value for the workload (the CUDA arm passes the same function's value through)."""
    sys.path.insert(0, ROOT)
    import bench
    from paper_1812_01396_b200 import inputs
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "C0", "--steps", "1",
                          "--warmup", "0"], capture_output=True, text=True, cwd=ROOT, timeout=300)
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["config"] == bench.config_dict(inputs.CONFIGS["C0"], 1)
    assert line["steps_timed"] == 1 and line["warmup_run"] == 0 and line["gpus_used"] == 0
    d = bench.config_dict(inputs.CONFIGS["C4"], 1)
    assert d["workload"] == "C4" and d["bs"] == 4096 and d["nb"] == 24 and d["n_energy_per_gpu"] == 4 and d["nrhs"] == 512
    assert "L2" in d["l2"]


def test_reference_sample_does_not_depend_on_the_number_of_repeats():
    """the two arms of one driver call must quote the same baseline.  The oracle sample is a function of the
    workload only; the reference arm keeps its run time bounded by repeating it fewer times, never by shrinking it."""
    sys.path.insert(0, ROOT)
    import bench
    from paper_1812_01396_b200 import inputs
    import inspect
    assert list(inspect.signature(bench.oracle_sample).parameters) == ["cfg"]
    _, scale1, desc1 = bench.oracle_sample(inputs.CONFIGS["C0"])
    _, scale2, desc2 = bench.oracle_sample(inputs.CONFIGS["C0"])
    assert (scale1, desc1) == (scale2, desc2) and scale1 == 2.0
    # repetitions: all of warm-up + steps when they fit the budget at the first repetition's pace, else what fits, >= 1
    assert bench.reference_repetitions(0.01, 3, 20) == 23
    assert bench.reference_repetitions(13.5, 3, 20, budget=150.0) == 11
    assert bench.reference_repetitions(500.0, 3, 20, budget=150.0) == 1
    assert bench.reference_repetitions(13.5, 3, 20, budget=150.0) == bench.reference_repetitions(13.5, 1, 50, budget=150.0)


def test_full_size_oracle_record_comes_from_the_fingerprint_headers():
    sys.path.insert(0, ROOT)
    import bench
    from paper_1812_01396_b200 import inputs
    for name in ("C3", "C4"):
        rec = bench.full_size_oracle_record(inputs.CONFIGS[name])
        head = open(os.path.join(ROOT, "tests", "golden", f"{name.lower()}_fingerprint.txt")).readlines()[1]
        assert rec is not None and f"in {rec['seconds_one_energy']} s on {rec['cores']} host cores" in head
        assert "not this box" in rec["source"]
    assert bench.full_size_oracle_record(inputs.CONFIGS["C0"]) is None    # no stored full-size run: nothing is made up
