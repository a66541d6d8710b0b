#!/usr/bin/env python
"""bench.py -- energy-point solves/s of the SplitSolve hot path (a0-a7) on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C4|C3|C2|C1|C0] [--impl ours|reference]

One "step" = one pass of the whole hot path over one batch of synthetic input: ss_solve (+ ss_transmission) over
all n_energy energy points of the workload.  Default workload: C4 (BASELINE.json configs[4], the largest single-GPU
configuration); at N = 1 the line also carries an "also" block with the same measurement on C3 (configs[3], the other
bs >= 2048 target configuration).  N > 1 (torchrun, one rank per GPU): the energy grid is n_energy*N
points and rank r owns every N-th point (energy points are independent: PAPER.md L204, L210, L262), each rank a
full replica of H and S; no collective in the data path, T(E) all-gathered at the end (8 B per energy).
Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1812_01396_b200 import inputs  # noqa: E402

METRIC = "energy_point_solves_per_s"
UNIT = "solves/s"
# FP64 roofline denominator: 148 SMs x 64 FP64 FMA/clk/SM x 2 flop x 1.965 GHz; the DMMA
# microbenchmark in the library (ss_fp64_peak_tflops) measures 37.07 on this pool's B200s and is printed beside it.
FP64_PEAK_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
# real flops executed per algorithmic (LAPACK-convention) flop: 4M executes 8 per complex multiply-add, 3M 6
EXECUTED_RATIO = {False: 1.0, True: 0.75}
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant GEMM kernel: read from the committed summary of
# the `ncu --set full` capture (profiles/*_gemm_traffic.csv: kernel,M,N,K,batch,dram_bytes_read,dram_bytes_write,source)
TRAFFIC_CSVS = [os.path.join(ROOT, "profiles", f) for f in ("r03_gemm_traffic.csv", "r02_gemm_traffic.csv")]


def ncu_traffic(is3m: bool, bs: int, batch: int):
    """(bytes per launch, over-fetch ratio, note) of the dominant GEMM launch of the timed workload -- M = N = K = bs, `batch`
    chains per launch (two chains per energy of a stream group) -- from the committed ncu summaries, or (None, None, why).
    Rows are matched by (kernel, M, N, K) and then by batch; a row of another batch size is used only when there is none of
    the same, and the note says so.  over-fetch = captured DRAM bytes / algorithmic bytes of the CAPTURED launch."""
    want = "zgemm3m_kernel" if is3m else "zgemm_kernel"
    rows = []
    for path in TRAFFIC_CSVS:
        try:
            with open(path) as f:
                for ln in f:
                    r = ln.strip().split(",")
                    if len(r) >= 8 and r[0] == want:
                        rows.append((r, path))
        except OSError:
            pass
    same = [(r, p) for r, p in rows if tuple(int(x) for x in r[1:4]) == (bs, bs, bs)]
    if not same:
        return None, None, f"no ncu capture of {want} at {bs}^3 in profiles/ (captured: {sorted({r[1] for r, _ in rows})})"
    exact = [(r, p) for r, p in same if int(r[4]) == batch]
    r, path = (exact or same)[0]
    M, N, K, b = (int(x) for x in r[1:5])
    rd, wr = float(r[5]), float(r[6])
    alg = 16.0 * (M * K + K * N + M * N) * b
    note = (f"{os.path.relpath(path, ROOT)}: {r[0]} {M}x{N}x{K} x{b}, read {rd:.4g} + write {wr:.4g} B per launch, algorithmic "
            f"{alg:.4g} B, over-fetch {(rd + wr) / alg:.2f}x; capture {','.join(r[7:])}" +
            ("" if exact else f"; NOTE: the timed step launches batch {batch}, no capture of that batch size is committed"))
    return rd + wr, (rd + wr) / alg, note


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="C4", choices=sorted(inputs.CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--gemm-variant", type=int, default=None, help="complex-GEMM kernel variant (binding.GEMM_VARIANTS); "
                    "default: the library default (3M)")
    ap.add_argument("--stream-groups", type=int, default=None, help="stream groups the energies are split over "
                    "(library default 4; 1 = single stream)")
    ap.add_argument("--option", action="append", default=[], metavar="NAME=INT", help="extra ss_set_option calls (tuning)")
    ap.add_argument("--trace", default=None, help="write the phase timeline of the last timed step to this CSV")
    ap.add_argument("--split", default="energy", choices=["energy", "column", "spatial"], help="N > 1: 'energy' = every rank its own "
                    "energies (default, SURVEY 8(e)); 'column' = pairs of ranks share their energies, first block column of "
                    "A^-1 on the even rank, last on the odd one; 'spatial' = pairs of ranks share their energies, top half of the device on the "
                    "even rank, bottom half on the odd one, SPIKE-style merge (SURVEY 8(f2), PAPER.md L167, L169)")
    ap.add_argument("--real-energies", action="store_true", help="variant of the workload with Im E = 0 and the energy grid moved "
                    "above the spectrum ([3.5, 4.5]: A definite), for the Hermitian modes of SURVEY 8(f1) (--option hermitian=1|2)")
    ap.add_argument("--emulate-split", default=None, choices=["column", "spatial"], help="ONE GPU: run the per-rank work of the "
                    "two-GPU splits of SURVEY 8(f2) rank after rank (two handles), time each rank's phases with CUDA events and "
                    "print the per-rank critical path; the exchanges are device copies here, their NVLink time is estimated "
                    "from the bytes (see profiles/r02_split_emulation.md)")
    ap.add_argument("--dist-backend", default="nccl", choices=["nccl", "gloo"], help="N > 1: torch.distributed backend.  'gloo' is "
                    "for exercising the N > 1 code paths on a box with fewer GPUs than ranks (ranks share GPUs; every collective "
                    "is a host-level call, no kernel waits for another rank's): a functional check, never a measurement")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-also", action="store_true", help="skip the second block (C3) of the default C4 line")
    ap.add_argument("--kernel", default=None, choices=["gemm", "density", "lu"], help="time ONE kernel alone through its C-ABI "
                    "entry point instead of the hot path (tuning, and the command of the ncu --set full captures in profiles/)")
    ap.add_argument("--dims", type=int, nargs="*", default=[], help="--kernel gemm: M N K batch [reps]; --kernel density: "
                    "n_energy n nrhs [reps]; --kernel lu: n batch [reps]")
    ap.add_argument("--beta", type=float, default=0.0, help="--kernel gemm: C = A B + beta C (1 = the in-place update form)")
    ap.add_argument("--sumplane", action="store_true", help="--kernel gemm: pass re + im planes of A and B (ss_zgemm_batched_sums)")
    ap.add_argument("--raster", type=int, default=None, help="--kernel gemm: tile rows per raster group (library default 16)")
    ap.add_argument("--variants", default=None, help="--kernel gemm: comma-separated GEMM variants (default: library default)")
    ap.add_argument("--calibrate-oracle", action="store_true", help="time the oracle on the full and on the truncated C2 "
                    "device (one energy, Inj columns only) and print the ratio that the extrapolated cpu_baseline rests on")
    return ap.parse_args()


# ---------------------------------------------------------------------------------------------------------
# clocks
# ---------------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.samples = []
        self._stop = threading.Event()
        self._t = None

    def _run(self):
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-i",
                                      str(self.index)], capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.samples.append([x.strip() for x in out.split(",")])
            except Exception:
                pass
            self._stop.wait(0.2)

    def __enter__(self):
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._t.join(timeout=6)

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for s in self.samples:
            try:
                sm.append(float(s[0])); mx.append(float(s[1]))
                for n, v in zip(names, s[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ---------------------------------------------------------------------------------------------------------
# the oracle legs (cpu_baseline and --impl reference): the only places bench.py executes oracle/
# ---------------------------------------------------------------------------------------------------------
def config_dict(cfg, world):
    """One spelling of `config` for both arms (the driver compares them)."""
    return {"workload": cfg.name, "bs": cfg.bs, "nb": cfg.nb, "n_energy_per_gpu": cfg.n_energy, "nrhs": cfg.nrhs,
            "parallelism": f"energy-parallel x{world}",
            "l2": "inputs larger than L2 (H,S,slots >> 126 MB)" if cfg.bs >= 512 else
            "small workload: inputs fit L2 (launch-bound config)"}


REFERENCE_BUDGET_S = 150.0     # --impl reference: host seconds the timed oracle repetitions may take in total


_sample_inputs = {}


def oracle_sample(cfg):
    """Times the oracle, as it stands, on a bounded sample of the workload: ONE energy point of the same generator
    with the device truncated to nb_s blocks (nb_s = 2 for bs >= 1024, else min(nb, 4)), solved by the plain definition
    (LU of the full matrix: oracle/dense.py when the truncated matrix is <= 8192 rows -- with 2 blocks the band of the
    block-tridiagonal matrix IS the whole matrix -- else oracle/banded.py).  The full-size oracle (banded LU, the only
    form that fits the host) costs 64 nb bs^3 flops for the factorisation, linear in nb, so the per-energy time is
    EXTRAPOLATED by nb / nb_s and flagged as such; `--calibrate-oracle` measures that ratio on C2, and the full-size
    Tier B times of one energy point of C3 / C4 are in the headers of tests/golden/c{3,4}_fingerprint.txt.
    The sample depends on the workload ONLY (never on --steps / --warmup), so the cpu_baseline of the CUDA arm and the
    --impl reference arm time the same thing and their values differ by timing noise alone; the reference arm bounds its
    run time by capping how often it repeats the sample (REFERENCE_BUDGET_S), not by shrinking it.
    Returns (sample seconds, scale, description)."""
    from oracle import banded, dense
    nb_s = 2 if cfg.bs >= 1024 else min(cfg.nb, 4)
    bs_s = cfg.bs
    if cfg.name not in _sample_inputs:
        if cfg.kind == "chain":
            _sample_inputs[cfg.name] = inputs.perfect_chain_problem(bs_s, nb_s, 1)
        else:
            _sample_inputs[cfg.name] = inputs.random_problem(bs_s, nb_s, 1, cfg.nrhs, seed=cfg.seed, threads=os.cpu_count() or 1)
    p = _sample_inputs[cfg.name]
    solver = dense if bs_s * nb_s <= 8192 else banded
    t0 = time.perf_counter()
    solver.solve_energy(p.E[0], p.H_diag, p.H_upper, p.S_diag, p.S_upper, p.Sigma_L[0], p.Sigma_R[0], p.Inj_first[0], None)
    dt = time.perf_counter() - t0
    scale = (cfg.nb / nb_s) * (cfg.bs / bs_s) ** 3
    desc = (f"1 energy point, device truncated to nb={nb_s} of {cfg.nb} blocks" +
            (f" of bs={bs_s} instead of {cfg.bs}" if bs_s != cfg.bs else f" (bs={cfg.bs})") + f", nrhs={cfg.nrhs}, "
            f"oracle/{'dense' if solver is dense else 'banded'}.py LU of the full matrix; solves/s EXTRAPOLATED to the full device "
            f"by x{scale:g} (cost linear in nb" + (", cubic in bs" if bs_s != cfg.bs else "") + "; see profiles/r02_oracle_scaling.md)")
    return dt, scale, desc


def reference_repetitions(first_seconds, warmup, steps, budget=REFERENCE_BUDGET_S):
    """How many times --impl reference repeats the (fixed) sample: warm-up + steps if that fits the budget at the pace of the
    first repetition, else as many as fit (at least one; at least two when a warm-up was asked for and two fit)."""
    want = warmup + steps
    fit = int(budget / max(first_seconds, 1e-9))
    return max(1, min(want, fit))


def full_size_oracle_record(cfg):
    """The one NOT extrapolated oracle time there is for C3 / C4: the run that wrote the Tier B fingerprint of one full energy
    point (tests/golden/make_golden_large.py: banded LU of the whole matrix, 16 columns of X and the last block column of
    T^-1), read from that file's header.  Measured once on the build container, not on this box: context, not a timing."""
    import re
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "tests", "golden", f"{cfg.name.lower()}_fingerprint.txt")
    try:
        head = open(path).readline() + open(path).readlines()[1]
    except (OSError, IndexError):
        return None
    m = re.search(r"in (\d+) s on (\d+) host cores", head)
    if not m:
        return None
    return {"seconds_one_energy": int(m.group(1)), "cores": int(m.group(2)), "kind": "oracle/banded.py, full device, no extrapolation",
            "source": os.path.relpath(path, os.path.dirname(os.path.abspath(__file__))) + " header (build container, not this box)"}


def cpu_baseline(cfg):
    dt, scale, desc = oracle_sample(cfg)
    out = {"value": 1.0 / (dt * scale), "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle", "sample": desc,
           "sample_seconds": dt, "extrapolated": scale != 1.0, "scale": scale}
    rec = full_size_oracle_record(cfg)
    if rec:
        out["full_size_record"] = rec
    return out


def cpu_baseline_full(cfg):
    """The oracle on the WHOLE device of `cfg`, one energy point, X for the workload's Inj columns: oracle/banded.py, LU with
    partial pivoting of the full matrix in band storage.  Nothing is truncated and nothing is extrapolated.  T(E) is NOT
    computed (want_G = False): it needs the last block column of the inverse, 2 bs more right-hand sides, which takes the C2
    sample from 16 s to 122 s on the box's 16 cores (profiles/r03_bench.md) -- so the sample is LESS work than one energy
    point of a GPU step, and says so.  Used for C2; C3 / C4 would take 40 min / 4 h per energy point
    (tests/golden/c{3,4}_fingerprint.txt headers)."""
    from oracle import banded
    p = inputs.random_problem(cfg.bs, cfg.nb, 1, cfg.nrhs, seed=cfg.seed, threads=os.cpu_count() or 1)
    t0 = time.perf_counter()
    banded.solve_energy(p.E[0], p.H_diag, p.H_upper, p.S_diag, p.S_upper, p.Sigma_L[0], p.Sigma_R[0], p.Inj_first[0], None,
                        want_G=False)
    dt = time.perf_counter() - t0
    return {"value": 1.0 / dt, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle",
            "sample": f"1 of {cfg.n_energy} energy points of {cfg.name}, the full device (nb={cfg.nb}, bs={cfg.bs}, nrhs={cfg.nrhs}), "
                      "X only (no T(E): less work than the GPU step's energy point), oracle/banded.py LU of the full matrix in band "
                      "storage; not truncated, not extrapolated",
            "sample_seconds": dt, "extrapolated": False, "scale": 1.0}


def run_reference(args, cfg):
    """--impl reference: the oracle, as it stands, on the host cores.  Each step is the bounded sample of oracle_sample;
    `ms_per_step` is what was actually timed, `value` the solves/s extrapolated to the full device (flagged)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    times, desc, scale = [], "", 1.0
    dt, scale, desc = oracle_sample(cfg)                                  # the first repetition sizes the run
    total = reference_repetitions(dt, args.warmup, args.steps)
    n_warm = min(args.warmup, max(0, total - 1), 1 if total < args.warmup + args.steps else args.warmup)
    if n_warm == 0:
        times.append(dt)
    for i in range(1, total):
        dt, scale, desc = oracle_sample(cfg)
        if i >= n_warm:
            times.append(dt)
    mean = sum(times) / max(1, len(times))
    val = 1.0 / (mean * scale) if mean > 0 else 0.0
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "steps_timed": len(times), "warmup_run": n_warm,
            "gpus_used": 0, "n_gpus_is": "the N of the run this line is paired with; the oracle runs on the host cores of rank 0 only",
            "ms_per_step": 1e3 * mean, "ms_per_step_is": "the timed sample (one truncated energy point)",
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "c128 (f64 re/im)", "data": "synthetic",
            "config": config_dict(cfg, max(1, args.gpus)),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle", "sample": desc,
                             "sample_seconds": mean, "extrapolated": scale != 1.0, "scale": scale},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def calibrate_oracle():
    """Full vs truncated C2 device, one energy point, Inj columns only (want_G = False on both): is 'linear in nb' true?"""
    from oracle import banded
    cfg = inputs.CONFIGS["C2"]
    out = {}
    for nb_s in (4, 8, cfg.nb):
        p = inputs.random_problem(cfg.bs, nb_s, 1, cfg.nrhs, seed=cfg.seed, threads=os.cpu_count() or 1)
        t0 = time.perf_counter()
        banded.solve_energy(p.E[0], p.H_diag, p.H_upper, p.S_diag, p.S_upper, p.Sigma_L[0], p.Sigma_R[0], p.Inj_first[0], None,
                            want_G=False)
        out[nb_s] = time.perf_counter() - t0
    full = out[cfg.nb]
    print(json.dumps({"calibrate_oracle": "C2, one energy, oracle/banded.py, Inj columns only", "cores": os.cpu_count(),
                      "seconds": out, "full_over_scaled_nb4": full / (out[4] * cfg.nb / 4),
                      "full_over_scaled_nb8": full / (out[8] * cfg.nb / 8)}), flush=True)


# ---------------------------------------------------------------------------------------------------------
# the CUDA arm
# ---------------------------------------------------------------------------------------------------------
def measure(args, cfg, world, rank, local, steps, warmup, want_e2e, want_clocks=True):
    """One workload on this rank's GPU: W warm-up + K timed steps (device-resident inputs), one serial step for the
    per-launch GEMM timing, optionally the end-to-end leg through the host-buffer entry points.  Returns the measurement
    as a dict (rank-local except for the max-over-ranks step time and the gathered T)."""
    import torch
    import torch.distributed as dist
    from paper_1812_01396_b200 import binding, sharding

    nE, bs, nb, m = cfg.n_energy, cfg.bs, cfg.nb, cfg.nrhs
    spatial_split = args.split == "spatial" and world > 1
    column_split = (args.split == "column" and world > 1) or spatial_split      # both: pairs of ranks share their energies
    if column_split:
        # ranks (2j, 2j+1) share the energies of shard j; every rank creates every pair's group
        if world % 2:
            raise SystemExit("--split column needs an even number of GPUs")
        pair_groups = [dist.new_group([2 * j, 2 * j + 1]) for j in range(world // 2)]
        pair_group = pair_groups[rank // 2]
        e_world, e_rank = world // 2, rank // 2
    else:
        pair_group = None
        e_world, e_rank = world, rank
    # inputs: same generator as the parity tests; energies sharded round-robin over ranks (weak scaling)
    if cfg.kind == "chain":
        p = inputs.perfect_chain_problem(bs, nb, nE * e_world)
        idx = sharding.energy_indices(nE * e_world, e_rank, e_world)
        p.E, p.Sigma_L, p.Sigma_R, p.Inj_first = p.E[idx], p.Sigma_L[idx], p.Sigma_R[idx], p.Inj_first[idx]
    else:
        if world > 1 and rank != 0:
            # H, S come from rank 0 by one NCCL broadcast per array (the paper's MPI_Bcast, L212)
            p = inputs.Problem(bs, nb, *(np.empty((k, bs, bs), dtype=np.complex128) for k in (nb, nb - 1, nb, nb - 1)),
                               None, None, None, None)
        else:
            p = inputs.random_problem(bs, nb, 1, 1, seed=cfg.seed, threads=os.cpu_count() or 1)      # H, S only
        grid = inputs.energy_grid(nE * e_world, cfg.e_lo, cfg.e_hi, cfg.eta)
        idx = sharding.energy_indices(nE * e_world, e_rank, e_world)
        p.E = grid[idx].copy()
        p.Sigma_L = np.stack([inputs.sigma_block(cfg.seed, int(e), bs, "L") for e in idx])
        p.Sigma_R = np.stack([inputs.sigma_block(cfg.seed, int(e), bs, "R") for e in idx])
        p.Inj_first = np.stack([inputs.inj_block(cfg.seed, int(e), bs, m) for e in idx])

    def pin(a):
        t = torch.from_numpy(np.ascontiguousarray(a))
        return t.pin_memory() if want_e2e else t

    host = {k: pin(getattr(p, k)) for k in ("H_diag", "H_upper", "S_diag", "S_upper", "Sigma_L", "Sigma_R", "Inj_first")}
    devt = {k: v.cuda(non_blocking=True) for k, v in host.items()}
    torch.cuda.synchronize()
    if world > 1 and cfg.kind != "chain":
        hs = ("H_diag", "H_upper", "S_diag", "S_upper")
        sharding.broadcast_hamiltonian([devt[k] for k in hs], 0, world)
        torch.cuda.synchronize()
        if rank != 0 and want_e2e:                        # the e2e leg uploads from host buffers: fill them
            for k in hs:
                host[k].copy_(devt[k])

    variant = binding.get_default_gemm_variant()
    is3m = variant != 0
    if spatial_split:
        # this rank's half of the device: rows [lo, hi) of the block stacks (the whole H, S were generated / broadcast above;
        # a production caller would only ever hold its slices)
        lo, hi = sharding.partition_bounds(nb, 2)[rank & 1]
        ss = binding.SplitSolve(hi - lo, bs, nE)
    else:
        ss = binding.SplitSolve(nb, bs, nE)
    groups = 4 if args.stream_groups is None else args.stream_groups
    ss.set_option("stream_groups", groups)
    for kv in args.option:
        k, v = kv.split("=")
        ss.set_option(k, int(v))
    if args.trace:
        ss.set_option("trace", 1)
    if spatial_split:
        ss.set_hamiltonian(devt["H_diag"][lo:hi].contiguous(), devt["H_upper"][lo:hi - 1].contiguous(),
                           devt["S_diag"][lo:hi].contiguous(), devt["S_upper"][lo:hi - 1].contiguous())
    else:
        ss.set_hamiltonian(devt["H_diag"], devt["H_upper"], devt["S_diag"], devt["S_upper"])
    X = torch.empty((nE, nb * bs, m), dtype=torch.complex128, device="cuda")

    col_T = [None]
    if spatial_split:
        def couple(hb):
            return devt["S_upper"][hb - 1].contiguous(), devt["H_upper"][hb - 1].contiguous()
        engine = sharding.LibraryPartitionEngine(ss, p.E, couple, devt["Sigma_L"], devt["Sigma_R"], devt["Inj_first"], None)

        def step():
            _, col_T[0] = sharding.spatial_split_solve(engine, nb, rank & 1, 2, group=pair_group)
    elif column_split:
        engine = sharding.LibraryColumnEngine(ss, p.E, devt["Sigma_L"], devt["Sigma_R"], devt["Inj_first"], None)

        def step():
            _, col_T[0] = sharding.column_split_solve(engine, rank, group=pair_group)
    else:
        def step():
            ss.solve(p.E, devt["Sigma_L"], devt["Sigma_R"], devt["Inj_first"], None, X)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(warmup):
        step()
    T_last = ss.transmission()
    sweep_ms, gemm_ms, gemm_fl, gemm_n = [], 0.0, 0.0, 0
    serial = min(groups, nE) <= 1 or column_split          # column split: no separate per-launch GEMM timing step
    # CUDA events around every GEMM launch.  On a single stream they are taken inside the timed region; with stream
    # groups kernels of different groups overlap, so a launch's event-to-event time is not the kernel's own duration:
    # then the per-launch GEMM timing comes from one extra step with stream_groups = 1, right after the timed region.
    ss.set_option("profile_gemm", 1 if (serial or args.trace) else 0)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    torch.cuda.profiler.start()                      # cudaProfilerStart: `ncu --profile-from-start off` sees the timed region only
    with ClockSampler(local) as clocks:
        ev0.record()
        for _ in range(steps):
            step()
            T_last = ss.transmission()               # the step's result: synchronises, 8 B per energy
            if not column_split:
                sweep_ms.append(ss.phase_ms(0))
            if serial and not column_split:
                a, b, c = ss.gemm_profile()
                gemm_ms += a; gemm_fl += b; gemm_n += c
        ev1.record()
        barrier()
    torch.cuda.profiler.stop()
    ms_total = ev0.elapsed_time(ev1)
    launches = ss.launch_count()
    gemm_ref_ms = ms_total
    if args.trace:
        ss.trace_write(args.trace)
        ss.set_option("trace", 0)
    if not serial:
        ss.set_option("stream_groups", 1)
        ss.set_option("profile_gemm", 1)
        step()
        ss.transmission()
        gemm_ms, gemm_fl, gemm_n = ss.gemm_profile()
        gemm_ref_ms = ss.phase_ms(2)
        ss.set_option("stream_groups", groups)
    ss.set_option("profile_gemm", 0)
    ms_total = sharding.max_over_ranks(ms_total, world, device="cuda")
    if column_split:
        T_all = T_last                                    # every pair holds its own energies' T(E); no global gather here
    else:
        T_all = sharding.gather_transmission(T_last, nE * world, rank, world, device="cuda")   # 8 B per energy
    ms_step = ms_total / steps
    value = nE * e_world / (ms_step * 1e-3)

    flops_step = ss.flops(m) * nE
    sweep_flops = ss.flops_sweep() * nE
    sweep_tf = sweep_flops / (np.mean(sweep_ms) * 1e-3) / 1e12 if sweep_ms else 0.0     # column split: not timed separately
    gemm_tf = gemm_fl / (gemm_ms * 1e-3) / 1e12 if gemm_ms > 0 else 0.0

    # ---- e2e: host buffers through the C ABI, H2D of every input and D2H of X and T inside the timed region
    e2e = None
    if want_e2e and not column_split:
        Xh = torch.empty((nE, nb * bs, m), dtype=torch.complex128).pin_memory()
        Th = torch.empty(nE, dtype=torch.float64).pin_memory()

        def e2e_step():
            ss.set_hamiltonian_host(host["H_diag"], host["H_upper"], host["S_diag"], host["S_upper"])
            ss.solve_host(p.E, host["Sigma_L"], host["Sigma_R"], host["Inj_first"], None, Xh, Th)
        e2e_step()                                    # warm-up (allocates the handle-owned device copies)
        barrier()
        n_e2e = max(1, min(steps, 2))
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            e2e_step()
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        dt = sharding.max_over_ranks(dt, world, device="cuda")
        h2d = sum(host[k].numel() * 16 for k in host) + nE * 16
        d2h = Xh.numel() * 16 + nE * 8
        e2e = {"value": nE * world * n_e2e / dt, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
               "steps": n_e2e}
        del Xh, Th
    T_first = float(T_all[0])
    ss.close()
    del X, devt, host
    torch.cuda.empty_cache()

    ratio = EXECUTED_RATIO[is3m]
    # dominant launch of the timed step: bs^3 with two chains (first / last column sweep) per energy of a stream group
    dom_batch = 2 * ((nE + min(groups, nE) - 1) // min(groups, nE))
    traffic, overfetch, traffic_note = ncu_traffic(is3m, bs, dom_batch)
    kern = ("zgemm3m_kernel" if is3m else "zgemm_kernel") + f" [{binding.GEMM_VARIANTS[variant]}] (DMMA.8x8x4, mma.sync f64)"
    out = {
        "value": value, "ms_per_step": ms_step, "steps": steps, "warmup": warmup,
        "config": config_dict(cfg, world), "launch": {"stream_groups": groups, "split": ("spatial pairs" if spatial_split else "column pairs") if column_split else "energy"},
        "tflops": {"whole_solve": flops_step / (ms_step * 1e-3) / 1e12,
                   "whole_solve_executed_frac_of_fp64_peak": flops_step / (ms_step * 1e-3) / 1e12 * ratio / FP64_PEAK_NOMINAL_TFLOPS,
                   "sweep_a1_a4": sweep_tf,
                   "sweep_executed": sweep_tf * ratio, "sweep_executed_frac_of_fp64_peak": sweep_tf * ratio / FP64_PEAK_NOMINAL_TFLOPS,
                   "flops_per_step": flops_step,
                   "convention": "LAPACK (complex multiply-add = 8 flops), closed form ss_flops; *_executed = x" + str(ratio) +
                   " (3M: 6 real flops per complex multiply-add)"},
        "roofline": {"bound": "tensor", "kernel": kern,
                     "achieved": gemm_tf * ratio if gemm_n else None, "peak": FP64_PEAK_NOMINAL_TFLOPS, "unit": "TFLOP/s",
                     "frac": gemm_tf * ratio / FP64_PEAK_NOMINAL_TFLOPS if gemm_n else None,
                     "flops_convention": "achieved = real FP64 flops the kernel executes (3M: 6 M N K per complex GEMM) per second, "
                     "summed over every GEMM launch of one step; achieved_lapack = the same launches at 8 M N K",
                     "achieved_lapack": gemm_tf, "executed_over_lapack": ratio,
                     "traffic": traffic, "traffic_overfetch": overfetch, "traffic_note": traffic_note,
                     "dominant_launch": f"{bs}x{bs}x{bs} x{dom_batch}",
                     "peak_source": "148 SM x 64 FP64 FMA/clk x 2 x 1.965 GHz (no FP64 entry in MEASURED_PEAKS.json); "
                     "peak_measured_dmma_microbench is the library's DMMA microbenchmark on this GPU",
                     "gemm_launches": gemm_n, "gemm_share_of_step": gemm_ms / gemm_ref_ms,
                     "ms_per_step_serial": None if (serial or column_split) else gemm_ref_ms,
                     "gemm_flops_share": gemm_fl / (flops_step * (steps if serial else 1)),
                     "measured_in": "not collected (--split column / spatial runs time the step only)" if column_split else
                     "timed region (single stream)" if serial else
                     "one extra step with stream_groups=1 right after the timed region (kernels of different stream "
                     f"groups overlap in the timed region); that serial step took {gemm_ref_ms:.1f} ms"},
        "gpu_launches": int(launches * steps),
        "clocks": clocks.summary(),
        "T_first_energy": T_first,
    }
    if column_split:                                      # a pair of GPUs shares one shard of energies
        out["config"].update({"n_energy_per_gpu": nE / 2, "parallelism": f"{args.split} split over GPU pairs x energy-parallel x{e_world}"})
    if e2e:
        out["e2e"] = e2e
    return out


def launch_ranks(n: int) -> int:
    """Re-executes this command line under torch.distributed.run with n ranks on this node (rendezvous on 127.0.0.1, a free
    port); rank r binds GPU r (LOCAL_RANK).  NCCL's own logging is left as the environment has it (NCCL_DEBUG is passed
    through), so a scaling run can count ranks and transports.  Returns the launcher's exit code."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.run(cmd).returncode


def run_ours(args, cfg):
    import torch
    import torch.distributed as dist
    from paper_1812_01396_b200 import binding, build

    if "WORLD_SIZE" not in os.environ and args.gpus > 1:
        # started without torchrun: start the N ranks here (one per GPU) and let rank 0 print the line
        if args.dist_backend != "gloo" and torch.cuda.device_count() < args.gpus:
            raise SystemExit(f"bench.py --gpus {args.gpus}: only {torch.cuda.device_count()} CUDA device(s) visible "
                             "(--dist-backend gloo lets ranks share GPUs for a functional check)")
        raise SystemExit(launch_ranks(args.gpus))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != max(1, args.gpus):
        raise SystemExit(f"bench.py --gpus {args.gpus} was started with WORLD_SIZE={world}: the two must agree")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    if args.dist_backend == "gloo":
        local %= torch.cuda.device_count()                # functional check: ranks may share a GPU
    torch.cuda.set_device(local)
    if world > 1:
        if args.dist_backend == "gloo":
            dist.init_process_group("gloo")
        else:
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    build.build()
    binding.load()
    if args.gemm_variant is not None:
        binding.set_default_gemm_variant(args.gemm_variant)
    peak_measured = binding.fp64_peak_tflops(300.0)

    r = measure(args, cfg, world, rank, local, args.steps, args.warmup, want_e2e=not args.no_e2e)
    also = None
    if cfg.name == "C4" and world == 1 and not args.no_also:
        # the other bs >= 2048 target configuration, same process, same measurement (>= 3 warm-up steps)
        c3 = inputs.CONFIGS["C3"]
        a = measure(args, c3, world, rank, local, max(1, min(args.steps, 5)), max(3, min(args.warmup, 3)), want_e2e=False)
        also = {"C3": {k: a[k] for k in ("value", "ms_per_step", "steps", "warmup", "config", "launch", "tflops", "roofline", "gpu_launches",
                                         "clocks")}}
        also["C3"]["unit"] = UNIT
        # the three small configurations (launch-latency-bound): every BASELINE.json config in one driver line
        for name in ("C2", "C1", "C0"):
            c = inputs.CONFIGS[name]
            a = measure(args, c, world, rank, local, max(1, min(args.steps, 5)), 3, want_e2e=False)
            also[name] = {k: a[k] for k in ("value", "ms_per_step", "steps", "warmup", "config", "launch", "tflops", "gpu_launches",
                                            "T_first_energy")}
            also[name]["unit"] = UNIT
            also[name]["launches_per_step"] = a["gpu_launches"] // max(1, a["steps"])
        if not args.no_cpu_baseline:
            # the one configuration whose FULL-size oracle run fits a bench run: GPU and oracle timed in the same run, same
            # box, same (whole) device -- the un-extrapolated counterpart of the flagged cpu_baseline of C4 / C3
            also["C2"]["cpu_baseline"] = cpu_baseline_full(inputs.CONFIGS["C2"])

    if rank == 0:
        line = {
            "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": r["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "c128 (f64 re/im)", "data": "synthetic",
            "config": r["config"], "launch": r["launch"], "tflops": r["tflops"], "roofline": r["roofline"], "gpu_launches": r["gpu_launches"],
            "clocks": r["clocks"], "T_first_energy": r["T_first_energy"],
        }
        line["roofline"]["peak_measured_dmma_microbench"] = peak_measured
        if world > 1 and args.dist_backend != "nccl":
            line["dist_backend"] = args.dist_backend + " (ranks may share GPUs: functional check of the N > 1 path, NOT a measurement)"
        if "e2e" in r:
            line["e2e"] = r["e2e"]
        if also:
            line["also"] = also
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = cpu_baseline(cfg)
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


# ---------------------------------------------------------------------------------------------------------
# single-kernel modes (tuning and the ncu captures under profiles/)
# ---------------------------------------------------------------------------------------------------------
def kernel_gemm(args):
    """ss_zgemm_batched alone: best-of-reps CUDA-event time, TFLOP/s in LAPACK convention (8 flops per complex
    multiply-add, whatever the variant executes) and the executed-flop fraction of the FP64 pipe."""
    import torch
    from paper_1812_01396_b200 import binding, build
    build.build()
    if args.raster is not None:
        binding.set_gemm_raster(args.raster)
    a = args.dims
    M, N, K, batch = (a + [2048, 2048, 2048, 16][len(a):])[:4]
    reps = a[4] if len(a) > 4 else 5
    variants = [binding.get_default_gemm_variant()] if args.variants is None else [int(v) for v in args.variants.split(",")]
    g = torch.Generator(device="cuda").manual_seed(0)
    A = torch.randn((batch, M, K), dtype=torch.complex128, device="cuda", generator=g)
    B = torch.randn((batch, K, N), dtype=torch.complex128, device="cuda", generator=g)
    C = torch.zeros((batch, M, N), dtype=torch.complex128, device="cuda")
    ref = A[0] @ B[0]
    if args.sumplane:
        As, Bs = (A.real + A.imag).contiguous(), (B.real + B.imag).contiguous()
        Cs = torch.zeros((batch, M, N), dtype=torch.float64, device="cuda")
        plain = binding.zgemm_batched

        def with_sums(A_, B_, C_, alpha, beta):
            return binding.zgemm_batched_sums(A_, As, B_, Bs, C_, Cs, alpha, beta)
        binding.zgemm_batched = with_sums
    for v in variants:
        binding.set_default_gemm_variant(v)
        C.zero_()
        for _ in range(3):
            binding.zgemm_batched(A, B, C, 1.0, args.beta)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        best = 1e30
        for _ in range(reps):
            e0.record()
            binding.zgemm_batched(A, B, C, 1.0, args.beta)
            e1.record()
            torch.cuda.synchronize()
            best = min(best, e0.elapsed_time(e1))
        if args.beta != 0.0:                       # accuracy is checked on a fresh beta = 0 product
            binding.zgemm_batched(A, B, C, 1.0, 0.0)
            torch.cuda.synchronize()
        err = (C[0] - ref).abs().max().item() / (K ** 0.5)
        tf = 8.0 * M * N * K * batch / best / 1e9
        print(f"zgemm[{binding.GEMM_VARIANTS[v]}] M={M} N={N} K={K} batch={batch} beta={args.beta:g}: {best:.3f} ms  "
              f"{tf:.2f} TFLOP/s (LAPACK conv.)  executed frac of 37.22: {tf * EXECUTED_RATIO[v != 0] / FP64_PEAK_NOMINAL_TFLOPS:.3f}  "
              f"max err/sqrt(K) {err:.2e}", flush=True)


def kernel_density(args):
    """ss_density alone against the HBM roofline: algorithmic bytes = 16 n_energy n nrhs + 8 n."""
    import torch
    from paper_1812_01396_b200 import binding, build
    build.build()
    a = args.dims
    n_energy, n, nrhs = (a + [8, 65536, 256][len(a):])[:3]          # config C3's X
    reps = a[3] if len(a) > 3 else 10
    X = torch.randn((n_energy, n, nrhs), dtype=torch.complex128, device="cuda")
    w = torch.rand(n_energy, dtype=torch.float64, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")  # > 126 MB L2
    for _ in range(3):
        rho = binding.density(X, w)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    best = 1e30
    for _ in range(reps):
        flush.zero_()
        e0.record()
        rho = binding.density(X, w)
        e1.record()
        torch.cuda.synchronize()
        best = min(best, e0.elapsed_time(e1))
    want = (w[:, None] * (X.real ** 2 + X.imag ** 2).sum(dim=2)).sum(dim=0)
    err = ((rho - want).abs().max() / want.abs().max()).item()
    gbs = (16.0 * n_energy * n * nrhs + 8.0 * n) / best / 1e6
    peak, src = None, "fallback"
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        peak, src = json.load(open(path)).get("hbm_gbs"), "measured"
    peak = peak or 6650.0
    print(f"density n_energy={n_energy} n={n} nrhs={nrhs}: {best:.3f} ms  {gbs:.0f} GB/s = {gbs / peak:.3f} of {src} {peak:.0f} GB/s  "
          f"rel err {err:.1e}")


def kernel_lu(args):
    """ss_zgetrf_batched alone (a2 of the sweep: `batch` chains of an n x n pivoted LU, the shape one block step of a
    stream group factors): best-of-reps CUDA-event time, TFLOP/s at (8/3) n^3 per matrix.  The command of the
    `ncu --set full -k regex:lu_panel` capture under profiles/ (the latency-bound panel kernel is its second kernel)."""
    import torch
    from paper_1812_01396_b200 import binding, build
    build.build()
    a = args.dims
    n, batch = (a + [2048, 16][len(a):])[:2]
    reps = a[2] if len(a) > 2 else 5
    g = torch.Generator(device="cuda").manual_seed(0)
    A0 = torch.randn((batch, n, n), dtype=torch.complex128, device="cuda", generator=g)
    A = A0.clone()
    for _ in range(2):
        A.copy_(A0)
        ipiv, info = binding.zgetrf_batched(A, n)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    best = 1e30
    for _ in range(reps):
        A.copy_(A0)
        e0.record()
        ipiv, info = binding.zgetrf_batched(A, n)
        e1.record()
        torch.cuda.synchronize()
        best = min(best, e0.elapsed_time(e1))
    assert int(info.abs().max()) == 0
    tf = 8.0 / 3.0 * n ** 3 * batch / best / 1e9
    print(f"zgetrf n={n} batch={batch}: {best:.3f} ms  {tf:.2f} TFLOP/s (LAPACK conv., (8/3) n^3)  "
          f"{(n + 127) // 128} panel launches of lu_panel_kernel per factorisation", flush=True)


def emulate_split(args, cfg):
    """Per-rank work of the 2-GPU splits, on one GPU (the ranks run one after the other, so nothing waits on anything)."""
    import torch
    from paper_1812_01396_b200 import binding, build, sharding
    build.build()
    nE, bs, nb, m = cfg.n_energy, cfg.bs, cfg.nb, cfg.nrhs
    p = inputs.random_problem(bs, nb, 1, 1, seed=cfg.seed, threads=os.cpu_count() or 1)
    E = inputs.energy_grid(nE, cfg.e_lo, cfg.e_hi, cfg.eta)
    d = {k: torch.from_numpy(getattr(p, k)).cuda() for k in ("H_diag", "H_upper", "S_diag", "S_upper")}
    sl = torch.from_numpy(np.stack([inputs.sigma_block(cfg.seed, e, bs, "L") for e in range(nE)])).cuda()
    sr = torch.from_numpy(np.stack([inputs.sigma_block(cfg.seed, e, bs, "R") for e in range(nE)])).cuda()
    inj = torch.from_numpy(np.stack([inputs.inj_block(cfg.seed, e, bs, m) for e in range(nE)])).cuda()
    spatial = args.emulate_split == "spatial"
    bounds = sharding.partition_bounds(nb, 2) if spatial else [(0, nb), (0, nb)]
    hs = []
    for lo, hi in bounds:
        ss = binding.SplitSolve(hi - lo, bs, nE)
        ss.set_hamiltonian(d["H_diag"][lo:hi].contiguous(), d["H_upper"][lo:hi - 1].contiguous(), d["S_diag"][lo:hi].contiguous(),
                           d["S_upper"][lo:hi - 1].contiguous())
        hs.append(ss)

    def timed(fn):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(); e0.record(); out = fn(); e1.record(); torch.cuda.synchronize()
        return out, e0.elapsed_time(e1)

    res = []
    for rep in range(args.warmup + args.steps):
        t = [dict(), dict()]
        if spatial:
            hcut = bounds[1][0]
            Sc, Hc = d["S_upper"][hcut - 1].contiguous(), d["H_upper"][hcut - 1].contiguous()
            for r in range(2):
                _, t[r]["sweep"] = timed(lambda: hs[r].sweep_partition(E))
            edges = [torch.stack([ss.edge_blocks(0), ss.edge_blocks(1)]) for ss in hs]
            iface = torch.stack([edges[0][1], edges[1][0]], dim=1).contiguous()
            for r in range(2):
                _, t[r]["merge"] = timed(lambda: hs[r].merge_partition(r, iface, Sc, Hc))
            corners = torch.stack([hs[0].edge_blocks(0), hs[1].edge_blocks(1)], dim=1).contiguous()
            for r in range(2):
                _, t[r]["post"] = timed(lambda: (hs[r].post_partition(corners, sl, sr, inj), hs[r].transmission()))
            link = 2 * nE * 4 * bs * bs * 16                       # two all-gathers of 4 blocks per energy and rank
        else:
            for r in range(2):
                _, t[r]["sweep"] = timed(lambda: hs[r].sweep_column(E, r))
            cb = [hs[r].corner_blocks(r) for r in range(2)]
            t[0]["merge"] = t[1]["merge"] = 0.0
            for r in range(2):
                _, t[r]["post"] = timed(lambda: (hs[r].post_column(r, cb[1 - r], sl, sr, inj), hs[r].transmission()))
            link = nE * 2 * bs * bs * 16 + nE * nb * bs * m * 16   # corner all-gather + sum-all-reduce of the X shares
        if rep >= args.warmup:
            res.append(t)
    per_rank = [{k: float(np.mean([t[r][k] for t in res])) for k in ("sweep", "merge", "post")} for r in range(2)]
    crit = max(sum(x.values()) for x in per_rank)
    link_ms = link / 770e9 * 1e3
    print(json.dumps({"emulate_split": args.emulate_split, "workload": cfg.name, "per_rank_ms": per_rank,
                      "critical_path_ms": crit, "link_bytes_per_rank": link, "link_ms_at_770GBps": link_ms,
                      "solves_per_s_two_gpus_estimate": nE / ((crit + link_ms) * 1e-3),
                      "note": "ranks run one after the other on ONE GPU; exchanges are device copies; not a 2-GPU measurement"}), flush=True)


def main():
    args = parse()
    cfg = inputs.CONFIGS[args.workload]
    if args.real_energies:
        import dataclasses
        cfg = dataclasses.replace(cfg, name=cfg.name + " (real energies 3.5..4.5)", e_lo=3.5, e_hi=4.5, eta=0.0)
    if args.calibrate_oracle:
        calibrate_oracle()
        return
    if args.kernel:
        {"gemm": kernel_gemm, "density": kernel_density, "lu": kernel_lu}[args.kernel](args)
        return
    if args.emulate_split:
        emulate_split(args, cfg)
        return
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
