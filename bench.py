#!/usr/bin/env python
"""bench.py -- energy-point solves/s of the SplitSolve hot path (a0-a7) on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C3|C4|C2|C1|C0] [--impl ours|reference]

One "step" = one pass of the whole hot path over one batch of synthetic input: ss_solve (+ ss_transmission) over
all n_energy energy points of the workload.  N > 1 (torchrun, one rank per GPU): the energy grid is n_energy*N
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
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant GEMM shape (a1/a4 of C3: M=N=K=2048,
# batch 16; algorithmic bytes 3 x 16 x 67.1 MB = 3.22e9) from the committed `ncu --set full` captures
NCU_TRAFFIC = {False: {"bytes": 7.14e9, "note": "profiles/r01_zgemm_ncu_full.md (4M, 2048^3 x16 launch; algorithmic 3.22e9 B)"},
               True: {"bytes": 7.48e9, "note": "profiles/r01_zgemm3m_ncu_full.md (3M, 2048^3 x16 launch; algorithmic 3.22e9 B)"}}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="C3", choices=sorted(inputs.CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--gemm-variant", type=int, default=None, help="complex-GEMM kernel variant (binding.GEMM_VARIANTS); "
                    "default: the library default (3M)")
    ap.add_argument("--stream-groups", type=int, default=None, help="stream groups the energies are split over "
                    "(library default 4; 1 = single stream)")
    ap.add_argument("--nb-lu", type=int, default=None, help="outer LU block (16..128, default 128)")
    ap.add_argument("--trace", default=None, help="write the phase timeline of the last timed step to this CSV")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
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
def oracle_sample(cfg):
    """Times the oracle, as it stands, on a bounded sample of the workload: ONE energy point of the same
    generator with the device truncated to nb_s blocks (nb_s = 2 for bs >= 1024, else min(nb, 4)), solved by
    the plain definition (LU of the full matrix: oracle/dense.py when the truncated matrix is <= 8192 rows --
    with 2 blocks the band of the block-tridiagonal matrix IS the whole matrix -- else oracle/banded.py).
    The time is scaled by nb / nb_s: the oracle's cost at full size (banded LU, the only form that fits the
    host) is linear in nb, and costs MORE per block than the truncated sample, so the scaled figure flatters
    the oracle.  Returns (sample seconds, scaled seconds, description)."""
    from oracle import banded, dense
    nb_s = 2 if cfg.bs >= 1024 else min(cfg.nb, 4)
    if cfg.kind == "chain":
        p = inputs.perfect_chain_problem(cfg.bs, nb_s, 1)
    else:
        p = inputs.random_problem(cfg.bs, nb_s, 1, cfg.nrhs, seed=cfg.seed, threads=os.cpu_count() or 1)
    solver = dense if cfg.bs * nb_s <= 8192 else banded
    t0 = time.perf_counter()
    solver.solve_energy(p.E[0], p.H_diag, p.H_upper, p.S_diag, p.S_upper, p.Sigma_L[0], p.Sigma_R[0], p.Inj_first[0], None)
    dt = time.perf_counter() - t0
    scale = cfg.nb / nb_s
    desc = (f"1 energy point, device truncated to nb={nb_s} of {cfg.nb} blocks (bs={cfg.bs}, nrhs={cfg.nrhs}), "
            f"oracle/{'dense' if solver is dense else 'banded'}.py LU of the full matrix; time scaled x{scale:g} (linear in nb)")
    return dt, dt * scale, desc


def cpu_baseline(cfg):
    dt, dt_full, desc = oracle_sample(cfg)
    return {"value": 1.0 / dt_full, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle", "sample": desc,
            "sample_seconds": dt}


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    times, desc = [], ""
    for i in range(args.warmup + args.steps):
        dt, dt_full, desc = oracle_sample(cfg)
        if i >= args.warmup:
            times.append(dt_full)
    tot = sum(times)
    val = len(times) / tot if tot > 0 else 0.0
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot / max(1, len(times)), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "c128 (f64 re/im)", "data": "synthetic",
            "config": {"workload": cfg.name, "bs": cfg.bs, "nb": cfg.nb, "n_energy": cfg.n_energy, "nrhs": cfg.nrhs},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle", "sample": desc},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------------------
# the CUDA arm
# ---------------------------------------------------------------------------------------------------------
def run_ours(args, cfg):
    import torch
    import torch.distributed as dist
    from paper_1812_01396_b200 import binding, build, sharding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    build.build()
    binding.load()

    nE, bs, nb, m = cfg.n_energy, cfg.bs, cfg.nb, cfg.nrhs
    # inputs: same generator as the parity tests; energies sharded round-robin over ranks (weak scaling)
    threads = max(1, (os.cpu_count() or 1) // max(1, world))
    if cfg.kind == "chain":
        p = inputs.perfect_chain_problem(bs, nb, nE * world)
        idx = sharding.energy_indices(nE * world, rank, world)
        p.E, p.Sigma_L, p.Sigma_R, p.Inj_first = p.E[idx], p.Sigma_L[idx], p.Sigma_R[idx], p.Inj_first[idx]
    else:
        if world > 1 and rank != 0:
            # H, S come from rank 0 by one NCCL broadcast per array (the paper's MPI_Bcast, L212)
            p = inputs.Problem(bs, nb, *(np.empty((k, bs, bs), dtype=np.complex128) for k in (nb, nb - 1, nb, nb - 1)),
                               None, None, None, None)
        else:
            p = inputs.random_problem(bs, nb, 1, 1, seed=cfg.seed, threads=os.cpu_count() or 1)      # H, S only
        grid = inputs.energy_grid(nE * world, cfg.e_lo, cfg.e_hi, cfg.eta)
        idx = sharding.energy_indices(nE * world, rank, world)
        p.E = grid[idx].copy()
        p.Sigma_L = np.stack([inputs.sigma_block(cfg.seed, int(e), bs, "L") for e in idx])
        p.Sigma_R = np.stack([inputs.sigma_block(cfg.seed, int(e), bs, "R") for e in idx])
        p.Inj_first = np.stack([inputs.inj_block(cfg.seed, int(e), bs, m) for e in idx])

    def pin(a):
        t = torch.from_numpy(np.ascontiguousarray(a))
        return t.pin_memory()

    host = {k: pin(getattr(p, k)) for k in ("H_diag", "H_upper", "S_diag", "S_upper", "Sigma_L", "Sigma_R", "Inj_first")}
    devt = {k: v.cuda(non_blocking=True) for k, v in host.items()}
    torch.cuda.synchronize()
    if world > 1 and cfg.kind != "chain":
        hs = ("H_diag", "H_upper", "S_diag", "S_upper")
        sharding.broadcast_hamiltonian([devt[k] for k in hs], 0, world)
        torch.cuda.synchronize()
        if rank != 0 and not args.no_e2e:                 # the e2e leg uploads from host buffers: fill them
            for k in hs:
                host[k].copy_(devt[k])

    if args.gemm_variant is not None:
        binding.set_default_gemm_variant(args.gemm_variant)
    variant = binding.get_default_gemm_variant()
    is3m = variant != 0
    ss = binding.SplitSolve(nb, bs, nE)
    groups = 4 if args.stream_groups is None else args.stream_groups
    ss.set_option("stream_groups", groups)
    if args.nb_lu is not None:
        ss.set_option("nb_lu", args.nb_lu)
    if args.trace:
        ss.set_option("trace", 1)
    ss.set_hamiltonian(devt["H_diag"], devt["H_upper"], devt["S_diag"], devt["S_upper"])
    X = torch.empty((nE, nb * bs, m), dtype=torch.complex128, device="cuda")

    def step():
        ss.solve(p.E, devt["Sigma_L"], devt["Sigma_R"], devt["Inj_first"], None, X)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    peak_measured = binding.fp64_peak_tflops(300.0)
    for _ in range(args.warmup):
        step()
    T_last = ss.transmission()
    sweep_ms, gemm_ms, gemm_fl, gemm_n = [], 0.0, 0.0, 0
    serial = min(groups, nE) <= 1
    # CUDA events around every GEMM launch.  On a single stream they are taken inside the timed region; with stream
    # groups kernels of different groups overlap, so a launch's event-to-event time is not the kernel's own duration:
    # then the per-launch GEMM timing comes from one extra step with stream_groups = 1, right after the timed region.
    ss.set_option("profile_gemm", 1 if (serial or args.trace) else 0)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    torch.cuda.profiler.start()                      # cudaProfilerStart: `ncu --profile-from-start off` sees the timed region only
    with ClockSampler(local) as clocks:
        ev0.record()
        for _ in range(args.steps):
            step()
            T_last = ss.transmission()               # the step's result: synchronises, 8 B per energy
            sweep_ms.append(ss.phase_ms(0))
            if serial:
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
    T_all = sharding.gather_transmission(T_last, nE * world, rank, world, device="cuda")   # 8 B per energy
    ms_step = ms_total / args.steps
    value = nE * world / (ms_step * 1e-3)

    flops_step = ss.flops(m) * nE
    sweep_flops = ss.flops_sweep() * nE
    sweep_tf = sweep_flops / (np.mean(sweep_ms) * 1e-3) / 1e12
    gemm_tf = gemm_fl / (gemm_ms * 1e-3) / 1e12 if gemm_ms > 0 else 0.0

    # ---- e2e: host buffers through the C ABI, H2D of every input and D2H of X and T inside the timed region
    e2e = None
    if not args.no_e2e:
        Xh = torch.empty((nE, nb * bs, m), dtype=torch.complex128).pin_memory()
        Th = torch.empty(nE, dtype=torch.float64).pin_memory()
        ss2 = ss                                      # same handle: workspace is reused
        def e2e_step():
            ss2.set_hamiltonian_host(host["H_diag"], host["H_upper"], host["S_diag"], host["S_upper"])
            ss2.solve_host(p.E, host["Sigma_L"], host["Sigma_R"], host["Inj_first"], None, Xh, Th)
        e2e_step()                                    # warm-up (allocates the handle-owned device copies)
        e2e_step()                                    # second warm-up: the library captures its CUDA graph here
        barrier()
        n_e2e = max(1, min(args.steps, 2))
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
        ss.set_hamiltonian(devt["H_diag"], devt["H_upper"], devt["S_diag"], devt["S_upper"])

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "c128 (f64 re/im)", "data": "synthetic",
            "config": {"workload": cfg.name, "bs": bs, "nb": nb, "n_energy_per_gpu": nE, "nrhs": m,
                       "parallelism": f"energy-parallel x{world}", "stream_groups": groups, "l2": "inputs larger than L2 (H,S,slots >> 126 MB)"
                       if bs >= 512 else "small workload: inputs fit L2 (launch-bound config)"},
            "tflops": {"whole_solve": flops_step / (ms_step * 1e-3) / 1e12, "sweep_a1_a4": sweep_tf,
                       "sweep_frac_of_fp64_peak": sweep_tf / FP64_PEAK_NOMINAL_TFLOPS, "flops_per_step": flops_step,
                       "convention": "LAPACK (complex multiply-add = 8 flops), closed form ss_flops"},
            "roofline": {"bound": "tensor",
                         "kernel": ("zgemm3m_kernel" if is3m else "zgemm_kernel") + f" [{binding.GEMM_VARIANTS[variant]}] "
                         "(DMMA.8x8x4, mma.sync f64)", "achieved": gemm_tf,
                         "peak": FP64_PEAK_NOMINAL_TFLOPS, "unit": "TFLOP/s", "frac": gemm_tf / FP64_PEAK_NOMINAL_TFLOPS,
                         "flops_convention": "algorithmic = 8 M N K per complex GEMM (LAPACK); the 3M kernel executes 6 real "
                         "flops per complex multiply-add, so frac may exceed the executed-flop pipe utilisation frac_executed",
                         "executed_over_algorithmic": EXECUTED_RATIO[is3m],
                         "frac_executed": gemm_tf * EXECUTED_RATIO[is3m] / FP64_PEAK_NOMINAL_TFLOPS,
                         "traffic": NCU_TRAFFIC[is3m]["bytes"], "traffic_note": NCU_TRAFFIC[is3m]["note"],
                         "peak_source": "148 SM x 64 FP64 FMA/clk x 2 x 1.965 GHz; no FP64 peak in "
                         "MEASURED_PEAKS.json", "peak_measured_dmma_microbench": peak_measured,
                         "gemm_launches": gemm_n, "gemm_share_of_step": gemm_ms / gemm_ref_ms,
                         "gemm_flops_share": gemm_fl / (flops_step * (args.steps if serial else 1)),
                         "measured_in": "timed region (single stream)" if serial else
                         "one extra step with stream_groups=1 right after the timed region (kernels of different stream "
                         f"groups overlap in the timed region); that serial step took {gemm_ref_ms:.1f} ms"},
            "gpu_launches": int(launches * args.steps),
            "clocks": clocks.summary(),
            "T_first_energy": float(T_all[0]),
        }
        if e2e:
            line["e2e"] = e2e
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = cpu_baseline(cfg)
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse()
    cfg = inputs.CONFIGS[args.workload]
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
