"""Times ss_density alone and prints its HBM roofline fraction.
  python -m paper_1812_01396_b200.density_bench [n_energy n nrhs [reps]]
Algorithmic bytes = 16 * n_energy * n * nrhs (X read once) + 8 * n (rho written); peak = MEASURED_PEAKS.json hbm_gbs."""
import json
import os
import sys

import torch

from . import binding


def main():
    a = [int(x) for x in sys.argv[1:]]
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
    bytes_alg = 16.0 * n_energy * n * nrhs + 8.0 * n
    gbs = bytes_alg / best / 1e6
    peak = None
    path = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "MEASURED_PEAKS.json")
    if os.path.exists(path):
        peak = json.load(open(path)).get("hbm_gbs")
    src = "measured" if peak else "fallback"
    peak = peak or 6650.0
    print(f"density n_energy={n_energy} n={n} nrhs={nrhs}: {best:.3f} ms  {gbs:.0f} GB/s = {gbs / peak:.3f} of {src} {peak:.0f} GB/s  "
          f"rel err {err:.1e}")


if __name__ == "__main__":
    main()
