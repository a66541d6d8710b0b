"""Times the library's batched complex-FP64 GEMM kernel alone (ss_zgemm_batched) and prints TFLOP/s
(LAPACK convention: 8 flops per complex multiply-add, whatever the variant executes).
  python -m paper_1812_01396_b200.gemm_bench [M N K batch [reps]] [--variant V[,V...]]
Used for the ncu `--set full` capture of the dominant kernel (profiles/) and for tuning."""
import argparse

import torch

from . import binding


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("dims", nargs="*", type=int)
    ap.add_argument("--beta", type=float, default=0.0, help="C = A B + beta C (beta = 1: the in-place update form of the LU/TRSM steps)")
    ap.add_argument("--variant", default=None, help="comma-separated GEMM variants (binding.GEMM_VARIANTS); default: library default")
    args = ap.parse_args()
    a = args.dims
    M, N, K, batch = (a + [2048, 2048, 2048, 16][len(a):])[:4]
    reps = a[4] if len(a) > 4 else 5
    variants = [binding.get_default_gemm_variant()] if args.variant is None else [int(v) for v in args.variant.split(",")]
    g = torch.Generator(device="cuda").manual_seed(0)
    A = torch.randn((batch, M, K), dtype=torch.complex128, device="cuda", generator=g)
    B = torch.randn((batch, K, N), dtype=torch.complex128, device="cuda", generator=g)
    C = torch.zeros((batch, M, N), dtype=torch.complex128, device="cuda")
    ref = A[0] @ B[0]
    for v in variants:
        binding.set_default_gemm_variant(v)
        C.zero_()
        for _ in range(2):
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
        print(f"zgemm[{binding.GEMM_VARIANTS[v]}] M={M} N={N} K={K} batch={batch} beta={args.beta:g}: {best:.3f} ms  "
              f"{8.0 * M * N * K * batch / best / 1e9:.2f} TFLOP/s  max err/sqrt(K) {err:.2e}", flush=True)


if __name__ == "__main__":
    main()
