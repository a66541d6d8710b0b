"""ss_zgesv_batched_noalloc (include/splitsolve.h): the batched LU solve for callers that cannot allocate device memory.

Some users of this library never get to call cudaMalloc: a plug-in that a host application hands device pointers to and
that owns no allocator, a run whose HBM has been given away completely (H, S and the block columns of a large device, or
another framework's pool), a latency-critical loop in which the device-wide stall of cudaMalloc / cudaFree is not
acceptable.  For them the library carries one fixed scratch array (SS_NOALLOC_SCRATCH_BYTES = 16 MiB per GPU, held until
the process exits) and this entry point uses it instead of a caller-owned work buffer.

What is checked: on two calls in a row (different sizes, so the second finds the first one's leftovers in the shared
array) the results equal those of the existing ss_zgesv_batched path, within the tolerances tests/test_parity_gpu.py uses
for that path and -- since the same kernels run in the same order -- bit for bit; a request beyond the limit is refused
with a clear error and touches nothing; a repeated call leaves the amount of free device memory unchanged.

The no-alloc call comes FIRST in the test, before the reference path, so that in a fresh process it is the first thing the
library does on the device (the one-time address look-up of the scratch array happens cold).  The file name sorts last on
purpose: pytest -x stops at the first failure, and a failure here must not hide the parity tests.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from paper_1812_01396_b200 import inputs  # noqa: E402

pytestmark = pytest.mark.gpu


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def outputs(batch, n, nrhs):
    """Caller-owned outputs, filled with sentinels so that an entry the library did not write shows up."""
    X = torch.full((batch, n, nrhs), complex(np.nan, np.nan), dtype=torch.complex128, device="cuda")
    ipiv = torch.full((batch, n), -7, dtype=torch.int32, device="cuda")
    info = torch.full((batch,), -7, dtype=torch.int32, device="cuda")
    return X, ipiv, info


def test_noalloc_solve_matches_the_existing_path_on_two_calls_in_a_row(lib):
    cases = [(513, 10, 1, 160), (200, 37, 2, 161)]      # n, nrhs, batch, seed: several 128-panels + a ragged tail, then smaller
    mats = []
    for n, nrhs, batch, seed in cases:
        A = inputs.complex_gaussian(2, seed, n, (batch, n, n), 1.0)
        B = inputs.complex_gaussian(2, seed + 50, n, (batch, n, nrhs), 1.0)
        mats.append((A, B))
        assert lib.load().ss_lu_workspace_bytes(n, batch) <= lib.NOALLOC_SCRATCH_BYTES

    # the two no-alloc calls, back to back on one stream, nothing else from the library in between
    got = []
    for (n, nrhs, batch, _), (A, B) in zip(cases, mats):
        AB = dev(np.concatenate([A, B], axis=2))
        got.append(lib.zgesv_batched_noalloc(AB, *outputs(batch, n, nrhs), n) + (AB,))
    torch.cuda.synchronize()

    for (n, nrhs, batch, _), (A, B), (X, ipiv, info, AB) in zip(cases, mats, got):
        AB_ref = dev(np.concatenate([A, B], axis=2))
        X_ref, ipiv_ref, info_ref = lib.zgesv_batched(AB_ref, n)
        torch.cuda.synchronize()
        assert int(info.abs().max()) == 0 and int(info_ref.abs().max()) == 0
        Xh, Xr = X.cpu().numpy(), X_ref.cpu().numpy()
        assert np.isfinite(Xh).all()
        for z in range(batch):
            # the tolerances of test_zgesv_batched_vs_numpy: relative 1e-9 on X, backward error 1e-13
            assert np.linalg.norm(Xh[z] - Xr[z]) <= 1e-9 * np.linalg.norm(Xr[z])
            res = np.linalg.norm(A[z] @ Xh[z] - B[z]) / (np.linalg.norm(A[z]) * np.linalg.norm(Xh[z]) + np.linalg.norm(B[z]))
            assert res <= 1e-13, (n, z, res)
        # same kernels, same order, only the scratch lives elsewhere: identical bits, pivots and factors included
        assert torch.equal(ipiv, ipiv_ref)
        assert torch.equal(X, X_ref)
        assert torch.equal(AB, AB_ref)


def test_noalloc_refuses_sizes_beyond_its_scratch_and_touches_nothing(lib):
    n, nrhs, batch = 1024, 4, 2                          # 2 x 12 MiB of scratch needed, 16 MiB built in
    assert lib.load().ss_lu_workspace_bytes(n, batch) > lib.NOALLOC_SCRATCH_BYTES
    assert lib.load().ss_lu_workspace_bytes(n, 1) <= lib.NOALLOC_SCRATCH_BYTES      # the documented n = 1024, batch 1 fits
    AB = torch.ones((batch, n, n + nrhs), dtype=torch.complex128, device="cuda")
    X, ipiv, info = outputs(batch, n, nrhs)
    with pytest.raises(lib.SplitSolveError, match="invalid argument") as err:
        lib.zgesv_batched_noalloc(AB, X, ipiv, info, n)
    assert err.value.status == lib.SS_ERR_INVALID_ARG
    torch.cuda.synchronize()
    assert int((info == -7).sum()) == batch and int((ipiv == -7).sum()) == batch * n
    assert bool(torch.isnan(X.real).all()) and bool((AB == 1).all())


def test_noalloc_repeat_call_leaves_free_device_memory_unchanged(lib):
    """After a first call of a shape (kernels loaded, scratch address known), calling it again must not lower the free
    device memory the driver reports: the entry point owns no allocation to grow."""
    n, nrhs, batch = 300, 8, 2
    A = inputs.complex_gaussian(2, 170, n, (batch, n, n), 1.0)
    B = inputs.complex_gaussian(2, 171, n, (batch, n, nrhs), 1.0)
    AB0 = dev(np.concatenate([A, B], axis=2))
    AB1, AB2 = AB0.clone(), AB0.clone()
    o1, o2 = outputs(batch, n, nrhs), outputs(batch, n, nrhs)
    lib.zgesv_batched_noalloc(AB1, *o1, n)
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    lib.zgesv_batched_noalloc(AB2, *o2, n)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after >= free_before
    assert torch.equal(o1[0], o2[0]) and torch.equal(o1[1], o2[1])
