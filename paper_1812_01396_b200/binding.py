"""Thin ctypes binding of libsplitsolve (include/splitsolve.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels.  torch is used for device buffers and streams
(`tensor.data_ptr()`, `torch.cuda.current_stream().cuda_stream`).  There is no CPU fallback: loading fails
loudly when the shared library is missing.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, byref, c_char_p, c_double, c_float, c_int, c_longlong, c_size_t, c_void_p

PKG_DIR = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(PKG_DIR, "libsplitsolve.so")

SS_OK, SS_ERR_INVALID_ARG, SS_ERR_NOT_READY, SS_ERR_ALLOC, SS_ERR_SINGULAR, SS_ERR_CUDA, SS_ERR_UNSTABLE = range(7)

# every symbol include/splitsolve.h declares: name -> (restype, argtypes)
SIGNATURES = {
    "ss_create": (c_int, [c_int, c_int, c_int, POINTER(c_void_p)]),
    "ss_destroy": (c_int, [c_void_p]),
    "ss_set_hamiltonian": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p]),
    "ss_set_hamiltonian_host": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p]),
    "ss_solve": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_int, c_void_p, c_void_p]),
    "ss_solve_host": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_int, c_void_p, c_void_p]),
    "ss_sweep_column": (c_int, [c_void_p, c_void_p, c_int, c_void_p]),
    "ss_get_corner_blocks": (c_int, [c_void_p, c_int, c_void_p, c_void_p]),
    "ss_post_column": (c_int, [c_void_p, c_int, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_int, c_void_p, c_void_p]),
    "ss_sweep_partition": (c_int, [c_void_p, c_void_p, c_void_p]),
    "ss_get_edge_blocks": (c_int, [c_void_p, c_int, c_void_p, c_void_p]),
    "ss_merge_partition": (c_int, [c_void_p, c_int, c_void_p, c_void_p, c_void_p, c_void_p]),
    "ss_post_partition": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_int, c_void_p, c_void_p]),
    "ss_synchronize": (c_int, [c_void_p]),
    "ss_transmission": (c_int, [c_void_p, c_void_p]),
    "ss_inverse_columns": (c_int, [c_void_p, c_int, POINTER(c_void_p), POINTER(c_void_p)]),
    "ss_copy_inverse_columns": (c_int, [c_void_p, c_int, c_void_p, c_void_p]),
    "ss_last_info": (c_int, [c_void_p, POINTER(c_int), POINTER(c_int), POINTER(c_int)]),
    "ss_last_mode": (c_int, [c_void_p, POINTER(c_int), POINTER(c_int)]),
    "ss_flops": (c_double, [c_void_p, c_int]),
    "ss_flops_sweep": (c_double, [c_void_p]),
    "ss_workspace_bytes": (c_size_t, [c_int, c_int, c_int, c_int]),
    "ss_phase_ms": (c_int, [c_void_p, c_int, POINTER(c_float)]),
    "ss_gemm_profile": (c_int, [c_void_p, POINTER(c_double), POINTER(c_double), POINTER(c_longlong)]),
    "ss_launch_count": (c_longlong, [c_void_p]),
    "ss_trace_write": (c_int, [c_void_p, c_char_p]),
    "ss_set_option": (c_int, [c_void_p, c_char_p, c_int]),
    "ss_strerror": (c_char_p, [c_int]),
    "ss_zgemm_batched": (c_int, [c_int, c_int, c_int, c_double, c_void_p, c_int, c_longlong, c_void_p, c_int, c_longlong,
                                 c_double, c_void_p, c_int, c_longlong, c_int, c_void_p]),
    "ss_zgemm_batched_sums": (c_int, [c_int, c_int, c_int, c_double, c_void_p, c_void_p, c_int, c_longlong, c_void_p, c_void_p, c_int,
                                      c_longlong, c_double, c_void_p, c_void_p, c_int, c_longlong, c_int, c_void_p]),
    "ss_lu_workspace_bytes": (c_size_t, [c_int, c_int]),
    "ss_zgetrf_batched": (c_int, [c_int, c_int, c_void_p, c_int, c_longlong, c_void_p, c_void_p, c_int, c_void_p, c_size_t,
                                  c_void_p]),
    "ss_zgesv_batched": (c_int, [c_int, c_int, c_void_p, c_int, c_longlong, c_void_p, c_int, c_longlong, c_void_p,
                                 c_void_p, c_int, c_void_p, c_size_t, c_void_p]),
    "ss_zgesv_batched_noalloc": (c_int, [c_int, c_int, c_void_p, c_int, c_longlong, c_void_p, c_int, c_longlong, c_void_p,
                                         c_void_p, c_int, c_void_p]),
    "ss_fp64_peak_tflops": (c_int, [c_double, POINTER(c_double)]),
    "ss_density": (c_int, [c_void_p, c_int, c_longlong, c_int, c_void_p, c_void_p, c_void_p]),
    "ss_bond_current": (c_int, [c_void_p, c_void_p, c_int, c_void_p]),
    "ss_set_default_gemm_variant": (c_int, [c_int]),
    "ss_get_default_gemm_variant": (c_int, []),
    "ss_set_gemm_raster": (c_int, [c_int]),
}

_lib = None


class SplitSolveError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = load().ss_strerror(status).decode() if _lib is not None else str(status)
        super().__init__(f"{where}: {msg} (status {status})")


def load() -> ctypes.CDLL:
    """Loads libsplitsolve.so (built in-tree by build.py).  No fallback."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_1812_01396_b200.build` "
                               "(the CUDA extension is required; there is no CPU fallback)")
        lib = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(lib, name)
            fn.restype = res
            fn.argtypes = args
        _lib = lib
    return _lib


def _check(status: int, where: str):
    if status != SS_OK:
        raise SplitSolveError(status, where)


def _dev(t, name):
    import torch
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.complex128 and t.is_contiguous()):
        raise TypeError(f"{name}: expected a contiguous CUDA complex128 tensor")
    return t.data_ptr()


def _stream():
    import torch
    return torch.cuda.current_stream().cuda_stream


class SplitSolve:
    """ss_create / ss_set_hamiltonian / ss_solve / ss_transmission with torch tensors as buffers."""

    def __init__(self, nb: int, bs: int, n_energy: int):
        self._h = c_void_p()
        self.nb, self.bs, self.n_energy = nb, bs, n_energy
        _check(load().ss_create(nb, bs, n_energy, byref(self._h)), "ss_create")
        self._keep = []

    def close(self):
        if self._h:
            load().ss_destroy(self._h)
            self._h = c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_option(self, name: str, value: int):
        _check(load().ss_set_option(self._h, name.encode(), int(value)), "ss_set_option")

    def set_hamiltonian(self, H_diag, H_upper, S_diag, S_upper):
        self._keep = [H_diag, H_upper, S_diag, S_upper]      # borrowed by the library: keep alive
        _check(load().ss_set_hamiltonian(self._h, _dev(H_diag, "H_diag"), _dev(H_upper, "H_upper"),
                                         _dev(S_diag, "S_diag"), _dev(S_upper, "S_upper")), "ss_set_hamiltonian")

    def set_hamiltonian_host(self, H_diag, H_upper, S_diag, S_upper):
        """Host buffers: numpy complex128 arrays or CPU torch tensors (C-contiguous).  Uploaded asynchronously (pinned
        memory): kept alive here until replaced."""
        self._keep = [H_diag, H_upper, S_diag, S_upper]
        _check(load().ss_set_hamiltonian_host(self._h, _host(H_diag), _host(H_upper), _host(S_diag), _host(S_upper)),
               "ss_set_hamiltonian_host")

    def solve(self, E, Sigma_L, Sigma_R, Inj_first, Inj_last=None, X=None):
        """E: host complex128 (numpy / list); other arguments CUDA complex128 tensors. Returns X (enqueued)."""
        import numpy as np
        import torch
        E = np.ascontiguousarray(np.asarray(E, dtype=np.complex128))
        assert E.shape == (self.n_energy,)
        nrhs = 0 if Inj_first is None else int(Inj_first.shape[-1])
        if X is None and nrhs > 0:
            X = torch.empty((self.n_energy, self.nb * self.bs, nrhs), dtype=torch.complex128, device=Sigma_L.device)
        self._keep_solve = [Sigma_L, Sigma_R, Inj_first, Inj_last, X]
        _check(load().ss_solve(self._h, E.ctypes.data, _dev(Sigma_L, "Sigma_L"), _dev(Sigma_R, "Sigma_R"),
                               _dev(Inj_first, "Inj_first"), _dev(Inj_last, "Inj_last"), nrhs, _dev(X, "X"),
                               _stream()), "ss_solve")
        return X

    def solve_host(self, E, Sigma_L, Sigma_R, Inj_first, Inj_last, X_out, T_out):
        """All host buffers (numpy or pinned CPU torch tensors); blocking; H2D/D2H copies inside the call."""
        import numpy as np
        E = np.ascontiguousarray(np.asarray(E, dtype=np.complex128))
        nrhs = 0 if Inj_first is None else int(Inj_first.shape[-1])
        _check(load().ss_solve_host(self._h, E.ctypes.data, _host(Sigma_L), _host(Sigma_R), _host(Inj_first),
                                    _host(Inj_last), nrhs, _host(X_out), _host(T_out)), "ss_solve_host")

    # ---- one block column of A^-1 per GPU ----
    def sweep_column(self, E, column: int):
        import numpy as np
        E = np.ascontiguousarray(np.asarray(E, dtype=np.complex128))
        assert E.shape == (self.n_energy,)
        _check(load().ss_sweep_column(self._h, E.ctypes.data, int(column), _stream()), "ss_sweep_column")

    def corner_blocks(self, column: int):
        """Blocks 1 and nb of that block column for every energy: CUDA tensor [n_energy, 2, bs, bs] (enqueued)."""
        import torch
        out = torch.empty((self.n_energy, 2, self.bs, self.bs), dtype=torch.complex128, device="cuda")
        _check(load().ss_get_corner_blocks(self._h, int(column), out.data_ptr(), _stream()), "ss_get_corner_blocks")
        return out

    def post_column(self, column: int, peer_corner, Sigma_L, Sigma_R, Inj_first, Inj_last=None, X_part=None):
        import torch
        nrhs = 0 if Inj_first is None else int(Inj_first.shape[-1])
        if X_part is None and nrhs > 0:
            X_part = torch.empty((self.n_energy, self.nb * self.bs, nrhs), dtype=torch.complex128, device=Sigma_L.device)
        self._keep_solve = [peer_corner, Sigma_L, Sigma_R, Inj_first, Inj_last, X_part]
        _check(load().ss_post_column(self._h, int(column), _dev(peer_corner, "peer_corner"), _dev(Sigma_L, "Sigma_L"),
                                     _dev(Sigma_R, "Sigma_R"), _dev(Inj_first, "Inj_first"), _dev(Inj_last, "Inj_last"), nrhs,
                                     _dev(X_part, "X_part"), _stream()), "ss_post_column")
        return X_part

    # ---- the device split into two halves, one per GPU ----
    def sweep_partition(self, E):
        import numpy as np
        E = np.ascontiguousarray(np.asarray(E, dtype=np.complex128))
        assert E.shape == (self.n_energy,)
        _check(load().ss_sweep_partition(self._h, E.ctypes.data, _stream()), "ss_sweep_partition")

    def edge_blocks(self, edge: int):
        """[n_energy, 2, bs, bs]: block `edge` (0 first, 1 last) of the first and of the last block column."""
        import torch
        out = torch.empty((self.n_energy, 2, self.bs, self.bs), dtype=torch.complex128, device="cuda")
        _check(load().ss_get_edge_blocks(self._h, int(edge), out.data_ptr(), _stream()), "ss_get_edge_blocks")
        return out

    def merge_partition(self, part: int, iface, S_couple, H_couple):
        """iface [n_energy, 2, 2, bs, bs]: [:, 0] = last block of both columns of the top partition, [:, 1] = first block of
        both columns of the bottom partition."""
        self._keep_merge = [iface, S_couple, H_couple]
        _check(load().ss_merge_partition(self._h, int(part), _dev(iface, "iface"), _dev(S_couple, "S_couple"),
                                         _dev(H_couple, "H_couple"), _stream()), "ss_merge_partition")

    def post_partition(self, corners, Sigma_L, Sigma_R, Inj_first, Inj_last=None, X_rows=None):
        """corners [n_energy, 2, 2, bs, bs]: [:, 0] = first block, [:, 1] = last block of the global (Q, P) columns."""
        peer_corner = corners
        import torch
        nrhs = 0 if Inj_first is None else int(Inj_first.shape[-1])
        if X_rows is None and nrhs > 0:
            X_rows = torch.empty((self.n_energy, self.nb * self.bs, nrhs), dtype=torch.complex128, device=Sigma_L.device)
        self._keep_solve = [peer_corner, Sigma_L, Sigma_R, Inj_first, Inj_last, X_rows]
        _check(load().ss_post_partition(self._h, _dev(peer_corner, "peer_corner"), _dev(Sigma_L, "Sigma_L"), _dev(Sigma_R, "Sigma_R"),
                                        _dev(Inj_first, "Inj_first"), _dev(Inj_last, "Inj_last"), nrhs, _dev(X_rows, "X_rows"),
                                        _stream()), "ss_post_partition")
        return X_rows

    def synchronize(self):
        _check(load().ss_synchronize(self._h), "ss_synchronize")

    def transmission(self):
        import numpy as np
        T = np.empty(self.n_energy, dtype=np.float64)
        _check(load().ss_transmission(self._h, T.ctypes.data), "ss_transmission")
        return T

    def inverse_columns(self, energy: int):
        """Copies of Q = (A^-1)[:, first block] and P = (A^-1)[:, last block], each [nb, bs, bs] (CUDA tensors)."""
        import torch
        Q = torch.empty((self.nb, self.bs, self.bs), dtype=torch.complex128, device="cuda")
        P = torch.empty_like(Q)
        _check(load().ss_copy_inverse_columns(self._h, energy, Q.data_ptr(), P.data_ptr()), "ss_copy_inverse_columns")
        torch.cuda.current_stream().synchronize()
        return Q, P

    def last_info(self):
        e, b, c = c_int(), c_int(), c_int()
        _check(load().ss_last_info(self._h, byref(e), byref(b), byref(c)), "ss_last_info")
        return e.value, b.value, c.value

    def last_mode(self):
        """(mode, retried) of the last solve: 0 general, 1 Hermitian Schur update, 2 + no-pivot L Delta L^H."""
        m, r = c_int(), c_int()
        _check(load().ss_last_mode(self._h, byref(m), byref(r)), "ss_last_mode")
        return m.value, r.value

    def flops(self, nrhs: int) -> float:
        return float(load().ss_flops(self._h, nrhs))

    def flops_sweep(self) -> float:
        return float(load().ss_flops_sweep(self._h))

    def phase_ms(self, phase: int) -> float:
        ms = c_float()
        _check(load().ss_phase_ms(self._h, phase, byref(ms)), "ss_phase_ms")
        return float(ms.value)

    def gemm_profile(self):
        """(device ms, algorithmic flops, launches) of the GEMM kernel in the last solve (option profile_gemm=1)."""
        ms, fl, n = c_double(), c_double(), c_longlong()
        _check(load().ss_gemm_profile(self._h, byref(ms), byref(fl), byref(n)), "ss_gemm_profile")
        return float(ms.value), float(fl.value), int(n.value)

    def bond_current(self, X):
        """J[e, i] = 2 Im Tr(X_i^H A_{i,i+1}(E_e) X_{i+1}) for the X of the last solve: numpy float64 [n_energy, nb-1]."""
        import numpy as np
        J = np.empty((self.n_energy, self.nb - 1), dtype=np.float64)
        _check(load().ss_bond_current(self._h, _dev(X, "X"), int(X.shape[-1]), J.ctypes.data), "ss_bond_current")
        return J

    def trace_write(self, path: str):
        _check(load().ss_trace_write(self._h, str(path).encode()), "ss_trace_write")

    def launch_count(self) -> int:
        return int(load().ss_launch_count(self._h))


def _host(a):
    if a is None:
        return None
    import numpy as np
    try:
        import torch
        if isinstance(a, torch.Tensor):
            assert not a.is_cuda and a.is_contiguous()
            return a.data_ptr()
    except ImportError:
        pass
    assert isinstance(a, np.ndarray) and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data


def workspace_bytes(nb, bs, n_energy, nrhs) -> int:
    return int(load().ss_workspace_bytes(nb, bs, n_energy, nrhs))


def zgemm_batched(A, B, C, alpha=1.0, beta=0.0):
    """C[z] = alpha A[z] B[z] + beta C[z]; A [batch,M,K], B [batch,K,N], C [batch,M,N] CUDA complex128."""
    batch, M, K = A.shape
    N = B.shape[2]
    _check(load().ss_zgemm_batched(M, N, K, alpha, _dev(A, "A"), K, M * K, _dev(B, "B"), N, K * N, beta,
                                   _dev(C, "C"), N, M * N, batch, _stream()), "ss_zgemm_batched")
    return C


def zgemm_batched_sums(A, As, B, Bs, C, Cs=None, alpha=1.0, beta=0.0):
    """zgemm_batched with sum planes As = A.real + A.imag, Bs likewise (float64 CUDA tensors, same shapes); Cs (optional,
    float64 [batch, M, N]) receives C.real + C.imag."""
    batch, M, K = A.shape
    N = B.shape[2]
    _check(load().ss_zgemm_batched_sums(M, N, K, alpha, _dev(A, "A"), As.data_ptr(), K, M * K, _dev(B, "B"), Bs.data_ptr(), N, K * N,
                                        beta, _dev(C, "C"), None if Cs is None else Cs.data_ptr(), N, M * N, batch, _stream()),
           "ss_zgemm_batched_sums")
    return C


def _lu_work(n, batch, device):
    """Caller-owned scratch of ss_zgetrf_batched / ss_zgesv_batched (torch keeps it alive until the stream has used it)."""
    import torch
    return torch.empty(int(load().ss_lu_workspace_bytes(n, batch)), dtype=torch.uint8, device=device)


def zgetrf_batched(AB, n):
    """In-place LU of the leading n x n part of AB [batch, n, ncols]; returns (ipiv, info) int32 CUDA tensors."""
    import torch
    batch, rows, ncols = AB.shape
    assert rows == n
    ipiv = torch.zeros((batch, n), dtype=torch.int32, device=AB.device)
    info = torch.zeros((batch,), dtype=torch.int32, device=AB.device)
    work = _lu_work(n, batch, AB.device)
    _check(load().ss_zgetrf_batched(n, ncols, _dev(AB, "AB"), ncols, n * ncols, ipiv.data_ptr(), info.data_ptr(), batch,
                                    work.data_ptr(), work.numel(), _stream()), "ss_zgetrf_batched")
    return ipiv, info


def zgesv_batched(AB, n):
    """Solves A X = B for AB = [A | B] [batch, n, n + nrhs] (overwritten); returns X [batch, n, nrhs], ipiv, info."""
    import torch
    batch, rows, ncols = AB.shape
    nrhs = ncols - n
    X = torch.empty((batch, n, nrhs), dtype=torch.complex128, device=AB.device)
    ipiv = torch.zeros((batch, n), dtype=torch.int32, device=AB.device)
    info = torch.zeros((batch,), dtype=torch.int32, device=AB.device)
    work = _lu_work(n, batch, AB.device)
    _check(load().ss_zgesv_batched(n, nrhs, _dev(AB, "AB"), ncols, n * ncols, _dev(X, "X"), nrhs, n * nrhs,
                                   ipiv.data_ptr(), info.data_ptr(), batch, work.data_ptr(), work.numel(), _stream()),
           "ss_zgesv_batched")
    return X, ipiv, info


NOALLOC_SCRATCH_BYTES = 16 << 20      # SS_NOALLOC_SCRATCH_BYTES of include/splitsolve.h


def zgesv_batched_noalloc(AB, X, ipiv, info, n):
    """ss_zgesv_batched_noalloc: zgesv_batched for callers that cannot allocate device memory (they were only handed
    pointers, the HBM is fully spoken for, or a cudaMalloc stall is not affordable where they run).  Nothing is allocated
    here either: the caller passes every buffer -- AB [batch, n, n + nrhs] (overwritten), X [batch, n, nrhs] out, ipiv
    [batch, n] int32 out, info [batch] int32 out, all CUDA tensors on the current device -- and the scratch is the library's
    built-in array of NOALLOC_SCRATCH_BYTES, which limits the size (load().ss_lu_workspace_bytes(n, batch) must fit, else
    SplitSolveError "invalid argument") and is shared by all calls on the device: calls whose GPU work could overlap must
    be ordered by the caller.  Make the first call on a device during set-up, before any stream capture."""
    import torch
    batch, rows, ncols = AB.shape
    nrhs = ncols - n
    assert rows == n and tuple(X.shape) == (batch, n, nrhs)
    for t, shape in ((ipiv, (batch, n)), (info, (batch,))):
        if not (t.is_cuda and t.dtype == torch.int32 and t.is_contiguous() and tuple(t.shape) == shape):
            raise TypeError(f"expected a contiguous CUDA int32 tensor of shape {shape}")
    _check(load().ss_zgesv_batched_noalloc(n, nrhs, _dev(AB, "AB"), ncols, n * ncols, _dev(X, "X"), nrhs, n * nrhs,
                                           ipiv.data_ptr(), info.data_ptr(), batch, _stream()), "ss_zgesv_batched_noalloc")
    return X, ipiv, info


def density(X, w=None):
    """rho[i] = sum_e w[e] sum_c |X[e, i, c]|^2 for X [n_energy, n, nrhs] (CUDA complex128); w CUDA float64 [n_energy] or None."""
    import torch
    n_energy, n, nrhs = X.shape
    rho = torch.empty(n, dtype=torch.float64, device=X.device)
    if w is not None and not (w.is_cuda and w.dtype == torch.float64 and w.is_contiguous() and w.numel() == n_energy):
        raise TypeError("w: expected a contiguous CUDA float64 tensor [n_energy]")
    _check(load().ss_density(_dev(X, "X"), n_energy, n, nrhs, None if w is None else w.data_ptr(), rho.data_ptr(), _stream()),
           "ss_density")
    return rho


GEMM_VARIANTS = {0: "4M 64x64", 1: "3M 64x32 (3 CTAs/SM for K<768, software-pipelined 2 CTAs/SM above)",
                 2: "3M 64x32 lean, every K", 3: "3M 64x32 software-pipelined, every K",
                 4: "3M 64x32 software-pipelined, TMA-staged operands, 2 CTAs/SM (experiment; uniformly strided batches only)",
                 5: "3M 64x32 software-pipelined, TMA-staged operands, 3 CTAs/SM (experiment)"}


def set_default_gemm_variant(variant: int):
    _check(load().ss_set_default_gemm_variant(int(variant)), "ss_set_default_gemm_variant")


def set_gemm_raster(tile_rows: int):
    _check(load().ss_set_gemm_raster(int(tile_rows)), "ss_set_gemm_raster")


def get_default_gemm_variant() -> int:
    return int(load().ss_get_default_gemm_variant())


def fp64_peak_tflops(ms: float = 200.0) -> float:
    out = c_double()
    _check(load().ss_fp64_peak_tflops(ms, byref(out)), "ss_fp64_peak_tflops")
    return float(out.value)
