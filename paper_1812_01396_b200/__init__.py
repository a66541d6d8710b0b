"""libsplitsolve on B200: the GPU half of SplitSolve (arxiv/paper_1812_01396, §3B) as hand-written
sm_100a CUDA kernels behind a C ABI (`include/splitsolve.h`), plus a thin ctypes binding (`binding`).

Importing the package does not load the shared library; `binding` does, and fails loudly when the
CUDA extension is missing.  There is no CPU fallback.  `inputs` holds the seeded synthetic input generators.
"""
__all__ = ["inputs", "binding", "build"]
