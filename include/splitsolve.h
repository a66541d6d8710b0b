/*
 * libsplitsolve -- the GPU half of the SplitSolve algorithm (arxiv/paper_1812_01396, §3B,
 * L125-175) for one NVIDIA B200 (sm_100a).  C ABI: plain pointers and sizes, no C++/torch types.
 *
 * For each energy point E the library solves the open-boundary Schroedinger equation (Eq. 5)
 *
 *        (E*S - H - Sigma_L - Sigma_R) * X = Inj ,
 *
 * H, S block tridiagonal with nb diagonal blocks of size bs x bs (L127), complex FP64 throughout:
 *   pre-processing  (Alg. 1, and its mirror, L167): forward/backward block-Schur sweeps over
 *                   A = E*S - H give Q_i = (A^-1)_{i,1} and P_i = (A^-1)_{i,nb}, i = 1..nb;
 *   post-processing (L141-146, L148, L155, L175): R = 1 - C*[Q P] (2bs x 2bs corner system),
 *                   w = R^-1 b',  X_i = Q_i w_top + P_i w_bot;
 *   transmission    T(E) = Re Tr(Gamma_L G_1N Gamma_R G_1N^H), Gamma = i(Sigma - Sigma^H),
 *                   G_1N = Q_1 (R^-1)_12 + P_1 (R^-1)_22      (BASELINE.json north_star; L23, L85).
 *
 * Conventions
 *   - ss_cplx is {double re, im}: identical to C99 `double _Complex`, numpy/torch complex128.
 *   - All matrices are ROW-MAJOR (C-contiguous), dense, leading dimension = number of columns unless a
 *     leading dimension argument says otherwise.  Blocks are 0-indexed in memory: H_diag[i] is the paper's
 *     H_{i+1,i+1}; H_upper[i] is H_{i+1,i+2}.  The lower blocks are implied: H_{i+1,i} = H_{i,i+1}^H (L154),
 *     and A_{i+1,i} = E*S_{i,i+1}^H - H_{i,i+1}^H with E NOT conjugated.
 *   - Pointers named *_dev are CUDA device pointers (16-byte aligned), *_host are host pointers.
 *     The caller owns every buffer it passes in.  Device inputs of ss_set_hamiltonian are BORROWED: they
 *     must stay valid and unchanged while the handle uses them.  The handle owns its workspace.
 *   - Every function returns an ss_status_t (except the pure queries); nothing throws or aborts.
 *   - A handle is not thread-safe.  Device work is enqueued on the stream given to ss_solve (NULL = the
 *     legacy default stream); ss_solve returns after enqueueing, results are complete after
 *     ss_synchronize / ss_transmission or a synchronisation of that stream by the caller.
 *   - ss_solve first waits (on the host) for the previous ss_solve of the SAME handle to finish: its per-solve scratch
 *     and the staged energies are reused.  Use one handle per concurrently running solve.
 *   - One process drives one GPU (the device current at ss_create); kernel attributes are set once per process.
 *   - Limits of this version: 2 <= nb, 1 <= bs <= 4096, 1 <= n_energy, 0 <= nrhs.
 *   - Accuracy.  With Im E > 0 (the configurations of BASELINE.json use 1e-3) the results meet: normwise backward error of
 *     X <= 1e-12, relative error of X <= 1e-8 and of T(E) <= 1e-9 against a dense LU of the whole matrix.  At Im E == 0 and
 *     E inside the band, A = E*S - H (WITHOUT the self-energies) is nearly singular at the resonances of the closed device
 *     although the matrix of Eq. 5 is not; the method's split (Eq. 11-13) then loses digits in proportion to kappa(A):
 *     backward errors up to ~1e-11 were measured on random devices (the paper's own sequence of steps evaluated in numpy
 *     shows the same).  A caller that needs the tight tolerances at real energies adds a small imaginary part to E (the
 *     physical broadening eta); the analytic perfect chain and energies outside the spectrum are not affected.
 */
#ifndef SPLITSOLVE_H
#define SPLITSOLVE_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct { double re, im; } ss_cplx;
typedef struct ss_handle_s* ss_handle_t;

typedef enum {
    SS_OK = 0,
    SS_ERR_INVALID_ARG = 1,   /* NULL pointer, size out of range */
    SS_ERR_NOT_READY = 2,     /* ss_solve before ss_set_hamiltonian, ss_transmission before ss_solve */
    SS_ERR_ALLOC = 3,         /* device or host allocation failed */
    SS_ERR_SINGULAR = 4,      /* an exactly zero pivot was met; see ss_last_info */
    SS_ERR_CUDA = 5,          /* a CUDA runtime call or kernel launch failed */
    SS_ERR_UNSTABLE = 6       /* split-phase calls with option "hermitian" = 2: the growth limit was exceeded (redo with 0) */
} ss_status_t;

/* ---- life cycle -------------------------------------------------------------------------------------- */

/* Creates a solver for nb diagonal blocks of size bs and up to n_energy energy points per ss_solve.
 * Allocates nothing on the device yet (workspace is allocated lazily by the first ss_solve, when nrhs is
 * known; see ss_workspace_bytes). */
ss_status_t ss_create(int nb, int bs, int n_energy, ss_handle_t* out);

/* Frees the handle and all device memory it owns.  NULL is allowed. */
ss_status_t ss_destroy(ss_handle_t h);

/* ---- inputs ------------------------------------------------------------------------------------------ */

/* Registers H and S (resident in HBM, borrowed -- L184 "stored in their memory").
 *   H_diag_dev, S_diag_dev   : [nb  ][bs][bs]
 *   H_upper_dev, S_upper_dev : [nb-1][bs][bs]  = blocks (i, i+1) */
ss_status_t ss_set_hamiltonian(ss_handle_t h, const ss_cplx* H_diag_dev, const ss_cplx* H_upper_dev,
                               const ss_cplx* S_diag_dev, const ss_cplx* S_upper_dev);

/* Same, from HOST buffers: the handle allocates device copies it owns and uploads them ASYNCHRONOUSLY, block by block in the
 * order the sweeps consume them; the next ss_solve waits per block step, so with pinned host memory the upload overlaps
 * the first block steps.  The host buffers must stay valid and unchanged until that solve has completed (ss_synchronize,
 * ss_transmission or ss_solve_host returned); pageable buffers are staged before the call returns. */
ss_status_t ss_set_hamiltonian_host(ss_handle_t h, const ss_cplx* H_diag_host, const ss_cplx* H_upper_host,
                                    const ss_cplx* S_diag_host, const ss_cplx* S_upper_host);

/* ---- the hot path ------------------------------------------------------------------------------------ */

/* Solves all n_energy energy points.
 *   E_host        : [n_energy] complex energies (host; copied before return)
 *   Sigma_L_dev   : [n_energy][bs][bs]  boundary self-energy of the left contact  (top-left block of C, L148)
 *   Sigma_R_dev   : [n_energy][bs][bs]  right contact (bottom-right block)
 *   Inj_first_dev : [n_energy][bs][nrhs] non-zero rows of Inj in the first block row (L127); may be NULL iff nrhs==0
 *   Inj_last_dev  : same for the last block row, or NULL = zeros
 *   X_dev         : out [n_energy][nb*bs][nrhs]; may be NULL iff nrhs == 0
 *   cuda_stream   : cudaStream_t (as void*), NULL = default stream.  All work is ordered after what is
 *                   already enqueued on it and is complete when it drains.
 * The sweep (a0-a4) reads neither Sigma nor Inj (pre-/post-processing split of L150-152).
 * Errors: argument checks synchronously; a zero pivot is reported by ss_synchronize / ss_transmission. */
ss_status_t ss_solve(ss_handle_t h, const ss_cplx* E_host, const ss_cplx* Sigma_L_dev, const ss_cplx* Sigma_R_dev,
                     const ss_cplx* Inj_first_dev, const ss_cplx* Inj_last_dev, int nrhs, ss_cplx* X_dev,
                     void* cuda_stream);

/* Same with HOST buffers for everything (pageable or pinned): uploads Sigma/Inj into device buffers the
 * handle owns, runs ss_solve on an internal stream, downloads X (may be NULL) and T (may be NULL), synchronises.
 * Returns SS_ERR_SINGULAR if a pivot was exactly zero. */
ss_status_t ss_solve_host(ss_handle_t h, const ss_cplx* E_host, const ss_cplx* Sigma_L_host,
                          const ss_cplx* Sigma_R_host, const ss_cplx* Inj_first_host, const ss_cplx* Inj_last_host,
                          int nrhs, ss_cplx* X_host, double* T_host);

/* ---- one energy batch on two GPUs (computing the first and the last block column of
 * A^-1 "naturally scale[s] to two accelerators"; L175: z is distributed to all accelerators) --------------------------
 * GPU 0 runs the first-column sweep, GPU 1 the last-column sweep, each on its own handle with the full H and S:
 *     ss_sweep_column(h, E, column)                 a0-a4 for that block column only (Q_i resp. P_i, i = 1..nb)
 *     ss_get_corner_blocks(h, column, out)          out[e][0] = block 1, out[e][1] = block nb of that column
 *     -- the two GPUs exchange their corner blocks (2 * n_energy * 2 blocks of bs x bs; NCCL / peer copy, caller's job) --
 *     ss_post_column(h, column, peer_corner, ...)   a5 and a7 redundantly on both GPUs (R needs all four corner blocks and is
 *                                                   only 2bs x 2bs), a6 for the own column only:
 *                                                   X_part = Q_i w_top (column 0) resp. P_i w_bot (column 1)
 *     -- X = X_part(GPU 0) + X_part(GPU 1): one sum-reduction of [n_energy][nb*bs][nrhs] (caller's job) --
 * ss_transmission / ss_synchronize work as after ss_solve (T(E) is complete on both GPUs).
 *   column          : 0 = first block column (Q), 1 = last block column (P)
 *   out_dev / peer_corner_dev : [n_energy][2][bs][bs], caller-owned device memory
 * Errors as for ss_solve; SS_ERR_NOT_READY if the calls come out of order or for another column than the one swept. */
ss_status_t ss_sweep_column(ss_handle_t h, const ss_cplx* E_host, int column, void* cuda_stream);
ss_status_t ss_get_corner_blocks(ss_handle_t h, int column, ss_cplx* out_dev, void* cuda_stream);
ss_status_t ss_post_column(ss_handle_t h, int column, const ss_cplx* peer_corner_dev, const ss_cplx* Sigma_L_dev,
                           const ss_cplx* Sigma_R_dev, const ss_cplx* Inj_first_dev, const ss_cplx* Inj_last_dev, int nrhs,
                           ss_cplx* X_part_dev, void* cuda_stream);

/* ---- one energy batch on 2^k GPUs, split ALONG THE DEVICE ("horizontal split", L169 SPIKE:
 * "power of 2" partitions merged recursively).  Every GPU owns a contiguous run of blocks and creates a handle for ITS
 * sub-device (its slices of H_diag/S_diag, H_upper/S_upper; >= 2 blocks) -- none holds the whole H, S or whole block columns.
 *     ss_sweep_partition(h, E)                       a0-a4 on the sub-device: first and last block column of its own inverse
 *     ss_get_edge_blocks(h, edge, out)               out[e][0] / out[e][1] = block `edge` (0 first, 1 last) of the first / last
 *                                                    block column the handle currently holds
 *     per merge level (teams of 2, 4, ... partitions; top half = part 0, bottom half = part 1):
 *       -- gather iface[e][0] = edge 1 of the LAST partition of the top half, iface[e][1] = edge 0 of the FIRST partition of the
 *          bottom half ([n_energy][2][2][bs][bs]) on every GPU of the team --
 *       ss_merge_partition(h, part, iface, S_c, H_c) S_c, H_c = the coupling blocks S_{h,h+1}, H_{h,h+1} of the boundary (device,
 *                                                    [bs][bs]).  With U = E S_c - H_c, L = E S_c^H - H_c^H, (QT_h, PT_h) = iface[e][0],
 *                                                    (QB_1, PB_1) = iface[e][1], every GPU solves
 *                                                        (1 - PT_h U QB_1 L) a = QT_h,  b = -QB_1 L a,
 *                                                        (1 - QB_1 L PT_h U) b' = PB_1, a' = -PT_h U b'
 *                                                    redundantly and updates ITS rows: in the top half Q_i = QT_i - PT_i (U b),
 *                                                    P_i = -PT_i (U b'); in the bottom half Q_i = -QB_i (L a), P_i = PB_i - QB_i (L a').
 *                                                    Afterwards the handles of the team hold the rows of the first / last block
 *                                                    column of the inverse of the JOINED sub-device.
 *     -- gather corners[e][0] = edge 0 of the first partition (Q_1, P_1), corners[e][1] = edge 1 of the last (Q_nb, P_nb) --
 *     ss_post_partition(h, corners, Sigma_L, Sigma_R, Inj_first, Inj_last, nrhs, X_rows)
 *                                                    a5, a7 redundantly on every GPU, a6 for the own rows:
 *                                                    X_rows [n_energy][nb_local*bs][nrhs]; X is the partitions stacked.
 * (The paper gives no equations for the merge -- its Fig. 6 is not in PAPER.md; these follow from the two halves being
 * coupled through U and L only: x_T = QT - PT U x_{B,1}, x_B = -QB L x_{T,h} for the first block column, and likewise for
 * the last.)  Not available together with option "offload_columns".  Buffers are caller-owned device memory. */
ss_status_t ss_sweep_partition(ss_handle_t h, const ss_cplx* E_host, void* cuda_stream);
ss_status_t ss_get_edge_blocks(ss_handle_t h, int edge, ss_cplx* out_dev, void* cuda_stream);
ss_status_t ss_merge_partition(ss_handle_t h, int part, const ss_cplx* iface_dev, const ss_cplx* S_couple_dev,
                               const ss_cplx* H_couple_dev, void* cuda_stream);
ss_status_t ss_post_partition(ss_handle_t h, const ss_cplx* corners_dev, const ss_cplx* Sigma_L_dev, const ss_cplx* Sigma_R_dev,
                              const ss_cplx* Inj_first_dev, const ss_cplx* Inj_last_dev, int nrhs, ss_cplx* X_rows_dev,
                              void* cuda_stream);

/* Waits for the last ss_solve; returns SS_ERR_SINGULAR if any pivot was exactly zero. */
ss_status_t ss_synchronize(ss_handle_t h);

/* T_host: out [n_energy], T_LR(E) of the last ss_solve.  Synchronises. */
ss_status_t ss_transmission(ss_handle_t h, double* T_host);

/* ---- queries ----------------------------------------------------------------------------------------- */

/* Borrowed device pointers to the inverse block columns of energy `energy` of the last ss_solve, each
 * [nb][bs][bs]: Q_first[i] = (A^-1)_{i+1,1}, Q_last[i] = (A^-1)_{i+1,nb}.  Valid until the next ss_solve. */
ss_status_t ss_inverse_columns(ss_handle_t h, int energy, const ss_cplx** Q_first_dev, const ss_cplx** Q_last_dev);

/* Copies the same two block columns into caller-owned device buffers [nb][bs][bs] (either may be NULL).  Synchronises: waits
 * for the handle's last solve, and the copies are complete on return.  With option "hermitian" = 2 the solve is checked
 * first (and redone on the general path if its growth limit was exceeded), so an error of ss_synchronize can be returned. */
ss_status_t ss_copy_inverse_columns(ss_handle_t h, int energy, ss_cplx* Q_first_out_dev, ss_cplx* Q_last_out_dev);

/* Location of the first exactly-zero pivot (or column without a finite candidate) of the last ss_solve (-1s if none): energy
 * index, 1-based block index i of Alg. 1 (0 = the corner system R; -2 = an interface system of ss_merge_partition, column then
 * 0 for the system of a, 1 for that of b'), column 0 = first-column sweep / 1 = mirror sweep.  Records of the sweep come
 * before those of the corner system and of the merges, and survive later merge levels.  Synchronises. */
ss_status_t ss_last_info(ss_handle_t h, int* energy, int* block, int* column);

/* Closed-form flop count of steps a1-a7 per energy point (LAPACK convention: complex multiply-add = 8 flops;
 * ZGEMM 8MNK, ZGETRF (8/3)n^3, ZTRSM 4n^2 nrhs) of the path the LAST ss_solve took (before any solve: the general
 * path).  ss_flops_sweep counts a1-a4 only: general path (160/3 nb - 32) bs^3; with the Hermitian Schur update
 * (modes 1, 2 of option "hermitian") a1 counts 4 bs^3 per block instead of 8, with L Delta L^H a2 counts 4/3 bs^3 instead of 8/3. */
double ss_flops(ss_handle_t h, int nrhs);
double ss_flops_sweep(ss_handle_t h);

/* Which path the last ss_solve took: *mode = 0 general, 1 Hermitian Schur update, 2 + no-pivot L Delta L^H;
  * *retried = 1 if a mode-2 solve exceeded its growth limit and was redone on the general path (then *mode = 0).
 * Meaningful after ss_synchronize / ss_transmission. */
ss_status_t ss_last_mode(ss_handle_t h, int* mode, int* retried);

/* Device bytes the handle allocates for the solve workspace of (nb, bs, n_energy, nrhs) in the default (fully device-
 * resident) mode.  Not included: caller-owned inputs/outputs; the device copies of H, S that ss_set_hamiltonian_host makes
 * (4 nb bs^2 * 16 B) and the staging buffers of ss_solve_host (Sigma, Inj, X); with option "offload_columns" the block
 * columns shrink from 2 (nb+1) to 2 * ring blocks per energy and move to pinned host memory instead. */
size_t ss_workspace_bytes(int nb, int bs, int n_energy, int nrhs);

/* Device time in milliseconds of the phases of the last ss_solve (CUDA events on its stream):
 * phase 0 = sweep a0-a4, 1 = post-processing a5-a7, 2 = whole call.  Synchronises. */
ss_status_t ss_phase_ms(ss_handle_t h, int phase, float* ms);

/* Number of kernel launches the last ss_solve enqueued. */
long long ss_launch_count(ss_handle_t h);

/* Writes the phase timeline of the last ss_solve (option "trace" = 1, stream_groups > 1) as CSV
 * "group,class,start_ms,end_ms" (times relative to the start of the solve) to `path`.  Synchronises. */
ss_status_t ss_trace_write(ss_handle_t h, const char* path);

/* With option "profile_gemm" = 1, every launch of the GEMM kernel in ss_solve is bracketed by CUDA events on the
 * solve's stream; this returns, for the last ss_solve, the summed device time of those launches (ms), their
 * algorithmic flops (8 M N K per complex GEMM) and their number.  Synchronises. */
ss_status_t ss_gemm_profile(ss_handle_t h, double* ms, double* flops, long long* launches);

/* Options: "hermitian" (0/1/2, default 0): what to exploit when EVERY energy of a
 * solve has Im E == 0, where A = E S - H and all Schur complements D_i are Hermitian in exact arithmetic.
 *   0: nothing (the general path: full Schur update, LU with partial pivoting).
 *   1: the Schur update D_i = A_ii - A_{i,i+1} X_{i+1} computes the lower triangle only (half the a1 flops) and mirrors it.
 *   2: additionally D_i is factored WITHOUT pivoting as L Delta L^H (the paper's zhesv_nopiv: half the a2 flops, no pivot
 *      search, no row interchanges); the largest multiplier met is monitored, and if it exceeds "hermitian_growth_limit"
 *      (default 64) -- or a pivot is exactly zero -- the results are discarded at the next ss_synchronize / ss_transmission /
 *      ss_solve_host and the whole solve is redone on the general path with the same arguments (which must therefore still
 *      be valid then).
 * NUMERICAL CAVEAT (measured): both modes replace the computed product A_{i,i+1} X_{i+1} by its
 * Hermitian part.  The discarded anti-Hermitian part is the forward error of X_{i+1} (~ kappa(D_{i+1}) u), and the general
 * path owes its small backward error to keeping it: at real energies INSIDE the band, where A itself is nearly singular,
 * modes 1 and 2 lose digits in proportion to kappa(A) (backward errors 1e-11 .. 1e-4 on the random test devices against
 * 1e-15 .. 1e-12 for mode 0).  They are exact on the perfect chain (config 1) and meet the tolerances when A is
 * definite (energies outside the spectrum).  Hence off by default.
 * "offload_columns" (0, 1 or a ring size 6..64; default 0; only before the first solve of the handle; SURVEY.md 8(f4),
 * part of Q kept on the host, "the time to transfer ... hidden"): the 2 nb blocks X_i / Y_i -> Q_i / P_i of
 * every energy live in pinned HOST memory owned by the handle (n_energy * 2 (nb+1) bs^2 * 16 B) and the device keeps a ring of
 * `ring` blocks per chain (default 6): every block is written back as soon as it is produced, fetched back two steps ahead
 * for the column recursion a4 and block by block for a6, on a copy stream per stream group, ordered by events only.
 * Device memory for the block columns drops from 2 (nb+1) to 2 * ring blocks per energy; results are bit-identical.
 * ss_inverse_columns is not available in this mode (use ss_copy_inverse_columns).
 * "transmission" (0/1, default 1:
 * compute T(E) in ss_solve), "profile_gemm" (0/1, default 0), "gemm_variant" (see ss_set_default_gemm_variant;
 * default = the process-wide default at ss_create), "trace" (0/1, default 0: record a CUDA-event
 * timeline of every group's high-/low-priority phases, see ss_trace_write), "stream_groups" (1..16,
 * default 4: the energy points are split
 * over that many groups, each with a high-priority stream for the latency-bound panel kernels and a low-priority
 * stream for the large GEMMs, forked from and joined back to the stream given to ss_solve; 1 = everything on that
 * stream). */
ss_status_t ss_set_option(ss_handle_t h, const char* name, int value);

const char* ss_strerror(ss_status_t s);

/* ---- building blocks (device pointers; the kernels the hot path is made of) ----------------------------- */

/* Batched complex-FP64 GEMM on the FP64 tensor pipe (mma.sync f64):
 *   C[z] = alpha * A[z] * B[z] + beta * C[z],  z = 0..batch-1,  A: M x K (lda), B: K x N (ldb), C: M x N (ldc),
 * row-major, matrices of batch z at base + z*stride (elements).  alpha, beta real.  M, N, K >= 0. */
ss_status_t ss_zgemm_batched(int M, int N, int K, double alpha, const ss_cplx* A_dev, int lda, long long strideA,
                             const ss_cplx* B_dev, int ldb, long long strideB, double beta, ss_cplx* C_dev, int ldc,
                             long long strideC, int batch, void* cuda_stream);

/* EXPERIMENT, not used by the solve path (profiles/r02_gemm_sumplane.md: bit-identical, slower); kept for bench.py --sumplane.
 * The same product with SUM PLANES: the 3M arithmetic needs re + im of every operand element; A_sum_dev / B_sum_dev (doubles,
 * same leading dimensions and batch strides as A / B, both or neither) supply them, so that the kernel stages them beside
 * the operands instead of adding per fragment on the FP64 pipe.  They take effect only where the software-pipelined 3M
 * kernel runs (GEMM variant 3, or variant 1 with K >= 768) and K, N, lda, ldb and the strides are even; everywhere else
 * they are ignored and the plain product runs -- C holds the same bits either way.  C_sum_dev (or NULL) receives re + im of
 * every element of C under every 3M variant (1..5); under variant 0 (4M) a non-NULL C_sum_dev is SS_ERR_INVALID_ARG. */
ss_status_t ss_zgemm_batched_sums(int M, int N, int K, double alpha, const ss_cplx* A_dev, const double* A_sum_dev, int lda,
                                  long long strideA, const ss_cplx* B_dev, const double* B_sum_dev, int ldb, long long strideB,
                                  double beta, ss_cplx* C_dev, double* C_sum_dev, int ldc, long long strideC, int batch,
                                  void* cuda_stream);

/* Batched blocked LU with partial pivoting (ZGETRF) of the leading n x n part of the n x ncols (ncols >= n, ld)
 * row-major matrices AB[z]; the row interchanges and the L-solve are applied to the trailing ncols - n columns too (so
 * that AB[:, n:] becomes L^-1 P B).  Recursive over column ranges down to 128-column panels (leaf panels of 16 columns
 * factored by a thread-block-cluster kernel: warp-shuffle / redux pivot search, rows in registers), every update a DMMA
 * GEMM.  ipiv_dev: [batch][n] 0-based row indices (LAPACK semantics: row j was swapped with row ipiv[j]); info_dev:
 * [batch], 0 or 1 + index of the first zero pivot.  n <= 8192.
 * work_dev: caller-owned device scratch of at least ss_lu_workspace_bytes(n, batch) bytes (the inverses of the 128 x 128
 * diagonal blocks of L and U); its contents are needed by nothing after the call's work has completed.
 * Asynchronous: everything is enqueued on cuda_stream, nothing is allocated, the host does not wait. */
size_t ss_lu_workspace_bytes(int n, int batch);
ss_status_t ss_zgetrf_batched(int n, int ncols, ss_cplx* AB_dev, int ld, long long stride, int* ipiv_dev,
                              int* info_dev, int batch, void* work_dev, size_t work_bytes, void* cuda_stream);

/* Batched solve A X = B (ZGESV): LU as above on AB = [A | B] (n x (n + nrhs), ld), then blocked ZTRSM back
 * substitution with the upper factor (left-looking over 128-row blocks, explicit block inverses: GEMMs); X[z]
 * (n x nrhs, ldx) at X_dev + z*strideX.  AB is overwritten.  Workspace and asynchrony as for ss_zgetrf_batched. */
ss_status_t ss_zgesv_batched(int n, int nrhs, ss_cplx* AB_dev, int ld, long long stride, ss_cplx* X_dev, int ldx,
                             long long strideX, int* ipiv_dev, int* info_dev, int batch, void* work_dev, size_t work_bytes,
                             void* cuda_stream);

/* ss_zgesv_batched for callers that are not in a position to allocate device memory.
 *
 * Who that is: code that is handed device pointers by a host application and owns no allocator of its own (a plug-in
 * inside a transport code whose GPU memory was carved up at start-up, a Fortran/C driver that only forwards pointers);
 * code running after the whole HBM has been given away (H, S and the block columns of a large device, or another
 * framework's memory pool, leave nothing for a cudaMalloc to find); and code inside a latency-critical loop, where
 * cudaMalloc / cudaFree stall the whole device while they run.  ss_zgesv_batched serves them only if somebody else has
 * set aside ss_lu_workspace_bytes(n, batch) of scratch beforehand; this variant brings its scratch with it.
 *
 * The scratch (block inverses of the factors, row-move buffer, permutation lists) is ONE fixed array of
 * SS_NOALLOC_SCRATCH_BYTES that is part of the library image: every GPU on which the library's kernels get loaded holds
 * that many bytes from then until the process exits, whether or not this function is ever called.  The function itself
 * calls no cudaMalloc, cudaFree, or any routine that allocates; the caller passes inputs and outputs only.
 *
 * Arguments, layout, results and asynchrony are those of ss_zgesv_batched without (work_dev, work_bytes); the results are
 * the same bits, because the same kernels run in the same order.  Differences the caller has to know about:
 *   - Size limit: ss_lu_workspace_bytes(n, batch) must not exceed SS_NOALLOC_SCRATCH_BYTES, otherwise the call does
 *     nothing and returns SS_ERR_INVALID_ARG (ss_strerror: "invalid argument").  16 MiB covers, for instance, n = 1024
 *     with batch 1, n = 512 with batch 3, n = 256 with batch 10, n = 128 with batch 21.  Check with ss_lu_workspace_bytes.
 *   - The device that is current at the call must be the one AB_dev, X_dev, ipiv_dev, info_dev and cuda_stream belong to:
 *     each device has its own copy of the array.
 *   - First call on a device: the function looks up where that device keeps its copy of the array (one
 *     cudaGetSymbolAddress, which also makes the runtime load the library's kernels onto that device) and remembers the
 *     answer.  Make that first call during set-up, before any stream capture is begun; later calls on the device only
 *     enqueue kernels and one memset of info_dev.
 *   - All calls on one device share the one array, and it keeps whatever the previous call left in it.  Nothing in it needs
 *     to start at zero (every part is written within a call before that call reads it), so nothing is cleared.  Two calls
 *     whose GPU work can overlap -- different streams without an event between them, or two host threads -- overwrite each
 *     other's scratch and give wrong results without any error: keep all calls of one device on one stream, or order them
 *     yourself.  The same goes for two processes only in the sense that each has its own copy; they do not interfere.
 * Errors: SS_ERR_INVALID_ARG (arguments as for ss_zgesv_batched, or the size limit), SS_ERR_CUDA (the address look-up or a
 * launch failed).  Singular matrices are reported through info_dev as usual. */
#define SS_NOALLOC_SCRATCH_BYTES (16u << 20)
ss_status_t ss_zgesv_batched_noalloc(int n, int nrhs, ss_cplx* AB_dev, int ld, long long stride, ss_cplx* X_dev, int ldx,
                                     long long strideX, int* ipiv_dev, int* info_dev, int batch, void* cuda_stream);

/* Carrier density from the solution ("charge and current densities can be directly
 * derived from ... c(E)"):  rho[i] = sum_e w[e] * sum_c |X[e][i][c]|^2,  i = 0..n-1.
 *   X_dev [n_energy][n][nrhs] (the output of ss_solve, n = nb*bs), w_dev [n_energy] doubles (occupation x energy
 *   integration weight) or NULL = all ones, rho_dev out [n] doubles.  Deterministic (no atomics); enqueued on cuda_stream. */
ss_status_t ss_density(const ss_cplx* X_dev, int n_energy, long long n, int nrhs, const double* w_dev, double* rho_dev,
                       void* cuda_stream);

/* Bond (spectral) current through every block interface, from the solution X of the LAST ss_solve
 * on this handle (its energies and H, S are used):
 *     J[e][i] = 2 Im Tr( X_i^H A_{i,i+1}(E_e) X_{i+1} ),   i = 0..nb-2,   A_{i,i+1} = E_e S_{i,i+1} - H_{i,i+1}  (Eq. 5).
 * At Im E = 0 the interior equations give J[e][i] = J[e][i+1] (current conservation).  X_dev [n_energy][nb*bs][nrhs] as
 * returned by that solve (nrhs <= its nrhs), J_host out [n_energy][nb-1].  Overwrites handle scratch; synchronises. */
ss_status_t ss_bond_current(ss_handle_t h, const ss_cplx* X_dev, int nrhs, double* J_host);

/* Arithmetic of the complex GEMM kernel (north_star: "4M or 3M ... whichever reaches the higher fraction of the chip's
 * FP64 peak"):  0 = 4M (four real products per complex product, 64x64 tile);  1 = 3M, the default (three real products,
 * P1 = Ar Br, P2 = Ai Bi, P3 = (Ar+Ai)(Br+Bi); 6 instead of 8 real flops per complex multiply-add; rounding differs,
 * normwise error stays O(u)), 64x32 CTA tile, kernel chosen by K (3 CTAs/SM for K < 768, software-pipelined main loop at
 * 2 CTAs/SM from K = 768);  2 / 3 = those two 3M kernels for every K;  4 / 5 = EXPERIMENTS (measured, not adopted:
 * profiles/r02_gemm_tma.md): variant 3's main loop with the operand tiles staged by TMA at 2 / 3 CTAs per SM, for uniformly
 * strided batches of whole matrices only -- any other operand layout, and a tensor map that cannot be encoded, silently take
 * variant 3.  Anything outside 0..5 is SS_ERR_INVALID_ARG.  The process-wide default (initially 1) applies to handles created
 * afterwards and to the handle-less building blocks above. */
ss_status_t ss_set_default_gemm_variant(int variant);

/* TUNING KNOB for bench.py --raster, not part of the stable interface: tile rows per raster group of the GEMM kernels (1..64,
 * default 16; process-wide): the CTAs of that many tile rows run side by side and share the B column tiles in L2;
 * profiles/r02_gemm_tma.md has the DRAM traffic it controls. */
ss_status_t ss_set_gemm_raster(int tile_rows);
int ss_get_default_gemm_variant(void);

/* FP64 pipe microbenchmark (register-resident mma.sync.m8n8k4.f64 chains on all SMs): returns sustained
 * TFLOP/s over about `ms` milliseconds; the measured roofline denominator bench.py prints beside the nominal one. */
ss_status_t ss_fp64_peak_tflops(double ms, double* tflops);

#ifdef __cplusplus
}
#endif
#endif /* SPLITSOLVE_H */
