// libsplitsolve: handle, workspace, the SplitSolve driver (Alg. 1 + mirror, post-processing, T(E)) and the C ABI
// declared in include/splitsolve.h.  Only the CUDA runtime is linked: no cuBLAS / cuSOLVER / torch, no CPU fallback.
#include "../../include/splitsolve.h"

#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>

#include "sweep.cuh"
#include "zgetrf.cuh"

using namespace ss;

static int g_default_variant = GV_3M;   // process-wide default GEMM variant (new handles, handle-less building blocks)

struct ss_handle_s {
    int nb = 0, bs = 0, n_energy = 0;
    const cplx *Hd = nullptr, *Hu = nullptr, *Sd = nullptr, *Su = nullptr;
    cplx* own_hs[4] = {nullptr, nullptr, nullptr, nullptr};
    bool have_h = false, solved = false;
    bool launched = false;           // some ss_solve has been enqueued: ev[2] is a valid event to wait on
    // options
    int want_T = 1;
    int hermitian = 0;               // SURVEY 8(f1) at real energies: 0 off, 1 Hermitian Schur update, 2 + no-pivot L Delta L^H
    int growth_limit = 64;           // mode 2: largest multiplier tolerated before the solve is redone with the pivoted LU
    int mode = 0;                    // what the last ss_solve used
    // block columns kept in pinned HOST memory, a ring of device slots per chain
    int offload = 0;                 // option "offload_columns"
    int ring = 6;                    // device slots per chain in that mode (>= 6: 3 in use + 2 prefetched + 1 slack)
    cplx* host_cols = nullptr;       // pinned [n_energy][2][nb+1][bs*bs]
    cplx* corner = nullptr;          // device [n_energy][2 columns][first / last block][bs*bs]
    struct GroupCopy { cudaStream_t st = nullptr; std::vector<cudaEvent_t> ev_slot[2]; std::vector<cudaEvent_t> ev_step; };
    std::vector<GroupCopy> gcopy;    // per stream group: its copy stream, one event per (column, ring slot), step events
    int slots_per_chain() const { return offload ? ring : nb + 1; }
    int part = -1;                   // spatial split (ss_*_partition): -1 whole device, 0 top half, 1 bottom half; set by ss_merge_partition
    int swept_cols = 0;              // block columns the last sweep computed (3 = both; 1 / 2: ss_sweep_column)
    bool whole_solve = true;         // the last post-processing belonged to an ss_solve (so a redo is possible)
    bool force_general = false;      // set while a solve is being redone
    int retried = 0;                 // that solve was redone on the pivoted path (growth limit exceeded)
    struct { const ss_cplx *sl, *sr, *i1, *i2; ss_cplx* x; int nrhs; void* stream; } last_args{};
    int profile_gemm = 0;
    int gemm_variant = g_default_variant;
    int stream_groups = 4;
    int want_trace = 0;
    std::vector<TraceRec> trace;
    cudaStream_t main_stream = nullptr;
    cudaEvent_t ev_in = nullptr, ev_out = nullptr;
    // asynchronous upload of H, S from host buffers (ss_set_hamiltonian_host)
    cudaStream_t copy_stream = nullptr;
    std::vector<cudaEvent_t> up_ev;
    bool upload_pending = false;     // the next solve must wait for the per-block upload events
    bool upload_consumed = false;    // a solve that waited for them has been enqueued: cleared once it has completed
    cudaEvent_t ev_sig = nullptr;    // ss_solve_host: Sigma / Inj uploads done (only the post-processing waits for it)
    bool post_wait = false;
    GemmProfile prof;
    // stream groups (created on first use): per group a high- and a low-priority stream and two events
    struct GroupRes { cudaStream_t hi = nullptr, lo = nullptr; cudaEvent_t ev_sw = nullptr, ev_mark = nullptr; };
    std::vector<GroupRes> groups;
    cudaEvent_t ev_fork = nullptr;
    // workspace (allocated for ws_nrhs)
    int ws_nrhs = -1;
    cplx *slots = nullptr, *aug = nullptr, *aop = nullptr, *tinv = nullptr, *raug = nullptr, *wz = nullptr;
    cplx *gam_l = nullptr, *gam_r = nullptr, *g1n = nullptr, *w1 = nullptr, *w2 = nullptr, *E_dev = nullptr;
    double *tpart = nullptr, *T_dev = nullptr, *J_dev = nullptr;
    int *ipiv = nullptr, *info = nullptr, *perm = nullptr;
    cplx* E_pinned = nullptr;
    // host-path buffers
    cplx *hp_sigl = nullptr, *hp_sigr = nullptr, *hp_inj1 = nullptr, *hp_inj2 = nullptr, *hp_x = nullptr;
    int hp_nrhs = -1;
    cudaStream_t own_stream = nullptr;
    // last solve
    cudaStream_t last_stream = nullptr;
    cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};
    long long launches = 0;
    int last_nrhs = 0;
};

static const int TRACE_PARTS = 592;   // 4 x 148 CTAs per energy for the trace reduction

static inline long long cdiv(long long a, long long b) { return (a + b - 1) / b; }

// Leading dimension of a handle-owned row-major work matrix with n columns.  A byte stride that is a multiple of 2 KB
// maps the rows a panel kernel walks down (one thread per row) onto the same cache sets: measured, the 16-column
// leaf panel ran 1.5x slower at ld = 4096 than at ld = 4112.  So such strides get 16 elements (256 B) of padding.
static inline int pad_ld(long long n) { return (int)((n >= 128 && n % 128 == 0) ? n + 16 : n); }

static void free_dev(void* p) { if (p) cudaFree(p); }

static void free_workspace(ss_handle_t h) {
    free_dev(h->slots); free_dev(h->aug); free_dev(h->aop); free_dev(h->tinv); free_dev(h->raug); free_dev(h->wz);
    free_dev(h->gam_l); free_dev(h->gam_r); free_dev(h->g1n); free_dev(h->w1); free_dev(h->w2); free_dev(h->E_dev);
    free_dev(h->tpart); free_dev(h->T_dev); free_dev(h->ipiv); free_dev(h->info); free_dev(h->perm); free_dev(h->corner);
    if (h->host_cols) cudaFreeHost(h->host_cols);
    h->corner = nullptr; h->host_cols = nullptr;
    h->slots = h->aug = h->aop = h->tinv = h->raug = h->wz = nullptr;
    h->gam_l = h->gam_r = h->g1n = h->w1 = h->w2 = h->E_dev = nullptr;
    h->tpart = h->T_dev = nullptr; h->ipiv = h->info = h->perm = nullptr;
    h->ws_nrhs = -1;
}

struct WsSizes {
    size_t slots, aug, aop, tinv, raug, wz, sq, E, tpart, T, ipiv, info, perm;
    size_t total() const { return slots + aug + aop + tinv + raug + wz + 5 * sq + E + tpart + T + ipiv + info + perm; }
};

// ints of row-permutation scratch per energy: enough for its two chains' sweeps (n = bs) and, afterwards, its corner
// system (n = 2bs); every stream group owns the slice of its energies
static inline size_t perm_ints_per_energy(int bs) { return ((size_t)2 * (3 * (size_t)bs + 1) + 7) / 4 * 4 + 4; }

static WsSizes ws_sizes(int nb, int bs, int nE, int nrhs, int slots_per_chain = 0) {
    WsSizes w;
    const size_t B2 = (size_t)bs * bs, C = sizeof(cplx);
    w.slots = (size_t)nE * 2 * (slots_per_chain ? slots_per_chain : nb + 1) * B2 * C;
    w.aug = (size_t)nE * 2 * bs * pad_ld(2 * bs) * C;
    w.aop = (size_t)nE * 2 * B2 * C;
    // the sweep and the corner system own disjoint regions: stream groups do not wait for one another between the two
    // phases, so one group's corner LU may run while another group's sweep still uses its triangular inverses
    w.tinv = (lu_tinv_elems(bs, 2 * nE) + lu_tinv_elems(2 * bs, nE)) * C;
    size_t W = (size_t)pad_ld(3LL * bs + nrhs), W2 = (size_t)pad_ld(2LL * bs + nrhs);   // with / without the e_2 columns
    if (W2 > W) W = W2;
    w.raug = (size_t)nE * 2 * bs * W * C;
    w.wz = (size_t)nE * 2 * bs * ((size_t)nrhs + bs) * C;
    w.sq = (size_t)nE * B2 * C;
    w.E = (size_t)nE * C;
    w.tpart = (size_t)nE * TRACE_PARTS * sizeof(double);
    w.T = (size_t)nE * sizeof(double);
    w.ipiv = (size_t)3 * nE * 2 * bs * sizeof(int);
    w.info = (size_t)8 * nE * sizeof(int);                     // 3 nE zero-pivot records, 2 nE growth monitors, nE single-column sweeps, 2 nE merge records
    w.perm = (size_t)nE * perm_ints_per_energy(bs) * sizeof(int);
    return w;
}

// The sizes of everything but the corner system [R | b' | e_2] and its solution do not depend on nrhs: that part is
// allocated once and survives a later call with more right-hand sides (ss_sweep_column knows no nrhs yet, and the sweep's
// results must outlive the allocation ss_post_column makes).
static ss_status_t ensure_workspace(ss_handle_t h, int nrhs) {
    WsSizes w = ws_sizes(h->nb, h->bs, h->n_energy, nrhs, h->slots_per_chain());
    bool ok = true;
    auto A = [&](void** p, size_t bytes) { if (ok && cudaMalloc(p, bytes ? bytes : 16) != cudaSuccess) ok = false; };
    if (!h->slots) {
        A((void**)&h->slots, w.slots); A((void**)&h->aug, w.aug); A((void**)&h->aop, w.aop); A((void**)&h->tinv, w.tinv);
        A((void**)&h->gam_l, w.sq); A((void**)&h->gam_r, w.sq); A((void**)&h->g1n, w.sq); A((void**)&h->w1, w.sq);
        A((void**)&h->w2, w.sq); A((void**)&h->E_dev, w.E); A((void**)&h->tpart, w.tpart); A((void**)&h->T_dev, w.T);
        A((void**)&h->ipiv, w.ipiv); A((void**)&h->info, w.info); A((void**)&h->perm, w.perm);
        if (h->offload) {
            A((void**)&h->corner, (size_t)h->n_energy * 4 * h->bs * h->bs * sizeof(cplx));
            if (ok && cudaMallocHost((void**)&h->host_cols, (size_t)h->n_energy * 2 * (h->nb + 1) * h->bs * h->bs * sizeof(cplx)) != cudaSuccess)
                ok = false;
        }
        if (!ok) { cudaGetLastError(); free_workspace(h); return SS_ERR_ALLOC; }
    }
    if (h->ws_nrhs < nrhs) {
        free_dev(h->raug); free_dev(h->wz); h->raug = h->wz = nullptr;
        A((void**)&h->raug, w.raug); A((void**)&h->wz, w.wz);
        if (!ok) { cudaGetLastError(); free_workspace(h); return SS_ERR_ALLOC; }
        h->ws_nrhs = nrhs;
    }
    return SS_OK;
}

extern "C" size_t ss_workspace_bytes(int nb, int bs, int n_energy, int nrhs) {
    if (nb < 2 || bs < 1 || n_energy < 1 || nrhs < 0) return 0;
    return ws_sizes(nb, bs, n_energy, nrhs).total();
}

extern "C" const char* ss_strerror(ss_status_t s) {
    switch (s) {
        case SS_OK: return "ok";
        case SS_ERR_INVALID_ARG: return "invalid argument";
        case SS_ERR_NOT_READY: return "not ready (call order)";
        case SS_ERR_ALLOC: return "allocation failed";
        case SS_ERR_SINGULAR: return "exactly zero pivot";
        case SS_ERR_CUDA: return "CUDA error";
        case SS_ERR_UNSTABLE: return "no-pivot factorisation exceeded its growth limit";
    }
    return "unknown status";
}

extern "C" ss_status_t ss_create(int nb, int bs, int n_energy, ss_handle_t* out) {
    if (!out) return SS_ERR_INVALID_ARG;
    *out = nullptr;
    if (nb < 2 || bs < 1 || bs > 4096 || n_energy < 1) return SS_ERR_INVALID_ARG;
    ss_handle_t h = new (std::nothrow) ss_handle_s();
    if (!h) return SS_ERR_ALLOC;
    h->nb = nb; h->bs = bs; h->n_energy = n_energy;
    for (int i = 0; i < 3; i++)
        if (cudaEventCreate(&h->ev[i]) != cudaSuccess) { cudaGetLastError(); delete h; return SS_ERR_CUDA; }
    if (cudaMallocHost((void**)&h->E_pinned, sizeof(cplx) * (size_t)n_energy) != cudaSuccess) {
        cudaGetLastError(); delete h; return SS_ERR_ALLOC;
    }
    *out = h;
    return SS_OK;
}

static void free_host_path(ss_handle_t h) {
    free_dev(h->hp_sigl); free_dev(h->hp_sigr); free_dev(h->hp_inj1); free_dev(h->hp_inj2); free_dev(h->hp_x);
    h->hp_sigl = h->hp_sigr = h->hp_inj1 = h->hp_inj2 = h->hp_x = nullptr;
    h->hp_nrhs = -1;
}

extern "C" ss_status_t ss_destroy(ss_handle_t h) {
    if (!h) return SS_OK;
    cudaDeviceSynchronize();
    free_workspace(h);
    free_host_path(h);
    for (int i = 0; i < 4; i++) free_dev(h->own_hs[i]);
    for (int i = 0; i < 3; i++) if (h->ev[i]) cudaEventDestroy(h->ev[i]);
    for (cudaEvent_t e : h->prof.ev) cudaEventDestroy(e);
    for (auto& r : h->trace) { cudaEventDestroy(r.t0); cudaEventDestroy(r.t1); }
    if (h->E_pinned) cudaFreeHost(h->E_pinned);
    free_dev(h->J_dev);
    if (h->own_stream) cudaStreamDestroy(h->own_stream);
    for (auto& g : h->groups) {
        if (g.hi) cudaStreamDestroy(g.hi);
        if (g.lo) cudaStreamDestroy(g.lo);
        if (g.ev_sw) cudaEventDestroy(g.ev_sw);
        if (g.ev_mark) cudaEventDestroy(g.ev_mark);
    }
    if (h->ev_fork) cudaEventDestroy(h->ev_fork);
    for (auto& c : h->gcopy) {
        if (c.st) cudaStreamDestroy(c.st);
        for (int q = 0; q < 2; q++) for (cudaEvent_t e : c.ev_slot[q]) cudaEventDestroy(e);
        for (cudaEvent_t e : c.ev_step) cudaEventDestroy(e);
    }
    if (h->main_stream) cudaStreamDestroy(h->main_stream);
    if (h->copy_stream) cudaStreamDestroy(h->copy_stream);
    for (cudaEvent_t e : h->up_ev) cudaEventDestroy(e);
    if (h->ev_sig) cudaEventDestroy(h->ev_sig);
    if (h->ev_in) cudaEventDestroy(h->ev_in);
    if (h->ev_out) cudaEventDestroy(h->ev_out);
    delete h;
    return SS_OK;
}

extern "C" ss_status_t ss_set_hamiltonian(ss_handle_t h, const ss_cplx* Hd, const ss_cplx* Hu, const ss_cplx* Sd,
                                          const ss_cplx* Su) {
    if (!h || !Hd || !Hu || !Sd || !Su) return SS_ERR_INVALID_ARG;
    h->Hd = (const cplx*)Hd; h->Hu = (const cplx*)Hu; h->Sd = (const cplx*)Sd; h->Su = (const cplx*)Su;
    h->have_h = true; h->solved = false;
    h->upload_pending = false;
    h->upload_consumed = false;
    return SS_OK;
}

// Host buffers: the blocks are uploaded asynchronously on a copy stream of the handle, in the order the two sweeps
// consume them (from both ends of the device towards the middle), with one event per pair of ends; block step s of the
// sweep waits for event s only, so that with pinned host memory the upload runs under the first block steps instead of
// in front of the solve.  (From pageable memory cudaMemcpyAsync stages synchronously: same result, no overlap.)
extern "C" ss_status_t ss_set_hamiltonian_host(ss_handle_t h, const ss_cplx* Hd, const ss_cplx* Hu, const ss_cplx* Sd,
                                               const ss_cplx* Su) {
    if (!h || !Hd || !Hu || !Sd || !Su) return SS_ERR_INVALID_ARG;
    const int nb = h->nb;
    const size_t B2e = (size_t)h->bs * h->bs, B2 = B2e * sizeof(cplx);
    const size_t bytes[4] = {B2 * nb, B2 * (nb - 1), B2 * nb, B2 * (nb - 1)};
    for (int i = 0; i < 4; i++)
        if (!h->own_hs[i] && cudaMalloc((void**)&h->own_hs[i], bytes[i]) != cudaSuccess) { cudaGetLastError(); return SS_ERR_ALLOC; }
    if (!h->copy_stream && cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking) != cudaSuccess) {
        cudaGetLastError(); return SS_ERR_CUDA;
    }
    while ((int)h->up_ev.size() < nb) {
        cudaEvent_t e;
        if (cudaEventCreateWithFlags(&e, cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); return SS_ERR_CUDA; }
        h->up_ev.push_back(e);
    }
    if (h->launched) cudaEventSynchronize(h->ev[2]);      // the previous solve may still read the old blocks
    std::vector<char> done_d((size_t)nb, 0), done_u((size_t)(nb > 1 ? nb - 1 : 0), 0);
    bool ok = true;
    auto put = [&](int which, const ss_cplx* src, int idx) {
        if (ok && cudaMemcpyAsync(h->own_hs[which] + (size_t)idx * B2e, src + (size_t)idx * B2e, B2, cudaMemcpyHostToDevice,
                                  h->copy_stream) != cudaSuccess) ok = false;
    };
    for (int k = 0; k < nb; k++) {
        const int dl[2] = {nb - 1 - k, k}, ul[2] = {nb - 2 - k, k};
        for (int q = 0; q < 2; q++) {
            if (dl[q] >= 0 && dl[q] < nb && !done_d[dl[q]]) { done_d[dl[q]] = 1; put(0, Hd, dl[q]); put(2, Sd, dl[q]); }
            if (ul[q] >= 0 && ul[q] < nb - 1 && !done_u[ul[q]]) { done_u[ul[q]] = 1; put(1, Hu, ul[q]); put(3, Su, ul[q]); }
        }
        if (ok && cudaEventRecord(h->up_ev[k], h->copy_stream) != cudaSuccess) ok = false;
    }
    if (!ok) { cudaGetLastError(); return SS_ERR_CUDA; }
    ss_status_t st = ss_set_hamiltonian(h, (ss_cplx*)h->own_hs[0], (ss_cplx*)h->own_hs[1], (ss_cplx*)h->own_hs[2],
                                        (ss_cplx*)h->own_hs[3]);
    h->upload_pending = true;
    h->upload_consumed = false;
    return st;
}

extern "C" ss_status_t ss_set_option(ss_handle_t h, const char* name, int value) {
    if (!h || !name) return SS_ERR_INVALID_ARG;
    if (!strcmp(name, "transmission")) { h->want_T = value ? 1 : 0; return SS_OK; }
    if (!strcmp(name, "profile_gemm")) { h->profile_gemm = value ? 1 : 0; return SS_OK; }
    if (!strcmp(name, "stream_groups")) {
        if (value < 1 || value > 16) return SS_ERR_INVALID_ARG;
        h->stream_groups = value; return SS_OK;
    }
    if (!strcmp(name, "trace")) { h->want_trace = value ? 1 : 0; return SS_OK; }
    if (!strcmp(name, "offload_columns")) {
        // changes the layout of the workspace: only before the first solve
        if (h->slots) return SS_ERR_NOT_READY;
        if (value != 0 && (value < 6 || value > 64) && value != 1) return SS_ERR_INVALID_ARG;
        h->offload = value ? 1 : 0;
        h->ring = value > 1 ? value : 6;
        return SS_OK;
    }
    if (!strcmp(name, "hermitian")) {
        if (value < 0 || value > 2) return SS_ERR_INVALID_ARG;
        h->hermitian = value; return SS_OK;
    }
    if (!strcmp(name, "hermitian_growth_limit")) {
        if (value < 1) return SS_ERR_INVALID_ARG;
        h->growth_limit = value; return SS_OK;
    }
    if (!strcmp(name, "gemm_raster")) {                                                       // process-wide (tuning)
        if (value < 1 || value > 64) return SS_ERR_INVALID_ARG;
        g_gemm_raster = value; return SS_OK;
    }
    if (!strcmp(name, "gemm_variant")) {
        if (value < 0 || value >= GV_COUNT) return SS_ERR_INVALID_ARG;
        h->gemm_variant = value; return SS_OK;
    }
    return SS_ERR_INVALID_ARG;
}

// Closed-form flop counts (LAPACK convention) of the path the LAST ss_solve took (before any solve: the general path).
// Per block and chain: a1 8 bs^3 (Hermitian Schur update, modes 1 and 2: 4 bs^3), a2 8/3 bs^3 (mode 2, L Delta L^H: 4/3 bs^3),
// a3 8 bs^3, a4 8 bs^3; the first block of a chain has no a1, the last no a4.
static double sweep_flops(const ss_handle_s* h) {
    const double bs3 = (double)h->bs * h->bs * h->bs, nb = h->nb;
    const double a1 = (h->mode >= 1 ? 4.0 : 8.0), a2 = (h->mode == 2 ? 4.0 / 3.0 : 8.0 / 3.0);
    return 2.0 * ((nb - 1) * a1 + nb * a2 + nb * 8.0 + (nb - 1) * 8.0) * bs3;
}

extern "C" double ss_flops_sweep(ss_handle_t h) {
    if (!h) return 0.0;
    return sweep_flops(h);
}

extern "C" double ss_flops(ss_handle_t h, int nrhs) {
    if (!h || nrhs < 0) return 0.0;
    const double bs = h->bs, nb = h->nb, m = nrhs;
    const double bs3 = bs * bs * bs;
    double sweep = sweep_flops(h);
    // a5: 4 GEMM (32 bs^3) + ZGETRF(2bs) (64/3 bs^3) + 2 ZTRSM with m rhs (2 * 4 (2bs)^2 m = 32 bs^2 m)
    double a5 = 32.0 * bs3 + 64.0 / 3.0 * bs3 + 32.0 * bs * bs * m;
    double a6 = 16.0 * nb * bs * bs * m;
    // a7: R^-1[:, bs:] (2 ZTRSM with bs rhs: 32 bs^3) + G (16 bs^3) + two Gamma products (16 bs^3) + trace (8 bs^2)
    double a7 = h->want_T ? (64.0 * bs3 + 8.0 * bs * bs) : 0.0;
    return sweep + a5 + a6 + a7;
}

extern "C" ss_status_t ss_last_mode(ss_handle_t h, int* mode, int* retried) {
    if (!h || !mode || !retried) return SS_ERR_INVALID_ARG;
    if (!h->solved) return SS_ERR_NOT_READY;
    *mode = h->mode; *retried = h->retried;
    return SS_OK;
}

// ---------------------------------------------------------------------------------------------------------
// the hot path
// ---------------------------------------------------------------------------------------------------------
static void launch_form(Ctx& ctx, FormSide s0, FormSide s1, const cplx* E, BPtr dst, int ld, int bs, int batch, int eshift = 1) {
    dim3 grid((unsigned)cdiv(bs, 32), (unsigned)cdiv(bs, 32), (unsigned)batch);
    form_kernel<<<grid, 256, 0, ctx.st>>>(s0, s1, E, dst, ld, bs, eshift);
    ctx.note(cudaGetLastError());
}

// ---- slot addressing.  Full mode: [n_energy][2][nb+1] blocks, logical slot = physical slot.  Offload mode (SURVEY.md 8(f4),
// part of Q on the host, "transfers overlapped"): [n_energy][2][ring] blocks, logical slot idx lives in
// ring slot idx % ring while it is in use; every block is also written to the pinned host array host_cols[e][col][idx].
static inline long long slot_stride_e(const ss_handle_s* h) { return 2LL * h->slots_per_chain() * h->bs * h->bs; }
static inline cplx* slot_ptr(const ss_handle_s* h, int e0, int col, int idx) {
    const long long B2 = (long long)h->bs * h->bs;
    const int spc = h->slots_per_chain();
    return h->slots + (long long)e0 * slot_stride_e(h) + ((long long)col * spc + (h->offload ? idx % spc : idx)) * B2;
}
static inline cplx* host_ptr(const ss_handle_s* h, int e0, int col, int idx) {
    const long long B2 = (long long)h->bs * h->bs;
    return h->host_cols + ((long long)e0 * 2 * (h->nb + 1) + (long long)col * (h->nb + 1) + idx) * B2;
}

static bool ensure_offload(ss_handle_t h, int nG) {
    while ((int)h->gcopy.size() < nG) {
        ss_handle_s::GroupCopy c;
        bool ok = cudaStreamCreateWithFlags(&c.st, cudaStreamNonBlocking) == cudaSuccess;
        for (int q = 0; q < 2 && ok; q++)
            for (int i = 0; i < h->ring && ok; i++) {
                cudaEvent_t e;
                ok = cudaEventCreateWithFlags(&e, cudaEventDisableTiming) == cudaSuccess;
                if (ok) c.ev_slot[q].push_back(e);
            }
        for (int i = 0; i < 4 && ok; i++) {
            cudaEvent_t e;
            ok = cudaEventCreateWithFlags(&e, cudaEventDisableTiming) == cudaSuccess;
            if (ok) c.ev_step.push_back(e);
        }
        h->gcopy.push_back(c);
        if (!ok) return false;
    }
    return true;
}

// a0-a4: Algorithm 1 and its mirror (L167) for the energies [e0, e0 + nEg) of one stream group, both
// columns in lockstep.  Chain z = 2*e + col.  Slot layout per chain (nb+1 slots of bs x bs): column 0 keeps X_i in slot i
// (X_1 in slot 0) and ends with Q_i in slot i-1; column 1 keeps Y_i in slot i-1 (Y_nb in slot nb) and ends with P_i in
// slot i.  sweep_step(s) is block step s of both sweeps (a0-a3), recursion_step(r) one product of a4.
// cols: 3 = both sweeps in lockstep (chain z = 2*e + col), 1 / 2 = only the first- / last-column sweep (chain z = e;
// "naturally scale to two accelerators", one block column per GPU).
struct Group {
    int e0 = 0, nE = 0;
    int cols = 3;
    Ctx ctx;
    bool dual() const { return cols == 3; }
    int batch() const { return dual() ? 2 * nE : nE; }
    // pointer of chain z: both columns (p0 first, p1 last) or the one of this group
    BPtr ch(const cplx* p0, const cplx* p1, long long s_energy) const {
        return dual() ? bp_chain(p0, p1, s_energy) : bp_strided(cols == 1 ? p0 : p1, s_energy);
    }
    // ---- offload mode: transfers of logical slot idx of column col for this group's energies, on the group's copy stream
    ss_handle_s::GroupCopy* cp = nullptr;
    std::vector<char>* slot_used = nullptr;           // [2][ring]: a transfer event has been recorded for that ring slot in this solve
    void wait_slot(ss_handle_t h, int col, int idx) { // the compute stream waits for the last transfer that touched that ring slot
        const int rs = idx % h->ring;
        if ((*slot_used)[col * h->ring + rs]) cudaStreamWaitEvent(ctx.st, cp->ev_slot[col][rs], 0);
    }
    void copy_after_compute(int which) {              // the copy stream waits for everything enqueued so far on the compute stream
        cudaEventRecord(cp->ev_step[which], ctx.st);
        cudaStreamWaitEvent(cp->st, cp->ev_step[which], 0);
    }
    void xfer(ss_handle_t h, int col, int idx, bool to_host) {
        const size_t B2b = sizeof(cplx) * (size_t)h->bs * h->bs;
        cplx* d = slot_ptr(h, e0, col, idx);
        cplx* hp = host_ptr(h, e0, col, idx);
        const size_t dp = sizeof(cplx) * (size_t)slot_stride_e(h), hpitch = 2 * (size_t)(h->nb + 1) * B2b;
        cudaError_t e = to_host ? cudaMemcpy2DAsync(hp, hpitch, d, dp, B2b, (size_t)nE, cudaMemcpyDeviceToHost, cp->st)
                                : cudaMemcpy2DAsync(d, dp, hp, hpitch, B2b, (size_t)nE, cudaMemcpyHostToDevice, cp->st);
        if (ctx.err == cudaSuccess && e != cudaSuccess) ctx.err = e;
        const int rs = idx % h->ring;
        cudaEventRecord(cp->ev_slot[col][rs], cp->st);
        (*slot_used)[col * h->ring + rs] = 1;
    }
    void save_corner(ss_handle_t h, int col, int which, int idx) {     // block 1 / nb of a column -> h->corner (compute stream)
        const size_t B2b = sizeof(cplx) * (size_t)h->bs * h->bs;
        cplx* dst = h->corner + (((long long)e0 * 2 + col) * 2 + which) * (long long)h->bs * h->bs;
        cudaError_t e = cudaMemcpy2DAsync(dst, 4 * B2b, slot_ptr(h, e0, col, idx), sizeof(cplx) * (size_t)slot_stride_e(h), B2b,
                                          (size_t)nE, cudaMemcpyDeviceToDevice, ctx.st);
        if (ctx.err == cudaSuccess && e != cudaSuccess) ctx.err = e;
    }
};

static void sweep_step(ss_handle_t h, Group& G, int s) {
    Ctx& ctx = G.ctx;
    const int nb = h->nb, bs = h->bs, e0 = G.e0, batch = G.batch(), eshift = G.dual() ? 1 : 0;
    const long long B2 = (long long)bs * bs;
    const long long s_slot_e = slot_stride_e(h);
    auto slot = [&](int col, int idx) { return slot_ptr(h, e0, col, idx); };
    const int ldg = pad_ld(2 * bs);
    const long long s_aug_e = 2LL * bs * ldg;
    const BPtr aug = G.ch(h->aug + e0 * s_aug_e, h->aug + e0 * s_aug_e + (long long)bs * ldg, s_aug_e);
    const BPtr aop = G.ch(h->aop + e0 * 2 * B2, h->aop + e0 * 2 * B2 + B2, 2 * B2);
    const cplx* E = h->E_dev + e0;
    LuWork w;
    w.tinv = h->tinv + lu_tinv_elems(bs, 2 * e0);
    w.ipiv = h->ipiv + (long long)2 * e0 * 2 * bs; w.ipiv_stride = 2 * bs;
    w.info = G.dual() ? h->info + 2 * e0 : h->info + 5 * h->n_energy + e0;
    w.growth = h->info + 3 * h->n_energy + 2 * e0;
    const int mode = h->mode;                                  // 0 general, 1 Hermitian Schur update, 2 + L Delta L^H (real energies)
    const int info_stride = 2 * bs + 2;

    w.perm = h->perm + (long long)e0 * perm_ints_per_energy(bs);
    w.tmp = h->aop + e0 * 2 * B2; w.tmp_elems = B2;            // the formed operand is consumed before the LU starts

    const int i_f = nb - s, i_m = s + 1;                       // 1-based block index of each chain
    ctx.use(CLS_HI);
    if (h->upload_pending) cudaStreamWaitEvent(ctx.st, h->up_ev[s], 0);   // H, S blocks of this step (ss_set_hamiltonian_host)
    // right-hand sides: A_{i,i-1} (column 0) / A_{i,i+1} (column 1); identity at the ends (L164, reading c1).  Formed into
    // the slot X_i / Y_i will occupy; the LU copies them into [D | B] with the row interchanges already applied.
    FormSide r0 = (i_f > 1) ? FormSide{h->Su + (long long)(i_f - 2) * B2, h->Hu + (long long)(i_f - 2) * B2, FORM_CONJT}
                            : FormSide{nullptr, nullptr, FORM_IDENT};
    FormSide r1 = (i_m < nb) ? FormSide{h->Su + (long long)(i_m - 1) * B2, h->Hu + (long long)(i_m - 1) * B2, FORM_PLAIN}
                             : FormSide{nullptr, nullptr, FORM_IDENT};
    if (G.cols == 2) r0 = r1;                                  // one sweep only: its side goes first
    const int widx[2] = {i_f >= 2 ? i_f : 0, i_m <= nb - 1 ? i_m - 1 : nb};      // logical slots X_i / Y_i go to
    const BPtr out = G.ch(slot(0, widx[0]), slot(1, widx[1]), s_slot_e);
    if (h->offload)
        for (int c = 0; c < 2; c++)
            if (G.cols & (1 << c)) G.wait_slot(h, c, widx[c]);   // the ring slot's previous content has reached the host
    if (mode == 2) launch_form(ctx, r0, r1, E, bp_offset(aug, bs), ldg, bs, batch, eshift);    // no interchanges: straight into [D | B]
    else launch_form(ctx, r0, r1, E, out, bs, bs, batch, eshift);
    GemmArgs g{};
    g.M = bs; g.N = bs; g.K = 0;
    g.A = aop; g.lda = bs; g.B = aop; g.ldb = bs;
    if (s > 0) {
        // left operands: A_{i,i+1} (column 0) / A_{i,i-1} (column 1)
        FormSide a0{h->Su + (long long)(i_f - 1) * B2, h->Hu + (long long)(i_f - 1) * B2, FORM_PLAIN};
        FormSide a1{h->Su + (long long)(i_m - 2) * B2, h->Hu + (long long)(i_m - 2) * B2, FORM_CONJT};
        if (G.cols == 2) a0 = a1;
        launch_form(ctx, a0, a1, E, aop, bs, bs, batch, eshift);
        g.K = bs;
        g.B = G.ch(slot(0, i_f + 1), slot(1, i_m - 2), s_slot_e);   // X_{i+1} / Y_{i-1}
    }
    // a1 (+ a0 for the diagonal block, fused in the epilogue): D = E S_ii - H_ii - A_op * X_prev
    ctx.use(CLS_LO);
    g.C = aug; g.ldc = ldg; g.Cin = aug; g.ldcin = ldg; g.alpha = 1.0; g.beta = 0.0;
    g.S = G.ch(h->Sd + (long long)(i_f - 1) * B2, h->Sd + (long long)(i_m - 1) * B2, 0);
    g.H = G.ch(h->Hd + (long long)(i_f - 1) * B2, h->Hd + (long long)(i_m - 1) * B2, 0);
    g.lds = bs; g.E = E; g.eshift = eshift;
    if (mode >= 1) g.tri = 1;                                  // D_i is Hermitian at real E (L154): lower triangle only
    gemm_run(ctx, g, batch, GEMM_BIG, EPI_SCHUR);
    // a2 + the L half of a3
    if (mode == 2) {
        lu_factor_herm(ctx, aug, ldg, bs, 2 * bs, batch, w, s * info_stride);
    } else {
        if (mode == 1) { ctx.use(CLS_HI); launch_mirror(ctx, aug, ldg, 0, 0, bs, bs, 0, 1, batch); }
        lu_factor(ctx, aug, ldg, bs, 2 * bs, batch, w, s * info_stride, &out, bs);
    }
    // U half of a3: X_i / Y_i into its slot
    back_substitute(ctx, aug, ldg, bs, bs, out, bs, batch, w);
    if (h->offload) {
        if ((G.cols & 1) && i_f == 1) G.save_corner(h, 0, 0, 0);        // Q_1 = X_1
        if ((G.cols & 2) && i_m == nb) G.save_corner(h, 1, 1, nb);      // P_nb = Y_nb
        G.copy_after_compute(s & 3);
        for (int c = 0; c < 2; c++)
            if (G.cols & (1 << c)) G.xfer(h, c, widx[c], true);
    }
}

// a4: Q_i = -X_i Q_{i-1} (i = 2..nb), P_i = -Y_i P_{i+1} (i = nb-1..1); r = 1..nb-1
static void recursion_step(ss_handle_t h, Group& G, int r) {
    const int nb = h->nb, bs = h->bs, batch = G.batch();
    const long long s_slot_e = slot_stride_e(h);
    auto slot = [&](int col, int idx) { return slot_ptr(h, G.e0, col, idx); };
    const int i0 = r + 1, i1 = nb - r;
    // logical slots of the product C = -A B: column 0 (X_i0, Q_{i0-1}) -> Q_i0, column 1 (Y_i1, P_{i1+1}) -> P_i1
    const int ia[2] = {i0, i1 - 1}, ib[2] = {i0 - 2, i1 + 1}, ic[2] = {i0 - 1, i1};
    G.ctx.use(CLS_LO);
    if (h->offload) {
        // prefetch the X / Y of step r + 2 from the host into its ring slot: that slot's last reader was step r - 2's product
        // and its last write-back is earlier on the same copy stream; the first two steps use blocks still resident from the sweep
        const int L = 2, rp = r + L;
        if (rp <= nb - 1) {
            G.copy_after_compute((r + 3) & 3);
            const int pa[2] = {rp + 1, nb - rp - 1};
            for (int c = 0; c < 2; c++)
                if (G.cols & (1 << c)) G.xfer(h, c, pa[c], false);
        }
        for (int c = 0; c < 2; c++)
            if (G.cols & (1 << c)) { G.wait_slot(h, c, ia[c]); G.wait_slot(h, c, ic[c]); }
    }
    GemmArgs g = gemm_std(bs, bs, bs, -1.0, G.ch(slot(0, ia[0]), slot(1, ia[1]), s_slot_e), bs,
                          G.ch(slot(0, ib[0]), slot(1, ib[1]), s_slot_e), bs, 0.0,
                          G.ch(slot(0, ic[0]), slot(1, ic[1]), s_slot_e), bs);
    gemm_run(G.ctx, g, batch, GEMM_BIG, EPI_STD);
    if (h->offload) {
        if (r == nb - 1) {
            if (G.cols & 1) G.save_corner(h, 0, 1, ic[0]);              // Q_nb
            if (G.cols & 2) G.save_corner(h, 1, 0, ic[1]);              // P_1
        }
        G.copy_after_compute(r & 3);
        for (int c = 0; c < 2; c++)
            if (G.cols & (1 << c)) G.xfer(h, c, ic[c], true);
    }
}

// G.cols == 3: both block columns are in this handle's slots.  G.cols == 1 / 2: only the first / last one
// is; blocks 1 and nb of the other column come from `peer` ([n_energy][2][bs][bs], written there by the caller after the
// exchange with the GPU that owns that column), and X receives only this column's share Q_i w_top resp. P_i w_bot.
static void run_post(ss_handle_t h, Group& G, const cplx* SigL, const cplx* SigR, const cplx* inj1, const cplx* inj2,
                     int m, cplx* X, const cplx* peer) {
    Ctx& ctx = G.ctx;
    const int nb = h->nb, bs = h->bs, nE = G.nE, e0 = G.e0;
    const long long B2 = (long long)bs * bs;
    const long long s_slot_e = slot_stride_e(h);
    auto slot = [&](int col, int idx) { return slot_ptr(h, e0, col, idx); };
    // corner blocks [column][first / last block] with their energy strides
    const cplx* cor[2][2] = {{slot(0, 0), slot(0, nb - 1)}, {slot(1, 1), slot(1, nb)}};
    long long cor_s[2] = {s_slot_e, s_slot_e};
    if (h->offload)                                   // saved aside when they were produced (the ring has moved on)
        for (int c = 0; c < 2; c++) {
            cor[c][0] = h->corner + ((long long)e0 * 2 + c) * 2 * B2; cor[c][1] = cor[c][0] + B2; cor_s[c] = 4 * B2;
        }
    if (G.cols != 3) {
        const int other = (G.cols == 1) ? 1 : 0;
        cor[other][0] = peer + (long long)e0 * 2 * B2; cor[other][1] = cor[other][0] + B2; cor_s[other] = 2 * B2;
    } else if (h->part >= 0) {
        // spatial split: this handle holds the rows of one partition of the device (merged: global Q_i, P_i); the corner
        // blocks of the whole device come gathered in peer[e][first / last][column]
        for (int c = 0; c < 2; c++)
            for (int q = 0; q < 2; q++) cor[c][q] = peer + (((long long)e0 * 2 + q) * 2 + c) * B2;
        cor_s[0] = cor_s[1] = 4 * B2;
    }
    const int zc = h->want_T ? bs : 0;                // columns of e_2 (for (R^-1)_{12}, (R^-1)_{22})
    const int W = 2 * bs + m + zc;
    const int nr = m + zc;
    const int ldW = pad_ld(W);
    const long long s_r = 2LL * bs * ldW, s_w = 2LL * bs * nr;
    cplx* raug = h->raug + e0 * s_r;
    cplx* wz = h->wz + e0 * s_w;
    SigL += e0 * B2; SigR += e0 * B2;
    if (inj1) inj1 += (long long)e0 * bs * m;
    if (inj2) inj2 += (long long)e0 * bs * m;
    if (X) X += (long long)e0 * nb * bs * m;
    cplx *g1n = h->g1n + e0 * B2, *w1 = h->w1 + e0 * B2, *w2 = h->w2 + e0 * B2;
    cplx *gam_l = h->gam_l + e0 * B2, *gam_r = h->gam_r + e0 * B2;
    ctx.use(CLS_HI);
    if (h->post_wait) cudaStreamWaitEvent(ctx.st, h->ev_sig, 0);          // Sigma, Inj uploaded by ss_solve_host
    {
        dim3 grid((unsigned)min((long long)8, cdiv(W, 256)), (unsigned)(2 * bs), (unsigned)nE);
        corner_init_kernel<<<grid, 256, 0, ctx.st>>>(raug, s_r, W, ldW, bs, m, inj1, inj2);
        ctx.note(cudaGetLastError());
    }
    ctx.use(CLS_LO);
    // R = 1 - C [Q P]:  R11 -= Sigma_L Q_1, R12 -= Sigma_L P_1, R21 -= Sigma_R Q_nb, R22 -= Sigma_R P_nb
    const cplx* sig[2] = {SigL, SigR};
    for (int br = 0; br < 2; br++)
        for (int bc = 0; bc < 2; bc++) {
            GemmArgs g = gemm_std(bs, bs, bs, -1.0, bp_strided(sig[br], B2), bs, bp_strided(cor[bc][br], cor_s[bc]), bs, 1.0,
                                  bp_strided(raug + (long long)br * bs * ldW + (long long)bc * bs, s_r), ldW);
            gemm_run(ctx, g, nE, GEMM_BIG, EPI_STD);
        }
    LuWork w;
    w.tinv = h->tinv + lu_tinv_elems(bs, 2 * h->n_energy) + lu_tinv_elems(2 * bs, e0);
    w.ipiv = h->ipiv + (long long)2 * h->n_energy * 2 * bs + (long long)e0 * 2 * bs; w.ipiv_stride = 2 * bs;
    w.info = h->info + 2 * h->n_energy + e0;
    w.perm = h->perm + (long long)e0 * perm_ints_per_energy(bs);
    w.tmp = h->aop + e0 * 2 * B2; w.tmp_elems = 2 * B2;
    lu_factor(ctx, bp_strided(raug, s_r), ldW, 2 * bs, W, nE, w, 0);
    back_substitute(ctx, bp_strided(raug, s_r), ldW, 2 * bs, nr, bp_strided(wz, s_w), nr, nE, w);
    // a6: X_i = Q_i w_top + P_i w_bot, batch z = e*nb + (i-1)
    if (m > 0 && h->offload) {
        // the block columns come back from the host block by block, two ring slots per column alternating: the copy of
        // block i+1 runs under the products of block i
        for (int i = 0; i < nb; i++) {
            const int li[2] = {i, i + 1};                        // logical slots of Q_{i+1}, P_{i+1}
            const long long xoff = (long long)i * bs * m, xs = (long long)nb * bs * m;
            if (i >= 2) cudaStreamWaitEvent(G.cp->st, G.cp->ev_step[i & 1], 0);   // the products of block i-2 are done with this ring slot
            else if (i == 0) G.copy_after_compute(3);            // ... and the recursion with all of them
            for (int c = 0; c < 2; c++) {
                if (!(G.cols & (1 << c))) continue;
                const size_t B2b = sizeof(cplx) * (size_t)B2;
                cplx* d = h->slots + (long long)e0 * s_slot_e + ((long long)c * h->ring + (i & 1)) * B2;
                cudaError_t e = cudaMemcpy2DAsync(d, sizeof(cplx) * (size_t)s_slot_e, host_ptr(h, e0, c, li[c]),
                                                  2 * (size_t)(nb + 1) * B2b, B2b, (size_t)nE, cudaMemcpyHostToDevice, G.cp->st);
                if (ctx.err == cudaSuccess && e != cudaSuccess) ctx.err = e;
                cudaEventRecord(G.cp->ev_slot[c][i & 1], G.cp->st);
                cudaStreamWaitEvent(ctx.st, G.cp->ev_slot[c][i & 1], 0);
                GemmArgs g = gemm_std(bs, m, bs, 1.0, bp_strided(d, s_slot_e), bs,
                                      bp_strided(wz + (c ? (long long)bs * nr : 0), s_w), nr, (c == 1 && (G.cols & 1)) ? 1.0 : 0.0,
                                      bp_strided(X + xoff, xs), m);
                gemm_run(ctx, g, nE, GEMM_BIG, EPI_STD);
            }
            cudaEventRecord(G.cp->ev_step[i & 1], ctx.st);
        }
    } else if (m > 0) {
        if (G.cols & 1) {
            GemmArgs g = gemm_std(bs, m, bs, 1.0, bp_two_level(slot(0, 0), nb, B2, s_slot_e), bs,
                                  bp_two_level(wz, nb, 0, s_w), nr, 0.0,
                                  bp_two_level(X, nb, (long long)bs * m, (long long)nb * bs * m), m);
            gemm_run(ctx, g, nE * nb, GEMM_BIG, EPI_STD);
        }
        if (G.cols & 2) {
            GemmArgs g2 = gemm_std(bs, m, bs, 1.0, bp_two_level(slot(1, 1), nb, B2, s_slot_e), bs,
                                   bp_two_level(wz + (long long)bs * nr, nb, 0, s_w), nr, (G.cols & 1) ? 1.0 : 0.0,
                                   bp_two_level(X, nb, (long long)bs * m, (long long)nb * bs * m), m);
            gemm_run(ctx, g2, nE * nb, GEMM_BIG, EPI_STD);
        }
    }
    // a7: G_1N = Q_1 (R^-1)_12 + P_1 (R^-1)_22;  T = Re Tr(Gamma_L G Gamma_R G^H)
    if (h->want_T) {
        GemmArgs g = gemm_std(bs, bs, bs, 1.0, bp_strided(cor[0][0], cor_s[0]), bs, bp_strided(wz + m, s_w), nr, 0.0,
                              bp_strided(g1n, B2), bs);
        gemm_run(ctx, g, nE, GEMM_BIG, EPI_STD);
        GemmArgs g2 = gemm_std(bs, bs, bs, 1.0, bp_strided(cor[1][0], cor_s[1]), bs,
                               bp_strided(wz + (long long)bs * nr + m, s_w), nr, 1.0, bp_strided(g1n, B2), bs);
        gemm_run(ctx, g2, nE, GEMM_BIG, EPI_STD);
        dim3 gg((unsigned)cdiv(bs, 32), (unsigned)cdiv(bs, 32), (unsigned)nE);
        gamma_kernel<<<gg, 256, 0, ctx.st>>>(SigL, gam_l, bs); ctx.note(cudaGetLastError());
        gamma_kernel<<<gg, 256, 0, ctx.st>>>(SigR, gam_r, bs); ctx.note(cudaGetLastError());
        GemmArgs g3 = gemm_std(bs, bs, bs, 1.0, bp_strided(gam_l, B2), bs, bp_strided(g1n, B2), bs, 0.0,
                               bp_strided(w1, B2), bs);
        gemm_run(ctx, g3, nE, GEMM_BIG, EPI_STD);
        GemmArgs g4 = gemm_std(bs, bs, bs, 1.0, bp_strided(w1, B2), bs, bp_strided(gam_r, B2), bs, 0.0,
                               bp_strided(w2, B2), bs);
        gemm_run(ctx, g4, nE, GEMM_BIG, EPI_STD);
        int parts = (int)min((long long)TRACE_PARTS, cdiv(B2, 256));
        trace_partial_kernel<<<dim3((unsigned)parts, (unsigned)nE), 256, 0, ctx.st>>>(w2, B2, g1n, B2, B2, 0,
                                                                                       h->tpart + (long long)e0 * TRACE_PARTS);
        ctx.note(cudaGetLastError());
        trace_final_kernel<<<nE, 32, 0, ctx.st>>>(h->tpart + (long long)e0 * TRACE_PARTS, parts, h->T_dev + e0);
        ctx.note(cudaGetLastError());
    }
}

static bool ensure_groups(ss_handle_t h, int n) {
    if (!h->ev_fork && cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming) != cudaSuccess) return false;
    int lo_prio = 0, hi_prio = 0;
    cudaDeviceGetStreamPriorityRange(&lo_prio, &hi_prio);     // numerically lower = higher priority
    while ((int)h->groups.size() < n) {
        ss_handle_s::GroupRes g;
        bool ok = cudaStreamCreateWithPriority(&g.hi, cudaStreamNonBlocking, hi_prio) == cudaSuccess &&
                  cudaStreamCreateWithPriority(&g.lo, cudaStreamNonBlocking, lo_prio) == cudaSuccess &&
                  cudaEventCreateWithFlags(&g.ev_sw, cudaEventDisableTiming) == cudaSuccess &&
                  cudaEventCreateWithFlags(&g.ev_mark, cudaEventDisableTiming) == cudaSuccess;
        h->groups.push_back(g);                               // pushed even on failure so that ss_destroy frees the parts
        if (!ok) return false;
    }
    return true;
}

// Everything ss_solve puts on the device, enqueued on `stream` (a non-default stream the handle owns).
enum { PH_SWEEP = 1, PH_POST = 2 };
static cudaError_t enqueue_solve(ss_handle_t h, cudaStream_t stream, int phases, int cols, const cplx* Sigma_L,
                                 const cplx* Sigma_R, const cplx* Inj_first, const cplx* Inj_last, int nrhs, cplx* X,
                                 const cplx* peer) {
    auto mark = [&](cudaEvent_t ev) { return cudaEventRecord(ev, stream); };
    const size_t nEs = (size_t)h->n_energy;
    if (phases & PH_SWEEP) {
        if (cudaMemcpyAsync(h->E_dev, h->E_pinned, sizeof(cplx) * nEs, cudaMemcpyHostToDevice, stream) != cudaSuccess ||
            cudaMemsetAsync(h->info, 0, sizeof(int) * 8 * nEs, stream) != cudaSuccess)
            return cudaErrorUnknown;
    } else if (cudaMemsetAsync(h->info + 2 * nEs, 0, sizeof(int) * nEs, stream) != cudaSuccess) {   // the corner's records
        return cudaErrorUnknown;
    }
    // Energy points are independent: split them over stream groups.  Group g owns the energies
    // [e0, e0 + nE); the host interleaves the groups' launches step by step so that every group's streams stay fed.
    const int nG = h->stream_groups < h->n_energy ? h->stream_groups : h->n_energy;
    std::vector<Group> G((size_t)nG);
    std::vector<std::vector<char>> slot_used((size_t)nG, std::vector<char>((size_t)2 * h->ring, 0));
    for (int g = 0; g < nG; g++) {
        G[g].e0 = (int)((long long)h->n_energy * g / nG);
        G[g].nE = (int)((long long)h->n_energy * (g + 1) / nG) - G[g].e0;
        G[g].cols = cols;
        if (h->offload) { G[g].cp = &h->gcopy[g]; G[g].slot_used = &slot_used[g]; }
        Ctx& c = G[g].ctx;
        c.variant = h->gemm_variant;
        c.group = g;
        c.prof = h->profile_gemm ? &h->prof : nullptr;
        c.st = stream;
    }
    mark(h->ev[0]);
    if (nG > 1) {
        cudaEventRecord(h->ev_fork, stream);
        for (int g = 0; g < nG; g++) {
            Ctx& c = G[g].ctx;
            c.s_hi = h->groups[g].hi; c.s_lo = h->groups[g].lo; c.ev_sw = h->groups[g].ev_sw;
            c.st = c.s_lo; c.cls = CLS_LO;
            cudaStreamWaitEvent(c.s_lo, h->ev_fork, 0);
        }
    }
    if (h->offload) {                                      // the copy streams join the solve behind its starting point
        cudaEventRecord(h->ev_in, stream);
        for (int g = 0; g < nG; g++) cudaStreamWaitEvent(h->gcopy[g].st, h->ev_in, 0);
    }
    for (auto& r : h->trace) { cudaEventDestroy(r.t0); cudaEventDestroy(r.t1); }
    h->trace.clear();
    if (h->want_trace)
        for (int g = 0; g < nG; g++) { G[g].ctx.trace = &h->trace; G[g].ctx.trace_open(); }
    const int nb = h->nb;
    if (phases & PH_SWEEP) {
        for (int s = 0; s < nb; s++)
            for (int g = 0; g < nG; g++) sweep_step(h, G[g], s);
        for (int r = 1; r < nb; r++)
            for (int g = 0; g < nG; g++) recursion_step(h, G[g], r);
    }
    if (nG > 1)
        for (int g = 0; g < nG; g++) {                     // marks the end of the sweep phase; the groups do not wait
            G[g].ctx.use(CLS_LO);
            cudaEventRecord(h->groups[g].ev_mark, G[g].ctx.st);
            cudaStreamWaitEvent(stream, h->groups[g].ev_mark, 0);
        }
    mark(h->ev[1]);
    if (phases & PH_POST)
        for (int g = 0; g < nG; g++) run_post(h, G[g], Sigma_L, Sigma_R, Inj_first, Inj_last, nrhs, X, peer);
    if (nG > 1)
        for (int g = 0; g < nG; g++) {
            G[g].ctx.use(CLS_LO);
            cudaEventRecord(h->groups[g].ev_mark, G[g].ctx.st);
            cudaStreamWaitEvent(stream, h->groups[g].ev_mark, 0);
        }
    if (h->offload)                                        // the write-backs to the host belong to the solve
        for (int g = 0; g < nG; g++) {
            cudaEventRecord(h->gcopy[g].ev_step[0], h->gcopy[g].st);
            cudaStreamWaitEvent(stream, h->gcopy[g].ev_step[0], 0);
        }
    for (int g = 0; g < nG; g++) G[g].ctx.trace_close();
    mark(h->ev[2]);
    h->launches = 0;
    cudaError_t err = cudaSuccess;
    for (int g = 0; g < nG; g++) {
        h->launches += G[g].ctx.launches;
        if (err == cudaSuccess) err = G[g].ctx.err;
    }
    return err;
}

static ss_status_t check_info(ss_handle_t h);

// Common body of ss_solve (both phases, both columns) and of the split-phase calls of SURVEY.md 8(f2).
static ss_status_t run_phases(ss_handle_t h, const ss_cplx* E_host, int phases, int cols, const ss_cplx* Sigma_L,
                              const ss_cplx* Sigma_R, const ss_cplx* Inj_first, const ss_cplx* Inj_last, int nrhs, ss_cplx* X,
                              const ss_cplx* peer, void* cuda_stream) {
    if (!h->have_h) return SS_ERR_NOT_READY;
    if (h->launched) cudaEventSynchronize(h->ev[2]);      // the previous call may still use the scratch this one may re-allocate
    ss_status_t st = ensure_workspace(h, nrhs);
    if (st != SS_OK) return st;
    const int nG = h->stream_groups < h->n_energy ? h->stream_groups : h->n_energy;
    if (nG > 1 && !ensure_groups(h, nG)) { cudaGetLastError(); return SS_ERR_CUDA; }
    if (h->offload && !ensure_offload(h, nG)) { cudaGetLastError(); return SS_ERR_CUDA; }
    if (!h->main_stream) {
        if (cudaStreamCreateWithFlags(&h->main_stream, cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&h->ev_in, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&h->ev_out, cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); return SS_ERR_CUDA; }
    }
    cudaStream_t user = (cudaStream_t)cuda_stream, main = h->main_stream;
    if (h->launched) cudaEventSynchronize(h->ev[2]);      // E_pinned and the per-solve scratch of the previous call are free again
    if (phases & PH_SWEEP) {
        if (h->upload_consumed) { h->upload_pending = false; h->upload_consumed = false; }   // that solve saw the whole upload
        if ((const void*)E_host != (const void*)h->E_pinned) memcpy(h->E_pinned, E_host, sizeof(cplx) * (size_t)h->n_energy);
        // A = E S - H is Hermitian when every energy is real
        bool all_real = true;
        for (int e = 0; e < h->n_energy; e++) all_real = all_real && (E_host[e].im == 0.0);
        int mode = all_real ? h->hermitian : 0;
        if (mode == 2 && h->bs > LEAF2_TPB * LEAF2_MAXC) mode = 1;
        if (h->force_general) mode = 0;
        h->mode = mode;
        if (!h->force_general) h->retried = 0;
        h->swept_cols = cols;
    }
    if (phases == (PH_SWEEP | PH_POST)) h->last_args = {Sigma_L, Sigma_R, Inj_first, Inj_last, X, nrhs, cuda_stream};
    h->prof.used = 0; h->prof.flops = 0.0; h->prof.launches = 0;
    // the solve runs on a stream of the handle, ordered after the caller's stream and joined back to it
    cudaEventRecord(h->ev_in, user);
    cudaStreamWaitEvent(main, h->ev_in, 0);

    cudaError_t err = enqueue_solve(h, main, phases, cols, (const cplx*)Sigma_L, (const cplx*)Sigma_R, (const cplx*)Inj_first,
                                    (const cplx*)Inj_last, nrhs, (cplx*)X, (const cplx*)peer);
    cudaEventRecord(h->ev_out, main);
    cudaStreamWaitEvent(user, h->ev_out, 0);
    if ((phases & PH_SWEEP) && h->upload_pending) h->upload_consumed = true;
    h->last_stream = user;
    h->launched = true;
    if (phases & PH_POST) { h->last_nrhs = nrhs; h->solved = true; h->whole_solve = (phases & PH_SWEEP) != 0; }
    else h->solved = false;
    if (err != cudaSuccess) { cudaGetLastError(); return SS_ERR_CUDA; }
    return SS_OK;
}

extern "C" ss_status_t ss_solve(ss_handle_t h, const ss_cplx* E_host, const ss_cplx* Sigma_L, const ss_cplx* Sigma_R,
                                const ss_cplx* Inj_first, const ss_cplx* Inj_last, int nrhs, ss_cplx* X,
                                void* cuda_stream) {
    if (!h || !E_host || !Sigma_L || !Sigma_R || nrhs < 0) return SS_ERR_INVALID_ARG;
    if (nrhs > 0 && (!Inj_first || !X)) return SS_ERR_INVALID_ARG;
    h->part = -1;
    return run_phases(h, E_host, PH_SWEEP | PH_POST, 3, Sigma_L, Sigma_R, Inj_first, Inj_last, nrhs, X, nullptr, cuda_stream);
}

// ---- one energy batch on two GPUs, one block column of A^-1 each ----------------
extern "C" ss_status_t ss_sweep_column(ss_handle_t h, const ss_cplx* E_host, int column, void* cuda_stream) {
    if (!h || !E_host || column < 0 || column > 1) return SS_ERR_INVALID_ARG;
    h->part = -1;
    return run_phases(h, E_host, PH_SWEEP, 1 << column, nullptr, nullptr, nullptr, nullptr, 0, nullptr, nullptr, cuda_stream);
}

extern "C" ss_status_t ss_get_corner_blocks(ss_handle_t h, int column, ss_cplx* out_dev, void* cuda_stream) {
    if (!h || !out_dev || column < 0 || column > 1) return SS_ERR_INVALID_ARG;
    if (!h->launched || !(h->swept_cols & (1 << column))) return SS_ERR_NOT_READY;
    const size_t B2 = (size_t)h->bs * h->bs, nb = h->nb;
    const cplx* base = h->offload ? h->corner + (size_t)column * 2 * B2      // saved aside when produced: [e][column][2][B2]
                                  : h->slots + (column ? (nb + 1) * B2 + B2 : 0);   // block 1 of that column of energy 0
    const size_t spitch = (h->offload ? 4 * B2 : 2 * (nb + 1) * B2) * sizeof(cplx);
    // [n_energy][2][bs][bs]: blocks 1 and nb; one strided 2-D copy per block position
    for (int q = 0; q < 2; q++) {
        const cplx* src = base + (q ? (h->offload ? B2 : (nb - 1) * B2) : 0);
        if (cudaMemcpy2DAsync((cplx*)out_dev + q * B2, 2 * B2 * sizeof(cplx), src, spitch, B2 * sizeof(cplx),
                              (size_t)h->n_energy, cudaMemcpyDeviceToDevice, (cudaStream_t)cuda_stream) != cudaSuccess) {
            cudaGetLastError(); return SS_ERR_CUDA;
        }
    }
    return SS_OK;
}

// ---- SURVEY.md 8(f2), second half: the device split into two halves along the transport axis ("horizontal
// split", L169 SPIKE), one half per GPU.  Each GPU sweeps ITS OWN sub-device (ss_sweep_partition: first and last block
// columns of A_T^-1 resp. A_B^-1); the halves are coupled only through U = A_{h,h+1} and L = A_{h+1,h}.  With
//   QT, PT = first / last block column of A_T^-1 (h blocks),  QB, PB = those of A_B^-1,
// the first block column x of the whole inverse solves  x_T = QT - PT U x_{B,1},  x_B = -QB L x_{T,h},  so the interface
// blocks a = x_{T,h}, b = x_{B,1} obey  (1 - PT_h U QB_1 L) a = QT_h,  b = -QB_1 L a;  the last block column likewise with
// (1 - QB_1 L PT_h U) b' = PB_1,  a' = -PT_h U b'.  Then
//   top half:     Q_i = QT_i - PT_i (U b),      P_i = -PT_i (U b')              i = 1..h
//   bottom half:  Q_{h+i} = -QB_i (L a),        P_{h+i} = PB_i - QB_i (L a')    i = 1..nb-h
// Both GPUs solve the two bs x bs interface systems redundantly from own + peer interface blocks (2 blocks per energy each
// way), then update their own rows; no other data crosses.  Afterwards each half holds the rows of the GLOBAL Q, P.
static void edge_ptrs(ss_handle_t h, int edge, const cplx* out[2]) {      // first (0) / last (1) block of both columns, energy 0
    out[0] = slot_ptr(h, 0, 0, edge ? h->nb - 1 : 0);
    out[1] = slot_ptr(h, 0, 1, edge ? h->nb : 1);
}

extern "C" ss_status_t ss_sweep_partition(ss_handle_t h, const ss_cplx* E_host, void* cuda_stream) {
    if (!h || !E_host) return SS_ERR_INVALID_ARG;
    if (h->offload) return SS_ERR_NOT_READY;
    h->part = -1;
    return run_phases(h, E_host, PH_SWEEP, 3, nullptr, nullptr, nullptr, nullptr, 0, nullptr, nullptr, cuda_stream);
}

extern "C" ss_status_t ss_get_edge_blocks(ss_handle_t h, int edge, ss_cplx* out_dev, void* cuda_stream) {
    if (!h || !out_dev || edge < 0 || edge > 1) return SS_ERR_INVALID_ARG;
    if (!h->launched || h->swept_cols != 3 || h->offload) return SS_ERR_NOT_READY;
    const size_t B2 = (size_t)h->bs * h->bs;
    const cplx* src[2];
    edge_ptrs(h, edge, src);
    for (int c = 0; c < 2; c++)
        if (cudaMemcpy2DAsync((cplx*)out_dev + c * B2, 2 * B2 * sizeof(cplx), src[c], sizeof(cplx) * (size_t)slot_stride_e(h),
                              B2 * sizeof(cplx), (size_t)h->n_energy, cudaMemcpyDeviceToDevice, (cudaStream_t)cuda_stream) != cudaSuccess) {
            cudaGetLastError(); return SS_ERR_CUDA;
        }
    return SS_OK;
}

extern "C" ss_status_t ss_merge_partition(ss_handle_t h, int part, const ss_cplx* iface_dev, const ss_cplx* S_couple_dev,
                                          const ss_cplx* H_couple_dev, void* cuda_stream) {
    if (!h || part < 0 || part > 1 || !iface_dev || !S_couple_dev || !H_couple_dev) return SS_ERR_INVALID_ARG;
    if (!h->launched || h->swept_cols != 3 || h->offload) return SS_ERR_NOT_READY;
    const int nb = h->nb, bs = h->bs, nE = h->n_energy;
    const long long B2 = (long long)bs * bs, sE = slot_stride_e(h);
    cudaStream_t user = (cudaStream_t)cuda_stream, main = h->main_stream;
    cudaEventSynchronize(h->ev[2]);
    cudaEventRecord(h->ev_in, user);
    cudaStreamWaitEvent(main, h->ev_in, 0);
    Ctx ctx; ctx.st = main; ctx.variant = h->gemm_variant;
    // interface blocks, gathered by the caller: iface[e][0] = (QT_h, PT_h), the LAST block of both columns of the top
    // partition; iface[e][1] = (QB_1, PB_1), the FIRST block of both columns of the bottom partition.  (In a merge of
    // partitions that are themselves spread over several GPUs, most ranks own neither.)
    const cplx* ifc = (const cplx*)iface_dev;
    const cplx *QTh = ifc, *PTh = ifc + B2, *QB1 = ifc + 2 * B2, *PB1 = ifc + 3 * B2;
    const long long sT = 4 * B2, sB = 4 * B2;
    cplx *U = h->gam_l, *Lc = h->gam_r, *W1 = h->g1n, *V1 = h->w1, *W2 = h->w2;
    auto gemm = [&](double alpha, const cplx* A, long long sA, const cplx* B, long long sB_, double beta, cplx* C, long long sC, int ldc) {
        GemmArgs g = gemm_std(bs, bs, bs, alpha, bp_strided(A, sA), bs, bp_strided(B, sB_), bs, beta, bp_strided(C, sC), ldc);
        gemm_run(ctx, g, nE, GEMM_BIG, EPI_STD);
    };
    // U = E S_c - H_c, L = E S_c^H - H_c^H for every energy (eshift 0: batch entry = energy)
    FormSide up{(const cplx*)S_couple_dev, (const cplx*)H_couple_dev, FORM_PLAIN}, lo{(const cplx*)S_couple_dev, (const cplx*)H_couple_dev, FORM_CONJT};
    launch_form(ctx, up, up, h->E_dev, bp_strided(U, B2), bs, bs, nE, 0);
    launch_form(ctx, lo, lo, h->E_dev, bp_strided(Lc, B2), bs, bs, nE, 0);
    gemm(1.0, QB1, sB, Lc, B2, 0.0, W1, B2, bs);                          // W1 = QB_1 L
    gemm(1.0, PTh, sT, U, B2, 0.0, V1, B2, bs);                           // V1 = PT_h U
    gemm(1.0, U, B2, W1, B2, 0.0, W2, B2, bs);                            // W2 = U QB_1 L
    // the two interface systems as chains z = 2 e + q of the sweep's work matrix: [1 - PT_h W2 | QT_h], [1 - W1 V1 | PB_1]
    const int ldg = pad_ld(2 * bs);
    const long long s_aug_e = 2LL * bs * ldg;
    const BPtr aug = bp_chain(h->aug, h->aug + (long long)bs * ldg, s_aug_e);
    {
        dim3 grid((unsigned)min((long long)8, cdiv(2 * bs, 256)), (unsigned)bs, (unsigned)(2 * nE));
        merge_init_kernel<<<grid, 256, 0, ctx.st>>>(aug, ldg, bs, QTh, sT, PB1, sB);
        ctx.note(cudaGetLastError());
    }
    gemm(-1.0, PTh, sT, W2, B2, 1.0, h->aug, s_aug_e, ldg);
    gemm(-1.0, W1, B2, V1, B2, 1.0, h->aug + (long long)bs * ldg, s_aug_e, ldg);
    LuWork w2;                                                            // the sweep's scratch: all of it is free now
    w2.tinv = h->tinv; w2.ipiv = h->ipiv; w2.ipiv_stride = 2 * bs; w2.info = h->info + 6 * (size_t)nE;
    // zero pivots of the interface systems go to the merge's own records [6 nE, 8 nE): the sweep's records [0, 2 nE) stay
    // readable, and since a record is written by compare-and-swap against 0 and cleared only by the next sweep, the first
    // failure of ANY merge level survives the levels after it (check_info, ss_last_info: block = -2)
    w2.perm = h->perm; w2.tmp = h->aop; w2.tmp_elems = B2;
    lu_factor(ctx, aug, ldg, bs, 2 * bs, 2 * nE, w2, 0);
    cplx *av = h->aop, *bpv = h->aop + B2;                                // a (chain 0) and b' (chain 1) per energy
    back_substitute(ctx, aug, ldg, bs, bs, bp_chain(av, bpv, 2 * B2), bs, 2 * nE, w2);
    // the two products each half needs: top U b, U b' (b = -W1 a); bottom L a, L a' (a' = -V1 b')
    cplx *F1 = V1, *F2 = (part == 0) ? Lc : U;
    if (part == 0) {
        gemm(-1.0, W1, B2, av, 2 * B2, 0.0, W2, B2, bs);                  // b
        gemm(1.0, U, B2, W2, B2, 0.0, F1, B2, bs);                        // F1 = U b    (V1 is free: a' is not needed here)
        gemm(1.0, U, B2, bpv, 2 * B2, 0.0, F2, B2, bs);                   // F2 = U b'
    } else {
        gemm(-1.0, V1, B2, bpv, 2 * B2, 0.0, W2, B2, bs);                 // a'
        gemm(1.0, Lc, B2, av, 2 * B2, 0.0, F1, B2, bs);                   // F1 = L a
        gemm(1.0, Lc, B2, W2, B2, 0.0, F2, B2, bs);                       // F2 = L a'
    }
    // row updates.  Column 0 lives in slots 0..nb-1, column 1 in slots 1..nb.
    const cplx* Qs = slot_ptr(h, 0, 0, 0);
    const cplx* Ps = slot_ptr(h, 0, 1, 1);
    auto batched = [&](double alpha, const cplx* A, const cplx* F, double beta, const cplx* C) {   // all blocks and energies at once
        GemmArgs g = gemm_std(bs, bs, bs, alpha, bp_two_level(A, nb, B2, sE), bs, bp_two_level(F, nb, 0, B2), bs, beta,
                              bp_two_level(C, nb, B2, sE), bs);
        gemm_run(ctx, g, nE * nb, GEMM_BIG, EPI_STD);
    };
    auto in_place = [&](const cplx* Col, const cplx* F) {                 // Col_i = -Col_i F, block by block through a scratch block
        for (int i = 0; i < nb; i++) {
            gemm(-1.0, Col + (long long)i * B2, sE, F, B2, 0.0, W1, B2, bs);
            ctx.note(cudaMemcpy2DAsync((cplx*)Col + (long long)i * B2, sizeof(cplx) * (size_t)sE, W1, sizeof(cplx) * (size_t)B2,
                                       sizeof(cplx) * (size_t)B2, (size_t)nE, cudaMemcpyDeviceToDevice, ctx.st));
        }
    };
    if (part == 0) {
        batched(-1.0, Ps, F1, 1.0, Qs);                                   // Q_i = QT_i - PT_i (U b)
        in_place(Ps, F2);                                                 // P_i = -PT_i (U b')
    } else {
        batched(-1.0, Qs, F2, 1.0, Ps);                                   // P_i = PB_i - QB_i (L a')
        in_place(Qs, F1);                                                 // Q_i = -QB_i (L a)
    }
    cudaEventRecord(h->ev[2], main);
    cudaEventRecord(h->ev_out, main);
    cudaStreamWaitEvent(user, h->ev_out, 0);
    h->part = part;
    h->last_stream = user;
    if (ctx.err != cudaSuccess) { cudaGetLastError(); return SS_ERR_CUDA; }
    return SS_OK;
}

extern "C" ss_status_t ss_post_partition(ss_handle_t h, const ss_cplx* corners_dev, const ss_cplx* Sigma_L,
                                         const ss_cplx* Sigma_R, const ss_cplx* Inj_first, const ss_cplx* Inj_last, int nrhs,
                                         ss_cplx* X_rows, void* cuda_stream) {
    if (!h || !corners_dev || !Sigma_L || !Sigma_R || nrhs < 0) return SS_ERR_INVALID_ARG;
    if (nrhs > 0 && (!Inj_first || !X_rows)) return SS_ERR_INVALID_ARG;
    if (!h->launched || h->part < 0) return SS_ERR_NOT_READY;
    return run_phases(h, nullptr, PH_POST, 3, Sigma_L, Sigma_R, Inj_first, Inj_last, nrhs, X_rows, corners_dev, cuda_stream);
}

extern "C" ss_status_t ss_post_column(ss_handle_t h, int column, const ss_cplx* peer_corner_dev, const ss_cplx* Sigma_L,
                                      const ss_cplx* Sigma_R, const ss_cplx* Inj_first, const ss_cplx* Inj_last, int nrhs,
                                      ss_cplx* X_part, void* cuda_stream) {
    if (!h || !peer_corner_dev || !Sigma_L || !Sigma_R || nrhs < 0 || column < 0 || column > 1) return SS_ERR_INVALID_ARG;
    if (nrhs > 0 && (!Inj_first || !X_part)) return SS_ERR_INVALID_ARG;
    if (!h->launched || h->swept_cols != (1 << column)) return SS_ERR_NOT_READY;
    return run_phases(h, nullptr, PH_POST, 1 << column, Sigma_L, Sigma_R, Inj_first, Inj_last, nrhs, X_part, peer_corner_dev,
                      cuda_stream);
}

static ss_status_t check_info(ss_handle_t h) {
    const int nE = h->n_energy, n = 8 * nE;
    int* host = (int*)malloc(sizeof(int) * (size_t)n);
    if (!host) return SS_ERR_ALLOC;
    cudaError_t e = cudaMemcpy(host, h->info, sizeof(int) * (size_t)n, cudaMemcpyDeviceToHost);
    ss_status_t st = SS_OK;
    bool grown = false;
    if (e != cudaSuccess) { cudaGetLastError(); st = SS_ERR_CUDA; }
    else {
        for (int i = 0; i < n; i++) if ((i < 3 * nE || i >= 5 * nE) && host[i] != 0) { st = SS_ERR_SINGULAR; break; }
        if (h->mode == 2) {
            const float lim = (float)h->growth_limit;
            for (int i = 3 * nE; i < 5 * nE; i++) {
                float g; memcpy(&g, &host[i], sizeof(float));
                if (!(g <= lim)) grown = true;
            }
        }
    }
    free(host);
    if (st != SS_ERR_CUDA && h->mode == 2 && (grown || st == SS_ERR_SINGULAR) && !h->force_general) {
        if (!h->whole_solve) return SS_ERR_UNSTABLE;          // split-phase calls: the caller redoes both phases with "hermitian" = 0
        // the no-pivot L Delta L^H met a multiplier above the limit (or a zero pivot): its results are discarded and the
        // whole solve is redone on the general path (mode 0), same arguments, same stream
        h->force_general = true;
        h->retried = 1;
        ss_status_t s2 = ss_solve(h, (const ss_cplx*)h->E_pinned, h->last_args.sl, h->last_args.sr, h->last_args.i1,
                                  h->last_args.i2, h->last_args.nrhs, h->last_args.x, h->last_args.stream);
        h->force_general = false;
        if (s2 != SS_OK) return s2;
        if (cudaEventSynchronize(h->ev[2]) != cudaSuccess) { cudaGetLastError(); return SS_ERR_CUDA; }
        return check_info(h);
    }
    return st;
}

extern "C" ss_status_t ss_synchronize(ss_handle_t h) {
    if (!h) return SS_ERR_INVALID_ARG;
    if (!h->solved) return SS_ERR_NOT_READY;
    if (cudaEventSynchronize(h->ev[2]) != cudaSuccess) { cudaGetLastError(); return SS_ERR_CUDA; }
    return check_info(h);
}

extern "C" ss_status_t ss_transmission(ss_handle_t h, double* T_host) {
    if (!h || !T_host) return SS_ERR_INVALID_ARG;
    if (!h->solved || !h->want_T) return SS_ERR_NOT_READY;
    if (cudaEventSynchronize(h->ev[2]) != cudaSuccess) { cudaGetLastError(); return SS_ERR_CUDA; }
    ss_status_t st = check_info(h);                       // may redo the solve (hermitian mode 2 above its growth limit)
    if (st == SS_ERR_CUDA || st == SS_ERR_ALLOC) return st;
    if (cudaMemcpy(T_host, h->T_dev, sizeof(double) * (size_t)h->n_energy, cudaMemcpyDeviceToHost) != cudaSuccess) {
        cudaGetLastError(); return SS_ERR_CUDA;
    }
    return st;
}

extern "C" ss_status_t ss_last_info(ss_handle_t h, int* energy, int* block, int* column) {
    if (!h || !energy || !block || !column) return SS_ERR_INVALID_ARG;
    if (!h->solved) return SS_ERR_NOT_READY;
    *energy = *block = *column = -1;
    if (cudaEventSynchronize(h->ev[2]) != cudaSuccess) { cudaGetLastError(); return SS_ERR_CUDA; }
    const int nE = h->n_energy, n = 8 * nE;
    int* host = (int*)malloc(sizeof(int) * (size_t)n);
    if (!host) return SS_ERR_ALLOC;
    if (cudaMemcpy(host, h->info, sizeof(int) * (size_t)n, cudaMemcpyDeviceToHost) != cudaSuccess) {
        cudaGetLastError(); free(host); return SS_ERR_CUDA;
    }
    const int info_stride = 2 * h->bs + 2;
    for (int i = 0; i < n; i++) {
        if (!host[i] || (i >= 3 * nE && i < 5 * nE)) continue;     // [3 nE, 5 nE) are the growth monitors
        if (i >= 6 * nE) {                                         // interface system of an ss_merge_partition
            *energy = (i - 6 * nE) >> 1; *column = (i - 6 * nE) & 1; *block = -2;
        } else if (i < 2 * nE || i >= 5 * nE) {
            const bool single = i >= 5 * nE;                       // ss_sweep_column: one record per energy
            int s = (host[i] - 1) / info_stride;
            *energy = single ? i - 5 * nE : i >> 1;
            *column = single ? (h->swept_cols == 2 ? 1 : 0) : (i & 1);
            *block = *column ? s + 1 : h->nb - s;
        } else {
            *energy = i - 2 * nE; *column = -1; *block = 0;
        }
        break;
    }
    free(host);
    return SS_OK;
}

extern "C" ss_status_t ss_inverse_columns(ss_handle_t h, int energy, const ss_cplx** Q_first, const ss_cplx** Q_last) {
    if (!h || !Q_first || !Q_last || energy < 0 || energy >= h->n_energy) return SS_ERR_INVALID_ARG;
    if (!h->solved || h->offload) return SS_ERR_NOT_READY;    // offload mode: the columns are on the host (ss_copy_inverse_columns)
    const long long B2 = (long long)h->bs * h->bs;
    const cplx* base = h->slots + (long long)energy * 2 * (h->nb + 1) * B2;
    *Q_first = (const ss_cplx*)base;                                   // column 0, slots 0..nb-1
    *Q_last = (const ss_cplx*)(base + (long long)(h->nb + 1) * B2 + B2);   // column 1, slots 1..nb
    return SS_OK;
}

extern "C" ss_status_t ss_copy_inverse_columns(ss_handle_t h, int energy, ss_cplx* Q_out, ss_cplx* P_out) {
    if (!h || energy < 0 || energy >= h->n_energy) return SS_ERR_INVALID_ARG;
    if (!h->launched || h->swept_cols != 3) return SS_ERR_NOT_READY;        // both block columns swept (ss_solve, ss_sweep_partition)
    // The columns are complete once the handle's last work is (ev[2]); waiting for it on the host makes the copies below
    // independent of which stream that work was joined to.  A no-pivot solve (mode 2) may still be discarded and redone:
    // decide that first, so that the columns returned are the ones the solve stands by.
    if (cudaEventSynchronize(h->ev[2]) != cudaSuccess) { cudaGetLastError(); return SS_ERR_CUDA; }
    if (h->mode == 2) {
        ss_status_t c = check_info(h);
        if (c != SS_OK) return c;
    }
    const size_t B2 = (size_t)h->bs * h->bs, bytes = sizeof(cplx) * (size_t)h->nb * B2;
    const cplx *q, *p;
    cudaMemcpyKind kind = cudaMemcpyDeviceToDevice;
    if (h->offload) {                                     // the block columns live in the handle's pinned host array
        q = host_ptr(h, energy, 0, 0); p = host_ptr(h, energy, 1, 1);
        kind = cudaMemcpyHostToDevice;
    } else {
        const cplx* base = h->slots + (size_t)energy * 2 * (h->nb + 1) * B2;
        q = base; p = base + (size_t)(h->nb + 1) * B2 + B2;
    }
    if (Q_out && cudaMemcpyAsync(Q_out, q, bytes, kind, h->last_stream) != cudaSuccess) { cudaGetLastError(); return SS_ERR_CUDA; }
    if (P_out && cudaMemcpyAsync(P_out, p, bytes, kind, h->last_stream) != cudaSuccess) { cudaGetLastError(); return SS_ERR_CUDA; }
    if (cudaStreamSynchronize(h->last_stream) != cudaSuccess) { cudaGetLastError(); return SS_ERR_CUDA; }   // complete on return
    return SS_OK;
}

extern "C" ss_status_t ss_phase_ms(ss_handle_t h, int phase, float* ms) {
    if (!h || !ms || phase < 0 || phase > 2) return SS_ERR_INVALID_ARG;
    if (!h->solved) return SS_ERR_NOT_READY;
    if (cudaEventSynchronize(h->ev[2]) != cudaSuccess) { cudaGetLastError(); return SS_ERR_CUDA; }
    cudaError_t e = (phase == 0) ? cudaEventElapsedTime(ms, h->ev[0], h->ev[1])
                  : (phase == 1) ? cudaEventElapsedTime(ms, h->ev[1], h->ev[2])
                                 : cudaEventElapsedTime(ms, h->ev[0], h->ev[2]);
    if (e != cudaSuccess) { cudaGetLastError(); return SS_ERR_CUDA; }
    return SS_OK;
}

extern "C" ss_status_t ss_gemm_profile(ss_handle_t h, double* ms, double* flops, long long* launches) {
    if (!h || !ms || !flops || !launches) return SS_ERR_INVALID_ARG;
    if (!h->solved || !h->profile_gemm) return SS_ERR_NOT_READY;
    if (cudaEventSynchronize(h->ev[2]) != cudaSuccess) { cudaGetLastError(); return SS_ERR_CUDA; }
    double total = 0.0;
    for (size_t i = 0; i + 1 < h->prof.used; i += 2) {
        float t = 0.f;
        if (cudaEventElapsedTime(&t, h->prof.ev[i], h->prof.ev[i + 1]) != cudaSuccess) { cudaGetLastError(); return SS_ERR_CUDA; }
        total += t;
    }
    *ms = total; *flops = h->prof.flops; *launches = h->prof.launches;
    return SS_OK;
}

extern "C" long long ss_launch_count(ss_handle_t h) { return h ? h->launches : 0; }

extern "C" ss_status_t ss_trace_write(ss_handle_t h, const char* path) {
    if (!h || !path) return SS_ERR_INVALID_ARG;
    if (!h->solved) return SS_ERR_NOT_READY;
    if (cudaEventSynchronize(h->ev[2]) != cudaSuccess) { cudaGetLastError(); return SS_ERR_CUDA; }
    FILE* f = fopen(path, "w");
    if (!f) return SS_ERR_INVALID_ARG;
    fprintf(f, "group,class,start_ms,end_ms\n");
    for (auto& r : h->trace) {
        float a = 0.f, b = 0.f;
        if (cudaEventElapsedTime(&a, h->ev[0], r.t0) != cudaSuccess || cudaEventElapsedTime(&b, h->ev[0], r.t1) != cudaSuccess) {
            cudaGetLastError(); continue;
        }
        fprintf(f, "%d,%s,%.4f,%.4f\n", r.group, r.cls == CLS_HI ? "hi" : "lo", a, b);
    }
    if (h->profile_gemm)                                   // every GEMM launch of the solve: class "gemm", group -1
        for (size_t i = 0; i + 1 < h->prof.used; i += 2) {
            float a = 0.f, b = 0.f;
            if (cudaEventElapsedTime(&a, h->ev[0], h->prof.ev[i]) != cudaSuccess ||
                cudaEventElapsedTime(&b, h->ev[0], h->prof.ev[i + 1]) != cudaSuccess) { cudaGetLastError(); continue; }
            fprintf(f, "-1,gemm,%.4f,%.4f\n", a, b);
        }
    fclose(f);
    return SS_OK;
}

extern "C" ss_status_t ss_solve_host(ss_handle_t h, const ss_cplx* E_host, const ss_cplx* SigL, const ss_cplx* SigR,
                                     const ss_cplx* Inj1, const ss_cplx* Inj2, int nrhs, ss_cplx* X_host, double* T_host) {
    if (!h || !E_host || !SigL || !SigR || nrhs < 0 || (nrhs > 0 && !Inj1)) return SS_ERR_INVALID_ARG;
    if (!h->have_h) return SS_ERR_NOT_READY;
    const size_t C = sizeof(cplx), B2 = (size_t)h->bs * h->bs, nE = h->n_energy;
    const size_t inj_bytes = nE * h->bs * (size_t)nrhs * C, x_bytes = nE * (size_t)h->nb * h->bs * nrhs * C;
    if (!h->own_stream && cudaStreamCreateWithFlags(&h->own_stream, cudaStreamNonBlocking) != cudaSuccess) {
        cudaGetLastError(); return SS_ERR_CUDA;
    }
    if (h->hp_nrhs < nrhs) {
        free_host_path(h);
        bool ok = cudaMalloc((void**)&h->hp_sigl, nE * B2 * C) == cudaSuccess && cudaMalloc((void**)&h->hp_sigr, nE * B2 * C) == cudaSuccess &&
                  cudaMalloc((void**)&h->hp_inj1, inj_bytes ? inj_bytes : 16) == cudaSuccess &&
                  cudaMalloc((void**)&h->hp_inj2, inj_bytes ? inj_bytes : 16) == cudaSuccess &&
                  cudaMalloc((void**)&h->hp_x, x_bytes ? x_bytes : 16) == cudaSuccess;
        if (!ok) { cudaGetLastError(); free_host_path(h); return SS_ERR_ALLOC; }
        h->hp_nrhs = nrhs;
    }
    cudaStream_t st = h->own_stream;
    // Sigma and Inj go up on the copy stream (behind a pending H, S upload, which shares the copy engine anyway); only the
    // post-processing waits for them, so the sweep starts at once (pre-/post-processing split of PAPER.md L150-152).
    if (!h->copy_stream && cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking) != cudaSuccess) {
        cudaGetLastError(); return SS_ERR_CUDA;
    }
    if (!h->ev_sig && cudaEventCreateWithFlags(&h->ev_sig, cudaEventDisableTiming) != cudaSuccess) {
        cudaGetLastError(); return SS_ERR_CUDA;
    }
    if (h->launched) cudaEventSynchronize(h->ev[2]);      // the previous solve may still read the staging buffers
    cudaStream_t cs = h->copy_stream;
    bool ok = cudaMemcpyAsync(h->hp_sigl, SigL, nE * B2 * C, cudaMemcpyHostToDevice, cs) == cudaSuccess &&
              cudaMemcpyAsync(h->hp_sigr, SigR, nE * B2 * C, cudaMemcpyHostToDevice, cs) == cudaSuccess;
    if (ok && nrhs > 0) ok = cudaMemcpyAsync(h->hp_inj1, Inj1, inj_bytes, cudaMemcpyHostToDevice, cs) == cudaSuccess;
    if (ok && nrhs > 0 && Inj2) ok = cudaMemcpyAsync(h->hp_inj2, Inj2, inj_bytes, cudaMemcpyHostToDevice, cs) == cudaSuccess;
    if (ok) ok = cudaEventRecord(h->ev_sig, cs) == cudaSuccess;
    if (!ok) { cudaGetLastError(); return SS_ERR_CUDA; }
    h->post_wait = true;
    ss_status_t s = ss_solve(h, E_host, (ss_cplx*)h->hp_sigl, (ss_cplx*)h->hp_sigr, nrhs ? (ss_cplx*)h->hp_inj1 : nullptr,
                             (nrhs && Inj2) ? (ss_cplx*)h->hp_inj2 : nullptr, nrhs, nrhs ? (ss_cplx*)h->hp_x : nullptr, st);
    h->post_wait = false;
    if (s != SS_OK) return s;
    if (h->mode == 2) {                                   // the no-pivot path may be redone: decide before downloading
        if (cudaStreamSynchronize(st) != cudaSuccess) { cudaGetLastError(); return SS_ERR_CUDA; }
        ss_status_t c = check_info(h);
        if (c == SS_ERR_CUDA || c == SS_ERR_ALLOC) return c;
    }
    if (X_host && nrhs > 0 && cudaMemcpyAsync(X_host, h->hp_x, x_bytes, cudaMemcpyDeviceToHost, st) != cudaSuccess) {
        cudaGetLastError(); return SS_ERR_CUDA;
    }
    if (T_host && h->want_T && cudaMemcpyAsync(T_host, h->T_dev, sizeof(double) * nE, cudaMemcpyDeviceToHost, st) != cudaSuccess) {
        cudaGetLastError(); return SS_ERR_CUDA;
    }
    if (cudaStreamSynchronize(st) != cudaSuccess) { cudaGetLastError(); return SS_ERR_CUDA; }
    return check_info(h);
}

// ---------------------------------------------------------------------------------------------------------
// building blocks
// ---------------------------------------------------------------------------------------------------------
extern "C" ss_status_t ss_zgemm_batched(int M, int N, int K, double alpha, const ss_cplx* A, int lda, long long sA,
                                        const ss_cplx* B, int ldb, long long sB, double beta, ss_cplx* C, int ldc,
                                        long long sC, int batch, void* stream) {
    if (M < 0 || N < 0 || K < 0 || batch < 0 || !C || (K > 0 && (!A || !B))) return SS_ERR_INVALID_ARG;
    if (lda < K || ldb < N || ldc < N) return SS_ERR_INVALID_ARG;
    GemmArgs g = gemm_std(M, N, K, alpha, bp_strided((const cplx*)(A ? A : C), sA), lda, bp_strided((const cplx*)(B ? B : C), sB), ldb,
                          beta, bp_strided((cplx*)C, sC), ldc);
    cudaError_t e = gemm_launch(g, batch, GEMM_BIG, EPI_STD, (cudaStream_t)stream, g_default_variant);
    if (e != cudaSuccess) { cudaGetLastError(); return SS_ERR_CUDA; }
    return SS_OK;
}

extern "C" size_t ss_lu_workspace_bytes(int n, int batch) {
    if (n < 1 || batch < 1) return 0;
    return (lu_tinv_elems(n, batch) + (size_t)lu_tmp_elems_default(n) * batch) * sizeof(cplx) + lu_perm_ints(n, batch) * sizeof(int);
}

// Same product with sum planes (zgemm.cuh, GemmArgs::sh*): A_sum / B_sum hold re + im of every element of A / B (same leading
// dimensions and batch strides, doubles), C_sum receives re + im of every element of C; any of the three may be NULL.
extern "C" ss_status_t ss_zgemm_batched_sums(int M, int N, int K, double alpha, const ss_cplx* A, const double* A_sum, int lda,
                                             long long sA, const ss_cplx* B, const double* B_sum, int ldb, long long sB,
                                             double beta, ss_cplx* C, double* C_sum, int ldc, long long sC, int batch, void* stream) {
    if (M < 0 || N < 0 || K < 0 || batch < 0 || !C || (K > 0 && (!A || !B))) return SS_ERR_INVALID_ARG;
    if (lda < K || ldb < N || ldc < N) return SS_ERR_INVALID_ARG;
    if (C_sum && g_default_variant == GV_4M) return SS_ERR_INVALID_ARG;   // only the 3M kernels' epilogue writes a sum plane
    GemmArgs g = gemm_std(M, N, K, alpha, bp_strided((const cplx*)(A ? A : C), sA), lda, bp_strided((const cplx*)(B ? B : C), sB), ldb,
                          beta, bp_strided((cplx*)C, sC), ldc);
    if (A_sum && B_sum) { g.shA_c = (const cplx*)A; g.shA_d = A_sum; g.shB_c = (const cplx*)B; g.shB_d = B_sum; }
    if (C_sum) { g.shC_c = (const cplx*)C; g.shC_d = C_sum; }
    cudaError_t e = gemm_launch(g, batch, GEMM_BIG, EPI_STD, (cudaStream_t)stream, g_default_variant);
    if (e != cudaSuccess) { cudaGetLastError(); return SS_ERR_CUDA; }
    return SS_OK;
}

static ss_status_t lu_common(int n, int nrhs_solve, int ncols, ss_cplx* AB, int ld, long long stride, ss_cplx* X, int ldx,
                             long long sX, int* ipiv, int* info, int batch, void* work, size_t work_bytes, void* stream) {
    if (n < 1 || n > LEAF_TPB * LEAF_MAXC || ncols < n || ld < ncols || batch < 1 || !AB || !ipiv || !info || !work)
        return SS_ERR_INVALID_ARG;
    if (work_bytes < ss_lu_workspace_bytes(n, batch)) return SS_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    LuWork w;
    w.tinv = (cplx*)work; w.ipiv = ipiv; w.ipiv_stride = n; w.info = info;
    w.tmp = w.tinv + lu_tinv_elems(n, batch); w.tmp_elems = lu_tmp_elems_default(n);
    w.perm = (int*)(w.tmp + (size_t)w.tmp_elems * batch);
    Ctx ctx; ctx.st = st; ctx.variant = g_default_variant;
    cudaMemsetAsync(info, 0, sizeof(int) * (size_t)batch, st);
    BPtr Ab = bp_strided((cplx*)AB, stride);
    lu_factor(ctx, Ab, ld, n, ncols, batch, w, 0);
    if (nrhs_solve > 0) back_substitute(ctx, Ab, ld, n, nrhs_solve, bp_strided((cplx*)X, sX), ldx, batch, w);
    if (ctx.err != cudaSuccess) { cudaGetLastError(); return SS_ERR_CUDA; }
    return SS_OK;
}

extern "C" ss_status_t ss_zgetrf_batched(int n, int ncols, ss_cplx* AB, int ld, long long stride, int* ipiv, int* info,
                                         int batch, void* work, size_t work_bytes, void* stream) {
    return lu_common(n, 0, ncols, AB, ld, stride, nullptr, 0, 0, ipiv, info, batch, work, work_bytes, stream);
}

extern "C" ss_status_t ss_zgesv_batched(int n, int nrhs, ss_cplx* AB, int ld, long long stride, ss_cplx* X, int ldx,
                                        long long sX, int* ipiv, int* info, int batch, void* work, size_t work_bytes,
                                        void* stream) {
    if (nrhs < 0 || (nrhs > 0 && (!X || ldx < nrhs))) return SS_ERR_INVALID_ARG;
    return lu_common(n, nrhs, n + nrhs, AB, ld, stride, X, ldx, sX, ipiv, info, batch, work, work_bytes, stream);
}

// ---------------------------------------------------------------------------------------------------------
// ss_zgesv_batched for callers that cannot allocate device memory (plug-ins that are only handed pointers, runs whose HBM
// is fully spoken for, latency-critical loops that cannot afford cudaMalloc's device-wide stall): the LU scratch is this
// fixed array inside the library image instead of a caller-owned buffer.  Every device that loads the library carries it
// until the process ends.  Nothing here allocates.
//
// ss_noalloc_scratch is a DEVICE symbol.  In host code its name is only a host-side shadow the runtime uses as a look-up
// key -- it is not an address the GPU can use: a kernel given `ss_noalloc_scratch` (or &ss_noalloc_scratch[0]) from host
// code would fault, or scribble over host memory on systems where the GPU can reach it.  The device address comes from
// cudaGetSymbolAddress, asked once per device with that device current (each device has its own copy at its own address).
// ---------------------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned char ss_noalloc_scratch[SS_NOALLOC_SCRATCH_BYTES];

constexpr int NOALLOC_MAX_DEVICES = 64;
static std::mutex g_noalloc_mu;
static void* g_noalloc_ptr[NOALLOC_MAX_DEVICES] = {};    // device address of ss_noalloc_scratch, per device ordinal

// Device address of the current device's copy of the scratch array; looked up on the first call per device.
static ss_status_t noalloc_scratch(void** out) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return SS_ERR_CUDA; }
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return SS_ERR_INVALID_ARG;
    std::lock_guard<std::mutex> lock(g_noalloc_mu);
    if (!g_noalloc_ptr[dev]) {
        void* p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&p, ss_noalloc_scratch);
        if (e != cudaSuccess || !p) { cudaGetLastError(); return SS_ERR_CUDA; }
        g_noalloc_ptr[dev] = p;
    }
    *out = g_noalloc_ptr[dev];
    return SS_OK;
}

extern "C" ss_status_t ss_zgesv_batched_noalloc(int n, int nrhs, ss_cplx* AB, int ld, long long stride, ss_cplx* X, int ldx,
                                                long long sX, int* ipiv, int* info, int batch, void* stream) {
    if (nrhs < 0 || (nrhs > 0 && (!X || ldx < nrhs))) return SS_ERR_INVALID_ARG;
    if (n < 1 || batch < 1) return SS_ERR_INVALID_ARG;
    // the size limit is checked first, from host arithmetic alone: an oversized request touches neither the device nor the array
    const size_t need = ss_lu_workspace_bytes(n, batch);
    if (need == 0 || need > (size_t)SS_NOALLOC_SCRATCH_BYTES) return SS_ERR_INVALID_ARG;
    void* work = nullptr;
    ss_status_t s = noalloc_scratch(&work);
    if (s != SS_OK) return s;
    // same host driver, same kernels, same order as ss_zgesv_batched: only where the scratch lives differs.  The scratch is
    // not cleared: the block inverses, the permutation lists and the row-move buffer are each written before they are read.
    return lu_common(n, nrhs, n + nrhs, AB, ld, stride, X, ldx, sX, ipiv, info, batch, work, (size_t)SS_NOALLOC_SCRATCH_BYTES, stream);
}

extern "C" ss_status_t ss_density(const ss_cplx* X, int n_energy, long long n, int nrhs, const double* w, double* rho,
                                  void* stream) {
    if (!X || !rho || n_energy < 1 || n < 1 || nrhs < 1) return SS_ERR_INVALID_ARG;
    const unsigned blocks = (unsigned)cdiv(n, 8);
    density_kernel<<<blocks, 256, 0, (cudaStream_t)stream>>>((const cplx*)X, n_energy, n, nrhs, w, rho);
    if (cudaGetLastError() != cudaSuccess) return SS_ERR_CUDA;
    return SS_OK;
}

// bond (spectral) current through every block interface, from the wave functions of the last solve:
//   J[e][i] = 2 Im Tr( X_i^H A_{i,i+1}(E_e) X_{i+1} ),  A_{i,i+1} = E S_{i,i+1} - H_{i,i+1}   (Eq. 5; L85).
// Per interface: a0's form kernel for all energies, one batched GEMM W = A_{i,i+1} X_{i+1}, one conj-dot reduction.
extern "C" ss_status_t ss_bond_current(ss_handle_t h, const ss_cplx* X, int nrhs, double* J_host) {
    if (!h || !X || !J_host || nrhs < 1) return SS_ERR_INVALID_ARG;
    if (!h->solved || nrhs > h->ws_nrhs) return SS_ERR_NOT_READY;
    if (cudaEventSynchronize(h->ev[2]) != cudaSuccess) { cudaGetLastError(); return SS_ERR_CUDA; }
    const int nb = h->nb, bs = h->bs, nE = h->n_energy, m = nrhs;
    const long long B2 = (long long)bs * bs, sX = (long long)nb * bs * m, sW = (long long)bs * m;
    if (!h->J_dev && cudaMalloc((void**)&h->J_dev, sizeof(double) * (size_t)nE * (nb - 1)) != cudaSuccess) {
        cudaGetLastError(); return SS_ERR_ALLOC;                  // handle-owned, allocated on first use
    }
    double* J_dev = h->J_dev;
    Ctx ctx; ctx.st = h->main_stream ? h->main_stream : h->last_stream; ctx.variant = h->gemm_variant;
    const BPtr aop = bp_chain(h->aop, h->aop + B2, 2 * B2);
    const int parts = (int)min((long long)TRACE_PARTS, cdiv(sW, 256));
    for (int i = 0; i + 1 < nb; i++) {
        FormSide up{h->Su + (long long)i * B2, h->Hu + (long long)i * B2, FORM_PLAIN}, none{nullptr, nullptr, FORM_NONE};
        launch_form(ctx, up, none, h->E_dev, aop, bs, bs, 2 * nE);
        GemmArgs g = gemm_std(bs, m, bs, 1.0, bp_strided(h->aop, 2 * B2), bs,
                              bp_strided((const cplx*)X + (long long)(i + 1) * bs * m, sX), m, 0.0, bp_strided(h->wz, sW), m);
        gemm_run(ctx, g, nE, GEMM_BIG, EPI_STD);
        trace_partial_kernel<<<dim3((unsigned)parts, (unsigned)nE), 256, 0, ctx.st>>>(
            h->wz, sW, (const cplx*)X + (long long)i * bs * m, sX, sW, 1, h->tpart);
        ctx.note(cudaGetLastError());
        trace_final_kernel<<<nE, 32, 0, ctx.st>>>(h->tpart, parts, J_dev + i, nb - 1, 2.0);
        ctx.note(cudaGetLastError());
    }
    cudaError_t e = cudaMemcpyAsync(J_host, J_dev, sizeof(double) * (size_t)nE * (nb - 1), cudaMemcpyDeviceToHost, ctx.st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx.st);    // J_host is a host result: the call returns it complete
    if (e != cudaSuccess || ctx.err != cudaSuccess) { cudaGetLastError(); return SS_ERR_CUDA; }
    return SS_OK;
}

extern "C" ss_status_t ss_set_gemm_raster(int tile_rows) {
    if (tile_rows < 1 || tile_rows > 64) return SS_ERR_INVALID_ARG;
    g_gemm_raster = tile_rows;
    return SS_OK;
}

extern "C" ss_status_t ss_set_default_gemm_variant(int variant) {
    if (variant < 0 || variant >= GV_COUNT) return SS_ERR_INVALID_ARG;
    g_default_variant = variant;
    return SS_OK;
}

extern "C" int ss_get_default_gemm_variant(void) { return g_default_variant; }

extern "C" ss_status_t ss_fp64_peak_tflops(double ms, double* tflops) {
    if (!tflops || ms <= 0) return SS_ERR_INVALID_ARG;
    int dev = 0, nsm = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    double* out = nullptr;
    if (cudaMalloc((void**)&out, 64) != cudaSuccess) { cudaGetLastError(); return SS_ERR_ALLOC; }
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int blocks = nsm * 4, iters = 20000;           // 16 warps per SM, 8 independent DMMA chains each
    const double fl_per_launch = 2.0 * 8 * 8 * 4 * 8 * (double)iters * blocks * 4;
    fp64_peak_kernel<<<blocks, 128>>>(out, iters);
    cudaDeviceSynchronize();
    double best = 0.0, spent = 0.0;
    while (spent < ms) {
        cudaEventRecord(e0); fp64_peak_kernel<<<blocks, 128>>>(out, iters); cudaEventRecord(e1);
        if (cudaEventSynchronize(e1) != cudaSuccess) break;
        float t = 0.f; cudaEventElapsedTime(&t, e0, e1);
        spent += t;
        double tf = fl_per_launch / (t * 1e-3) * 1e-12;
        if (tf > best) best = tf;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(out);
    if (cudaGetLastError() != cudaSuccess) return SS_ERR_CUDA;
    *tflops = best;
    return SS_OK;
}

#ifdef SS_PANEL_TIMING
extern "C" int ss_debug_panel_clocks(long long* out16, int reset) {
    cudaDeviceSynchronize();
    if (out16 && cudaMemcpyFromSymbol(out16, ss_panel_clk, sizeof(long long) * 16) != cudaSuccess) return 1;
    if (reset) { long long z[16] = {0}; cudaMemcpyToSymbol(ss_panel_clk, z, sizeof(z)); }
    return 0;
}
#endif
