// Batched blocked right-looking ZGETRF with partial pivoting + blocked ZTRSM back substitution (sm_100a).
//
// "Solve (A_ii - A_{i,i+1} X_{i+1}) X_i = A_{i,i-1}" of Algorithm 1;
// the paper used MAGMA zgesv_nopiv_gpu (L186) and names "the LU factorization and backward substitution"
// as the bottleneck (L266).  Here: partial pivoting (north_star), everything on the GPU, batched over all
// independent chains (energies x {first, last} column, L167/L204), and organised so that all O(n^3) work is
// DMMA GEMM (zgemm.cuh):
//
//   LU of the augmented matrix [D | B] (n x ncols, row-major): the row interchanges and the L-solve are applied
//   to B by the same trailing updates, so only the U-solve remains afterwards.
//     outer block NB (<=128):  panel (inner blocks of JB=16 columns)  ->  L11^-1 (trtri)  ->  U12 = L11^-1 A12 (GEMM,
//     in place, one CTA owns all rows of its columns)  ->  A22 -= L21 U12 (GEMM).
//     inner block JB=16:  leaf panel kernel  ->  row swaps on all other columns  ->  16 x w triangular solve  ->
//     rank-16 GEMM update of the rest of the panel.
//   Leaf panel kernel: one thread owns one matrix ROW of the 16-column panel in registers; one thread-block
//   cluster (<=16 CTAs x 512 threads, up to 8192 rows) per matrix.  Per column: warp-shuffle arg-max, CTA
//   candidate through shared memory, candidates + candidate rows exchanged through DISTRIBUTED shared memory,
//   one cluster barrier, rank-1 update in registers.  Pivoting is implicit (no data moves until the final
//   store), bookkeeping reproduces LAPACK's sequential-swap ipiv.
//   Back substitution (left-looking, block rows of NB): T_j = Y_j - U_{j,>j} X_{>j} (GEMM), X_j = U_jj^-1 T_j (GEMM).
#pragma once
#include <cooperative_groups.h>
#include <cstddef>
#include <vector>
#include "zgemm3m.cuh"
#include "sweep.cuh"

namespace ss {
namespace cg = cooperative_groups;

constexpr int LEAF_JB = 16;       // columns per leaf panel
constexpr int LEAF_TPB = 512;     // threads (= rows) per CTA
constexpr int LEAF_MAXC = 16;     // max cluster size

struct LeafCand {                 // one CTA's pivot candidate for one column
    double val;                   // |re| + |im| (LAPACK izamax metric), -1 if the CTA has no active row
    int pos;                      // current row position inside the panel
    int pad;
    cplx row[LEAF_JB];
};

// Factor the m x jb panel at (row0, col0) of each batch matrix.  grid = (csize, batch), cluster (csize,1,1).
__global__ void __launch_bounds__(LEAF_TPB, 1)
lu_leaf_kernel(BPtr Ab, int ld, int row0, int col0, int m, int jb, int* __restrict__ ipiv, int ipiv_stride,
               int* __restrict__ info, int info_base) {
    cg::cluster_group cluster = cg::this_cluster();
    const int csize = (int)cluster.num_blocks();
    const int crank = (int)cluster.block_rank();
    const int z = blockIdx.y;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NW = LEAF_TPB / 32;

    __shared__ LeafCand slots[2][LEAF_MAXC];
    __shared__ double w_val[NW];
    __shared__ int w_pos[NW];
    __shared__ int w_tid[NW];
    __shared__ int cta_owner;

    cplx* __restrict__ A = bptr(Ab, z) + (long long)row0 * ld + col0;
    const int r = crank * LEAF_TPB + tid;       // my row inside the panel
    const bool valid = r < m;

    cplx a[LEAF_JB];
#pragma unroll
    for (int k = 0; k < LEAF_JB; k++) a[k] = make_c(0.0, 0.0);
    if (valid) {
        const cplx* src = A + (long long)r * ld;
#pragma unroll
        for (int k = 0; k < LEAF_JB; k++)
            if (k < jb) a[k] = src[k];
    }
    int cur_pos = r;
    bool done = !valid;
    int final_pos = r;

#pragma unroll
    for (int j = 0; j < LEAF_JB; j++) {
        if (j < jb) {
            const int buf = j & 1;
            // ---- local arg-max (ties -> lowest position)
            double v = done ? -1.0 : (fabs(a[j].re) + fabs(a[j].im));
            int pp = cur_pos, tt = tid;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                double ov = __shfl_xor_sync(0xffffffffu, v, o);
                int op = __shfl_xor_sync(0xffffffffu, pp, o);
                int ot = __shfl_xor_sync(0xffffffffu, tt, o);
                if (ov > v || (ov == v && op < pp)) { v = ov; pp = op; tt = ot; }
            }
            if (lane == 0) { w_val[warp] = v; w_pos[warp] = pp; w_tid[warp] = tt; }
            __syncthreads();
            if (warp == 0) {
                double v2 = lane < NW ? w_val[lane] : -2.0;
                int p2 = lane < NW ? w_pos[lane] : 0x7fffffff;
                int t2 = lane < NW ? w_tid[lane] : 0;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    double ov = __shfl_xor_sync(0xffffffffu, v2, o);
                    int op = __shfl_xor_sync(0xffffffffu, p2, o);
                    int ot = __shfl_xor_sync(0xffffffffu, t2, o);
                    if (ov > v2 || (ov == v2 && op < p2)) { v2 = ov; p2 = op; t2 = ot; }
                }
                if (lane == 0) cta_owner = (v2 >= 0.0) ? t2 : -1;
            }
            __syncthreads();
            // ---- publish this CTA's candidate to every CTA of the cluster (DSMEM)
            const int owner = cta_owner;
            if (owner < 0) {
                if (tid == 0)
                    for (int c = 0; c < csize; c++) {
                        LeafCand* dst = cluster.map_shared_rank(&slots[buf][crank], c);
                        dst->val = -1.0; dst->pos = 0x7fffffff;
                    }
            } else if (tid == owner) {
                double myv = fabs(a[j].re) + fabs(a[j].im);
                for (int c = 0; c < csize; c++) {
                    LeafCand* dst = cluster.map_shared_rank(&slots[buf][crank], c);
                    dst->val = myv; dst->pos = cur_pos;
#pragma unroll
                    for (int k = 0; k < LEAF_JB; k++) dst->row[k] = a[k];
                }
            }
            cluster.sync();
            // ---- winner among the csize candidates
            int win = 0; double wv = slots[buf][0].val; int wp = slots[buf][0].pos;
            for (int c = 1; c < csize; c++) {
                double cv = slots[buf][c].val; int cp = slots[buf][c].pos;
                if (cv > wv || (cv == wv && cp < wp)) { wv = cv; wp = cp; win = c; }
            }
            if (wv < 0.0) { wp = j; }                     // no rows left (m < jb): nothing to do
            const bool singular = !(wv > 0.0);
            if (crank == 0 && tid == 0) {
                ipiv[(long long)z * ipiv_stride + row0 + j] = row0 + wp;
                if (singular && wv >= 0.0) atomicCAS(&info[z], 0, info_base + row0 + j + 1);
            }
            if (!done) {
                if (cur_pos == wp && wv >= 0.0) {
                    done = true; final_pos = j;           // I am the pivot row: becomes row j of U
                } else {
                    if (cur_pos == j) cur_pos = wp;       // LAPACK swap bookkeeping
                    if (!singular) {
                        const cplx* prow = slots[buf][win].row;
                        cplx rinv = crecip(prow[j]);
                        cplx l = cmul(a[j], rinv);
                        a[j] = l;
#pragma unroll
                        for (int k = j + 1; k < LEAF_JB; k++) a[k] = cfnma(a[k], l, prow[k]);
                    }
                }
            }
        }
    }
    if (valid) {
        if (!done) final_pos = cur_pos;
        cplx* dst = A + (long long)final_pos * ld;
#pragma unroll
        for (int k = 0; k < LEAF_JB; k++)
            if (k < jb) dst[k] = a[k];
    }
}

// ---- helpers of the fused panel kernel (lu_panel_kernel below): 256 rows per CTA, cluster of up to 16 CTAs = 4096 rows.
// Warp arg-max by three redux.sync on the bit pattern of |re|+|im| (non-negative doubles order like unsigned integers)
// and the row position.
constexpr int LEAF2_TPB = 256;
constexpr int LEAF2_MAXC = 16;

// 1 / a.  |a|^2 in the normal range: hardware reciprocal approximation (rcp.approx.ftz.f64, ~2^-23) + two Newton steps
// (relative error ~1 ulp: ample for a pivot reciprocal), no IEEE division on the critical path of a pivot step
__device__ __forceinline__ cplx crecip_fast(cplx a) {
    double n = fma(a.re, a.re, a.im * a.im);
    if (n > 1e-280 && n < 1e280) {
        double r;
        asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(n));
        r = fma(r, fma(-n, r, 1.0), r);
        r = fma(r, fma(-n, r, 1.0), r);
        return make_c(a.re * r, -a.im * r);
    }
    return crecip(a);
}

// (value, position) arg-max over the lanes of a warp; ties -> lowest position.  value >= 0 or -1 (no row).
// Returns true on the single winning lane (false on all lanes if no lane has a row).
__device__ __forceinline__ bool warp_argmax(double v, int pos, double& wv, int& wp) {
    unsigned long long key = (v >= 0.0) ? ((unsigned long long)__double_as_longlong(v) + 1ull) : 0ull;
    unsigned hi = (unsigned)(key >> 32), lo = (unsigned)key;
    unsigned mh = __reduce_max_sync(0xffffffffu, hi);
    unsigned ml = __reduce_max_sync(0xffffffffu, hi == mh ? lo : 0u);
    bool cand = (hi == mh) && (lo == ml);
    unsigned mp = __reduce_min_sync(0xffffffffu, cand ? (unsigned)pos : 0xffffffffu);
    unsigned long long mk = ((unsigned long long)mh << 32) | ml;
    wv = mk ? __longlong_as_double((long long)(mk - 1ull)) : -1.0;
    wp = (int)mp;
    return cand && (unsigned)pos == mp && mk != 0ull;
}

// ---- cluster-scope mbarrier / distributed-shared-memory primitives of the fused panel kernel
__device__ __forceinline__ unsigned smem_addr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ unsigned mapa_cluster(unsigned local, int cta) {
    unsigned r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local), "r"(cta));
    return r;
}
__device__ __forceinline__ void mbar_init(unsigned bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
// 16 bytes into another CTA's shared memory; the store itself completes 16 transaction bytes on that CTA's mbarrier
// (no fence, no barrier: the receiver's mbarrier wait is the only synchronisation)
__device__ __forceinline__ void st_async_16(unsigned remote_addr, unsigned long long a, unsigned long long b, unsigned remote_bar) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.b64 [%0], {%1, %2}, [%3];"
                 ::"r"(remote_addr), "l"(a), "l"(b), "r"(remote_bar) : "memory");
}

// ---- the whole 128-column panel in ONE launch (panels of up to 4096 rows): the thread-block cluster stays resident over
// the 8 inner blocks of 16 columns instead of being re-scheduled for every one of them (4 launches per inner block before:
// leaf, row swaps, 16-row triangular solve, rank-16 update).  One thread = one matrix row for the whole panel; pivoting is
// IMPLICIT for the whole panel (no row moves until the end), with the position bookkeeping of LAPACK's sequential swaps.
// Per inner block:
//  (1) the 16 active columns of the own row -> registers;
//  (2) 16 pivot steps WITHOUT any CTA or cluster barrier, two message hops each, both by st.async with mbarrier
//      transaction counts (no arrive, no release/acquire pair, no remote load):
//        keys: every warp finds its candidate (warp arg-max of |re|+|im| with the position), stages that row in its own
//              shared memory, and lane c pushes the warp's 16-byte key into CTA c's key array (st.async.shared::cluster,
//              completing 16 transaction bytes on CTA c's key barrier of the step's parity); thread 0 of every CTA has
//              armed that barrier with expect_tx = 16 x (8 warps x csize) bytes, every thread waits on its own CTA's;
//        row:  every warp reduces the keys (per lane over its keys, then redux.sync max / min on the bit pattern); the
//              warp holding the winner PUSHES its staged row, the pivot's reciprocal and the row number to every CTA's
//              row buffer (st.async again, expect_tx = one row message on the row barrier of that parity); every thread
//              waits on its own CTA's row barrier and applies the rank-1 update to the row in its registers -- column
//              j+1 at once, the rest deferred into the wait of the next step (software pipelining).
//      Keys, row messages and both barriers are double-buffered by step parity: a warp can be at most one step ahead of
//      the slowest warp of the cluster, because the key barrier of step j+1 cannot complete without that warp's key.
//  (3) the pivot rows' remaining panel columns are read by every CTA, U12 = L11^-1 A12 is solved redundantly in shared
//      memory (one thread per column), the owners write it back;
//  (4) rank-16 update of the own row's remaining panel columns with the multipliers still in registers (four columns
//      per trip, the next four prefetched).
// At the end the rows that moved (at most 2 x 128) are carried to their final positions, 16 columns at a time through
// registers with a cluster barrier between the reads and the writes of a chunk.
constexpr int PANEL_W = 128;
// Rank-jb update of up to 32 rows (bit mask act) of one warp: x[row][col] -= sum_k L[k][row] * U[k][col], 4 rows at a time,
// lane l owns columns l + 32 t, t < NT.  L: per-warp tile [16][32], U: [16][112] (shared memory).
template <int NT>
__device__ __forceinline__ void panel_rank_update(cplx* Awarp, int ld, const cplx* Lw, const cplx* U, unsigned act, int jb,
                                                  int wrest, int lane) {
    constexpr int UW = 128 - LEAF_JB;
    while (act) {
        int rho[4]; bool on[4];
#pragma unroll
        for (int i = 0; i < 4; i++) {
            on[i] = act != 0u;
            rho[i] = on[i] ? (__ffs(act) - 1) : 0;
            if (on[i]) act &= act - 1u;
        }
        cplx x[4][NT];
#pragma unroll
        for (int i = 0; i < 4; i++)
#pragma unroll
            for (int t = 0; t < NT; t++) {
                const int col = lane + 32 * t;
                x[i][t] = (on[i] && col < wrest) ? Awarp[(long long)rho[i] * ld + col] : make_c(0.0, 0.0);
            }
#pragma unroll 4
        for (int k = 0; k < LEAF_JB; k++) {
            if (k < jb) {
                cplx l[4], u[NT];
#pragma unroll
                for (int i = 0; i < 4; i++) l[i] = Lw[k * 32 + rho[i]];
#pragma unroll
                for (int t = 0; t < NT; t++) u[t] = U[k * UW + min(lane + 32 * t, UW - 1)];
#pragma unroll
                for (int i = 0; i < 4; i++)
#pragma unroll
                    for (int t = 0; t < NT; t++) x[i][t] = cfnma(x[i][t], l[i], u[t]);
            }
        }
#pragma unroll
        for (int i = 0; i < 4; i++)
#pragma unroll
            for (int t = 0; t < NT; t++) {
                const int col = lane + 32 * t;
                if (on[i] && col < wrest) Awarp[(long long)rho[i] * ld + col] = x[i][t];
            }
    }
}

constexpr int PANEL_DYN_SMEM = (LEAF2_TPB / 32) * LEAF_JB * 32 * (int)sizeof(cplx);   // Lsm: 64 KB

#ifdef SS_PANEL_TIMING
__device__ long long ss_panel_clk[16];                    // tuning aid: accumulated clock64 deltas of CTA 0, thread 0, matrix 0
#define PCLK_BEGIN long long pclk_t = clock64(); long long pclk_acc[11] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
#define PCLK(i) { long long t1 = clock64(); pclk_acc[i] += t1 - pclk_t; pclk_t = t1; }
#define PCLK_END if (tid == 0 && crank == 0 && z == 0) { for (int i = 0; i < 11; i++) ss_panel_clk[i] += pclk_acc[i]; }
#else
#define PCLK_BEGIN
#define PCLK(i)
#define PCLK_END
#endif

__global__ void __launch_bounds__(LEAF2_TPB, 2)
lu_panel_kernel(BPtr Ab, int ld, int j0, int m, int nbw, int* __restrict__ ipiv, int ipiv_stride,
                int* __restrict__ info, int info_base, int nopiv, int* __restrict__ growth) {
    cg::cluster_group cluster = cg::this_cluster();
    const int csize = (int)cluster.num_blocks();
    const int crank = (int)cluster.block_rank();
    const int z = blockIdx.y;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NW = LEAF2_TPB / 32, JB = LEAF_JB;
    double lmax = 0.0;                                    // nopiv: largest multiplier met (growth monitor)

    constexpr int MSG = JB + 2;                                        // pivot-row message: 16 entries, 1/pivot, {physical row}
    __shared__ __align__(16) ulonglong2 keys[2][NW * LEAF2_MAXC];      // [src CTA * NW + src warp]: {value bits, position}
    __shared__ __align__(16) cplx rowmsg[2][MSG];                      // the winner's row, pushed by its warp
    __shared__ __align__(16) cplx wstage[NW][MSG];                     // every warp's candidate, staged for that push
    __shared__ __align__(16) cplx Lpiv[JB][JB];                        // row k: the k-th pivot row's active entries (multipliers | U)
    __shared__ int piv_phys[JB];                                       // its physical row inside the panel
    __shared__ __align__(16) cplx U12[JB][PANEL_W - JB];
    __shared__ __align__(8) unsigned long long bars[4];                // [0..1] keys of even / odd steps, [2..3] row messages
    extern __shared__ __align__(16) unsigned char panel_dyn[];
    cplx* Lsm = reinterpret_cast<cplx*>(panel_dyn);                    // [NW][JB][32] multipliers of the warp's rows

    cplx* A = bptr(Ab, z) + (long long)j0 * ld + j0;      // no __restrict__/const: other CTAs write rows this CTA reads
    const int r = crank * LEAF2_TPB + tid;                // my (physical) row inside the panel
    const bool valid = r < m;
    cplx* Arow = A + (long long)r * ld;
    int cur_pos = r;
    bool done = !valid;
    int final_pos = r;

    const unsigned bars_a = smem_addr(bars);
    if (tid == 0) {
        for (int i = 0; i < 4; i++) mbar_init(bars_a + 8u * i, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    cluster.sync();
    const int nkeys = NW * csize;
    const int dest = lane & (LEAF2_MAXC - 1), half = lane >> 4;        // lane -> (destination CTA, half of a message)
    const unsigned r_bars = mapa_cluster(bars_a, dest < csize ? dest : 0);
    const unsigned r_keys = mapa_cluster(smem_addr(&keys[0][crank * NW + warp]), dest < csize ? dest : 0);
    const unsigned r_rowmsg = mapa_cluster(smem_addr(&rowmsg[0][0]), dest < csize ? dest : 0);

    PCLK_BEGIN
    for (int c = 0; c < nbw; c += JB) {
        const int jb = min(JB, nbw - c), wrest = nbw - c - jb;
        cplx a[JB];
#pragma unroll
        for (int k = 0; k < JB; k++) a[k] = (valid && k < jb) ? Arow[c + k] : make_c(0.0, 0.0);
        PCLK(0)
        // Pivot steps, software-pipelined: after the pivot row of step j has arrived, only column j+1 of the own row is
        // updated before the arg-max of step j+1 starts; the rest of step j's rank-1 update (columns j+2 ..) and the staging
        // of the candidate row run while the keys of step j+1 are in flight.
        bool pend = false; cplx lp = make_c(0.0, 0.0);    // deferred part of the previous step's update: a[k] -= lp * pp[k]
        const cplx* pp = rowmsg[0];
#pragma unroll
        for (int j = 0; j < JB; j++) {
            if (j < jb) {
                const int q = c + j;                      // pivot step = position inside the panel
                const int par = j & 1;
                const unsigned ph = (unsigned)(q >> 1) & 1u;
                if (tid == 0) {                           // this step's transaction bytes: csize * NW keys, one row message
                    mbar_expect_tx(bars_a + 8u * par, 16u * (unsigned)nkeys);
                    mbar_expect_tx(bars_a + 8u * (2 + par), 16u * MSG);
                }
                double wv; int wp;
                const double myv = done ? -1.0 : (nopiv ? (cur_pos == q ? (fabs(a[j].re) + fabs(a[j].im)) : -1.0)
                                                        : (fabs(a[j].re) + fabs(a[j].im)));
                const bool iwin = warp_argmax(myv, cur_pos, wv, wp);
                if (lane < csize) {
                    const unsigned long long kb = (wv >= 0.0) ? (unsigned long long)__double_as_longlong(wv) + 1ull : 0ull;
                    st_async_16(r_keys + (unsigned)(par * sizeof(ulonglong2) * NW * LEAF2_MAXC), kb, (unsigned long long)(unsigned)wp,
                                r_bars + 8u * par);
                }
                if (pend) {                               // the previous step's update, columns j+1 .. (column j went ahead)
#pragma unroll
                    for (int k = j + 1; k < JB; k++) a[k] = cfnma(a[k], lp, pp[k]);
                }
                if (iwin) {                               // stage my row, the pivot's reciprocal and my row number
                    cplx* st = wstage[warp];
#pragma unroll
                    for (int k = 0; k < JB; k++) st[k] = a[k];
                    st[JB] = crecip_fast(a[j]);
                    st[JB + 1] = make_c(__longlong_as_double((long long)r), 0.0);
                }
                PCLK(1)
                mbar_wait(bars_a + 8u * par, ph);
                PCLK(2)
                // ---- winner among the NW * csize keys: per lane over its keys, then one redux pass
                unsigned long long bk = 0ull; unsigned bp = 0xffffffffu; int bi = 0;
                for (int i = lane; i < nkeys; i += 32) {
                    const ulonglong2 kk = keys[par][i];
                    const unsigned kp = (unsigned)kk.y;
                    if (kk.x > bk || (kk.x == bk && kk.x != 0ull && kp < bp)) { bk = kk.x; bp = kp; bi = i; }
                }
                const unsigned hi = (unsigned)(bk >> 32), lo = (unsigned)bk;
                const unsigned mh = __reduce_max_sync(0xffffffffu, hi);
                const unsigned ml = __reduce_max_sync(0xffffffffu, hi == mh ? lo : 0u);
                const bool cand = (hi == mh) && (lo == ml);
                const unsigned mp = __reduce_min_sync(0xffffffffu, cand ? bp : 0xffffffffu);
                const unsigned long long gk = ((unsigned long long)mh << 32) | ml;
                const bool have = gk != 0ull;                 // some row is left
                const bool zero_piv = (gk == 1ull);           // best |value| is exactly 0
                const unsigned wl = __ballot_sync(0xffffffffu, cand && bp == mp);
                const int widx = __shfl_sync(0xffffffffu, bi, wl ? (__ffs(wl) - 1) : 0);
                const int gp = have ? (int)mp : q;
                // ---- the warp that holds the winner pushes its staged row to every CTA (with no row left: CTA 0's warp 0
                // pushes zeros, so that the row barrier of the step completes everywhere)
                const bool pusher = have ? (widx == crank * NW + warp) : (crank == 0 && warp == 0);
                if (pusher) {
                    __syncwarp();
                    if (dest < csize) {
                        const cplx* st = wstage[warp];
#pragma unroll
                        for (int i = 0; i < MSG / 2; i++) {
                            const int e = half * (MSG / 2) + i;
                            cplx v = have ? st[e] : make_c(0.0, 0.0);
                            st_async_16(r_rowmsg + (unsigned)((par * MSG + e) * sizeof(cplx)), (unsigned long long)__double_as_longlong(v.re),
                                        (unsigned long long)__double_as_longlong(v.im), r_bars + 8u * (2 + par));
                        }
                    }
                }
                PCLK(3)
                mbar_wait(bars_a + 8u * (2 + par), ph);
                PCLK(4)
                const cplx* prow = rowmsg[par];
                if (warp == 0) {
                    if (lane < JB) Lpiv[j][lane] = prow[lane];
                    else if (lane == JB) piv_phys[j] = have ? (int)__double_as_longlong(prow[JB + 1].re) : 0;
                }
                const bool singular = !have || zero_piv;
                if (crank == 0 && tid == 0) {
                    ipiv[(long long)z * ipiv_stride + j0 + q] = j0 + gp;
                    if (singular) atomicCAS(&info[z], 0, info_base + j0 + q + 1);   // exact zero, or every candidate NaN (no key)
                }
                pend = false;
                if (!done) {
                    if (cur_pos == gp && have) {
                        done = true; final_pos = q;       // I am the pivot row: becomes row q of the panel's U
                    } else {
                        if (cur_pos == q) cur_pos = gp;   // LAPACK swap bookkeeping
                        if (!singular) {
                            cplx l = cmul(a[j], prow[JB]);
                            a[j] = l;
                            if (nopiv) lmax = fmax(lmax, fabs(l.re) + fabs(l.im));
                            if (j + 1 < JB) a[j + 1] = cfnma(a[j + 1], l, prow[j + 1]);
                            pend = true; lp = l; pp = prow;
                        }
                    }
                }
                PCLK(5)
            }
        }
        if (pend) {                                       // jb < 16 only: nothing is left to update when jb == 16
#pragma unroll
            for (int k = 0; k < JB; k++)
                if (k > jb) a[k] = cfnma(a[k], lp, pp[k]);
        }
        if (valid) {
#pragma unroll
            for (int k = 0; k < JB; k++)
                if (k < jb) Arow[c + k] = a[k];
        }
        PCLK(6)
        if (wrest > 0) {
            const int cr = c + jb;                        // first remaining column
            __syncthreads();                              // Lpiv, piv_phys (written by warp 0) complete
            // A12: the pivot rows' remaining columns (every CTA reads all of them; .cg: written by their owner CTAs)
            for (int idx = tid; idx < jb * wrest; idx += LEAF2_TPB) {
                int k = idx / wrest, cc = idx - k * wrest;
                const double2 v = __ldcg(reinterpret_cast<const double2*>(A + (long long)piv_phys[k] * ld + cr + cc));
                U12[k][cc] = make_c(v.x, v.y);
            }
            cluster.sync();                               // all CTAs have read A12 before any owner overwrites it
            PCLK(7)
            if (tid < wrest) {                            // U12 = L11^-1 A12 in place, one thread per column
                for (int k = 1; k < jb; k++) {
                    cplx acc = U12[k][tid];
                    for (int kk = 0; kk < k; kk++) acc = cfnma(acc, Lpiv[k][kk], U12[kk][tid]);
                    U12[k][tid] = acc;
                }
            }
            __syncthreads();
            for (int idx = tid; idx < jb * wrest; idx += LEAF2_TPB) {
                int k = idx / wrest, cc = idx - k * wrest;
                int pr = piv_phys[k];
                if (pr / LEAF2_TPB == crank) A[(long long)pr * ld + cr + cc] = U12[k][cc];
            }
            PCLK(8)
            // ---- A22 -= L21 U12 on the rows of this warp.  A thread walking along its own row touches 32 different cache
            // lines per warp instruction (measured: half of the whole panel time went here), so the warp works row-wise
            // instead: the multipliers go through a per-warp shared-memory tile Lsm[k][lane], then 4 rows at a time, lane
            // l owns columns l, l+32, .. of each (512-byte coalesced accesses), 4 + NT shared loads per 4 NT complex
            // multiply-adds; NT = ceil(wrest / 32) column slots, so that narrow remainders do no masked work.
            {
                cplx* Lw = Lsm + (size_t)warp * (JB * 32);
#pragma unroll
                for (int k = 0; k < JB; k++) Lw[k * 32 + lane] = a[k];
                const unsigned act = __ballot_sync(0xffffffffu, valid && !done);
                __syncwarp();
                cplx* Awarp = A + (long long)(crank * LEAF2_TPB + warp * 32) * ld + cr;
                switch ((wrest + 31) >> 5) {
                    case 1: panel_rank_update<1>(Awarp, ld, Lw, &U12[0][0], act, jb, wrest, lane); break;
                    case 2: panel_rank_update<2>(Awarp, ld, Lw, &U12[0][0], act, jb, wrest, lane); break;
                    case 3: panel_rank_update<3>(Awarp, ld, Lw, &U12[0][0], act, jb, wrest, lane); break;
                    default: panel_rank_update<4>(Awarp, ld, Lw, &U12[0][0], act, jb, wrest, lane); break;
                }
                __syncwarp();
            }
            __syncthreads();                              // U12 / Lpiv / piv_phys are rewritten by the next inner block
            PCLK(9)
        }
    }
    if (nopiv && growth) {                                // largest |l| (as |re|+|im|) of the panel -> growth[z] (float bits order like ints)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) lmax = fmax(lmax, __shfl_xor_sync(0xffffffffu, lmax, o));
        if (lane == 0 && lmax > 0.0) atomicMax(&growth[z], __float_as_int(__double2float_ru(lmax)));
    }
    // ---- carry the moved rows to their final positions
    if (!done) final_pos = cur_pos;
    const bool moved = valid && final_pos != r;
    cplx* Adst = A + (long long)final_pos * ld;
    for (int c = 0; c < nbw; c += JB) {
        cplx a[JB];
        if (moved) {
#pragma unroll
            for (int k = 0; k < JB; k++)
                if (c + k < nbw) a[k] = Arow[c + k];
        }
        cluster.sync();
        if (moved) {
#pragma unroll
            for (int k = 0; k < JB; k++)
                if (c + k < nbw) Adst[c + k] = a[k];
        }
    }
    cluster.sync();                                       // no CTA may exit while another still reads its shared memory
    PCLK(10)
    PCLK_END
}

// Apply the row interchanges ipiv[row0 .. row0+jb) to the columns [c_lo, skip_lo) U [skip_hi, c_hi) of each matrix.
// One thread per column: consecutive threads touch consecutive elements of a row (coalesced in row-major).
__global__ void __launch_bounds__(256)
laswp_kernel(BPtr Ab, int ld, int c_lo, int c_hi, int row0, int jb, int skip_lo, int skip_hi,
             const int* __restrict__ ipiv, int ipiv_stride) {
    const int z = blockIdx.y;
    int c = blockIdx.x * blockDim.x + threadIdx.x;
    const int nleft = skip_lo - c_lo;
    const int total = nleft + (c_hi - skip_hi);
    if (c >= total) return;
    c = (c >= nleft) ? skip_hi + (c - nleft) : c_lo + c;
    cplx* __restrict__ A = bptr(Ab, z);
    const int* piv = ipiv + (long long)z * ipiv_stride + row0;
    for (int j = 0; j < jb; j++) {
        int p = piv[j];
        if (p != row0 + j) {
            cplx* x = A + (long long)(row0 + j) * ld + c;
            cplx* y = A + (long long)p * ld + c;
            cplx tx = *x, ty = *y;
            *x = ty; *y = tx;
        }
    }
}

// ---- row interchanges as a permutation.  A pivot list of p entries applied swap by swap costs p dependent
// read-modify-write trips per column thread (latency-bound: the recursive LU applies up to n/2 pivots to a sibling half at
// once).  Instead: one small kernel turns ipiv[piv_lo .. piv_lo+npiv) into the permutation it amounts to (rowsrc[r] = the
// row whose content ends up in row r, plus the compact list of rows that move), then the moved rows are copied through a
// scratch buffer by two fully parallel, coalesced kernels (gather, scatter).
__global__ void __launch_bounds__(256)
perm_build_kernel(const int* __restrict__ ipiv, int ipiv_stride, int piv_lo, int npiv, int n,
                  int* __restrict__ rowsrc, int* __restrict__ moves, int* __restrict__ count) {
    extern __shared__ int perm_sh[];                  // idx[n - piv_lo], piv[npiv], counter
    const int z = blockIdx.x, nrows = n - piv_lo;
    int* idx = perm_sh;
    int* piv = perm_sh + nrows;
    int* cnt = piv + npiv;
    for (int i = threadIdx.x; i < nrows; i += blockDim.x) idx[i] = i;
    for (int j = threadIdx.x; j < npiv; j += blockDim.x) piv[j] = ipiv[(long long)z * ipiv_stride + piv_lo + j] - piv_lo;
    if (threadIdx.x == 0) *cnt = 0;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int j = 0; j < npiv; j++) {
            const int p = piv[j];
            if (p != j) { int t = idx[j]; idx[j] = idx[p]; idx[p] = t; }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < nrows; i += blockDim.x) {
        rowsrc[(long long)z * n + piv_lo + i] = piv_lo + idx[i];
        if (idx[i] != i) {
            int k = atomicAdd(cnt, 1);
            moves[((long long)z * n + k) * 2] = piv_lo + i;             // destination row
            moves[((long long)z * n + k) * 2 + 1] = piv_lo + idx[i];    // source row
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) count[z] = *cnt;
}

// dir 0: tmp[a][c] = A[src(a)][c_lo + c];  dir 1: A[dst(a)][c_lo + c] = tmp[a][c];  a = blockIdx.y-th moved row
__global__ void __launch_bounds__(256)
row_move_kernel(BPtr Ab, int ld, int c_lo, int ncols, int n, const int* __restrict__ moves, const int* __restrict__ count,
                cplx* __restrict__ tmp, long long tmp_stride, int dir) {
    const int z = blockIdx.z, a = blockIdx.y;
    if (a >= count[z]) return;
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncols) return;
    const int row = moves[((long long)z * n + a) * 2 + (dir ? 0 : 1)];
    cplx* A = bptr(Ab, z) + (long long)row * ld + c_lo + c;
    cplx* t = tmp + (long long)z * tmp_stride + (long long)a * ncols + c;
    if (dir) *A = *t; else *t = *A;
}

// dst[r][c] = src[rowsrc[r]][c] for all n rows (out of place): the right-hand-side block formed elsewhere, permuted on the way in
__global__ void __launch_bounds__(256)
row_gather_ext_kernel(BPtr Dst, int ldd, BPtr Src, int lds, int ncols, int n, const int* __restrict__ rowsrc) {
    const int z = blockIdx.z, r = blockIdx.y;
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncols) return;
    const int sr = rowsrc[(long long)z * n + r];
    bptr(Dst, z)[(long long)r * ldd + c] = bptr(Src, z)[(long long)sr * lds + c];
}

// A12 <- L11^-1 A12 for the jb x w block right of a leaf (L11 = unit lower jb x jb at (row0, row0), jb <= 16).
// One thread per column of A12.
__global__ void __launch_bounds__(128)
trsm_leaf_kernel(BPtr Ab, int ld, int row0, int jb, int c0, int w) {
    __shared__ cplx L[LEAF_JB][LEAF_JB];
    const int z = blockIdx.y;
    cplx* __restrict__ A = bptr(Ab, z);
    for (int i = threadIdx.x; i < jb * jb; i += blockDim.x) {
        int rr = i / jb, cc = i % jb;
        L[rr][cc] = A[(long long)(row0 + rr) * ld + row0 + cc];
    }
    __syncthreads();
    int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= w) return;
    cplx x[LEAF_JB];
#pragma unroll
    for (int rr = 0; rr < LEAF_JB; rr++)
        if (rr < jb) x[rr] = A[(long long)(row0 + rr) * ld + c0 + c];
#pragma unroll
    for (int rr = 1; rr < LEAF_JB; rr++) {
        if (rr < jb) {
            cplx s = x[rr];
#pragma unroll
            for (int k = 0; k < LEAF_JB; k++)
                if (k < rr) s = cfnma(s, L[rr][k], x[k]);
            x[rr] = s;
        }
    }
#pragma unroll
    for (int rr = 1; rr < LEAF_JB; rr++)
        if (rr < jb) A[(long long)(row0 + rr) * ld + c0 + c] = x[rr];
}

// Inverse of an nt x nt (nt <= 128) triangular block T (row-major, ld) into Tinv (row-major, ldo = 128-padded):
// lower (unit or not) or upper.  16x16 blocked forward substitution, one CTA (256 threads) per (block column, matrix):
// the 8 diagonal 16x16 blocks are inverted up front (one thread per block column of each), the off-diagonal block rows
// are prefetched one step ahead, every step is two 16x16 products out of shared memory.
// Upper is handled as the index-reversed lower problem.  Everything outside the triangle of Tinv (up to the
// padded size pad) is written as zero, the padded diagonal as one.
struct TrtriArgs {
    BPtr T; int ld;            // source matrices
    long long t_step;          // element offset between consecutive diagonal blocks of one matrix (blockIdx.y)
    int n_total;               // order of the whole triangular matrix (diag block y has min(128, n_total - 128 y) rows)
    cplx* out;                 // [batch][nblocks][128*128]
    int nblocks;
    int upper, unit;
};

__global__ void __launch_bounds__(256)
trtri_kernel(TrtriArgs p) {
    constexpr int B = 16, NBK = 8, P = 128;
    extern __shared__ __align__(16) unsigned char trtri_smem[];
    typedef cplx Tile[B][B + 1];
    Tile* X = reinterpret_cast<Tile*>(trtri_smem);          // [NBK] inverse blocks of my block column
    Tile* Di = X + NBK;                                     // [NBK] first the diagonal blocks, then their inverses
    Tile* Lr = Di + NBK;                                    // [NBK-1] block row ib of the matrix, columns jbk .. ib-1
    Tile& S = *(Lr + (NBK - 1));
    const int jbk = blockIdx.x, yb = blockIdx.y, z = blockIdx.z;
    const int nt = min(P, p.n_total - P * yb);
    const cplx* __restrict__ T = bptr(p.T, z) + (long long)yb * p.t_step;
    cplx* __restrict__ O = p.out + ((long long)z * p.nblocks + yb) * (P * P);
    const int tid = threadIdx.x, tr = tid / B, tc = tid % B;
    const int upper = p.upper, unit = p.unit;
    // element (i, j) of the (index-reversed if upper) lower-triangular matrix, identity-padded to 128
    auto elem = [&](int i, int j) -> cplx {
        if (i >= nt || j >= nt) return make_c(i == j ? 1.0 : 0.0, 0.0);
        if (j > i) return make_c(0.0, 0.0);
        if (unit && i == j) return make_c(1.0, 0.0);
        int ii = upper ? nt - 1 - i : i, jj = upper ? nt - 1 - j : j;
        return T[(long long)ii * p.ld + jj];
    };
    // ---- all diagonal blocks jbk .. 7 at once: load, then one thread per (block, column) inverts by substitution
    for (int bk = jbk; bk < NBK; bk++) Di[bk][tr][tc] = elem(bk * B + tr, bk * B + tc);
    cplx pre[NBK - 1];                     // prefetch of block row jbk + 1
#pragma unroll
    for (int kb = 0; kb < NBK - 1; kb++)
        pre[kb] = (jbk + 1 < NBK && jbk + kb < jbk + 1) ? elem((jbk + 1) * B + tr, (jbk + kb) * B + tc) : make_c(0.0, 0.0);
    __syncthreads();
    {
        const int bk = jbk + tid / B, c = tid % B;
        cplx x[B];
#pragma unroll
        for (int i = 0; i < B; i++) x[i] = make_c(0.0, 0.0);
        if (bk < NBK) {
#pragma unroll
            for (int i = 0; i < B; i++) {
                if (i >= c) {
                    cplx s = make_c(i == c ? 1.0 : 0.0, 0.0);
#pragma unroll
                    for (int k = 0; k < B; k++)
                        if (k >= c && k < i) s = cfnma(s, Di[bk][i][k], x[k]);
                    x[i] = cmul(s, crecip(Di[bk][i][i]));
                }
            }
        }
        __syncthreads();                   // everyone has read the blocks: overwrite them with the inverses
        if (bk < NBK) {
#pragma unroll
            for (int i = 0; i < B; i++) Di[bk][i][c] = x[i];
        }
    }
    __syncthreads();
    X[jbk][tr][tc] = Di[jbk][tr][tc];
    // ---- block forward substitution down my block column; block row ib + 1 is prefetched while row ib is used
    for (int ib = jbk + 1; ib < NBK; ib++) {
        const int nk = ib - jbk;
#pragma unroll
        for (int kb = 0; kb < NBK - 1; kb++)
            if (kb < nk) Lr[kb][tr][tc] = pre[kb];
        if (ib + 1 < NBK) {
#pragma unroll
            for (int kb = 0; kb < NBK - 1; kb++)
                if (kb < nk + 1) pre[kb] = elem((ib + 1) * B + tr, (jbk + kb) * B + tc);
        }
        __syncthreads();
        cplx s0 = make_c(0.0, 0.0), s1 = make_c(0.0, 0.0);
        for (int kb = 0; kb < nk; kb++) {
#pragma unroll
            for (int k = 0; k < B; k += 2) {
                s0 = cfma(s0, Lr[kb][tr][k], X[jbk + kb][k][tc]);
                s1 = cfma(s1, Lr[kb][tr][k + 1], X[jbk + kb][k + 1][tc]);
            }
        }
        S[tr][tc] = make_c(s0.re + s1.re, s0.im + s1.im);
        __syncthreads();
        cplx o0 = make_c(0.0, 0.0), o1 = make_c(0.0, 0.0);
#pragma unroll
        for (int k = 0; k < B; k += 2) {
            o0 = cfnma(o0, Di[ib][tr][k], S[k][tc]);
            o1 = cfnma(o1, Di[ib][tr][k + 1], S[k + 1][tc]);
        }
        X[ib][tr][tc] = make_c(o0.re + o1.re, o0.im + o1.im);
        // the next iteration's first barrier orders these writes before anyone reads X[ib] or rewrites Lr / S
    }
    __syncthreads();
    // write block column jbk of the inverse (zeros above the diagonal blocks), undoing the index reversal.
    // Reversal applies to the nt x nt part only; the identity padding stays in place.
    for (int ib = 0; ib < NBK; ib++) {
        int i = ib * B + tr, j = jbk * B + tc;
        cplx v = (ib >= jbk) ? X[ib][tr][tc] : make_c(0.0, 0.0);
        int oi = i, oj = j;
        if (upper && i < nt && j < nt) { oi = nt - 1 - i; oj = nt - 1 - j; }
        if (upper && ((i < nt) != (j < nt))) v = make_c(0.0, 0.0);
        O[(long long)oi * P + oj] = v;
    }
}

constexpr int TRTRI_SMEM = (8 + 8 + 7 + 1) * 16 * 17 * (int)sizeof(cplx);

static void launch_trtri(cudaStream_t st, const TrtriArgs& t, int yblocks, int batch) {
    static bool configured = false;
    if (!configured) {
        cudaFuncSetAttribute(trtri_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, TRTRI_SMEM);
        configured = true;
    }
    trtri_kernel<<<dim3(8, (unsigned)yblocks, (unsigned)batch), 256, TRTRI_SMEM, st>>>(t);
}

// ---------------------------------------------------------------------------------------------------------
// host drivers
// ---------------------------------------------------------------------------------------------------------
struct GemmProfile {                 // optional per-launch CUDA-event timing of the GEMM kernel (bench.py's roofline)
    std::vector<cudaEvent_t> ev;     // pairs: start, stop
    size_t used = 0;                 // events used by the last solve
    double flops = 0.0;              // 8 M N K batch summed over the timed launches
    long long launches = 0;
};

// Launch context of one group of chains.  With stream groups (splitsolve.cu) every group owns two streams: a
// HIGH-priority one for the short latency-bound kernels of the panel factorisation (leaf, row swaps, small
// triangular solves and inverses, rank-16 updates) and a LOW-priority one for the large GEMMs, so that one group's
// panel runs in the shadow of another group's GEMMs (the block scheduler places pending high-priority CTAs first).
// use() moves the launch point between the two, ordering them with an event.  Without groups both are the caller's
// stream and use() does nothing.
enum { CLS_LO = 0, CLS_HI = 1 };
struct TraceRec { int group, cls; cudaEvent_t t0, t1; };      // one phase of one group (option "trace")
struct Ctx {
    std::vector<TraceRec>* trace = nullptr;
    int group = 0;
    void trace_open() {
        if (!trace) return;
        TraceRec r{group, cls, nullptr, nullptr};
        cudaEventCreate(&r.t0); cudaEventCreate(&r.t1);
        cudaEventRecord(r.t0, st);
        trace->push_back(r);
    }
    void trace_close() {
        if (!trace) return;
        for (size_t i = trace->size(); i-- > 0;)
            if ((*trace)[i].group == group) { cudaEventRecord((*trace)[i].t1, st); break; }
    }
    cudaStream_t st = nullptr;
    cudaStream_t s_hi = nullptr, s_lo = nullptr;
    cudaEvent_t ev_sw = nullptr;
    int cls = CLS_LO;
    long long launches = 0;
    cudaError_t err = cudaSuccess;
    GemmProfile* prof = nullptr;
    int variant = GV_4M;            // GEMM arithmetic / tile variant (zgemm3m.cuh)
    void note(cudaError_t e) { if (err == cudaSuccess && e != cudaSuccess) err = e; launches++; }
    void use(int c) {
        if (c == cls) return;
        if (!ev_sw) { trace_close(); cls = c; trace_open(); return; }      // single stream: phases only marked
        cudaStream_t to = (c == CLS_HI) ? s_hi : s_lo;
        trace_close();
        cudaError_t e = cudaEventRecord(ev_sw, st);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(to, ev_sw, 0);
        if (err == cudaSuccess && e != cudaSuccess) err = e;
        st = to; cls = c;
        trace_open();
    }
};

static void gemm_run(Ctx& ctx, const GemmArgs& g, int batch, int cfg, int epi) {
    GemmProfile* pr = ctx.prof;
    if (pr && g.M > 0 && g.N > 0 && batch > 0) {
        if (pr->used + 2 > pr->ev.size()) {
            cudaEvent_t a, b;
            if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) { ctx.note(cudaErrorMemoryAllocation); return; }
            pr->ev.push_back(a); pr->ev.push_back(b);
        }
        cudaEventRecord(pr->ev[pr->used], ctx.st);
        ctx.note(gemm_launch(g, batch, cfg, epi, ctx.st, ctx.variant));
        cudaEventRecord(pr->ev[pr->used + 1], ctx.st);
        pr->used += 2;
        double area = (double)g.M * g.N;
        if (g.tri) {                                      // only the tiles that touch the lower triangle are computed
            const int BM = 64, BN = (ctx.variant == GV_4M) ? 64 : 32;
            area = 0.0;
            for (int m0 = 0; m0 < g.M; m0 += BM)
                for (int n0 = 0; n0 < g.N; n0 += BN)
                    if (n0 + g.tri_col0 <= m0 + BM - 1 + g.tri_row0) area += (double)min(BM, g.M - m0) * min(BN, g.N - n0);
        }
        pr->flops += 8.0 * area * g.K * batch;
        pr->launches++;
    } else {
        ctx.note(gemm_launch(g, batch, cfg, epi, ctx.st, ctx.variant));
    }
}

struct LuWork {
    cplx* tinv = nullptr;       // [batch][2 * nblk(n)][128*128]: inverses of the 128 x 128 diagonal blocks of L, then of U
    int* ipiv = nullptr;        // [batch][ipiv_stride]
    int ipiv_stride = 0;
    int* info = nullptr;        // [batch]
    int* growth = nullptr;      // [batch] no-pivot factorisation: float bits of the largest multiplier (|re|+|im|) met
    int* perm = nullptr;        // [batch][3 n + 4] ints: rowsrc [batch][n], moves [batch][2n], count [batch]
    cplx* tmp = nullptr;        // [batch][tmp_elems] scratch of the row moves
    long long tmp_elems = 0;    // per matrix
};
static inline int lu_nblk(int n) { return (n + 127) / 128; }
static inline size_t lu_tinv_elems(int n, int batch) { return (size_t)2 * lu_nblk(n) * 128 * 128 * (size_t)batch; }
static inline size_t lu_perm_ints(int n, int batch) { return ((size_t)batch * (3 * (size_t)n + 1) + 3) / 4 * 4; }
static inline long long lu_tmp_elems_default(int n) { return (long long)n * (((n + 1) / 2 + 127) / 128 * 128); }

static inline GemmArgs gemm_std(int M, int N, int K, double alpha, BPtr A, int lda, BPtr B, int ldb, double beta,
                                BPtr C, int ldc) {
    GemmArgs g{};
    g.M = M; g.N = N; g.K = K; g.A = A; g.lda = lda; g.B = B; g.ldb = ldb; g.C = C; g.ldc = ldc;
    g.Cin = C; g.ldcin = ldc; g.alpha = alpha; g.beta = beta; g.E = nullptr;
    return g;
}

// The 16-column leaf kernel (512 rows per CTA, cluster of up to 16 CTAs): panels of more than 4096 rows only
static void launch_leaf(Ctx& ctx, BPtr Ab, int ld, int row0, int col0, int m, int jb, const LuWork& w, int info_base,
                        int batch) {
    static bool configured = false;
    if (!configured) {
        cudaFuncSetAttribute(lu_leaf_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        configured = true;
    }
    int need = (m + LEAF_TPB - 1) / LEAF_TPB, csize = 1;
    while (csize < need) csize <<= 1;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)csize, (unsigned)batch, 1);
    cfg.blockDim = dim3((unsigned)LEAF_TPB, 1, 1);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = ctx.st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)csize;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    ctx.note(cudaLaunchKernelEx(&cfg, lu_leaf_kernel, Ab, ld, row0, col0, m, jb, w.ipiv, w.ipiv_stride, w.info, info_base));
}

// ---------------------------------------------------------------------------------------------------------
// LU with partial pivoting of the leading n x n part of the n x ncols matrices (row-major, ld); the interchanges and the
// L-solve are applied to the trailing ncols - n columns too.  n <= LEAF_TPB * LEAF_MAXC.
//
// Recursive over column ranges (Toledo's recursive LU down to 128-column panels), so that the O(n^3) work runs in GEMMs
// with long K instead of rank-128 trailing updates:
//     rlu([c0, c1)):  rlu(left half) -> swaps on the right half -> A12 = L11^-1 A12 -> A22 -= A21 A12 (K = width of the
//     left half) -> rlu(right half) -> swaps on the left half.
// Triangular solves are left-looking over 128-row blocks with explicit inverses of the 128 x 128 diagonal blocks
// (trtri_kernel, one per panel), so they are GEMMs with K growing from 128 to the size of the triangle:
//     X_k = L_kk^-1 (A_k - L_{k,<k} X_{<k}).
// The right-hand-side columns [n, ncols) get all n interchanges at the end, then one left-looking L-solve.
// ---------------------------------------------------------------------------------------------------------
struct LuCall {
    Ctx& ctx; BPtr Ab; int ld, n, ncols, batch; const LuWork& w; int info_base;
    int nblk() const { return lu_nblk(n); }
    BPtr tinvL(int blk) const { return bp_strided(w.tinv + (long long)blk * 128 * 128, 2LL * nblk() * 128 * 128); }
    BPtr tinvU(int blk) const { return bp_strided(w.tinv + (long long)(nblk() + blk) * 128 * 128, 2LL * nblk() * 128 * 128); }
};

static void lu_perm_build(const LuCall& L, int piv_lo, int piv_hi) {
    static bool configured = false;
    if (!configured) {
        cudaFuncSetAttribute(perm_build_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 80 * 1024);   // n, npiv <= 8192: (2 * 8192 + 1) ints
        configured = true;
    }
    const int n = L.n, npiv = piv_hi - piv_lo;
    int* rowsrc = L.w.perm;
    int* moves = rowsrc + (long long)L.batch * n;
    int* count = moves + 2LL * L.batch * n;
    const size_t sh = sizeof(int) * ((size_t)(n - piv_lo) + npiv + 1);
    perm_build_kernel<<<L.batch, 256, sh, L.ctx.st>>>(L.w.ipiv, L.w.ipiv_stride, piv_lo, npiv, n, rowsrc, moves, count);
    L.ctx.note(cudaGetLastError());
}

// Apply the interchanges ipiv[piv_lo .. piv_hi) to the columns [c_lo, skip_lo) U [skip_hi, c_hi).
static void lu_swaps(const LuCall& L, int piv_lo, int piv_hi, int c_lo, int c_hi, int skip_lo, int skip_hi) {
    const int total = (skip_lo - c_lo) + (c_hi - skip_hi);
    const int npiv = piv_hi - piv_lo;
    if (total <= 0 || npiv <= 0) return;
    if (npiv <= 32 || !L.w.perm || !L.w.tmp) {                 // short list: swap by swap
        dim3 grid((unsigned)((total + 255) / 256), (unsigned)L.batch);
        laswp_kernel<<<grid, 256, 0, L.ctx.st>>>(L.Ab, L.ld, c_lo, c_hi, piv_lo, npiv, skip_lo, skip_hi, L.w.ipiv, L.w.ipiv_stride);
        L.ctx.note(cudaGetLastError());
        return;
    }
    lu_perm_build(L, piv_lo, piv_hi);
    const int n = L.n;
    const int* moves = L.w.perm + (long long)L.batch * n;
    const int* count = moves + 2LL * L.batch * n;
    const int cap = min(2 * npiv, n - piv_lo);                 // rows that can move
    const int ranges[2][2] = {{c_lo, skip_lo}, {skip_hi, c_hi}};
    for (int q = 0; q < 2; q++) {
        long long chunk = L.w.tmp_elems / cap;
        if (chunk >= 32) chunk = chunk / 32 * 32;
        if (chunk < 1) chunk = 1;
        for (int c0 = ranges[q][0]; c0 < ranges[q][1]; c0 += (int)chunk) {
            const int nc = (int)min((long long)(ranges[q][1] - c0), chunk);
            dim3 grid((unsigned)((nc + 255) / 256), (unsigned)cap, (unsigned)L.batch);
            for (int dir = 0; dir < 2; dir++) {
                row_move_kernel<<<grid, 256, 0, L.ctx.st>>>(L.Ab, L.ld, c0, nc, n, moves, count, L.w.tmp, L.w.tmp_elems, dir);
                L.ctx.note(cudaGetLastError());
            }
        }
    }
}

static void launch_panel_fused(Ctx& ctx, BPtr Ab, int ld, int j0, int m, int nbw, const LuWork& w, int info_base, int batch,
                               int nopiv = 0) {
    static bool configured = false;
    if (!configured) {
        cudaFuncSetAttribute(lu_panel_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        cudaFuncSetAttribute(lu_panel_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, PANEL_DYN_SMEM);
        configured = true;
    }
    int need = (m + LEAF2_TPB - 1) / LEAF2_TPB, csize = 1;
    while (csize < need) csize <<= 1;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)csize, (unsigned)batch, 1);
    cfg.blockDim = dim3((unsigned)LEAF2_TPB, 1, 1);
    cfg.dynamicSmemBytes = PANEL_DYN_SMEM;
    cfg.stream = ctx.st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)csize;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    ctx.note(cudaLaunchKernelEx(&cfg, lu_panel_kernel, Ab, ld, j0, m, nbw, w.ipiv, w.ipiv_stride, w.info, info_base, nopiv, w.growth));
}

// Panel of nbw <= 128 columns at (j0, j0), rows j0 .. n-1, swaps applied inside the panel only; then the inverse of its
// unit-lower 128 x 128 block for the solves that follow.  Up to 4096 rows: one fused launch (lu_panel_kernel); above
// (the 2bs corner system at bs > 2048): inner blocks of 16 columns by separate launches (leaf kernel, row swaps,
// 16-row triangular solve, rank-16 GEMM).
static void lu_panel(const LuCall& L, int j0, int nbw) {
    Ctx& ctx = L.ctx;
    ctx.use(CLS_HI);
    if (L.n - j0 <= LEAF2_TPB * LEAF2_MAXC) {
        launch_panel_fused(ctx, L.Ab, L.ld, j0, L.n - j0, nbw, L.w, L.info_base, L.batch);
    } else {
        for (int c = j0; c < j0 + nbw; c += LEAF_JB) {
            const int jb = min(LEAF_JB, j0 + nbw - c);
            const int m = L.n - c;
            launch_leaf(ctx, L.Ab, L.ld, c, c, m, jb, L.w, L.info_base, L.batch);
            lu_swaps(L, c, c + jb, j0, j0 + nbw, c, c + jb);
            const int wcols = j0 + nbw - (c + jb);
            if (wcols > 0) {
                dim3 grid((unsigned)((wcols + 127) / 128), (unsigned)L.batch);
                trsm_leaf_kernel<<<grid, 128, 0, ctx.st>>>(L.Ab, L.ld, c, jb, c + jb, wcols);
                ctx.note(cudaGetLastError());
                if (m - jb > 0) {
                    GemmArgs g = gemm_std(m - jb, wcols, jb, -1.0, bp_offset(L.Ab, (long long)(c + jb) * L.ld + c), L.ld,
                                          bp_offset(L.Ab, (long long)c * L.ld + c + jb), L.ld, 1.0,
                                          bp_offset(L.Ab, (long long)(c + jb) * L.ld + c + jb), L.ld);
                    gemm_run(ctx, g, L.batch, GEMM_BIG, EPI_STD);
                }
            }
        }
    }
    TrtriArgs t{};
    t.T = bp_offset(L.Ab, (long long)j0 * L.ld + j0); t.ld = L.ld; t.t_step = 0; t.n_total = nbw;
    t.out = L.w.tinv + (long long)(j0 / 128) * 128 * 128; t.nblocks = 2 * L.nblk(); t.upper = 0; t.unit = 1;
    launch_trtri(ctx.st, t, 1, L.batch);
    ctx.note(cudaGetLastError());
}

// A[r0:r1, ca:cb] <- L[r0:r1, r0:r1]^-1 A[r0:r1, ca:cb], L = unit lower factor in place; r0 a multiple of 128.
static void lu_trsm_lower(const LuCall& L, int r0, int r1, int ca, int cb) {
    if (cb <= ca) return;
    Ctx& ctx = L.ctx;
    ctx.use(CLS_LO);
    for (int k = r0; k < r1; k += 128) {
        const int nk = min(128, r1 - k);
        BPtr Ak = bp_offset(L.Ab, (long long)k * L.ld + ca);
        if (k > r0) {
            GemmArgs g = gemm_std(nk, cb - ca, k - r0, -1.0, bp_offset(L.Ab, (long long)k * L.ld + r0), L.ld,
                                  bp_offset(L.Ab, (long long)r0 * L.ld + ca), L.ld, 1.0, Ak, L.ld);
            gemm_run(ctx, g, L.batch, GEMM_BIG, EPI_STD);
        }
        GemmArgs g2 = gemm_std(nk, cb - ca, nk, 1.0, L.tinvL(k / 128), 128, Ak, L.ld, 0.0, Ak, L.ld);
        gemm_run(ctx, g2, L.batch, GEMM_TALL, EPI_STD);
    }
}

static void lu_recursive(const LuCall& L, int c0, int c1) {
    const int wd = c1 - c0;
    if (wd <= 128) { lu_panel(L, c0, wd); return; }
    const int mid = c0 + ((wd / 2 + 127) / 128) * 128;
    lu_recursive(L, c0, mid);
    L.ctx.use(CLS_HI);
    lu_swaps(L, c0, mid, mid, c1, mid, mid);
    lu_trsm_lower(L, c0, mid, mid, c1);
    if (L.n > mid) {
        GemmArgs u = gemm_std(L.n - mid, c1 - mid, mid - c0, -1.0, bp_offset(L.Ab, (long long)mid * L.ld + c0), L.ld,
                              bp_offset(L.Ab, (long long)c0 * L.ld + mid), L.ld, 1.0,
                              bp_offset(L.Ab, (long long)mid * L.ld + mid), L.ld);
        L.ctx.use(CLS_LO);
        gemm_run(L.ctx, u, L.batch, GEMM_BIG, EPI_STD);
    }
    lu_recursive(L, mid, c1);
    L.ctx.use(CLS_HI);
    lu_swaps(L, mid, c1, c0, mid, mid, mid);
}

// Bext (optional): the right-hand-side block lives elsewhere ((n x (ncols - n)), leading dimension ldb) and is copied into
// columns [n, ncols) with the rows already permuted, instead of being swapped in place.
static void lu_factor(Ctx& ctx, BPtr Ab, int ld, int n, int ncols, int batch, const LuWork& w, int info_base,
                      const BPtr* Bext = nullptr, int ldb = 0) {
    LuCall L{ctx, Ab, ld, n, ncols, batch, w, info_base};
    lu_recursive(L, 0, n);
    if (ncols > n) {
        ctx.use(CLS_HI);
        if (Bext && w.perm) {
            lu_perm_build(L, 0, n);
            dim3 grid((unsigned)((ncols - n + 255) / 256), (unsigned)n, (unsigned)batch);
            row_gather_ext_kernel<<<grid, 256, 0, ctx.st>>>(bp_offset(Ab, n), ld, *Bext, ldb, ncols - n, n, w.perm);
            ctx.note(cudaGetLastError());
        } else {
            lu_swaps(L, 0, n, n, ncols, ncols, ncols);
        }
        lu_trsm_lower(L, 0, n, n, ncols);
    }
}

// ---------------------------------------------------------------------------------------------------------
// Hermitian D (A = E S - H at real E) factored WITHOUT pivoting as L Delta L^H -- the paper's
// zhesv_nopiv_gpu (L266: 241 -> 228 TFLOP per energy point) -- at half the flops of the LU: only the lower triangle of D
// is read and updated (lower-triangle-only GEMMs), U = Delta L^H is written into the upper triangle panel by panel, so the
// result has the same [L \ U] layout as lu_factor (ipiv = identity) and the solves that follow are shared.
//     rec([c0, c1)):  rec(left half) -> lower(A22) -= L21 U12 (K = width of the left half) -> rec(right half)
//     panel (<= 128 columns): upper triangle of the diagonal block filled from the lower one; lu_panel_kernel with the
//     pivot search switched off (the diagonal row is the only candidate), which also records the largest multiplier met
//     (growth monitor); L11^-1; U12 = Delta L21^H (scaled conjugate transpose of the panel's sub-diagonal part).
// Panels of more than 4096 rows are not supported here (the caller uses the pivoted LU there).
// ---------------------------------------------------------------------------------------------------------
static void launch_mirror(Ctx& ctx, BPtr Ab, int ld, int rs, int cs, int nr, int nc, int scaled, int strict, int batch) {
    if (nr <= 0 || nc <= 0) return;
    dim3 grid((unsigned)((nc + 31) / 32), (unsigned)((nr + 31) / 32), (unsigned)batch);
    herm_mirror_kernel<<<grid, 256, 0, ctx.st>>>(Ab, ld, rs, cs, nr, nc, scaled, strict);
    ctx.note(cudaGetLastError());
}

static void herm_recursive(const LuCall& L, int c0, int c1) {
    Ctx& ctx = L.ctx;
    const int wd = c1 - c0;
    if (wd <= 128) {
        ctx.use(CLS_HI);
        launch_mirror(ctx, L.Ab, L.ld, c0, c0, wd, wd, 0, 1, L.batch);
        launch_panel_fused(ctx, L.Ab, L.ld, c0, L.n - c0, wd, L.w, L.info_base, L.batch, 1);
        TrtriArgs t{};
        t.T = bp_offset(L.Ab, (long long)c0 * L.ld + c0); t.ld = L.ld; t.t_step = 0; t.n_total = wd;
        t.out = L.w.tinv + (long long)(c0 / 128) * 128 * 128; t.nblocks = 2 * L.nblk(); t.upper = 0; t.unit = 1;
        launch_trtri(ctx.st, t, 1, L.batch);
        ctx.note(cudaGetLastError());
        launch_mirror(ctx, L.Ab, L.ld, c0 + wd, c0, L.n - c0 - wd, wd, 1, 0, L.batch);
        return;
    }
    const int mid = c0 + ((wd / 2 + 127) / 128) * 128;
    herm_recursive(L, c0, mid);
    if (L.n > mid) {
        GemmArgs u = gemm_std(L.n - mid, c1 - mid, mid - c0, -1.0, bp_offset(L.Ab, (long long)mid * L.ld + c0), L.ld,
                              bp_offset(L.Ab, (long long)c0 * L.ld + mid), L.ld, 1.0,
                              bp_offset(L.Ab, (long long)mid * L.ld + mid), L.ld);
        u.tri = 1; u.tri_row0 = mid; u.tri_col0 = mid;
        ctx.use(CLS_LO);
        gemm_run(ctx, u, L.batch, GEMM_BIG, EPI_STD);
    }
    herm_recursive(L, mid, c1);
}

// Same contract as lu_factor for Hermitian leading n x n parts given by their LOWER triangle (n <= 4096); no interchanges.
static void lu_factor_herm(Ctx& ctx, BPtr Ab, int ld, int n, int ncols, int batch, const LuWork& w, int info_base) {
    LuCall L{ctx, Ab, ld, n, ncols, batch, w, info_base};
    herm_recursive(L, 0, n);
    if (ncols > n) lu_trsm_lower(L, 0, n, n, ncols);
}

// X = U^-1 Y with U = upper factor in AB[:, 0:n], Y = AB[:, n:n+nrhs] (overwritten).  Left-looking over block rows.
static void back_substitute(Ctx& ctx, BPtr Ab, int ld, int n, int nrhs, BPtr X, int ldx, int batch, const LuWork& w) {
    if (nrhs <= 0 || n <= 0) return;
    const int P = 128;
    LuCall L{ctx, Ab, ld, n, n + nrhs, batch, w, 0};
    const int nblk = L.nblk();
    TrtriArgs t{};
    t.T = Ab; t.ld = ld; t.t_step = (long long)P * ld + P; t.n_total = n; t.out = w.tinv + (long long)nblk * P * P; t.nblocks = 2 * nblk;
    t.upper = 1; t.unit = 0;
    ctx.use(CLS_HI);
    launch_trtri(ctx.st, t, nblk, batch);
    ctx.note(cudaGetLastError());
    ctx.use(CLS_LO);
    for (int jb = nblk - 1; jb >= 0; jb--) {
        const int j = jb * P, nbj = min(P, n - j), kk = n - j - nbj;
        BPtr Yj = bp_offset(Ab, (long long)j * ld + n);
        if (kk > 0) {
            GemmArgs g = gemm_std(nbj, nrhs, kk, -1.0, bp_offset(Ab, (long long)j * ld + j + nbj), ld,
                                  bp_offset(X, (long long)(j + nbj) * ldx), ldx, 1.0, Yj, ld);
            gemm_run(ctx, g, batch, GEMM_BIG, EPI_STD);
        }
        GemmArgs g2 = gemm_std(nbj, nrhs, nbj, 1.0, L.tinvU(jb), P, Yj, ld, 0.0, bp_offset(X, (long long)j * ldx), ldx);
        gemm_run(ctx, g2, batch, GEMM_BIG, EPI_STD);
    }
}

}  // namespace ss
