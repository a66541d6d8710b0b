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
#include <vector>
#include "zgemm3m.cuh"

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

// ---- helpers of the second leaf panel kernel (lu_leaf3_kernel below): 256 rows per CTA, cluster of up to 16 CTAs = 4096
// rows.  Warp arg-max by three redux.sync on the bit pattern of |re|+|im| (non-negative doubles order like unsigned
// integers) and the row position.
constexpr int LEAF2_TPB = 256;
constexpr int LEAF2_MAXC = 16;

__device__ __forceinline__ cplx crecip_fast(cplx a) {
    double n = fma(a.re, a.re, a.im * a.im);
    if (n > 1e-280 && n < 1e280) {
        double r = 1.0 / n;
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

// ---- leaf panel for up to 4096 rows: one thread = one row, 16 columns in registers, sized to run in the shadow of the
// GEMM kernel of other stream groups (256 threads x 80 registers = one GEMM CTA slot).  Per column: the warp winner
// deposits (value, position, row) in shared memory; warp 0 picks the CTA winner and pushes only its 16-byte key (value,
// position, warp slot) to every CTA of the cluster (distributed shared memory); one cluster barrier; each warp finds the
// global winner with one redux pass over the keys and warp 0 PULLS the winner's row (16 x 16 B) out of the winning
// CTA's shared memory; rank-1 update in registers.  Measured 2.7 (4 CTAs) - 4.3 (16 CTAs) us per column against 4.9 - 9.0
// for lu_leaf_kernel, which remains for panels of more than 4096 rows (the 2bs corner system at bs = 4096).
struct LeafKey { double val; int pos; int warp; };

__global__ void __launch_bounds__(LEAF2_TPB, 3)
lu_leaf3_kernel(BPtr Ab, int ld, int row0, int col0, int m, int jb, int* __restrict__ ipiv, int ipiv_stride,
                int* __restrict__ info, int info_base) {
    cg::cluster_group cluster = cg::this_cluster();
    const int csize = (int)cluster.num_blocks();
    const int crank = (int)cluster.block_rank();
    const int z = blockIdx.y;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NW = LEAF2_TPB / 32;

    __shared__ __align__(16) LeafCand wcand[2][NW];
    __shared__ __align__(16) LeafKey keys[2][LEAF2_MAXC];
    __shared__ __align__(16) cplx prow[LEAF_JB];

    cplx* __restrict__ A = bptr(Ab, z) + (long long)row0 * ld + col0;
    const int r = crank * LEAF2_TPB + tid;       // my row inside the panel
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
            const int par = j & 1;
            double wv; int wp;
            const double myv = done ? -1.0 : (fabs(a[j].re) + fabs(a[j].im));
            if (warp_argmax(myv, cur_pos, wv, wp)) {
                LeafCand* c = &wcand[par][warp];
                c->val = myv; c->pos = cur_pos;
#pragma unroll
                for (int k = 0; k < LEAF_JB; k++) c->row[k] = a[k];
            }
            if (lane == 0 && wv < 0.0) { wcand[par][warp].val = -1.0; wcand[par][warp].pos = 0x7fffffff; }
            __syncthreads();
            if (warp == 0) {
                double v2 = lane < NW ? wcand[par][lane].val : -1.0;
                int p2 = lane < NW ? wcand[par][lane].pos : 0x7fffffff;
                double cv; int cp;
                bool win = warp_argmax(v2, p2, cv, cp);
                unsigned bal = __ballot_sync(0xffffffffu, win);
                LeafKey k; k.val = cv; k.pos = cp; k.warp = bal ? (__ffs(bal) - 1) : 0;
                if (lane < csize) *cluster.map_shared_rank(&keys[par][crank], lane) = k;
            }
            cluster.sync();
            // ---- winner among the csize keys (every warp, one redux pass)
            double kv = -1.0; int kp = 0x7fffffff, kw = 0;
            if (lane < csize) { LeafKey k = keys[par][lane]; kv = k.val; kp = k.pos; kw = k.warp; }
            double gv; int gp;
            bool gwin = warp_argmax(kv, kp, gv, gp);
            unsigned gbal = __ballot_sync(0xffffffffu, gwin);
            const int wcta = gbal ? (__ffs(gbal) - 1) : 0;
            const int wslot = __shfl_sync(0xffffffffu, kw, wcta);
            if (warp == 0 && lane < LEAF_JB && gv >= 0.0)
                prow[lane] = cluster.map_shared_rank(&wcand[par][wslot], wcta)->row[lane];
            if (gv < 0.0) { gp = j; }                     // no rows left (m < jb): nothing to do
            const bool singular = !(gv > 0.0);
            if (crank == 0 && tid == 0) {
                ipiv[(long long)z * ipiv_stride + row0 + j] = row0 + gp;
                if (singular && gv >= 0.0) atomicCAS(&info[z], 0, info_base + row0 + j + 1);
            }
            __syncthreads();
            if (!done) {
                if (cur_pos == gp && gv >= 0.0) {
                    done = true; final_pos = j;           // I am the pivot row: becomes row j of U
                } else {
                    if (cur_pos == j) cur_pos = gp;       // LAPACK swap bookkeeping
                    if (!singular) {
                        cplx rinv = crecip_fast(prow[j]);
                        cplx l = cmul(a[j], rinv);
                        a[j] = l;
#pragma unroll
                        for (int k = j + 1; k < LEAF_JB; k++) a[k] = cfnma(a[k], l, prow[k]);
                    }
                }
            }
        }
    }
    cluster.sync();                                   // no CTA may exit while another still reads its shared memory
    if (valid) {
        if (!done) final_pos = cur_pos;
        cplx* dst = A + (long long)final_pos * ld;
#pragma unroll
        for (int k = 0; k < LEAF_JB; k++)
            if (k < jb) dst[k] = a[k];
    }
}

// ---- the whole 128-column panel in ONE launch (panels of up to 4096 rows): the thread-block cluster stays resident over
// the 8 inner blocks of 16 columns instead of being re-scheduled for every one of them (4 launches per inner block before:
// leaf, row swaps, 16-row triangular solve, rank-16 update).  One thread = one matrix row for the whole panel; pivoting is
// IMPLICIT for the whole panel (no row moves until the end), with the same position bookkeeping as the leaf kernel.
// Per inner block:  (1) the 16 active columns of the own row -> registers;  (2) 16 pivot steps exactly as in
// lu_leaf3_kernel (redux arg-max, key exchange through distributed shared memory, one cluster barrier, winner row pulled);
// every CTA keeps the 16 pivot rows' active entries (L11 \ U11) and their physical row numbers;  (3) the pivot rows'
// remaining panel columns are read by every CTA, U12 = L11^-1 A12 is solved redundantly in shared memory (one thread per
// column), the owners write it back;  (4) rank-16 update of the own row's remaining panel columns with the multipliers
// still in registers.  At the end the rows that moved (at most 2 x 128) are carried to their final positions, 16 columns at
// a time through registers with a cluster barrier between the reads and the writes of a chunk.
constexpr int PANEL_W = 128;

__global__ void __launch_bounds__(LEAF2_TPB, 2)
lu_panel_kernel(BPtr Ab, int ld, int j0, int m, int nbw, int* __restrict__ ipiv, int ipiv_stride,
                int* __restrict__ info, int info_base) {
    cg::cluster_group cluster = cg::this_cluster();
    const int csize = (int)cluster.num_blocks();
    const int crank = (int)cluster.block_rank();
    const int z = blockIdx.y;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NW = LEAF2_TPB / 32, JB = LEAF_JB;

    __shared__ __align__(16) LeafCand wcand[2][NW];
    __shared__ __align__(16) LeafKey keys[2][LEAF2_MAXC];
    __shared__ __align__(16) cplx prow[JB];
    __shared__ __align__(16) cplx Lpiv[JB][JB];          // row k: the k-th pivot row's active entries (multipliers | U)
    __shared__ int piv_phys[JB];                          // its physical row inside the panel
    __shared__ __align__(16) cplx U12[JB][PANEL_W - JB];

    cplx* A = bptr(Ab, z) + (long long)j0 * ld + j0;      // no __restrict__/const: other CTAs write rows this CTA reads
    const int r = crank * LEAF2_TPB + tid;                // my (physical) row inside the panel
    const bool valid = r < m;
    cplx* Arow = A + (long long)r * ld;
    int cur_pos = r;
    bool done = !valid;
    int final_pos = r;

    for (int c = 0; c < nbw; c += JB) {
        const int jb = min(JB, nbw - c), wrest = nbw - c - jb;
        cplx a[JB];
#pragma unroll
        for (int k = 0; k < JB; k++) a[k] = (valid && k < jb) ? Arow[c + k] : make_c(0.0, 0.0);
#pragma unroll
        for (int j = 0; j < JB; j++) {
            if (j < jb) {
                const int q = c + j;                      // pivot step = position inside the panel
                const int par = j & 1;
                double wv; int wp;
                const double myv = done ? -1.0 : (fabs(a[j].re) + fabs(a[j].im));
                if (warp_argmax(myv, cur_pos, wv, wp)) {
                    LeafCand* cd = &wcand[par][warp];
                    cd->val = myv; cd->pos = cur_pos; cd->pad = r;
#pragma unroll
                    for (int k = 0; k < JB; k++) cd->row[k] = a[k];
                }
                if (lane == 0 && wv < 0.0) { wcand[par][warp].val = -1.0; wcand[par][warp].pos = 0x7fffffff; wcand[par][warp].pad = 0; }
                __syncthreads();
                if (warp == 0) {
                    double v2 = lane < NW ? wcand[par][lane].val : -1.0;
                    int p2 = lane < NW ? wcand[par][lane].pos : 0x7fffffff;
                    double cv; int cp;
                    bool win = warp_argmax(v2, p2, cv, cp);
                    unsigned bal = __ballot_sync(0xffffffffu, win);
                    LeafKey k; k.val = cv; k.pos = cp; k.warp = bal ? (__ffs(bal) - 1) : 0;
                    if (lane < csize) *cluster.map_shared_rank(&keys[par][crank], lane) = k;
                }
                cluster.sync();
                double kv = -1.0; int kp = 0x7fffffff, kw = 0;
                if (lane < csize) { LeafKey k = keys[par][lane]; kv = k.val; kp = k.pos; kw = k.warp; }
                double gv; int gp;
                bool gwin = warp_argmax(kv, kp, gv, gp);
                unsigned gbal = __ballot_sync(0xffffffffu, gwin);
                const int wcta = gbal ? (__ffs(gbal) - 1) : 0;
                const int wslot = __shfl_sync(0xffffffffu, kw, wcta);
                if (warp == 0 && lane < JB) {
                    const LeafCand* src = cluster.map_shared_rank(&wcand[par][wslot], wcta);
                    cplx v = (gv >= 0.0) ? src->row[lane] : make_c(0.0, 0.0);
                    prow[lane] = v;
                    Lpiv[j][lane] = v;
                    if (lane == 0) piv_phys[j] = (gv >= 0.0) ? src->pad : 0;
                }
                if (gv < 0.0) { gp = q; }                 // no rows left: nothing to do
                const bool singular = !(gv > 0.0);
                if (crank == 0 && tid == 0) {
                    ipiv[(long long)z * ipiv_stride + j0 + q] = j0 + gp;
                    if (singular && gv >= 0.0) atomicCAS(&info[z], 0, info_base + j0 + q + 1);
                }
                __syncthreads();
                if (!done) {
                    if (cur_pos == gp && gv >= 0.0) {
                        done = true; final_pos = q;       // I am the pivot row: becomes row q of the panel's U
                    } else {
                        if (cur_pos == q) cur_pos = gp;   // LAPACK swap bookkeeping
                        if (!singular) {
                            cplx rinv = crecip_fast(prow[j]);
                            cplx l = cmul(a[j], rinv);
                            a[j] = l;
#pragma unroll
                            for (int k = j + 1; k < JB; k++) a[k] = cfnma(a[k], l, prow[k]);
                        }
                    }
                }
            }
        }
        if (valid) {
#pragma unroll
            for (int k = 0; k < JB; k++)
                if (k < jb) Arow[c + k] = a[k];
        }
        if (wrest > 0) {
            const int cr = c + jb;                        // first remaining column
            // A12: the pivot rows' remaining columns (every CTA reads all of them; .cg: written by their owner CTAs)
            for (int idx = tid; idx < jb * wrest; idx += LEAF2_TPB) {
                int k = idx / wrest, cc = idx - k * wrest;
                const double2 v = __ldcg(reinterpret_cast<const double2*>(A + (long long)piv_phys[k] * ld + cr + cc));
                U12[k][cc] = make_c(v.x, v.y);
            }
            cluster.sync();                               // all CTAs have read A12 before any owner overwrites it
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
            if (valid && !done) {                         // A22 -= L21 U12 on my row (multipliers a[0..jb) in registers)
                for (int cc = 0; cc < wrest; cc++) {
                    cplx x = Arow[cr + cc];
#pragma unroll
                    for (int k = 0; k < JB; k++)
                        if (k < jb) x = cfnma(x, a[k], U12[k][cc]);
                    Arow[cr + cc] = x;
                }
            }
            __syncthreads();                              // U12 / Lpiv / piv_phys are rewritten by the next inner block
        }
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
        pr->flops += 8.0 * g.M * g.N * g.K * batch;
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
};
static inline int lu_nblk(int n) { return (n + 127) / 128; }
static inline size_t lu_tinv_elems(int n, int batch) { return (size_t)2 * lu_nblk(n) * 128 * 128 * (size_t)batch; }

static inline GemmArgs gemm_std(int M, int N, int K, double alpha, BPtr A, int lda, BPtr B, int ldb, double beta,
                                BPtr C, int ldc) {
    GemmArgs g{};
    g.M = M; g.N = N; g.K = K; g.A = A; g.lda = lda; g.B = B; g.ldb = ldb; g.C = C; g.ldc = ldc;
    g.Cin = C; g.ldcin = ldc; g.alpha = alpha; g.beta = beta; g.E = nullptr;
    return g;
}

static int g_leaf_version = 3;       // 1 = always lu_leaf_kernel (512 rows / CTA), 3 = lu_leaf3_kernel (256 rows / CTA) up to 4096 rows

static void launch_leaf(Ctx& ctx, BPtr Ab, int ld, int row0, int col0, int m, int jb, const LuWork& w, int info_base,
                        int batch) {
    static bool configured = false;
    if (!configured) {
        cudaFuncSetAttribute(lu_leaf_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        cudaFuncSetAttribute(lu_leaf3_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        configured = true;
    }
    const bool v3 = (g_leaf_version == 3) && m <= LEAF2_TPB * LEAF2_MAXC;
    const int tpb = v3 ? LEAF2_TPB : LEAF_TPB;
    int need = (m + tpb - 1) / tpb;
    int csize = 1;
    while (csize < need) csize <<= 1;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)csize, (unsigned)batch, 1);
    cfg.blockDim = dim3((unsigned)tpb, 1, 1);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = ctx.st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)csize;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (v3)
        ctx.note(cudaLaunchKernelEx(&cfg, lu_leaf3_kernel, Ab, ld, row0, col0, m, jb, w.ipiv, w.ipiv_stride, w.info, info_base));
    else
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

static void lu_swaps(const LuCall& L, int piv_lo, int piv_hi, int c_lo, int c_hi, int skip_lo, int skip_hi) {
    const int total = (skip_lo - c_lo) + (c_hi - skip_hi);
    if (total <= 0 || piv_hi <= piv_lo) return;
    dim3 grid((unsigned)((total + 255) / 256), (unsigned)L.batch);
    laswp_kernel<<<grid, 256, 0, L.ctx.st>>>(L.Ab, L.ld, c_lo, c_hi, piv_lo, piv_hi - piv_lo, skip_lo, skip_hi, L.w.ipiv, L.w.ipiv_stride);
    L.ctx.note(cudaGetLastError());
}

static int g_panel_fused = 1;        // 1: lu_panel_kernel for panels of up to 4096 rows; 0: always the per-16-column launches

static void launch_panel_fused(Ctx& ctx, BPtr Ab, int ld, int j0, int m, int nbw, const LuWork& w, int info_base, int batch) {
    static bool configured = false;
    if (!configured) {
        cudaFuncSetAttribute(lu_panel_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        configured = true;
    }
    int need = (m + LEAF2_TPB - 1) / LEAF2_TPB, csize = 1;
    while (csize < need) csize <<= 1;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)csize, (unsigned)batch, 1);
    cfg.blockDim = dim3((unsigned)LEAF2_TPB, 1, 1);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = ctx.st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)csize;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    ctx.note(cudaLaunchKernelEx(&cfg, lu_panel_kernel, Ab, ld, j0, m, nbw, w.ipiv, w.ipiv_stride, w.info, info_base));
}

// Panel of nbw <= 128 columns at (j0, j0), rows j0 .. n-1, swaps applied inside the panel only; then the inverse of its
// unit-lower 128 x 128 block for the solves that follow.  Up to 4096 rows: one fused launch (lu_panel_kernel); above
// (the 2bs corner system at bs > 2048): inner blocks of 16 columns by separate launches (leaf kernel, row swaps,
// 16-row triangular solve, rank-16 GEMM).
static void lu_panel(const LuCall& L, int j0, int nbw) {
    Ctx& ctx = L.ctx;
    ctx.use(CLS_HI);
    if (g_panel_fused && L.n - j0 <= LEAF2_TPB * LEAF2_MAXC) {
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

static void lu_factor(Ctx& ctx, BPtr Ab, int ld, int n, int ncols, int batch, const LuWork& w, int info_base) {
    LuCall L{ctx, Ab, ld, n, ncols, batch, w, info_base};
    lu_recursive(L, 0, n);
    if (ncols > n) {
        ctx.use(CLS_HI);
        lu_swaps(L, 0, n, n, ncols, ncols, ncols);
        lu_trsm_lower(L, 0, n, n, ncols);
    }
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
