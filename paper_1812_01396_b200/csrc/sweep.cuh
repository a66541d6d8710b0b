// Elementwise / reduction kernels of the SplitSolve sweep and post-processing (sm_100a): memory-bound,
// coalesced 16-byte accesses (one complex128 per thread per access).
//   form_kernel      a0: off-diagonal blocks A_{i,i+1} = E S_up - H_up, A_{i+1,i} = E S_up^H - H_up^H (Eq. 5;
//                    E not conjugated), or the identity that stands for A_{1,0} / A_{nb,nb+1} (Alg. 1)
//   corner_init      a5: [R | b' | e_2] initialised to [1 | Inj_first;Inj_last | 0;1] (L141, L148)
//   gamma_kernel     a7: Gamma = i (Sigma - Sigma^H)
//   trace kernels    a7: T = Re sum_ij W_ij conj(G_ij) = Re Tr(W G^H), two-pass deterministic reduction
#pragma once
#include "ss_common.cuh"

namespace ss {

enum { FORM_NONE = 0, FORM_PLAIN = 1, FORM_CONJT = 2, FORM_IDENT = 3 };

struct FormSide {
    const cplx* S;
    const cplx* H;
    int mode;
};

// dst(z)[r][c] (ld) for the bs x bs block.  eshift = 1: z = 2*e + column, side = s0 for column 0, s1 for column 1 (both
// sweeps in lockstep); eshift = 0: z = e, side s0 (one sweep only: SURVEY.md 8(f2), one column per GPU).
__global__ void __launch_bounds__(256)
form_kernel(FormSide s0, FormSide s1, const cplx* __restrict__ E, BPtr dst, int ld, int bs, int eshift) {
    __shared__ cplx tile[32][33];
    const int z = blockIdx.z;
    const FormSide s = (eshift && (z & 1)) ? s1 : s0;
    if (s.mode == FORM_NONE) return;
    cplx* __restrict__ D = bptr(dst, z);
    const int r0 = blockIdx.y * 32, c0 = blockIdx.x * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;      // 32 x 8
    const cplx Ee = E[z >> eshift];
    if (s.mode == FORM_PLAIN) {
        for (int rr = ty; rr < 32; rr += 8) {
            int r = r0 + rr, c = c0 + tx;
            if (r < bs && c < bs) {
                long long o = (long long)r * bs + c;
                cplx v = cmul(Ee, s.S[o]);
                cplx h = s.H[o];
                D[(long long)r * ld + c] = make_c(v.re - h.re, v.im - h.im);
            }
        }
    } else if (s.mode == FORM_IDENT) {
        for (int rr = ty; rr < 32; rr += 8) {
            int r = r0 + rr, c = c0 + tx;
            if (r < bs && c < bs) D[(long long)r * ld + c] = make_c(r == c ? 1.0 : 0.0, 0.0);
        }
    } else {
        // out[r][c] = E conj(S[c][r]) - conj(H[c][r]) = conj( conj(E) S[c][r] - H[c][r] ): read the source tile
        // (rows c0.., cols r0..) coalesced, transpose through shared memory.
        const cplx Ec = cconj(Ee);
        for (int cc = ty; cc < 32; cc += 8) {
            int sr = c0 + cc, sc = r0 + tx;
            cplx v = make_c(0.0, 0.0);
            if (sr < bs && sc < bs) {
                long long o = (long long)sr * bs + sc;
                cplx m = cmul(Ec, s.S[o]);
                cplx h = s.H[o];
                v = make_c(m.re - h.re, m.im - h.im);
            }
            tile[cc][tx] = v;
        }
        __syncthreads();
        for (int rr = ty; rr < 32; rr += 8) {
            int r = r0 + rr, c = c0 + tx;
            if (r < bs && c < bs) D[(long long)r * ld + c] = cconj(tile[tx][rr]);
        }
    }
}

// SURVEY.md 8(f1) (A Hermitian at real E): mirror of a block across the diagonal of a batch matrix.
// Source S = A[rs .. rs+nr) x [cs .. cs+nc) (below or on the diagonal), destination its mirror image:
//     A[cs + k][rs + r] = f_k * conj(A[rs + r][cs + k]),   f_k = A[cs+k][cs+k] if scaled (U12 = Delta * L21^H of an LDL^H), else 1;
// strict: only r > k is written (source and destination are the same diagonal block).  Tiles through shared memory so that
// both the reads and the writes are coalesced.
__global__ void __launch_bounds__(256)
herm_mirror_kernel(BPtr Ab, int ld, int rs, int cs, int nr, int nc, int scaled, int strict) {
    __shared__ cplx tile[32][33];
    cplx* __restrict__ A = bptr(Ab, blockIdx.z);
    const int r0 = blockIdx.y * 32, k0 = blockIdx.x * 32;        // tile of the SOURCE block: rows r0.., columns k0..
    if (strict && k0 > r0 + 31) return;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;      // 32 x 8
    for (int rr = ty; rr < 32; rr += 8) {
        int r = r0 + rr, k = k0 + tx;
        tile[rr][tx] = (r < nr && k < nc) ? A[(long long)(rs + r) * ld + cs + k] : make_c(0.0, 0.0);
    }
    __syncthreads();
    for (int kk = ty; kk < 32; kk += 8) {
        int k = k0 + kk, r = r0 + tx;
        if (k < nc && r < nr && (!strict || r > k)) {
            cplx v = cconj(tile[tx][kk]);
            if (scaled) v = cmul(A[(long long)(cs + k) * ld + cs + k], v);
            A[(long long)(cs + k) * ld + rs + r] = v;
        }
    }
}

// Raug[e] : 2bs x W row-major (leading dimension ld >= W), W = 2bs + m + bs:  [ 1_{2bs} | Inj_first ; Inj_last | 0 ; 1_bs ]
__global__ void __launch_bounds__(256)
corner_init_kernel(cplx* __restrict__ Raug, long long stride, int W, int ld, int bs, int m, const cplx* __restrict__ inj_first,
                   const cplx* __restrict__ inj_last) {
    const int e = blockIdx.z;
    const int r = blockIdx.y;
    cplx* __restrict__ row = Raug + (long long)e * stride + (long long)r * ld;
    for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < W; c += gridDim.x * blockDim.x) {
        cplx v = make_c(0.0, 0.0);
        if (c < 2 * bs) {
            if (c == r) v.re = 1.0;
        } else if (c < 2 * bs + m) {
            int cc = c - 2 * bs;
            if (r < bs) v = inj_first[((long long)e * bs + r) * m + cc];
            else if (inj_last) v = inj_last[((long long)e * bs + (r - bs)) * m + cc];
        } else {
            int cc = c - 2 * bs - m;
            if (r >= bs && cc == r - bs) v.re = 1.0;
        }
        row[c] = v;
    }
}

// Spatial split: [M | rhs] of the two interface systems of the merge, per chain z = 2 e + q:
// dst(z) (bs x 2bs, ld) = [ 1 | rhs_q[e] ]; the products are subtracted from the left half afterwards.
__global__ void __launch_bounds__(256)
merge_init_kernel(BPtr dst, int ld, int bs, const cplx* __restrict__ rhs0, long long s0, const cplx* __restrict__ rhs1, long long s1) {
    const int z = blockIdx.z, r = blockIdx.y;
    cplx* __restrict__ row = bptr(dst, z) + (long long)r * ld;
    const cplx* __restrict__ rhs = ((z & 1) ? rhs1 + (long long)(z >> 1) * s1 : rhs0 + (long long)(z >> 1) * s0) + (long long)r * bs;
    for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < 2 * bs; c += gridDim.x * blockDim.x)
        row[c] = (c < bs) ? make_c(c == r ? 1.0 : 0.0, 0.0) : rhs[c - bs];
}

// out[e][r][c] = i (Sigma[e][r][c] - conj(Sigma[e][c][r]))
__global__ void __launch_bounds__(256)
gamma_kernel(const cplx* __restrict__ Sigma, cplx* __restrict__ out, int bs) {
    __shared__ cplx tile[32][33];
    const int e = blockIdx.z;
    const cplx* __restrict__ S = Sigma + (long long)e * bs * bs;
    cplx* __restrict__ O = out + (long long)e * bs * bs;
    const int r0 = blockIdx.y * 32, c0 = blockIdx.x * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    for (int cc = ty; cc < 32; cc += 8) {
        int sr = c0 + cc, sc = r0 + tx;
        tile[cc][tx] = (sr < bs && sc < bs) ? S[(long long)sr * bs + sc] : make_c(0.0, 0.0);
    }
    __syncthreads();
    for (int rr = ty; rr < 32; rr += 8) {
        int r = r0 + rr, c = c0 + tx;
        if (r < bs && c < bs) {
            cplx a = S[(long long)r * bs + c];
            cplx b = tile[tx][rr];                 // Sigma[c][r]
            // i * ((a.re - b.re) + i (a.im + b.im)) = -(a.im + b.im) + i (a.re - b.re)
            O[(long long)r * bs + c] = make_c(-(a.im + b.im), a.re - b.re);
        }
    }
}

// partial[e][blockIdx.x] = sum over this block's grid-stride slice of
//   mode 0:  Re(W conj(G)) = W.re G.re + W.im G.im        (a7: T = Re Tr(W G^H))
//   mode 1:  Im(conj(G) W) = G.re W.im - G.im W.re        (f3: bond current, Im Tr(X_i^H W))
__global__ void __launch_bounds__(256)
trace_partial_kernel(const cplx* __restrict__ Wm, long long strideW, const cplx* __restrict__ G, long long strideG,
                     long long count, int mode, double* __restrict__ partial) {
    const int e = blockIdx.y;
    const double2* __restrict__ w = reinterpret_cast<const double2*>(Wm + (long long)e * strideW);
    const double2* __restrict__ g = reinterpret_cast<const double2*>(G + (long long)e * strideG);
    double acc = 0.0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < count; i += (long long)gridDim.x * blockDim.x) {
        double2 a = w[i], b = g[i];
        if (mode == 0) {
            acc = fma(a.x, b.x, acc);
            acc = fma(a.y, b.y, acc);
        } else {
            acc = fma(b.x, a.y, acc);
            acc = fma(-b.y, a.x, acc);
        }
    }
    __shared__ double red[8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int i = 0; i < 8; i++) s += red[i];
        partial[(long long)e * gridDim.x + blockIdx.x] = s;
    }
}

// T[e * t_stride] = scale * sum of the nparts partials of e
__global__ void trace_final_kernel(const double* __restrict__ partial, int nparts, double* __restrict__ T, int t_stride = 1,
                                   double scale = 1.0) {
    const int e = blockIdx.x;
    double acc = 0.0;
    for (int i = threadIdx.x; i < nparts; i += 32) acc += partial[(long long)e * nparts + i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (threadIdx.x == 0) T[(long long)e * t_stride] = scale * acc;
}

// carrier density from the wave functions c(E) = X ("charge and current densities can be
// directly derived from ... c(E)"):  rho[i] = sum_e w[e] sum_c |X[e][i][c]|^2  (w = occupation x integration weight,
// supplied by the caller).  HBM-bound: every element of X is read once, 16-byte coalesced; one warp per orbital row,
// energies accumulated in order in a register (deterministic, no atomics).
__global__ void __launch_bounds__(256)
density_kernel(const cplx* __restrict__ X, int n_energy, long long n, int m, const double* __restrict__ w, double* __restrict__ rho) {
    const int lane = threadIdx.x & 31;
    const long long row = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (row >= n) return;
    double total = 0.0;
    for (int e = 0; e < n_energy; e++) {
        const double2* __restrict__ x = reinterpret_cast<const double2*>(X + ((long long)e * n + row) * m);
        double acc = 0.0;
        for (int c = lane; c < m; c += 32) {
            double2 v = x[c];
            acc = fma(v.x, v.x, acc);
            acc = fma(v.y, v.y, acc);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        total = fma(w ? w[e] : 1.0, acc, total);
    }
    if (lane == 0) rho[row] = total;
}

// FP64 pipe microbenchmark: register-resident DMMA chains (the roofline denominator, measured live).
__global__ void __launch_bounds__(128) fp64_peak_kernel(double* out, int iters) {
    double c[8][2];
#pragma unroll
    for (int i = 0; i < 8; i++) { c[i][0] = 0.0; c[i][1] = 0.0; }
    double a = threadIdx.x * 1e-9, b = 1e-9 * (threadIdx.x % 7);
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 8; i++)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; i++) s += c[i][0] + c[i][1];
    if (s == 12345.678) out[0] = s;
}

}  // namespace ss
