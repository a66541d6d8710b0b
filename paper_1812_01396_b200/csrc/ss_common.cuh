// Common device/host helpers of libsplitsolve (sm_100a).  No dependency on torch, cuBLAS or cuSOLVER.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>

namespace ss {

struct __align__(16) cplx {
    double re, im;
};

__host__ __device__ __forceinline__ cplx make_c(double r, double i) { cplx z; z.re = r; z.im = i; return z; }
__device__ __forceinline__ cplx cmul(cplx a, cplx b) {
    return make_c(fma(a.re, b.re, -(a.im * b.im)), fma(a.re, b.im, a.im * b.re));
}
// a - b*c
__device__ __forceinline__ cplx cfnma(cplx a, cplx b, cplx c) {
    double r = fma(-b.re, c.re, a.re);
    r = fma(b.im, c.im, r);
    double i = fma(-b.re, c.im, a.im);
    i = fma(-b.im, c.re, i);
    return make_c(r, i);
}
// a + b*c
__device__ __forceinline__ cplx cfma(cplx a, cplx b, cplx c) {
    double r = fma(b.re, c.re, a.re);
    r = fma(-b.im, c.im, r);
    double i = fma(b.re, c.im, a.im);
    i = fma(b.im, c.re, i);
    return make_c(r, i);
}
__device__ __forceinline__ cplx cconj(cplx a) { return make_c(a.re, -a.im); }
__device__ __forceinline__ cplx csub(cplx a, cplx b) { return make_c(a.re - b.re, a.im - b.im); }
__device__ __forceinline__ cplx cneg(cplx a) { return make_c(-a.re, -a.im); }
// 1/a, scaled (Smith) to avoid overflow/underflow
__device__ __forceinline__ cplx crecip(cplx a) {
    if (fabs(a.re) >= fabs(a.im)) {
        double r = a.im / a.re, d = a.re + a.im * r;
        return make_c(1.0 / d, -r / d);
    } else {
        double r = a.re / a.im, d = a.re * r + a.im;
        return make_c(r / d, -1.0 / d);
    }
}

// Pointer of batch entry z.  two != 0: chains (energy e = z>>1, sweep column z&1) -> (z&1 ? p1 : p0) + e*s_out.
// two == 0: p0 + (z % n_in)*s_in + (z / n_in)*s_out.
struct BPtr {
    cplx* p0;
    cplx* p1;
    long long s_in;
    long long s_out;
    int n_in;
    int two;
};
__host__ __device__ __forceinline__ cplx* bptr(const BPtr& b, int z) {
    if (b.two) return ((z & 1) ? b.p1 : b.p0) + (long long)(z >> 1) * b.s_out;
    int zi = z % b.n_in, zo = z / b.n_in;
    return b.p0 + (long long)zi * b.s_in + (long long)zo * b.s_out;
}
inline BPtr bp_strided(const cplx* p, long long stride) {
    BPtr b; b.p0 = const_cast<cplx*>(p); b.p1 = nullptr; b.s_in = stride; b.s_out = 0; b.n_in = 1 << 30; b.two = 0; return b;
}
inline BPtr bp_two_level(const cplx* p, int n_in, long long s_in, long long s_out) {
    BPtr b; b.p0 = const_cast<cplx*>(p); b.p1 = nullptr; b.s_in = s_in; b.s_out = s_out; b.n_in = n_in; b.two = 0; return b;
}
inline BPtr bp_chain(const cplx* p0, const cplx* p1, long long s_energy) {
    BPtr b; b.p0 = const_cast<cplx*>(p0); b.p1 = const_cast<cplx*>(p1); b.s_in = 0; b.s_out = s_energy; b.n_in = 1; b.two = 1; return b;
}
inline BPtr bp_offset(BPtr b, long long off) {
    b.p0 += off; if (b.p1) b.p1 += off; return b;
}

}  // namespace ss
