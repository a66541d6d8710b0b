// Standalone probe (not part of libsplitsolve.so): FP64 DFMA vs DMMA (mma.sync f64, all four shapes) peak and fragment-layout check on B200.
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -o probe_fp64 probe_fp64.cu ; run: ./probe_fp64 sustained
// It decided the GEMM design: every f64 mma shape lowers to DMMA.8x8x4 and sustains 37.07 TFLOP/s vs 34.1 for plain DFMA.
#include <cstdio>
#include <cstdlib>
#include <vector>
#include <cmath>
#include <cuda_runtime.h>

#define CK(x) do { cudaError_t e = (x); if (e != cudaSuccess) { printf("CUDA error %s at %d\n", cudaGetErrorString(e), __LINE__); exit(1);} } while(0)

template <int NCH>
__global__ void k_dfma(double* out, int iters, double a, double b) {
    double acc[NCH];
#pragma unroll
    for (int i = 0; i < NCH; i++) acc[i] = threadIdx.x * 1e-3 + i;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < NCH; i++) acc[i] = fma(acc[i], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < NCH; i++) s += acc[i];
    if (s == 12345.678) out[0] = s;
}

__device__ __forceinline__ void mma884(double (&c)[2], double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}
__device__ __forceinline__ void mma1684(double (&c)[4], const double (&a)[2], double b) {
    asm volatile("mma.sync.aligned.m16n8k4.row.col.f64.f64.f64.f64 {%0,%1,%2,%3}, {%4,%5}, {%6}, {%0,%1,%2,%3};"
                 : "+d"(c[0]), "+d"(c[1]), "+d"(c[2]), "+d"(c[3]) : "d"(a[0]), "d"(a[1]), "d"(b));
}
__device__ __forceinline__ void mma1688(double (&c)[4], const double (&a)[4], const double (&b)[2]) {
    asm volatile("mma.sync.aligned.m16n8k8.row.col.f64.f64.f64.f64 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+d"(c[0]), "+d"(c[1]), "+d"(c[2]), "+d"(c[3])
                 : "d"(a[0]), "d"(a[1]), "d"(a[2]), "d"(a[3]), "d"(b[0]), "d"(b[1]));
}
__device__ __forceinline__ void mma16816(double (&c)[4], const double (&a)[8], const double (&b)[4]) {
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f64.f64.f64.f64 {%0,%1,%2,%3}, {%4,%5,%6,%7,%8,%9,%10,%11}, {%12,%13,%14,%15}, {%0,%1,%2,%3};"
                 : "+d"(c[0]), "+d"(c[1]), "+d"(c[2]), "+d"(c[3])
                 : "d"(a[0]), "d"(a[1]), "d"(a[2]), "d"(a[3]), "d"(a[4]), "d"(a[5]), "d"(a[6]), "d"(a[7]),
                   "d"(b[0]), "d"(b[1]), "d"(b[2]), "d"(b[3]));
}

// Mixed: even warps issue DMMA chains, odd warps DFMA chains (are the two FP64 paths one physical pipe or two?).
// flops counted for both; if the sum exceeds the single-path peak the pipes are separate.
__global__ void k_mixed(double* out, int iters, double fa, double fb, int dfma_every) {
    const int warp = threadIdx.x >> 5;
    double s = 0;
    if (dfma_every > 0 && (warp % dfma_every) == dfma_every - 1) {
        double acc[8];
#pragma unroll
        for (int i = 0; i < 8; i++) acc[i] = threadIdx.x * 1e-3 + i;
        for (int it = 0; it < iters; it++) {
#pragma unroll
            for (int i = 0; i < 8; i++) acc[i] = fma(acc[i], fa, fb);
        }
#pragma unroll
        for (int i = 0; i < 8; i++) s += acc[i];
    } else {
        double c[8][2];
#pragma unroll
        for (int i = 0; i < 8; i++) { c[i][0] = 0; c[i][1] = 0; }
        double a = threadIdx.x * 1e-9, b = 1e-9 * (threadIdx.x % 7);
        for (int it = 0; it < iters; it++) {
#pragma unroll
            for (int i = 0; i < 8; i++) mma884(c[i], a, b);
        }
#pragma unroll
        for (int i = 0; i < 8; i++) s += c[i][0] + c[i][1];
    }
    if (s == 12345.678) out[0] = s;
}

template <int NACC>
__global__ void k_mma884(double* out, int iters) {
    double c[NACC][2];
    for (int i = 0; i < NACC; i++) { c[i][0] = 0; c[i][1] = 0; }
    double a = threadIdx.x * 1e-9, b = 1e-9 * (threadIdx.x % 7);
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < NACC; i++) mma884(c[i], a, b);
    }
    double s = 0;
    for (int i = 0; i < NACC; i++) s += c[i][0] + c[i][1];
    if (s == 12345.678) out[0] = s;
}
template <int NACC>
__global__ void k_mma1684(double* out, int iters) {
    double c[NACC][4];
    for (int i = 0; i < NACC; i++) for (int j = 0; j < 4; j++) c[i][j] = 0;
    double a[2] = {threadIdx.x * 1e-9, 2e-9}; double b = 1e-9 * (threadIdx.x % 7);
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < NACC; i++) mma1684(c[i], a, b);
    }
    double s = 0;
    for (int i = 0; i < NACC; i++) for (int j = 0; j < 4; j++) s += c[i][j];
    if (s == 12345.678) out[0] = s;
}
template <int NACC>
__global__ void k_mma1688(double* out, int iters) {
    double c[NACC][4];
    for (int i = 0; i < NACC; i++) for (int j = 0; j < 4; j++) c[i][j] = 0;
    double a[4] = {threadIdx.x * 1e-9, 2e-9, 3e-9, 4e-9}; double b[2] = {1e-9 * (threadIdx.x % 7), 1e-9};
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < NACC; i++) mma1688(c[i], a, b);
    }
    double s = 0;
    for (int i = 0; i < NACC; i++) for (int j = 0; j < 4; j++) s += c[i][j];
    if (s == 12345.678) out[0] = s;
}
template <int NACC>
__global__ void k_mma16816(double* out, int iters) {
    double c[NACC][4];
    for (int i = 0; i < NACC; i++) for (int j = 0; j < 4; j++) c[i][j] = 0;
    double a[8]; for (int j = 0; j < 8; j++) a[j] = threadIdx.x * 1e-9 + j * 1e-10;
    double b[4]; for (int j = 0; j < 4; j++) b[j] = 1e-9 * (threadIdx.x % 7) + j * 1e-10;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < NACC; i++) mma16816(c[i], a, b);
    }
    double s = 0;
    for (int i = 0; i < NACC; i++) for (int j = 0; j < 4; j++) s += c[i][j];
    if (s == 12345.678) out[0] = s;
}

// layout check: each shape computes D = A(16xK) * B(Kx8) with assumed fragment layout
__global__ void k_layout(const double* A, const double* B, double* D884, double* D1684, double* D1688, double* D16816) {
    int lane = threadIdx.x, g = lane >> 2, t = lane & 3;
    // A is 16x16 row-major, B is 16x8 row-major (k,n)
    {   // m8n8k4 : rows 0..7, k 0..3
        double c[2] = {0, 0};
        mma884(c, A[g * 16 + t], B[t * 8 + g]);
        D884[g * 8 + 2 * t] = c[0]; D884[g * 8 + 2 * t + 1] = c[1];
    }
    {   // m16n8k4
        double c[4] = {0, 0, 0, 0};
        double a[2] = {A[g * 16 + t], A[(g + 8) * 16 + t]};
        mma1684(c, a, B[t * 8 + g]);
        D1684[g * 8 + 2 * t] = c[0]; D1684[g * 8 + 2 * t + 1] = c[1];
        D1684[(g + 8) * 8 + 2 * t] = c[2]; D1684[(g + 8) * 8 + 2 * t + 1] = c[3];
    }
    {   // m16n8k8
        double c[4] = {0, 0, 0, 0};
        double a[4] = {A[g * 16 + t], A[(g + 8) * 16 + t], A[g * 16 + t + 4], A[(g + 8) * 16 + t + 4]};
        double b[2] = {B[t * 8 + g], B[(t + 4) * 8 + g]};
        mma1688(c, a, b);
        D1688[g * 8 + 2 * t] = c[0]; D1688[g * 8 + 2 * t + 1] = c[1];
        D1688[(g + 8) * 8 + 2 * t] = c[2]; D1688[(g + 8) * 8 + 2 * t + 1] = c[3];
    }
    {   // m16n8k16
        double c[4] = {0, 0, 0, 0};
        double a[8], b[4];
        for (int i = 0; i < 8; i++) a[i] = A[(g + 8 * (i & 1)) * 16 + t + 4 * (i >> 1)];
        for (int i = 0; i < 4; i++) b[i] = B[(t + 4 * i) * 8 + g];
        mma16816(c, a, b);
        D16816[g * 8 + 2 * t] = c[0]; D16816[g * 8 + 2 * t + 1] = c[1];
        D16816[(g + 8) * 8 + 2 * t] = c[2]; D16816[(g + 8) * 8 + 2 * t + 1] = c[3];
    }
}

template <typename F>
double timeit(F f, int reps = 3) {
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    f(); CK(cudaDeviceSynchronize());
    float best = 1e30f;
    for (int r = 0; r < reps; r++) {
        cudaEventRecord(e0); f(); cudaEventRecord(e1); CK(cudaEventSynchronize(e1));
        float ms; cudaEventElapsedTime(&ms, e0, e1); if (ms < best) best = ms;
    }
    return best * 1e-3;
}

int main(int argc, char** argv) {
    cudaDeviceProp p; CK(cudaGetDeviceProperties(&p, 0));
    int clk = 0; cudaDeviceGetAttribute(&clk, cudaDevAttrClockRate, 0);
    printf("device %s SMs %d clock %d kHz\n", p.name, p.multiProcessorCount, clk);
    int nsm = p.multiProcessorCount;
    double* out; CK(cudaMalloc(&out, 1024));

    // layout check
    {
        std::vector<double> A(256), B(128), ref(128, 0.0);
        for (int i = 0; i < 256; i++) A[i] = sin(i * 0.37) + 0.1 * i;
        for (int i = 0; i < 128; i++) B[i] = cos(i * 0.91) - 0.05 * i;
        double *dA, *dB, *dD; CK(cudaMalloc(&dA, 256 * 8)); CK(cudaMalloc(&dB, 128 * 8)); CK(cudaMalloc(&dD, 4 * 128 * 8));
        CK(cudaMemset(dD, 0, 4 * 128 * 8));
        CK(cudaMemcpy(dA, A.data(), 256 * 8, cudaMemcpyHostToDevice)); CK(cudaMemcpy(dB, B.data(), 128 * 8, cudaMemcpyHostToDevice));
        k_layout<<<1, 32>>>(dA, dB, dD, dD + 128, dD + 256, dD + 384); CK(cudaDeviceSynchronize());
        std::vector<double> D(512); CK(cudaMemcpy(D.data(), dD, 512 * 8, cudaMemcpyDeviceToHost));
        int Ms[4] = {8, 16, 16, 16}, Ks[4] = {4, 4, 8, 16}; const char* nm[4] = {"m8n8k4", "m16n8k4", "m16n8k8", "m16n8k16"};
        for (int s = 0; s < 4; s++) {
            double err = 0;
            for (int m = 0; m < Ms[s]; m++) for (int n = 0; n < 8; n++) {
                double r = 0; for (int k = 0; k < Ks[s]; k++) r += A[m * 16 + k] * B[k * 8 + n];
                err = fmax(err, fabs(r - D[s * 128 + m * 8 + n]));
            }
            printf("layout %s max err %.3e\n", nm[s], err);
        }
    }

    int threads_list[3] = {128, 256, 512};
    // DFMA
    for (int ti = 0; ti < 3; ti++) {
        int th = threads_list[ti]; int blocks = nsm * (1024 / th); int iters = 20000;
        double t = timeit([&] { k_dfma<8><<<blocks, th>>>(out, iters, 1.0000001, 1e-9); });
        double fl = 2.0 * 8 * iters * (double)th * blocks;
        printf("DFMA NCH=8 threads=%d blocks=%d : %.3f ms  %.2f TFLOP/s\n", th, blocks, t * 1e3, fl / t * 1e-12);
        t = timeit([&] { k_dfma<16><<<blocks, th>>>(out, iters, 1.0000001, 1e-9); });
        fl = 2.0 * 16 * iters * (double)th * blocks;
        printf("DFMA NCH=16 threads=%d blocks=%d : %.3f ms  %.2f TFLOP/s\n", th, blocks, t * 1e3, fl / t * 1e-12);
    }
    // DMMA shapes; warps per SM sweep
    int wps_list[4] = {4, 8, 16, 32};
    for (int wi = 0; wi < 4; wi++) {
        int wps = wps_list[wi]; int th = 128; int blocks = nsm * wps / 4; int iters = 4000;
        double nw = (double)blocks * th / 32;
        double t;
        t = timeit([&] { k_mma884<8><<<blocks, th>>>(out, iters); });
        printf("DMMA m8n8k4  x8acc warps/SM=%d : %.3f ms %.2f TFLOP/s\n", wps, t * 1e3, 2.0 * 8 * 8 * 4 * 8 * iters * nw / t * 1e-12);
        t = timeit([&] { k_mma1684<8><<<blocks, th>>>(out, iters); });
        printf("DMMA m16n8k4 x8acc warps/SM=%d : %.3f ms %.2f TFLOP/s\n", wps, t * 1e3, 2.0 * 16 * 8 * 4 * 8 * iters * nw / t * 1e-12);
        t = timeit([&] { k_mma1688<8><<<blocks, th>>>(out, iters); });
        printf("DMMA m16n8k8 x8acc warps/SM=%d : %.3f ms %.2f TFLOP/s\n", wps, t * 1e3, 2.0 * 16 * 8 * 8 * 8 * iters * nw / t * 1e-12);
        t = timeit([&] { k_mma16816<8><<<blocks, th>>>(out, iters); });
        printf("DMMA m16n8k16 x8acc warps/SM=%d : %.3f ms %.2f TFLOP/s\n", wps, t * 1e3, 2.0 * 16 * 8 * 16 * 8 * iters * nw / t * 1e-12);
        t = timeit([&] { k_mma16816<2><<<blocks, th>>>(out, iters); });
        printf("DMMA m16n8k16 x2acc warps/SM=%d : %.3f ms %.2f TFLOP/s\n", wps, t * 1e3, 2.0 * 16 * 8 * 16 * 2 * iters * nw / t * 1e-12);
        t = timeit([&] { k_mma16816<1><<<blocks, th>>>(out, iters); });
        printf("DMMA m16n8k16 x1acc warps/SM=%d : %.3f ms %.2f TFLOP/s\n", wps, t * 1e3, 2.0 * 16 * 8 * 16 * 1 * iters * nw / t * 1e-12);
    }
    // mixed DMMA + DFMA warps: one pipe or two?
    for (int every = 2; every <= 4; every *= 2) {
        int th = 512, blocks = nsm * 2, iters = 4000;     // 32 warps per SM
        double nw = (double)blocks * th / 32;
        double nw_dfma = nw / every, nw_dmma = nw - nw_dfma;
        double t = timeit([&] { k_mixed<<<blocks, th>>>(out, iters, 1.0000001, 1e-9, every); });
        double fl_dmma = 2.0 * 8 * 8 * 4 * 8 * iters * nw_dmma, fl_dfma = 2.0 * 8 * iters * 32 * nw_dfma;
        printf("MIXED 1 DFMA warp in %d (same iters): %.3f ms  DMMA %.2f + DFMA %.2f = %.2f TFLOP/s\n", every, t * 1e3,
               fl_dmma / t * 1e-12, fl_dfma / t * 1e-12, (fl_dmma + fl_dfma) / t * 1e-12);
    }
    // sustained: run ~4 s of DFMA and ~4 s of DMMA m16n8k16, report TF in 0.5 s slices
    if (argc > 1) {
        for (int mode = 0; mode < 2; mode++) {
            for (int slice = 0; slice < 8; slice++) {
                double t, fl;
                if (mode == 0) {
                    int th = 256, blocks = nsm * 4, iters = 400000;
                    t = timeit([&] { k_dfma<8><<<blocks, th>>>(out, iters, 1.0000001, 1e-9); }, 1);
                    fl = 2.0 * 8 * iters * (double)th * blocks;
                } else {
                    int th = 128, blocks = nsm * 4, iters = 100000; double nw = (double)blocks * th / 32;
                    t = timeit([&] { k_mma16816<8><<<blocks, th>>>(out, iters); }, 1);
                    fl = 2.0 * 16 * 8 * 16 * 8 * iters * nw;
                }
                printf("sustained mode=%s slice %d: %.1f ms %.2f TFLOP/s\n", mode ? "DMMA16816" : "DFMA", slice, t * 1e3, fl / t * 1e-12);
                fflush(stdout);
            }
        }
    }
    return 0;
}
