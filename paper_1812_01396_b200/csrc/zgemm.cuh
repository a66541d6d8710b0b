// Batched complex-FP64 GEMM on the FP64 tensor pipe (DMMA.8x8x4 via mma.sync.m8n8k4.f64), sm_100a.
//
// Serves SURVEY.md §8(a) a1 (Schur update, fused with a0's diagonal block formation in the epilogue),
// a4 (column recursion), the trailing updates inside a2/a3 (blocked ZGETRF / ZTRSM), and a5-a7's products
// ("two matrix-matrix multiplications" per Q_i; L175).
//
// Complex product as ONE real product on interleaved data ("4M", no de-interleave pass):
//   C~ (M x 2N real, interleaved re/im) = A~ (M x 2K real, interleaved as stored) * B~ (2K x 2N real), with
//   B~[2k  ][2n] = Re b_kn   B~[2k  ][2n+1] = Im b_kn
//   B~[2k+1][2n] = -Im b_kn  B~[2k+1][2n+1] = Re b_kn
// so the A fragments are plain LDS.64 of the staged tile, the B fragments are LDS.64 of one component of
// the staged complex element (sign flipped on a per-thread-constant mask), and each thread's two
// accumulators of an m8n8 tile are exactly (re, im) of one complex element of C.
//
// Staging: cp.async (LDGSTS) 16 B = one complex element per request, zero-filled out of range, so M, N, K,
// leading dimensions and sub-matrix offsets are arbitrary.  STAGES-deep ring, one __syncthreads per K chunk.
#pragma once
#include "ss_common.cuh"

namespace ss {

enum { EPI_STD = 0, EPI_SCHUR = 1 };

struct GemmArgs {
    int M, N, K;
    BPtr A; int lda;
    BPtr B; int ldb;
    BPtr C; int ldc;
    BPtr Cin; int ldcin;       // EPI_STD: C = alpha*acc + beta*Cin (Cin may alias C; ignored when beta == 0)
    double alpha, beta;
    BPtr S; BPtr H; int lds;   // EPI_SCHUR: C = (E[z>>eshift]*S - H) - acc   (a0 fused into a1's epilogue)
    const cplx* E; int eshift; // eshift 1: batch entry z = 2*energy + column, 0: z = energy
    int tiles_m, tiles_n;
    // tri != 0: only the tiles that touch the lower triangle are computed (Hermitian updates): element
    // (i, j) of C is at global position (tri_row0 + i, tri_col0 + j); a tile whose every column lies right of its last row is skipped
    int tri, tri_row0, tri_col0;
    int raster_gm;             // tile rows per raster group (set by the launcher)
    // Sum planes (3M only).  The three real products of 3M need re + im of every operand element; formed per fragment in the
    // main loop these DADDs share the FP64 pipe with the DMMAs and cost 9 % of it (profiles/r02_gemm_sumplane.md).  An
    // operand that lies inside a region with a "shadow" array of doubles holding re + im of every element (same element
    // offsets: shadow address = sh*_d + (element pointer - sh*_c)) is staged together with its sum tile instead.  shC:
    // the epilogue also writes re + im of every output element (the producer side of the same scheme).
    const cplx* shA_c; const double* shA_d;
    const cplx* shB_c; const double* shB_d;
    const cplx* shC_c; double* shC_d;
};

static int g_gemm_raster = 16; // process-wide (tuning): 16 tile rows read 20 % less DRAM than 8 at equal speed, 32 thrash L2 (profiles/r02_gemm_tma.md)

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc, int src_bytes) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gsrc), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c0), "+d"(c1)
        : "d"(a), "d"(b));
}

template <int BM, int BN, int WARPS_M, int WARPS_N, int KC, int STAGES>
struct GemmCfg {
    static constexpr int NT = WARPS_M * WARPS_N * 32;
    static constexpr int WM = BM / WARPS_M, WN = BN / WARPS_N;   // warp tile, complex elements
    static constexpr int MI = WM / 8;                            // m8 tiles per warp
    static constexpr int NJ = WN / 4;                            // n8 (real) tiles per warp = 4 complex columns each
    static constexpr int LDA_S = 2 * KC + 4;                     // doubles; == 4 (mod 16): conflict-free A fragments
    static constexpr int LDB_S = 2 * (BN + 2);                   // doubles; == 4 (mod 16): conflict-free B fragments
    static constexpr int STAGE_D = BM * LDA_S + KC * LDB_S;      // doubles per stage
    static constexpr int SMEM_BYTES = STAGES * STAGE_D * 8;
    static constexpr int ITER_A = (BM * KC) / NT, ITER_B = (KC * BN) / NT;
    static_assert((BM * KC) % NT == 0 && (KC * BN) % NT == 0, "tile/thread mismatch");
    static_assert(WM % 8 == 0 && WN % 4 == 0 && KC % 2 == 0, "warp tile");
    static_assert((2 * KC) % 16 == 0 && (2 * BN) % 16 == 0, "bank layout");
};

template <class Cfg, int BM, int BN, int WARPS_M, int WARPS_N, int KC, int STAGES, int EPI, int MINB>
__global__ void __launch_bounds__(Cfg::NT, MINB) zgemm_kernel(const GemmArgs p) {
    extern __shared__ __align__(16) double smem[];
    constexpr int NT = Cfg::NT, MI = Cfg::MI, NJ = Cfg::NJ, LDA_S = Cfg::LDA_S, LDB_S = Cfg::LDB_S;
    constexpr int STAGE_D = Cfg::STAGE_D;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, t = lane & 3;
    const int z = blockIdx.y;

    // grouped rasterisation: raster_gm tile rows share the B columns in L2
    int tile_m, tile_n;
    {
        const int GM = p.raster_gm;
        int pid = blockIdx.x;
        int per_group = GM * p.tiles_n;
        int group = pid / per_group;
        int first_m = group * GM;
        int gsize = min(p.tiles_m - first_m, GM);
        int r = pid - group * per_group;
        tile_m = first_m + r % gsize;
        tile_n = r / gsize;
    }
    const int m0 = tile_m * BM, n0 = tile_n * BN;
    const int M = p.M, N = p.N, K = p.K;
    if (p.tri && (n0 + p.tri_col0) > (m0 + BM - 1 + p.tri_row0)) return;

    const cplx* __restrict__ Ag = bptr(p.A, z);
    const cplx* __restrict__ Bg = bptr(p.B, z);

    // ---- per-thread staging descriptors
    const cplx* a_src[Cfg::ITER_A]; int a_dst[Cfg::ITER_A]; int a_kc[Cfg::ITER_A]; bool a_ok[Cfg::ITER_A];
#pragma unroll
    for (int q = 0; q < Cfg::ITER_A; q++) {
        int c = tid + q * NT;
        int row = c / KC, kc = c % KC;
        a_kc[q] = kc;
        a_ok[q] = (m0 + row) < M;
        a_src[q] = Ag + (long long)(a_ok[q] ? (m0 + row) : 0) * p.lda + kc;
        a_dst[q] = row * LDA_S + 2 * kc;
    }
    const cplx* b_src[Cfg::ITER_B]; int b_dst[Cfg::ITER_B]; int b_kr[Cfg::ITER_B]; bool b_ok[Cfg::ITER_B];
#pragma unroll
    for (int q = 0; q < Cfg::ITER_B; q++) {
        int c = tid + q * NT;
        int kr = c / BN, col = c % BN;
        b_kr[q] = kr;
        b_ok[q] = (n0 + col) < N;
        b_src[q] = Bg + (long long)kr * p.ldb + (b_ok[q] ? (n0 + col) : 0);
        b_dst[q] = BM * LDA_S + kr * LDB_S + 2 * col;
    }

    auto load_stage = [&](int kt, int stage) {
        double* sbase = smem + stage * STAGE_D;
        const int k0 = kt * KC;
#pragma unroll
        for (int q = 0; q < Cfg::ITER_A; q++) {
            bool ok = a_ok[q] && (k0 + a_kc[q] < K);
            cp_async16(sbase + a_dst[q], ok ? (const void*)(a_src[q] + k0) : (const void*)Ag, ok ? 16 : 0);
        }
#pragma unroll
        for (int q = 0; q < Cfg::ITER_B; q++) {
            bool ok = b_ok[q] && (k0 + b_kr[q] < K);
            cp_async16(sbase + b_dst[q], ok ? (const void*)(b_src[q] + (long long)k0 * p.ldb) : (const void*)Bg, ok ? 16 : 0);
        }
    };

    // ---- fragment offsets
    const int wm0 = (warp / WARPS_N) * Cfg::WM, wn0 = (warp % WARPS_N) * Cfg::WN;
    int a_off[MI];
#pragma unroll
    for (int i = 0; i < MI; i++) a_off[i] = (wm0 + 8 * i + g) * LDA_S + t;
    int b_off[NJ];
#pragma unroll
    for (int j = 0; j < NJ; j++)
        b_off[j] = BM * LDA_S + (t >> 1) * LDB_S + 2 * (wn0 + 4 * j + (g >> 1)) + ((t & 1) ^ (g & 1));
    const int b_sign = ((t & 1) == 1 && (g & 1) == 0) ? (int)0x80000000 : 0;

    double acc[MI][NJ][2];
#pragma unroll
    for (int i = 0; i < MI; i++)
#pragma unroll
        for (int j = 0; j < NJ; j++) { acc[i][j][0] = 0.0; acc[i][j][1] = 0.0; }

    const int KT = (K + KC - 1) / KC;
#pragma unroll
    for (int s = 0; s < STAGES - 1; s++) {
        if (s < KT) load_stage(s, s);
        cp_async_commit();
    }

    for (int kt = 0; kt < KT; kt++) {
        cp_async_wait<STAGES - 2>();
        __syncthreads();
        {
            int nk = kt + STAGES - 1;
            if (nk < KT) load_stage(nk, nk % STAGES);
            cp_async_commit();
        }
        const double* sA = smem + (kt % STAGES) * STAGE_D;
#pragma unroll
        for (int ks = 0; ks < KC / 2; ks++) {
            double a[MI], b[NJ];
#pragma unroll
            for (int i = 0; i < MI; i++) a[i] = sA[a_off[i] + 4 * ks];
#pragma unroll
            for (int j = 0; j < NJ; j++) {
                double v = sA[b_off[j] + 2 * ks * LDB_S];
                b[j] = __hiloint2double(__double2hiint(v) ^ b_sign, __double2loint(v));
            }
#pragma unroll
            for (int i = 0; i < MI; i++)
#pragma unroll
                for (int j = 0; j < NJ; j++) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
        }
    }
    cp_async_wait<0>();

    // ---- epilogue: thread owns complex C[m0+wm0+8i+g][n0+wn0+4j+t] = (acc[i][j][0], acc[i][j][1])
    cplx* __restrict__ Cg = bptr(p.C, z);
    if (EPI == EPI_STD) {
        const cplx* Cin = (p.beta != 0.0) ? bptr(p.Cin, z) : nullptr;
        const double alpha = p.alpha, beta = p.beta;
#pragma unroll
        for (int i = 0; i < MI; i++) {
            int row = m0 + wm0 + 8 * i + g;
            if (row >= M) continue;
#pragma unroll
            for (int j = 0; j < NJ; j++) {
                int col = n0 + wn0 + 4 * j + t;
                if (col >= N) continue;
                cplx o = make_c(alpha * acc[i][j][0], alpha * acc[i][j][1]);
                if (Cin) {
                    cplx c = Cin[(long long)row * p.ldcin + col];
                    o.re = fma(beta, c.re, o.re);
                    o.im = fma(beta, c.im, o.im);
                }
                Cg[(long long)row * p.ldc + col] = o;
            }
        }
    } else {
        const cplx Ee = p.E[z >> p.eshift];
        const cplx* __restrict__ Sg = bptr(p.S, z);
        const cplx* __restrict__ Hg = bptr(p.H, z);
#pragma unroll
        for (int i = 0; i < MI; i++) {
            int row = m0 + wm0 + 8 * i + g;
            if (row >= M) continue;
#pragma unroll
            for (int j = 0; j < NJ; j++) {
                int col = n0 + wn0 + 4 * j + t;
                if (col >= N) continue;
                long long off = (long long)row * p.lds + col;
                cplx s = Sg[off], h = Hg[off];
                cplx d = cmul(Ee, s);
                cplx o = make_c(d.re - h.re - acc[i][j][0], d.im - h.im - acc[i][j][1]);
                Cg[(long long)row * p.ldc + col] = o;
            }
        }
    }
}

// tile configurations
using CfgBig = GemmCfg<64, 64, 2, 2, 8, 4>;      // general: 64x64 complex tile, 4 warps of 32x32
using CfgTall = GemmCfg<128, 32, 4, 1, 8, 4>;    // one CTA owns all (<=128) rows of its columns: in-place L^-1 * A12

enum { GEMM_BIG = 0, GEMM_TALL = 1 };

template <class Cfg, int BM, int BN, int WM_, int WN_, int KC, int ST, int EPI, int MINB>
static cudaError_t gemm_launch_t(GemmArgs a, int batch, cudaStream_t st) {
    auto kern = zgemm_kernel<Cfg, BM, BN, WM_, WN_, KC, ST, EPI, MINB>;
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::SMEM_BYTES);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    a.tiles_m = (a.M + BM - 1) / BM;
    a.tiles_n = (a.N + BN - 1) / BN;
    a.raster_gm = g_gemm_raster;
    if (a.tiles_m == 0 || a.tiles_n == 0 || batch == 0) return cudaSuccess;
    dim3 grid((unsigned)(a.tiles_m * a.tiles_n), (unsigned)batch, 1);
    kern<<<grid, Cfg::NT, Cfg::SMEM_BYTES, st>>>(a);
    return cudaGetLastError();
}

static cudaError_t gemm4m_launch(const GemmArgs& a, int batch, int cfg, int epi, cudaStream_t st) {
    if (cfg == GEMM_TALL) return gemm_launch_t<CfgTall, 128, 32, 4, 1, 8, 4, EPI_STD, 2>(a, batch, st);
    if (epi == EPI_SCHUR) return gemm_launch_t<CfgBig, 64, 64, 2, 2, 8, 4, EPI_SCHUR, 2>(a, batch, st);
    return gemm_launch_t<CfgBig, 64, 64, 2, 2, 8, 4, EPI_STD, 2>(a, batch, st);
}

}  // namespace ss
