// Batched complex-FP64 GEMM, "3M" arithmetic on the FP64 tensor pipe (DMMA.8x8x4 via mma.sync.m8n8k4.f64), sm_100a.
//
// Same contract and epilogues as zgemm.cuh (the updates inside a2/a3, a5-a7's products;
// PAPER.md L186 "two matrix-matrix multiplications" per Q_i).  north_star: "a complex-FP64 GEMM (4M or 3M over real
// FP64 MMA or FMA, whichever ... reach[es] the higher fraction of the chip's FP64 peak)".
//
// 3M: with A = Ar + i Ai, B = Br + i Bi, three REAL products
//       P1 = Ar Br,   P2 = Ai Bi,   P3 = (Ar + Ai)(Br + Bi)
//     give  Re C = P1 - P2,  Im C = P3 - P1 - P2 :  6 instead of 8 real flops per complex multiply-add.
// The operands stay interleaved (re, im) exactly as stored: one LDS.128 of the staged tile IS the (Ar, Ai) -- resp.
// (Br, Bi) -- fragment pair of m8n8k4 (A: lane holds row lane>>2, k lane&3; B: k lane&3, column lane>>2), the sum
// fragment costs one DADD, and every DMMA covers 8 x 8 COMPLEX outputs x 4 complex k.  Each thread owns, per m8n8
// tile, the complex outputs (row lane>>2, columns 2(lane&3), 2(lane&3)+1) -- a 32-byte contiguous store.
//
// Staging: cp.async 16 B = one complex element per request, zero-filled out of range (M, N, K, leading dimensions
// and sub-matrix offsets arbitrary), STAGES-deep ring, one __syncthreads per K chunk.  Shared-memory row strides are
// chosen so that both fragment LDS.128 patterns are bank-conflict-free: A stride == 8 (mod 16) doubles, B stride
// == 4 (mod 16) doubles.
#pragma once
#include <cuda.h>
#include <cstring>
#include "zgemm.cuh"

namespace ss {

// ---- TMA staging (experiment, profiles/r02_gemm_tma.md): cp.async.bulk.tensor + mbarrier instead of cp.async
__device__ __forceinline__ void g_mbar_init(unsigned bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void g_mbar_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void g_mbar_wait(unsigned bar, unsigned parity) {
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
__device__ __forceinline__ void tma_load_3d(unsigned smem_dst, const CUtensorMap* map, int c0, int c1, int c2, unsigned bar) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"(smem_dst), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(bar) : "memory");
}

template <int BM_, int BN_, int WARPS_M_, int WARPS_N_, int KC_, int STAGES_, int MINB_, int PF_ = 0, int TMA_ = 0, int SH_ = 0>
struct Gemm3Cfg {
    // 1: both operands come with a sum plane (GemmArgs::shA / shB): a tile of re + im is staged beside every operand tile
    // (row strides LDAS_S, LDBS_S == 4 mod 16 doubles: conflict-free LDS.64 fragments) and the main loop issues no DADD
    static constexpr int SH = SH_;
    static_assert(SH_ == 0 || (PF_ == 1 && TMA_ == 0), "sum planes: software-pipelined cp.async build only");
    static constexpr int BM = BM_, BN = BN_, WARPS_M = WARPS_M_, WARPS_N = WARPS_N_, KC = KC_, STAGES = STAGES_, MINB = MINB_;
    static constexpr int PF = PF_;     // 1: fragments of the next k-step are prefetched across the stage boundary
    // 1: operand tiles staged by TMA (cp.async.bulk.tensor, SWIZZLE_128B boxes of 128-byte rows: the A tile as one box of
    // BM rows x 8 complex k, the B tile as BN/8 boxes of 8 k-rows x 8 complex columns) and published by one mbarrier per
    // stage; unpadded tiles, fragment addresses XOR-swizzled; the 8 k of a stage are consumed as {0,2,4,6} then {1,3,5,7}
    // so that both fragment LDS.128 patterns stay bank-conflict-free under the swizzle.  Needs PF = 1 and KC = 8.
    static constexpr int TMA = TMA_;
    static_assert(TMA_ == 0 || (PF_ == 1 && KC_ == 8 && BN_ % 8 == 0), "TMA staging");
    static constexpr int TMA_STAGE_D = BM * 16 + (BN / 8) * 128;          // doubles per stage (unpadded boxes)
    static constexpr int TMA_SMEM_BYTES = STAGES * TMA_STAGE_D * 8 + 1024 + 8 * STAGES;   // + alignment slack + mbarriers
    static_assert(PF_ == 0 || STAGES_ >= 3, "cross-stage prefetch shortens the cp.async distance by one stage");
    static constexpr int NT = WARPS_M * WARPS_N * 32;
    static constexpr int WM = BM / WARPS_M, WN = BN / WARPS_N;   // warp tile, complex elements
    static constexpr int MI = WM / 8, NJ = WN / 8;               // m8 / n8 tiles per warp
    static constexpr int LDA_S = 2 * KC + 8;                     // doubles
    static constexpr int LDB_S = 2 * BN + 4;                     // doubles
    static constexpr int LDAS_S = KC + 4, LDBS_S = BN + 4;       // doubles: sum tiles
    static constexpr int SUM_A_OFF = BM * LDA_S + KC * LDB_S, SUM_B_OFF = SUM_A_OFF + BM * LDAS_S;
    static constexpr int STAGE_D = BM * LDA_S + KC * LDB_S + (SH_ ? BM * LDAS_S + KC * LDBS_S : 0);      // doubles per stage
    static constexpr int SMEM_BYTES = STAGES * STAGE_D * 8;
    static constexpr int CH_AS = BM * KC / 2, CH_BS = KC * BN / 2;   // 16-byte chunks (2 sums) of the sum tiles per stage
    static constexpr int ITER_AS = (CH_AS + (WARPS_M_ * WARPS_N_ * 32) - 1) / (WARPS_M_ * WARPS_N_ * 32);
    static constexpr int ITER_BS = (CH_BS + (WARPS_M_ * WARPS_N_ * 32) - 1) / (WARPS_M_ * WARPS_N_ * 32);
    static_assert(SH_ == 0 || (LDAS_S % 16 == 4 || LDAS_S % 16 == 12) , "bank layout of the A sum tile");
    static_assert(SH_ == 0 || (LDBS_S % 16 == 4 || LDBS_S % 16 == 12), "bank layout of the B sum tile");
    static constexpr int CH_A = BM * KC, CH_B = KC * BN;         // 16-byte chunks per stage
    static constexpr int ITER_A = (CH_A + NT - 1) / NT, ITER_B = (CH_B + NT - 1) / NT;
    static_assert(WM % 8 == 0 && WN % 8 == 0 && KC % 4 == 0, "warp tile");
    static_assert((2 * KC) % 16 == 0 && (2 * BN) % 16 == 0, "bank layout");
    static_assert(LDA_S % 16 == 8 && LDB_S % 16 == 4, "bank layout");
};

struct GemmTmaMaps { CUtensorMap a, b; };

template <class Cfg, int EPI>
__global__ void __launch_bounds__(Cfg::NT, Cfg::MINB) zgemm3m_kernel(const GemmArgs p, const __grid_constant__ GemmTmaMaps tm) {
    extern __shared__ __align__(16) double smem_raw[];
    constexpr int BM = Cfg::BM, BN = Cfg::BN, KC = Cfg::KC, STAGES = Cfg::STAGES;
    constexpr int NT = Cfg::NT, MI = Cfg::MI, NJ = Cfg::NJ, LDA_S = Cfg::LDA_S, LDB_S = Cfg::LDB_S;
    constexpr int STAGE_D = Cfg::TMA ? Cfg::TMA_STAGE_D : Cfg::STAGE_D;
    // TMA boxes with the 128-byte swizzle need 1024-byte aligned destinations
    double* smem = Cfg::TMA ? reinterpret_cast<double*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023) : smem_raw;

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
    const double* __restrict__ As_g = Cfg::SH ? p.shA_d + (Ag - p.shA_c) : nullptr;      // re + im of the operands' elements
    const double* __restrict__ Bs_g = Cfg::SH ? p.shB_d + (Bg - p.shB_c) : nullptr;

    // ---- per-thread staging state (chunk c of the A tile: row c / KC, k c % KC; of the B tile: k c / BN, col c % BN).
    // Stages are loaded in increasing k order, so each chunk keeps a running global pointer; shared-memory destinations
    // are 32-bit shared-space addresses; the per-chunk size (16 or 0 = zero fill for rows / columns beyond M / N) is loop
    // invariant, and only the last, partial k-chunk takes the predicated path.  (The first version recomputed pointers,
    // predicates and selects for every chunk of every stage: ~85 integer instructions per 48 DMMA.)
    constexpr bool LEAN = (Cfg::PF == 0);
    const cplx* a_p[Cfg::ITER_A]; unsigned a_sd[Cfg::ITER_A]; int a_sz[Cfg::ITER_A];
    const unsigned smem_u32 = (unsigned)__cvta_generic_to_shared(smem);
#pragma unroll
    for (int q = 0; q < Cfg::ITER_A; q++) {
        int c = tid + q * NT;
        int row = c / KC, kc = c % KC;
        bool in = (c < Cfg::CH_A);
        bool ok = in && (m0 + row) < M;
        a_sz[q] = ok ? 16 : (in ? 0 : -1);                   // -1: no such chunk
        a_p[q] = Ag + (long long)(ok ? (m0 + row) : 0) * p.lda + kc;
        a_sd[q] = smem_u32 + 8u * (unsigned)(row * LDA_S + 2 * kc);
    }
    const cplx* b_p[Cfg::ITER_B]; unsigned b_sd[Cfg::ITER_B]; int b_sz[Cfg::ITER_B];
#pragma unroll
    for (int q = 0; q < Cfg::ITER_B; q++) {
        int c = tid + q * NT;
        int kr = c / BN, col = c % BN;
        bool in = (c < Cfg::CH_B);
        bool ok = in && (n0 + col) < N;
        b_sz[q] = ok ? 16 : (in ? 0 : -1);
        b_p[q] = Bg + (long long)kr * p.ldb + (ok ? (n0 + col) : 0);
        b_sd[q] = smem_u32 + 8u * (unsigned)(BM * LDA_S + kr * LDB_S + 2 * col);
    }
    const long long b_step = (long long)KC * p.ldb;

    auto cp16 = [](unsigned sdst, const void* g, int bytes) {
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(sdst), "l"(g), "r"(bytes));
    };
    auto load_stage_lean = [&](int kt, int stage) {            // called with kt = 0, 1, 2, ... in order
        const unsigned soff = (unsigned)(stage * STAGE_D * 8);
        const int k0 = kt * KC;
        if (__builtin_expect(k0 + KC <= K, 1)) {
#pragma unroll
            for (int q = 0; q < Cfg::ITER_A; q++) {
                if (a_sz[q] >= 0) cp16(a_sd[q] + soff, a_p[q], a_sz[q]);
                a_p[q] += KC;
            }
#pragma unroll
            for (int q = 0; q < Cfg::ITER_B; q++) {
                if (b_sz[q] >= 0) cp16(b_sd[q] + soff, b_p[q], b_sz[q]);
                b_p[q] += b_step;
            }
        } else {                                               // last, partial k-chunk: zero-fill k >= K
            asm volatile("" ::: "memory");                       // keep this rare path a real branch
#pragma unroll
            for (int q = 0; q < Cfg::ITER_A; q++) {
                int kc = (tid + q * NT) % KC;
                bool ok = (k0 + kc < K);
                if (a_sz[q] >= 0) cp16(a_sd[q] + soff, ok ? (const void*)a_p[q] : (const void*)Ag, ok ? a_sz[q] : 0);
                a_p[q] += KC;
            }
#pragma unroll
            for (int q = 0; q < Cfg::ITER_B; q++) {
                int kr = (tid + q * NT) / BN;
                bool ok = (k0 + kr < K);
                if (b_sz[q] >= 0) cp16(b_sd[q] + soff, ok ? (const void*)b_p[q] : (const void*)Bg, ok ? b_sz[q] : 0);
                b_p[q] += b_step;
            }
        }
    };

    // ---- staging of the software-pipelined build (PF = 1): descriptors kept per chunk, address and predicate formed per
    // stage.  Measured, that kernel is faster with this form (44.2 vs 43.6 TFLOP/s at 2048^3 x 16) and the plain loop with
    // the running pointers above (43.6 vs 42.0); only the state of the form an instantiation uses survives in it.
    const cplx* a_src[Cfg::ITER_A]; int a_dst[Cfg::ITER_A]; int a_kc[Cfg::ITER_A]; bool a_ok[Cfg::ITER_A];
    const cplx* b_src[Cfg::ITER_B]; int b_dst[Cfg::ITER_B]; int b_kr[Cfg::ITER_B]; bool b_ok[Cfg::ITER_B];
    if constexpr (!LEAN) {
#pragma unroll
        for (int q = 0; q < Cfg::ITER_A; q++) {
            int c = tid + q * NT;
            int row = c / KC, kc = c % KC;
            a_kc[q] = (c < Cfg::CH_A) ? kc : (1 << 28);          // beyond the tile: never in range
            a_ok[q] = (c < Cfg::CH_A) && (m0 + row) < M;
            a_src[q] = Ag + (long long)(a_ok[q] ? (m0 + row) : 0) * p.lda + kc;
            a_dst[q] = (c < Cfg::CH_A) ? row * LDA_S + 2 * kc : -1;
        }
#pragma unroll
        for (int q = 0; q < Cfg::ITER_B; q++) {
            int c = tid + q * NT;
            int kr = c / BN, col = c % BN;
            b_kr[q] = (c < Cfg::CH_B) ? kr : (1 << 28);
            b_ok[q] = (c < Cfg::CH_B) && (n0 + col) < N;
            b_src[q] = Bg + (long long)kr * p.ldb + (b_ok[q] ? (n0 + col) : 0);
            b_dst[q] = (c < Cfg::CH_B) ? BM * LDA_S + kr * LDB_S + 2 * col : -1;
        }
    }
    auto load_stage_desc = [&](int kt, int stage) {
        double* sbase = smem + stage * STAGE_D;
        const int k0 = kt * KC;
#pragma unroll
        for (int q = 0; q < Cfg::ITER_A; q++) {
            if (a_dst[q] < 0) continue;
            bool ok = a_ok[q] && (k0 + a_kc[q] < K);
            cp_async16(sbase + a_dst[q], ok ? (const void*)(a_src[q] + k0) : (const void*)Ag, ok ? 16 : 0);
        }
#pragma unroll
        for (int q = 0; q < Cfg::ITER_B; q++) {
            if (b_dst[q] < 0) continue;
            bool ok = b_ok[q] && (k0 + b_kr[q] < K);
            cp_async16(sbase + b_dst[q], ok ? (const void*)(b_src[q] + (long long)k0 * p.ldb) : (const void*)Bg, ok ? 16 : 0);
        }
        if constexpr (Cfg::SH) {                          // the sum tiles: 16-byte chunks = two sums (K, N, lda, ldb even)
#pragma unroll
            for (int q = 0; q < Cfg::ITER_AS; q++) {
                const int c = tid + q * NT;
                if (c >= Cfg::CH_AS) continue;
                const int row = c / (KC / 2), k2 = 2 * (c % (KC / 2));
                const bool ok = (m0 + row) < M && (k0 + k2) < K;
                cp_async16(sbase + Cfg::SUM_A_OFF + row * Cfg::LDAS_S + k2,
                           ok ? (const void*)(As_g + (long long)(m0 + row) * p.lda + k0 + k2) : (const void*)Ag, ok ? 16 : 0);
            }
#pragma unroll
            for (int q = 0; q < Cfg::ITER_BS; q++) {
                const int c = tid + q * NT;
                if (c >= Cfg::CH_BS) continue;
                const int kr = c / (BN / 2), c2 = 2 * (c % (BN / 2));
                const bool ok = (k0 + kr) < K && (n0 + c2) < N;
                cp_async16(sbase + Cfg::SUM_B_OFF + kr * Cfg::LDBS_S + c2,
                           ok ? (const void*)(Bs_g + (long long)(k0 + kr) * p.ldb + n0 + c2) : (const void*)Bg, ok ? 16 : 0);
            }
        }
    };

    const unsigned tma_bars = (unsigned)__cvta_generic_to_shared(smem + STAGES * STAGE_D);     // STAGES mbarriers behind the tiles
    auto load_stage = [&](int kt, int stage) {
        if constexpr (Cfg::TMA) {
            if (tid == 0) {
                const unsigned bar = tma_bars + 8u * stage;
                const unsigned dst = (unsigned)__cvta_generic_to_shared(smem + stage * STAGE_D);
                g_mbar_expect_tx(bar, (unsigned)(STAGE_D * 8));
                tma_load_3d(dst, &tm.a, 2 * kt * KC, m0, z, bar);
#pragma unroll
                for (int jb = 0; jb < BN / 8; jb++)
                    tma_load_3d(dst + (unsigned)((BM * 16 + jb * 128) * 8), &tm.b, 2 * (n0 + 8 * jb), kt * KC, z, bar);
            }
        } else if constexpr (LEAN) load_stage_lean(kt, stage); else load_stage_desc(kt, stage);
    };
    if constexpr (Cfg::TMA) {
        if (tid == 0) {
            for (int i = 0; i < STAGES; i++) g_mbar_init(tma_bars + 8u * i, 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        __syncthreads();
    }

    // ---- fragment offsets (doubles, within a stage)
    const int wm0 = (warp / Cfg::WARPS_N) * Cfg::WM, wn0 = (warp % Cfg::WARPS_N) * Cfg::WN;
    const int a_off = (wm0 + g) * LDA_S + 2 * t;                        // + 8 i LDA_S + 8 ks
    const int b_off = BM * LDA_S + t * LDB_S + 2 * (wn0 + g);           // + 16 j + 4 ks LDB_S

    double P1[MI][NJ][2], P2[MI][NJ][2], P3[MI][NJ][2];
#pragma unroll
    for (int i = 0; i < MI; i++)
#pragma unroll
        for (int j = 0; j < NJ; j++) {
            P1[i][j][0] = P1[i][j][1] = 0.0;
            P2[i][j][0] = P2[i][j][1] = 0.0;
            P3[i][j][0] = P3[i][j][1] = 0.0;
        }

    const int KT = (K + KC - 1) / KC;
#pragma unroll
    for (int s = 0; s < STAGES - 1; s++) {
        if (s < KT) load_stage(s, s);
        cp_async_commit();
    }

    if (Cfg::PF == 0) {
        for (int kt = 0; kt < KT; kt++) {
            cp_async_wait<STAGES - 2>();
            __syncthreads();
            {
                int nk = kt + STAGES - 1;
                if (nk < KT) load_stage(nk, nk % STAGES);
                cp_async_commit();
            }
            const double* sS = smem + (kt % STAGES) * STAGE_D;
    #pragma unroll
            for (int ks = 0; ks < KC / 4; ks++) {
                double ar[MI], ai[MI], as[MI], br[NJ], bi[NJ], bs[NJ];
    #pragma unroll
                for (int i = 0; i < MI; i++) {
                    double2 v = *reinterpret_cast<const double2*>(sS + a_off + 8 * i * LDA_S + 8 * ks);
                    ar[i] = v.x; ai[i] = v.y; as[i] = v.x + v.y;
                }
    #pragma unroll
                for (int j = 0; j < NJ; j++) {
                    double2 v = *reinterpret_cast<const double2*>(sS + b_off + 16 * j + 4 * ks * LDB_S);
                    br[j] = v.x; bi[j] = v.y; bs[j] = v.x + v.y;
                }
    #pragma unroll
                for (int i = 0; i < MI; i++)
    #pragma unroll
                    for (int j = 0; j < NJ; j++) {
                        dmma884(P1[i][j][0], P1[i][j][1], ar[i], br[j]);
                        dmma884(P2[i][j][0], P2[i][j][1], ai[i], bi[j]);
                        dmma884(P3[i][j][0], P3[i][j][1], as[i], bs[j]);
                    }
            }
        }
    } else {
        // Same product, software-pipelined across the stage boundary: the CTA barrier that publishes stage kt+1 sits
        // BEFORE the last k-step of stage kt, so that the first fragments of stage kt+1 are already in registers when
        // stage kt's last DMMAs issue -- no warp starts a stage by waiting for its LDS.
        constexpr int KS = KC / 4;
        double fa[2][MI][2], fb[2][NJ][2];
        double fsa[2][Cfg::SH ? MI : 1], fsb[2][Cfg::SH ? NJ : 1];
        const int sa_off = Cfg::SUM_A_OFF + (wm0 + g) * Cfg::LDAS_S + t, sb_off = Cfg::SUM_B_OFF + t * Cfg::LDBS_S + wn0 + g;
        // TMA layout (doubles within a stage): A row r at 16 r, complex k chunk c at ((c ^ (r & 7)) << 1); B box jb at
        // 16 BM + 128 jb, k row kk at 16 kk, complex column cc at ((cc ^ (kk & 7)) << 1).  k-step ks uses the chunks 2t + ks.
        const int ta_off0 = (wm0 + g) * 16 + (((2 * t) ^ g) << 1), ta_off1 = (wm0 + g) * 16 + (((2 * t + 1) ^ g) << 1);
        const int tb_off0 = BM * 16 + (wn0 >> 3) * 128 + (2 * t) * 16 + ((g ^ (2 * t)) << 1);
        const int tb_off1 = BM * 16 + (wn0 >> 3) * 128 + (2 * t + 1) * 16 + ((g ^ (2 * t + 1)) << 1);
        auto load_frag = [&](int buf, const double* sS, int ks) {
            if constexpr (Cfg::TMA) {
                const int ao = ks ? ta_off1 : ta_off0, bo = ks ? tb_off1 : tb_off0;
#pragma unroll
                for (int i = 0; i < MI; i++) {
                    double2 v = *reinterpret_cast<const double2*>(sS + ao + 8 * 16 * i);
                    fa[buf][i][0] = v.x; fa[buf][i][1] = v.y;
                }
#pragma unroll
                for (int j = 0; j < NJ; j++) {
                    double2 v = *reinterpret_cast<const double2*>(sS + bo + 128 * j);
                    fb[buf][j][0] = v.x; fb[buf][j][1] = v.y;
                }
            } else {
#pragma unroll
                for (int i = 0; i < MI; i++) {
                    double2 v = *reinterpret_cast<const double2*>(sS + a_off + 8 * i * LDA_S + 8 * ks);
                    fa[buf][i][0] = v.x; fa[buf][i][1] = v.y;
                }
#pragma unroll
                for (int j = 0; j < NJ; j++) {
                    double2 v = *reinterpret_cast<const double2*>(sS + b_off + 16 * j + 4 * ks * LDB_S);
                    fb[buf][j][0] = v.x; fb[buf][j][1] = v.y;
                }
                if constexpr (Cfg::SH) {
#pragma unroll
                    for (int i = 0; i < MI; i++) fsa[buf][i] = sS[sa_off + 8 * i * Cfg::LDAS_S + 4 * ks];
#pragma unroll
                    for (int j = 0; j < NJ; j++) fsb[buf][j] = sS[sb_off + 4 * ks * Cfg::LDBS_S + 8 * j];
                }
            }
        };
        auto stage_landed = [&](int kt) {                 // stage kt is complete in shared memory (for this thread)
            if constexpr (Cfg::TMA) g_mbar_wait(tma_bars + 8u * (kt % STAGES), (unsigned)((kt / STAGES) & 1));
        };
        if constexpr (Cfg::TMA) { if (KT > 0) stage_landed(0); } else cp_async_wait<STAGES - 2>();
        __syncthreads();
        if (KT > 0) load_frag(0, smem, 0);
        int cur = 0;
        for (int kt = 0; kt < KT; kt++) {
            const double* sS = smem + (kt % STAGES) * STAGE_D;
#pragma unroll
            for (int ks = 0; ks < KS; ks++) {
                if (ks == KS - 1) {
                    // stage kt+1 must have landed (groups committed so far: STAGES-1+kt; needed complete: kt+2)
                    if constexpr (Cfg::TMA) { if (kt + 1 < KT) stage_landed(kt + 1); } else cp_async_wait<STAGES - 3>();
                    __syncthreads();
                    int nk = kt + STAGES - 1;
                    if (nk < KT) load_stage(nk, nk % STAGES);      // slot (kt-1) % STAGES: everyone is past stage kt-1
                    cp_async_commit();
                    if (kt + 1 < KT) load_frag(cur ^ 1, smem + ((kt + 1) % STAGES) * STAGE_D, 0);
                } else {
                    load_frag(cur ^ 1, sS, ks + 1);
                }
                double as[MI], bs[NJ];
#ifdef SS_EXP_NOSUM          // experiment only (WRONG results): the main loop without the fragment-sum DADDs, profiles/r02_gemm_sumplane.md
                if constexpr (true) {
#pragma unroll
                    for (int i = 0; i < MI; i++) as[i] = fa[cur][i][0];
#pragma unroll
                    for (int j = 0; j < NJ; j++) bs[j] = fb[cur][j][1];
                } else
#endif
                if constexpr (Cfg::SH) {                  // the sums were staged with the operands: no DADD on the DMMA pipe
#pragma unroll
                    for (int i = 0; i < MI; i++) as[i] = fsa[cur][i];
#pragma unroll
                    for (int j = 0; j < NJ; j++) bs[j] = fsb[cur][j];
                } else {
#pragma unroll
                    for (int i = 0; i < MI; i++) as[i] = fa[cur][i][0] + fa[cur][i][1];
#pragma unroll
                    for (int j = 0; j < NJ; j++) bs[j] = fb[cur][j][0] + fb[cur][j][1];
                }
#pragma unroll
                for (int i = 0; i < MI; i++)
#pragma unroll
                    for (int j = 0; j < NJ; j++) {
                        dmma884(P1[i][j][0], P1[i][j][1], fa[cur][i][0], fb[cur][j][0]);
                        dmma884(P2[i][j][0], P2[i][j][1], fa[cur][i][1], fb[cur][j][1]);
                        dmma884(P3[i][j][0], P3[i][j][1], as[i], bs[j]);
                    }
                cur ^= 1;
            }
        }
    }
    cp_async_wait<0>();

    // ---- epilogue: thread owns complex C[m0+wm0+8i+g][n0+wn0+8j+2t+h], h = 0, 1
    cplx* __restrict__ Cg = bptr(p.C, z);
    if (EPI == EPI_STD) {
        const cplx* Cin = (p.beta != 0.0) ? bptr(p.Cin, z) : nullptr;
        const double alpha = p.alpha, beta = p.beta;
        // C += alpha A B in place (the LU / TRSM updates): red.global.add.f64 instead of load-add-store.  Every element
        // is written by exactly one thread and receives exactly one addition, so the result is the same correctly
        // rounded c + alpha*acc, deterministic -- but no warp waits for a global load at the end of its tile.
        const bool red = (beta == 1.0) && (Cin == Cg) && (p.ldcin == p.ldc);
#pragma unroll
        for (int i = 0; i < MI; i++) {
            int row = m0 + wm0 + 8 * i + g;
            if (row >= M) continue;
#pragma unroll
            for (int j = 0; j < NJ; j++) {
#pragma unroll
                for (int h = 0; h < 2; h++) {
                    int col = n0 + wn0 + 8 * j + 2 * t + h;
                    if (col >= N) continue;
                    // alpha = +-1 (every product of the path): no multiplies -- each FP64 instruction of the epilogue
                    // costs the DMMA pipe ~6 cycles, 5 per element were 8 % of a K = 128 tile.  -(x) is exact, so the
                    // results are bit-identical to alpha * (...)
                    cplx o;
                    if (alpha == -1.0) {
                        o = make_c(P2[i][j][h] - P1[i][j][h], (P1[i][j][h] - P3[i][j][h]) + P2[i][j][h]);
                    } else {
                        o = make_c(P1[i][j][h] - P2[i][j][h], (P3[i][j][h] - P1[i][j][h]) - P2[i][j][h]);
                        if (alpha != 1.0) { o.re *= alpha; o.im *= alpha; }
                    }
                    if (red) {
                        double* dst = reinterpret_cast<double*>(Cg + (long long)row * p.ldc + col);
                        atomicAdd(dst, o.re);
                        atomicAdd(dst + 1, o.im);
                        continue;
                    }
                    if (Cin) {
                        cplx c = Cin[(long long)row * p.ldcin + col];
                        o.re = fma(beta, c.re, o.re);
                        o.im = fma(beta, c.im, o.im);
                    }
                    Cg[(long long)row * p.ldc + col] = o;
                    if (p.shC_d) p.shC_d[(Cg - p.shC_c) + (long long)row * p.ldc + col] = o.re + o.im;
                }
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
#pragma unroll
                for (int h = 0; h < 2; h++) {
                    int col = n0 + wn0 + 8 * j + 2 * t + h;
                    if (col >= N) continue;
                    double re = P1[i][j][h] - P2[i][j][h];
                    double im = P3[i][j][h] - P1[i][j][h] - P2[i][j][h];
                    long long off = (long long)row * p.lds + col;
                    cplx s = Sg[off], hh = Hg[off];
                    cplx d = cmul(Ee, s);
                    Cg[(long long)row * p.ldc + col] = make_c(d.re - hh.re - re, d.im - hh.im - im);
                }
            }
        }
    }
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda)
typedef CUresult (*TmapEncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                 const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static TmapEncodeFn tmap_encode_fn() {
    static TmapEncodeFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
            fn = (TmapEncodeFn)p;
    }
    return fn;
}
// rows x cols complex (row-major, ld) x batch (stride in complex elements) seen as FLOAT64 [batch][rows][2 cols]
static bool tmap_make(CUtensorMap* m, const cplx* base, long long rows, long long cols, long long ld, long long bstride, int batch,
                      int box_rows) {
    TmapEncodeFn fn = tmap_encode_fn();
    if (!fn || rows < 1 || cols < 1) return false;
    if (batch <= 1 || bstride <= 0) bstride = rows * ld;
    cuuint64_t dims[3] = {(cuuint64_t)(2 * cols), (cuuint64_t)rows, (cuuint64_t)(batch < 1 ? 1 : batch)};
    cuuint64_t strides[2] = {(cuuint64_t)ld * 16, (cuuint64_t)bstride * 16};
    cuuint32_t box[3] = {16, (cuuint32_t)box_rows, 1}, es[3] = {1, 1, 1};
    return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, (void*)base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
              CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <class Cfg, int EPI>
static cudaError_t gemm3m_launch_t(GemmArgs a, int batch, cudaStream_t st) {
    auto kern = zgemm3m_kernel<Cfg, EPI>;
    constexpr int SMEM = Cfg::TMA ? Cfg::TMA_SMEM_BYTES : Cfg::SMEM_BYTES;
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    a.tiles_m = (a.M + Cfg::BM - 1) / Cfg::BM;
    a.tiles_n = (a.N + Cfg::BN - 1) / Cfg::BN;
    a.raster_gm = g_gemm_raster;
    if (a.tiles_m == 0 || a.tiles_n == 0 || batch == 0) return cudaSuccess;
    GemmTmaMaps tm;
    if constexpr (Cfg::TMA) {
        if (!tmap_make(&tm.a, a.A.p0, a.M, a.K, a.lda, a.A.s_in, batch, Cfg::BM) ||
            !tmap_make(&tm.b, a.B.p0, a.K, a.N, a.ldb, a.B.s_in, batch, 8))
            return cudaErrorInvalidValue;
    } else {
        memset(&tm, 0, sizeof(tm));
    }
    dim3 grid((unsigned)(a.tiles_m * a.tiles_n), (unsigned)batch, 1);
    kern<<<grid, Cfg::NT, SMEM, st>>>(a, tm);
    return cudaGetLastError();
}

// tile configurations.  Measured on B200 at M=N=K=2048 x 16 (profiles/r01_gemm_variants.md): the small tile with
// several independent CTAs per SM wins (43.6 TFLOP/s LAPACK-convention, 44.2 with the prefetching main loop, vs 34.1
// for 4M): with one CTA per SM every __syncthreads idles the whole DMMA pipe, and larger warp tiles do not fit 3
// accumulator sets in registers.  The other tile shapes tried in round 1 (64x64, 64x96, 128x48, 64x48, 96x32, 3-stage
// ring) are recorded in that file and are no longer built.
using C3_64x32s4 = Gemm3Cfg<64, 32, 2, 2, 8, 4, 3>;      // 4 warps of 32x16, 4-stage ring, 3 CTAs/SM
using C3_64x32pf = Gemm3Cfg<64, 32, 2, 2, 8, 4, 2, 1>;   // 4 warps of 32x16, cross-stage fragment prefetch, 220 registers, 2 CTAs/SM
using C3_64x32sh = Gemm3Cfg<64, 32, 2, 2, 8, 4, 2, 1, 0, 1>; // the same main loop fed with staged sum tiles (no fragment-sum DADDs)
using C3_64x32tma = Gemm3Cfg<64, 32, 2, 2, 8, 4, 2, 1, 1>;  // the same main loop, operand tiles staged by TMA (experiment)
using C3_64x32tma3 = Gemm3Cfg<64, 32, 2, 2, 8, 4, 3, 1, 1>; // same at 3 CTAs/SM (the TMA build needs 168 registers)
using C3_Tall = Gemm3Cfg<128, 16, 4, 1, 8, 4, 2>;        // one CTA owns all (<=128) rows of its 16 columns: in-place L^-1 * A12

// GEMM variants: 0 = 4M (zgemm.cuh), 1 = 3M, kernel chosen by K (the default), 2 / 3 = the two 3M kernels for every K.
// GEMM_TALL always maps to the one-CTA-per-column configuration of the same arithmetic.
enum { GV_4M = 0, GV_3M = 1, GV_3M_LEAN = 2, GV_3M_PF = 3, GV_3M_TMA = 4, GV_3M_TMA3 = 5, GV_COUNT = 6 };

template <class Cfg>
static cudaError_t gemm3m_epi(const GemmArgs& a, int batch, int epi, cudaStream_t st) {
    if (epi == EPI_SCHUR) return gemm3m_launch_t<Cfg, EPI_SCHUR>(a, batch, st);
    return gemm3m_launch_t<Cfg, EPI_STD>(a, batch, st);
}

static cudaError_t gemm_launch(const GemmArgs& a, int batch, int cfg, int epi, cudaStream_t st, int variant) {
    if (variant == GV_4M) return gemm4m_launch(a, batch, cfg, epi, st);
    if (cfg == GEMM_TALL) return gemm3m_launch_t<C3_Tall, EPI_STD>(a, batch, st);
    // default: the 64x32 tile at 3 CTAs/SM (lean staging code: 43.6 TFLOP/s at 2048^3 x 16, 38.9 at K = 128); for long K the
    // software-pipelined main loop (fragments of the next k-step prefetched across the stage boundary, 2 CTAs/SM) is
    // another 1-2 % faster (44.2 / 44.6 at 2048^3 / 4096^3); the crossover measured on isolated launches lies near
    // K = 1200, inside the solve (4 stream groups) K >= 768 is at least as good (profiles/r01_gemm_variants.md)
    if (variant == GV_3M) variant = (a.K >= 768) ? GV_3M_PF : GV_3M_LEAN;
    if (variant == GV_3M_TMA || variant == GV_3M_TMA3) {
        // TMA tensor maps describe uniformly strided batches of whole matrices; anything else takes the cp.async kernel
        const bool ok = !a.A.two && !a.B.two && a.A.n_in >= batch && a.B.n_in >= batch && a.K > 0 &&
                        (batch <= 1 || (a.A.s_in > 0 && a.B.s_in > 0));
        if (ok) {
            cudaError_t e = variant == GV_3M_TMA3 ? gemm3m_epi<C3_64x32tma3>(a, batch, epi, st) : gemm3m_epi<C3_64x32tma>(a, batch, epi, st);
            if (e != cudaErrorInvalidValue) return e;     // cudaErrorInvalidValue = the tensor maps could not be encoded (nothing was
            cudaGetLastError();                           // launched): take the cp.async kernel instead of failing the product
        }
        variant = GV_3M_PF;
    }
    if (variant == GV_3M_PF) {
        // both operands inside regions with sum planes, everything even (two sums per 16-byte staging request)
        auto even = [](const BPtr& b, const cplx* base) {
            return ((b.p0 - base) % 2 == 0) && (!b.p1 || (b.p1 - base) % 2 == 0) && b.s_in % 2 == 0 && b.s_out % 2 == 0;
        };
        const bool sh = a.shA_d && a.shB_d && a.K % 2 == 0 && a.N % 2 == 0 && a.lda % 2 == 0 && a.ldb % 2 == 0 &&
                        even(a.A, a.shA_c) && even(a.B, a.shB_c);
        if (sh) return gemm3m_epi<C3_64x32sh>(a, batch, epi, st);
        return gemm3m_epi<C3_64x32pf>(a, batch, epi, st);
    }
    return gemm3m_epi<C3_64x32s4>(a, batch, epi, st);
}

}  // namespace ss
