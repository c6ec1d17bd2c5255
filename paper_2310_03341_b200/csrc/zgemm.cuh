// zgemm.cuh -- complex-FP64 GEMM engine on the FP64 tensor-core path (mma.sync m8n8k4 -> DMMA.8x8x4).
//
//   C <- alpha * opA(A1) opB(B1) [+ alpha * opA(A2) opB(B2)] + beta * C            (ZMODE_GEMM)
//   C <- Herm(A1) * B1,  A1 Hermitian with only the lower triangle + 64-aligned diagonal
//        blocks valid                                                                (ZMODE_HEMM)
//
// Used by S1 (V^H V, V T, HEMM-lower, V^H X, W, HER2K-lower) and S4b (WY application),
// SURVEY.md 8(a) rows S1.2-S1.5, S4b.  One complex MAC = 4 real DMMAs on (re, im) fragments;
// conjugation is folded into fragment sign flips.  Tiles are staged global -> shared with a
// 4-stage cp.async (LDGSTS) pipeline; shared-memory strides are padded so that every 128-bit
// fragment load of a quarter warp hits 8 distinct 16-byte bank groups.
#pragma once
#include "common.cuh"

namespace eigh {

struct ZgemmArgs {
    int M, N;
    int K1, K2;                       // inner lengths of pair 1 and (optional) pair 2
    const c128 *A1, *B1, *A2, *B2;
    int64_t lda1, ldb1, lda2, ldb2;
    c128* C;
    int64_t ldc;
    double alpha, beta;
    int lower_only;                   // skip tiles strictly above the diagonal
    int splitk;                       // >= 1
    c128* partial;                    // [splitk][N][M] raw accumulators when splitk > 1
};

enum { ZMODE_GEMM = 0, ZMODE_HEMM = 1 };

constexpr int ZG_BK = 8;
constexpr int ZG_STAGES = 4;
constexpr int ZG_KSTRIDE = ZG_BK + 4;   // K-contiguous tiles: stride == 4 (mod 8) 16B-units

// NJ = 8-column fragments per warp in N (warp tile 32 x 8 NJ): 4 for the 4-multiplication kernel, 2 for the 3M one
template <int WARPS_M, int WARPS_N, bool TA, bool TB, int MODE, int NJ = 4>
struct ZgemmCfg {
    static constexpr int BM = 32 * WARPS_M, BN = 8 * NJ * WARPS_N, NT = 32 * WARPS_M * WARPS_N;
    static constexpr int SA_N = BM + 2;                       // M-contiguous A tile: As[k][m]
    static constexpr int SB_C = BN + 2;                       // N-contiguous B tile: Bs[k][n]
    static constexpr int A_N_SIZE = ZG_BK * SA_N, A_C_SIZE = BM * ZG_KSTRIDE;
    static constexpr int A_STAGE = (MODE == ZMODE_HEMM) ? (A_N_SIZE > A_C_SIZE ? A_N_SIZE : A_C_SIZE)
                                                         : (TA ? A_C_SIZE : A_N_SIZE);
    static constexpr int B_STAGE = TB ? ZG_BK * SB_C : BN * ZG_KSTRIDE;
    static constexpr int STAGE = A_STAGE + B_STAGE;
    static constexpr size_t SMEM_BYTES = (size_t)ZG_STAGES * STAGE * sizeof(c128);
};

// One k-step (4 complex k) x 2 per stage.  ACT: A tile is K-contiguous (As[m][k]); CONJA: conj(A).
template <int BM, int BN, bool ACT, bool CONJA, bool BCT, bool CONJB>
__device__ __forceinline__ void zgemm_compute_stage(const c128* __restrict__ As, const c128* __restrict__ Bs,
                                                    int wm0, int wn0, int g, int t,
                                                    double (&cr)[4][4][2], double (&ci)[4][4][2]) {
    constexpr int SA_N = BM + 2, SB_C = BN + 2;
#pragma unroll
    for (int kk = 0; kk < ZG_BK; kk += 4) {
        double ar[4], ai[4], nai[4], br[4], bi[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int m = wm0 + 8 * i + g;
            const c128 a = ACT ? As[m * ZG_KSTRIDE + kk + t] : As[(kk + t) * SA_N + m];
            ar[i] = a.x;
            ai[i] = CONJA ? -a.y : a.y;
            nai[i] = CONJA ? a.y : -a.y;
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int n = wn0 + 8 * j + g;
            const c128 b = BCT ? Bs[(kk + t) * SB_C + n] : Bs[n * ZG_KSTRIDE + kk + t];
            br[j] = b.x;
            bi[j] = CONJB ? -b.y : b.y;
        }
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) dmma884p(cr[i][j][0], cr[i][j][1], ar[i], br[j]);
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) dmma884p(ci[i][j][0], ci[i][j][1], ar[i], bi[j]);
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) dmma884p(cr[i][j][0], cr[i][j][1], nai[i], bi[j]);
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) dmma884p(ci[i][j][0], ci[i][j][1], ai[i], br[j]);
    }
}

// 3M variant (Karatsuba / "zgemm3m"): three real products per complex multiply-add,
//   S1 += ar br,  S2 += ai bi,  S3 += (ar + ai)(br + bi);   Re = S1 - S2,  Im = S3 - S1 - S2  (combined once, after the K loop).
// 25 % fewer DMMAs for two extra DADDs per fragment; normwise error bound of the same order as the conventional
// product (the imaginary part loses componentwise, not normwise, accuracy).  Warp tile 32 x 8 NJ.
template <int BM, int BN, int NJ, bool ACT, bool CONJA, bool BCT, bool CONJB>
__device__ __forceinline__ void zgemm_compute_stage_3m(const c128* __restrict__ As, const c128* __restrict__ Bs,
                                                       int wm0, int wn0, int g, int t, double (&s1)[4][NJ][2],
                                                       double (&s2)[4][NJ][2], double (&s3)[4][NJ][2]) {
    constexpr int SA_N = BM + 2, SB_C = BN + 2;
#pragma unroll
    for (int kk = 0; kk < ZG_BK; kk += 4) {
        double ar[4], ai[4], as[4], br[NJ], bi[NJ], bs[NJ];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int m = wm0 + 8 * i + g;
            const c128 a = ACT ? As[m * ZG_KSTRIDE + kk + t] : As[(kk + t) * SA_N + m];
            ar[i] = a.x;
            ai[i] = CONJA ? -a.y : a.y;
            as[i] = ar[i] + ai[i];
        }
#pragma unroll
        for (int j = 0; j < NJ; ++j) {
            const int n = wn0 + 8 * j + g;
            const c128 b = BCT ? Bs[(kk + t) * SB_C + n] : Bs[n * ZG_KSTRIDE + kk + t];
            br[j] = b.x;
            bi[j] = CONJB ? -b.y : b.y;
            bs[j] = br[j] + bi[j];
        }
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < NJ; ++j) dmma884p(s1[i][j][0], s1[i][j][1], ar[i], br[j]);
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < NJ; ++j) dmma884p(s2[i][j][0], s2[i][j][1], ai[i], bi[j]);
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < NJ; ++j) dmma884p(s3[i][j][0], s3[i][j][1], as[i], bs[j]);
    }
}

template <int WARPS_M, int WARPS_N, bool TA, bool TB, int MODE, int MINB, int NJ = 4, bool M3 = false>
__global__ void __launch_bounds__(32 * WARPS_M * WARPS_N, MINB) zgemm_kernel(const ZgemmArgs p) {
    using Cfg = ZgemmCfg<WARPS_M, WARPS_N, TA, TB, MODE, NJ>;
    constexpr int BM = Cfg::BM, BN = Cfg::BN, NT = Cfg::NT, BK = ZG_BK;
    static_assert(M3 || NJ == 4, "the 4-multiplication kernel uses 32 x 32 warp tiles");
    extern __shared__ __align__(16) unsigned char zg_smem_raw[];
    c128* smem = reinterpret_cast<c128*>(zg_smem_raw);

    const int m0 = blockIdx.x * BM, n0 = blockIdx.y * BN;
    if (p.lower_only && m0 + BM - 1 < n0) return;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, t = lane & 3;
    const int wm0 = (warp % WARPS_M) * 32, wn0 = (warp / WARPS_M) * (8 * NJ);

    const int nkb1 = (p.K1 + BK - 1) / BK;
    const int nkb2 = (p.A2 != nullptr) ? (p.K2 + BK - 1) / BK : 0;
    const int nkb = nkb1 + nkb2;
    const int per = (nkb + p.splitk - 1) / p.splitk;
    const int kb_begin = blockIdx.z * per;
    const int kb_end = min(nkb, kb_begin + per);

    // 4-multiplication kernel: cr, ci.  3M kernel: cr = S1, ci = S3 and s2 = S2 (combined in the epilogue).
    double cr[4][NJ][2], ci[4][NJ][2], s2[M3 ? 4 : 1][M3 ? NJ : 1][2];
    if (M3) {
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < NJ; ++j) s2[M3 ? i : 0][M3 ? j : 0][0] = s2[M3 ? i : 0][M3 ? j : 0][1] = 0.0;
    }
    // beta == +-alpha: start the accumulators at (beta/alpha) C (exact), so that the read of C overlaps
    // the pipeline prologue instead of serialising the epilogue
    const bool preload = (p.splitk == 1) && (p.beta != 0.0) && (p.beta == p.alpha || p.beta == -p.alpha);
    if (preload) {
        const double sg = (p.beta == p.alpha) ? 1.0 : -1.0;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int row = m0 + wm0 + 8 * i + g;
#pragma unroll
            for (int j = 0; j < NJ; ++j)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int col = n0 + wn0 + 8 * j + 2 * t + e;
                    c128 v = cmake(0.0, 0.0);
                    if (row < p.M && col < p.N) v = p.C[row + (int64_t)col * p.ldc];
                    cr[i][j][e] = sg * v.x;
                    ci[i][j][e] = M3 ? sg * (v.x + v.y) : sg * v.y;      // 3M: Im = S3 - S1 - S2
                }
        }
    } else {
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < NJ; ++j) cr[i][j][0] = cr[i][j][1] = ci[i][j][0] = ci[i][j][1] = 0.0;
    }

    auto a_ctype = [&](int kb) -> bool {
        if (MODE == ZMODE_HEMM) return kb * BK >= m0 + BM;
        return TA;
    };

    // Sequential tile loader.  The blocks kb_begin, kb_begin + 1, ... are requested in order, so every thread keeps, for
    // its NA + NB elements of a stage, the global pointer, the shared-memory slot and the validity of its row / column, and
    // only advances the pointers from block to block.  The state is rebuilt where the operands change: at the start, at
    // the switch to the second (A2, B2) pair and, in HEMM mode, where the A tile turns from "as stored" to "mirrored".
    constexpr int NA = BM * BK / NT, NB = BN * BK / NT;
    const c128* pA[NA];
    const c128* pB[NB];
    int sA[NA], sB[NB], kA[NA], kB[NB];
    bool vA[NA], vB[NB];
    int64_t dA = 0, dB = 0;
    int ld_kb = kb_begin, ld_switch = kb_begin, ld_krem = 0;
    const c128* ld_safe = p.A1;
    auto ld_setup = [&](int kb) {
        const bool second = kb >= nkb1;
        const c128* A = second ? p.A2 : p.A1;
        const c128* B = second ? p.B2 : p.B1;
        const int64_t lda = second ? p.lda2 : p.lda1, ldb = second ? p.ldb2 : p.ldb1;
        const int Kp = second ? p.K2 : p.K1;
        const int k0 = (second ? kb - nkb1 : kb) * BK;
        const bool act = a_ctype(kb);
#pragma unroll
        for (int it = 0; it < NA; ++it) {
            const int idx = tid + it * NT;
            int m, k;
            if (!act) { m = idx % BM; k = idx / BM; }        // A element (m,k) at A[m + k*lda], M-contiguous
            else      { k = idx % BK; m = idx / BK; }        // A element (m,k) = conj(A[k + m*lda]), K-contiguous
            const int gm = m0 + m;
            vA[it] = gm < p.M;
            kA[it] = k;
            pA[it] = !act ? A + gm + (int64_t)(k0 + k) * lda : A + (k0 + k) + (int64_t)gm * lda;
            sA[it] = !act ? k * Cfg::SA_N + m : m * ZG_KSTRIDE + k;
        }
        dA = !act ? (int64_t)BK * lda : BK;
#pragma unroll
        for (int it = 0; it < NB; ++it) {
            const int idx = tid + it * NT;
            int n, k;
            if (!TB) { k = idx % BK; n = idx / BK; }         // B element (k,n) at B[k + n*ldb], K-contiguous
            else     { n = idx % BN; k = idx / BN; }         // B element (k,n) = conj(B[n + k*ldb]), N-contiguous
            const int gn = n0 + n;
            vB[it] = gn < p.N;
            kB[it] = k;
            pB[it] = !TB ? B + (k0 + k) + (int64_t)gn * ldb : B + gn + (int64_t)(k0 + k) * ldb;
            sB[it] = !TB ? n * ZG_KSTRIDE + k : k * Cfg::SB_C + n;
        }
        dB = !TB ? BK : (int64_t)BK * ldb;
        ld_krem = Kp - k0;
        ld_switch = 0x7fffffff;
        if (!second && nkb2 > 0) ld_switch = nkb1;
        if (MODE == ZMODE_HEMM && !act) ld_switch = min(ld_switch, (m0 + BM) / BK);
    };
    auto load_next = [&](int stage) {          // requests block ld_kb into `stage`
        if (ld_kb == ld_switch) ld_setup(ld_kb);
        c128* As = smem + (size_t)stage * Cfg::STAGE;
        c128* Bs = As + Cfg::A_STAGE;
#pragma unroll
        for (int it = 0; it < NA; ++it) {
            const bool ok = vA[it] && kA[it] < ld_krem;
            cp_async16(As + sA[it], ok ? pA[it] : ld_safe, ok ? 16 : 0);
            pA[it] += dA;
        }
#pragma unroll
        for (int it = 0; it < NB; ++it) {
            const bool ok = vB[it] && kB[it] < ld_krem;
            cp_async16(Bs + sB[it], ok ? pB[it] : ld_safe, ok ? 16 : 0);
            pB[it] += dB;
        }
        ld_krem -= BK;
        ++ld_kb;
    };

    // prologue
#pragma unroll
    for (int s = 0; s < ZG_STAGES - 1; ++s) {
        if (kb_begin + s < kb_end) load_next(s);
        cp_async_commit();
    }
    for (int kb = kb_begin; kb < kb_end; ++kb) {
        cp_async_wait<ZG_STAGES - 2>();
        __syncthreads();
        {
            const int nxt = kb + ZG_STAGES - 1;
            if (nxt < kb_end) load_next((nxt - kb_begin) % ZG_STAGES);
            cp_async_commit();
        }
        const int stage = (kb - kb_begin) % ZG_STAGES;
        const c128* As = smem + (size_t)stage * Cfg::STAGE;
        const c128* Bs = As + Cfg::A_STAGE;
        if constexpr (M3) {
            if (MODE == ZMODE_HEMM) {
                if (a_ctype(kb))
                    zgemm_compute_stage_3m<BM, BN, NJ, true, true, TB, TB>(As, Bs, wm0, wn0, g, t, cr, s2, ci);
                else
                    zgemm_compute_stage_3m<BM, BN, NJ, false, false, TB, TB>(As, Bs, wm0, wn0, g, t, cr, s2, ci);
            } else {
                zgemm_compute_stage_3m<BM, BN, NJ, TA, TA, TB, TB>(As, Bs, wm0, wn0, g, t, cr, s2, ci);
            }
        } else {
            if (MODE == ZMODE_HEMM) {
                if (a_ctype(kb))
                    zgemm_compute_stage<BM, BN, true, true, TB, TB>(As, Bs, wm0, wn0, g, t, cr, ci);
                else
                    zgemm_compute_stage<BM, BN, false, false, TB, TB>(As, Bs, wm0, wn0, g, t, cr, ci);
            } else {
                zgemm_compute_stage<BM, BN, TA, TA, TB, TB>(As, Bs, wm0, wn0, g, t, cr, ci);
            }
        }
    }
    cp_async_wait<0>();
    if constexpr (M3) {
        // Re = S1 - S2, Im = S3 - S1 - S2
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < NJ; ++j)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const double a1 = cr[i][j][e], a2 = s2[i][j][e], a3 = ci[i][j][e];
                    cr[i][j][e] = a1 - a2;
                    ci[i][j][e] = (a3 - a1) - a2;
                }
    }

    // epilogue
    if (p.splitk > 1) {
        c128* P = p.partial + (size_t)blockIdx.z * p.M * p.N;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int row = m0 + wm0 + 8 * i + g;
#pragma unroll
            for (int j = 0; j < NJ; ++j)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int col = n0 + wn0 + 8 * j + 2 * t + e;
                    if (row < p.M && col < p.N) P[row + (size_t)col * p.M] = cmake(cr[i][j][e], ci[i][j][e]);
                }
        }
    } else {
        const double alpha = p.alpha, beta = preload ? 0.0 : p.beta;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int row = m0 + wm0 + 8 * i + g;
#pragma unroll
            for (int j = 0; j < NJ; ++j)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int col = n0 + wn0 + 8 * j + 2 * t + e;
                    if (row < p.M && col < p.N) {
                        c128* dst = p.C + row + (int64_t)col * p.ldc;
                        c128 v = cmake(alpha * cr[i][j][e], alpha * ci[i][j][e]);
                        if (beta != 0.0) {
                            const c128 o = *dst;
                            v.x = fma(beta, o.x, v.x);
                            v.y = fma(beta, o.y, v.y);
                        }
                        *dst = v;
                    }
                }
        }
    }
}

// C = alpha * sum_s partial[s] + beta * C   (deterministic order s = 0..splitk-1)
static __global__ void zgemm_splitk_reduce_kernel(int M, int N, int splitk, const c128* __restrict__ partial,
                                           double alpha, double beta, c128* __restrict__ C, int64_t ldc,
                                           int lower_only_tiles, int BM, int BN) {
    const int64_t total = (int64_t)M * N;
    for (int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; idx < total;
         idx += (int64_t)gridDim.x * blockDim.x) {
        const int row = (int)(idx % M), col = (int)(idx / M);
        if (lower_only_tiles) {
            const int m0 = (row / BM) * BM, n0 = (col / BN) * BN;
            if (m0 + BM - 1 < n0) continue;
        }
        double sx = 0.0, sy = 0.0;
        for (int s = 0; s < splitk; ++s) {
            const c128 v = partial[(size_t)s * total + idx];
            sx += v.x; sy += v.y;
        }
        c128* dst = C + row + (int64_t)col * ldc;
        c128 v = cmake(alpha * sx, alpha * sy);
        if (beta != 0.0) { const c128 o = *dst; v.x = fma(beta, o.x, v.x); v.y = fma(beta, o.y, v.y); }
        *dst = v;
    }
}

// Host launcher (zgemm.cu).  Tiles are 64x64 (4 warps, 2 CTAs/SM) unless g_zgemm_big_tiles is set and
// small_tile is false (then 128x64, 8 warps, 1 CTA/SM).
// Returns a cudaError_t as int (0 = ok).  `launches` (optional) is incremented per kernel launch.
int zgemm_launch(const ZgemmArgs& a, bool ta, bool tb, int mode, bool small_tile, cudaStream_t stream,
                 int64_t* launches);
extern bool g_zgemm_big_tiles;
extern bool g_zgemm_3m;       // 3M kernels (default) or the 4-multiplication ones (option "gemm_3m" = 0)

}  // namespace eigh
