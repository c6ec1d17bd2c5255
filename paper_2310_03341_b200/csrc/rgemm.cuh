// rgemm.cuh -- real FP64 GEMM engine on the FP64 tensor-core path (mma.sync m8n8k4 -> DMMA.8x8x4): the real-symmetric
// counterpart of zgemm.cuh, used by the real instance of the 1-stage solver (SURVEY.md 8(f)2; PAPER.md:140, :158-160:
// the paper benchmarks real FP64).
//
//   C <- alpha * opA(A1) opB(B1) [+ alpha * opA(A2) opB(B2)] + beta * C,   op = N (as stored) or T (transposed)
//
// Same feature set as the complex engine: a second (A2, B2) pair in the same K loop (SYR2K: C -= V W^T + W V^T as one
// product), `lower_only` tile skipping, deterministic split-K (partials + ordered reduction, no FP64 atomics).
// CTA tile 128 x 64, BK = 16, 8 warps of 32 x 32, 4-stage cp.async pipeline with 8-byte copies (no alignment or
// even-ld requirement), two CTAs per SM.  Shared-memory strides are chosen so that the 64-bit fragment loads of a
// half warp touch 16 distinct banks pairs (conflict-free).
#pragma once
#include "common.cuh"

namespace eigh {

struct RgemmArgs {
    int M, N;
    int K1, K2;
    const double *A1, *B1, *A2, *B2;
    int64_t lda1, ldb1, lda2, ldb2;
    double* C;
    int64_t ldc;
    double alpha, beta;
    int lower_only;
    int splitk;
    double* partial;       // [splitk][N][M] raw accumulators when splitk > 1
};

constexpr int RG_BM = 128, RG_BN = 64, RG_BK = 16, RG_STAGES = 4, RG_NT = 256;
constexpr int RG_SA_N = RG_BM + 4;      // As[k][m]   (A as stored, M-contiguous)
constexpr int RG_SK = RG_BK + 4;        // As[m][k] / Bs[n][k]  (K-contiguous)
constexpr int RG_SB_T = RG_BN + 4;      // Bs[k][n]   (B transposed, N-contiguous)
constexpr int RG_A_STAGE = (RG_BK * RG_SA_N > RG_BM * RG_SK) ? RG_BK * RG_SA_N : RG_BM * RG_SK;
constexpr int RG_B_STAGE = (RG_BK * RG_SB_T > RG_BN * RG_SK) ? RG_BK * RG_SB_T : RG_BN * RG_SK;
constexpr int RG_STAGE = RG_A_STAGE + RG_B_STAGE;
constexpr size_t RG_SMEM_BYTES = (size_t)RG_STAGES * RG_STAGE * sizeof(double);

template <bool TA, bool TB>
__global__ void __launch_bounds__(RG_NT, 2) rgemm_kernel(const RgemmArgs p) {
    extern __shared__ __align__(16) unsigned char rg_smem_raw[];
    double* smem = reinterpret_cast<double*>(rg_smem_raw);
    const int m0 = blockIdx.x * RG_BM, n0 = blockIdx.y * RG_BN;
    if (p.lower_only && m0 + RG_BM - 1 < n0) return;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, t = lane & 3;
    const int wm0 = (warp & 3) * 32, wn0 = (warp >> 2) * 32;

    const int nkb1 = (p.K1 + RG_BK - 1) / RG_BK;
    const int nkb2 = (p.A2 != nullptr) ? (p.K2 + RG_BK - 1) / RG_BK : 0;
    const int nkb = nkb1 + nkb2;
    const int per = (nkb + p.splitk - 1) / p.splitk;
    const int kb_begin = blockIdx.z * per;
    const int kb_end = min(nkb, kb_begin + per);

    double acc[4][4][2];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    constexpr int NA = RG_BM * RG_BK / RG_NT, NB = RG_BN * RG_BK / RG_NT;
    auto load_block = [&](int stage, int kb) {
        const bool second = kb >= nkb1;
        const double* A = second ? p.A2 : p.A1;
        const double* B = second ? p.B2 : p.B1;
        const int64_t lda = second ? p.lda2 : p.lda1, ldb = second ? p.ldb2 : p.ldb1;
        const int Kp = second ? p.K2 : p.K1;
        const int k0 = (second ? kb - nkb1 : kb) * RG_BK;
        double* As = smem + (size_t)stage * RG_STAGE;
        double* Bs = As + RG_A_STAGE;
#pragma unroll
        for (int it = 0; it < NA; ++it) {
            const int idx = tid + it * RG_NT;
            int m, k;
            if (!TA) { m = idx % RG_BM; k = idx / RG_BM; } else { k = idx % RG_BK; m = idx / RG_BK; }
            const int gm = m0 + m, gk = k0 + k;
            const bool ok = gm < p.M && gk < Kp;
            const double* src = ok ? (!TA ? A + gm + (int64_t)gk * lda : A + gk + (int64_t)gm * lda) : A;
            cp_async8(As + (!TA ? k * RG_SA_N + m : m * RG_SK + k), src, ok ? 8 : 0);
        }
#pragma unroll
        for (int it = 0; it < NB; ++it) {
            const int idx = tid + it * RG_NT;
            int n, k;
            if (!TB) { k = idx % RG_BK; n = idx / RG_BK; } else { n = idx % RG_BN; k = idx / RG_BN; }
            const int gn = n0 + n, gk = k0 + k;
            const bool ok = gn < p.N && gk < Kp;
            const double* src = ok ? (!TB ? B + gk + (int64_t)gn * ldb : B + gn + (int64_t)gk * ldb) : B;
            cp_async8(Bs + (!TB ? n * RG_SK + k : k * RG_SB_T + n), src, ok ? 8 : 0);
        }
    };

#pragma unroll
    for (int s = 0; s < RG_STAGES - 1; ++s) {
        if (kb_begin + s < kb_end) load_block(s, kb_begin + s);
        cp_async_commit();
    }
    for (int kb = kb_begin; kb < kb_end; ++kb) {
        cp_async_wait<RG_STAGES - 2>();
        __syncthreads();
        {
            const int nxt = kb + RG_STAGES - 1;
            if (nxt < kb_end) load_block((nxt - kb_begin) % RG_STAGES, nxt);
            cp_async_commit();
        }
        const double* As = smem + (size_t)((kb - kb_begin) % RG_STAGES) * RG_STAGE;
        const double* Bs = As + RG_A_STAGE;
#pragma unroll
        for (int kk = 0; kk < RG_BK; kk += 4) {
            double a[4], b[4];
#pragma unroll
            for (int i = 0; i < 4; ++i)
                a[i] = !TA ? As[(kk + t) * RG_SA_N + wm0 + 8 * i + g] : As[(wm0 + 8 * i + g) * RG_SK + kk + t];
#pragma unroll
            for (int j = 0; j < 4; ++j)
                b[j] = !TB ? Bs[(wn0 + 8 * j + g) * RG_SK + kk + t] : Bs[(kk + t) * RG_SB_T + wn0 + 8 * j + g];
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) dmma884p(acc[i][j][0], acc[i][j][1], a[i], b[j]);
        }
    }
    cp_async_wait<0>();

    if (p.splitk > 1) {
        double* P = p.partial + (size_t)blockIdx.z * p.M * p.N;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int row = m0 + wm0 + 8 * i + g;
#pragma unroll
            for (int j = 0; j < 4; ++j)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int col = n0 + wn0 + 8 * j + 2 * t + e;
                    if (row < p.M && col < p.N) P[row + (size_t)col * p.M] = acc[i][j][e];
                }
        }
    } else {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int row = m0 + wm0 + 8 * i + g;
#pragma unroll
            for (int j = 0; j < 4; ++j)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int col = n0 + wn0 + 8 * j + 2 * t + e;
                    if (row < p.M && col < p.N) {
                        double* dst = p.C + row + (int64_t)col * p.ldc;
                        double v = p.alpha * acc[i][j][e];
                        if (p.beta != 0.0) v = fma(p.beta, *dst, v);
                        *dst = v;
                    }
                }
        }
    }
}

// C = alpha * sum_s partial[s] + beta * C   (deterministic order s = 0..splitk-1)
static __global__ void rgemm_splitk_reduce_kernel(int M, int N, int splitk, const double* __restrict__ partial, double alpha,
                                                  double beta, double* __restrict__ C, int64_t ldc, int lower_only) {
    const int64_t total = (int64_t)M * N;
    for (int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
        const int row = (int)(idx % M), col = (int)(idx / M);
        if (lower_only) {
            const int m0 = (row / RG_BM) * RG_BM, n0 = (col / RG_BN) * RG_BN;
            if (m0 + RG_BM - 1 < n0) continue;
        }
        double s = 0.0;
        for (int k = 0; k < splitk; ++k) s += partial[(size_t)k * total + idx];
        double* dst = C + row + (int64_t)col * ldc;
        double v = alpha * s;
        if (beta != 0.0) v = fma(beta, *dst, v);
        *dst = v;
    }
}

// Host launcher (rgemm.cu).  Returns a cudaError_t as int (0 = ok).
int rgemm_launch(const RgemmArgs& a, bool ta, bool tb, cudaStream_t stream, int64_t* launches);

}  // namespace eigh
