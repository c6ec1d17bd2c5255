// dgemm.cuh -- real FP64 GEMM on the FP64 tensor-core path (mma.sync m8n8k4 -> DMMA.8x8x4),
// batched over device-resident problem descriptors.  Used by the merge step of the tridiagonal
// divide & conquer:  Q_new[:, 0:k] = Q_old[:, idx[0:k]] * U.
//
//   C (M x N) <- A[:, idx] (M x K) * B (K x N),  all column-major, inner length K.
//
// Requirements: A, B, C base pointers 16-byte aligned and lda, ldb even (16-byte cp.async);
// problem sizes come from device memory so that sizes decided on the device (deflation counts)
// never need a host round trip: the grid is sized for the worst case and surplus CTAs exit.
#pragma once
#include "common.cuh"

namespace eigh {

struct DgemmDesc {           // one problem; lives in device memory
    int64_t offA, offB, offC;  // element offsets from the base pointers
    int64_t offIdx;            // offset into a_col_idx
    int M, N, K;
    int pad;
};

struct DgemmArgs {
    const double* A; int64_t lda;
    const double* B; int64_t ldb;
    double* C;       int64_t ldc;
    const int32_t* a_col_idx;     // may be NULL (identity)
    const DgemmDesc* desc;        // [gridDim.z] descriptors, or NULL -> use the inline one
    DgemmDesc one;
};

constexpr int DG_BM = 128, DG_BN = 64, DG_BK = 16, DG_STAGES = 4;   // 108 KB of shared memory: 2 thread blocks per SM
constexpr int DG_SA = DG_BM + 4;     // As[k][m], stride == 4 (mod 16) doubles
constexpr int DG_SB = DG_BK + 4;     // Bs[n][k]
constexpr int DG_STAGE = DG_BK * DG_SA + DG_BN * DG_SB;    // doubles
constexpr size_t DG_SMEM_BYTES = (size_t)DG_STAGES * DG_STAGE * sizeof(double);

// MI = 8-row fragments per warp along M: 4 = warp tile 32 x 32, 8 warps (the default); 8 = warp tile 64 x 32, 4 warps
template <int MI>
static __global__ void __launch_bounds__(MI == 4 ? 256 : 128, 2) dgemm_kernel_t(const DgemmArgs p) {
    constexpr int DG_NT = MI == 4 ? 256 : 128;
    extern __shared__ __align__(16) unsigned char dg_smem_raw[];
    double* smem = reinterpret_cast<double*>(dg_smem_raw);

    const DgemmDesc d = p.desc ? p.desc[blockIdx.z] : p.one;
    const int m0 = blockIdx.x * DG_BM, n0 = blockIdx.y * DG_BN;
    if (m0 >= d.M || n0 >= d.N || d.K <= 0) {
        if (m0 < d.M && n0 < d.N) {   // K == 0: C = 0
            for (int idx = threadIdx.x; idx < DG_BM * DG_BN; idx += DG_NT) {
                const int r = m0 + idx % DG_BM, c = n0 + idx / DG_BM;
                if (r < d.M && c < d.N) p.C[d.offC + r + (int64_t)c * p.ldc] = 0.0;
            }
        }
        return;
    }
    const double* A = p.A + d.offA;
    const double* B = p.B + d.offB;
    double* C = p.C + d.offC;
    const int32_t* cidx = p.a_col_idx ? p.a_col_idx + d.offIdx : nullptr;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, t = lane & 3;
    const int wm0 = MI == 4 ? (warp & 3) * 32 : (warp & 1) * 64, wn0 = (MI == 4 ? (warp >> 2) : (warp >> 1)) * 32;

    double acc[MI][4][2];
#pragma unroll
    for (int i = 0; i < MI; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    const int nkb = (d.K + DG_BK - 1) / DG_BK;

    // Per-thread loader state (fixed over the k-blocks): row pair / k of its A elements, column / k pair of its B
    // elements, their shared-memory slots; only the gathered column of A and the B pointer change from block to block.
    constexpr int NA = DG_BM * DG_BK / 2 / DG_NT, NB = DG_BN * DG_BK / 2 / DG_NT;
    const double* pA[NA];
    const double* pB[NB];
    int kA[NA], sA[NA], bA[NA], kB[NB], sB[NB];
    bool vB[NB];
#pragma unroll
    for (int it = 0; it < NA; ++it) {
        const int idx = tid + it * DG_NT;
        const int mp = idx % (DG_BM / 2), k = idx / (DG_BM / 2);
        const int gm = m0 + 2 * mp;
        kA[it] = k;
        sA[it] = k * DG_SA + 2 * mp;
        bA[it] = gm >= d.M ? 0 : (gm + 1 < d.M ? 16 : 8);
        pA[it] = A + (gm < d.M ? gm : 0);
    }
#pragma unroll
    for (int it = 0; it < NB; ++it) {
        const int idx = tid + it * DG_NT;
        const int kp = idx % (DG_BK / 2), n = idx / (DG_BK / 2);
        const int gn = n0 + n;
        kB[it] = 2 * kp;
        sB[it] = n * DG_SB + 2 * kp;
        vB[it] = gn < d.N;
        pB[it] = B + 2 * kp + (int64_t)(gn < d.N ? gn : 0) * p.ldb;
    }
    // gathered columns of A: the indices of the NEXT requested k-block are fetched one request ahead, so that no
    // cp.async address waits for an index load (the blocks are requested strictly in order 0, 1, 2, ...)
    int cpre[NA];
    auto fetch_idx = [&](int kb) {
#pragma unroll
        for (int it = 0; it < NA; ++it) {
            const int k = kb * DG_BK + kA[it];
            cpre[it] = (cidx && k < d.K) ? __ldg(cidx + k) : k;
        }
    };
    fetch_idx(0);
    auto load_stage = [&](int stage, int kb) {
        double* As = smem + (size_t)stage * DG_STAGE;
        double* Bs = As + DG_BK * DG_SA;
        const int k0 = kb * DG_BK;
        const int krem = d.K - k0;
#pragma unroll
        for (int it = 0; it < NA; ++it) {
            int bytes = 0;
            const double* src = A;
            if (kA[it] < krem && bA[it]) {
                src = pA[it] + (int64_t)cpre[it] * p.lda;
                bytes = bA[it];
            }
            cp_async16(As + sA[it], src, bytes);
        }
#pragma unroll
        for (int it = 0; it < NB; ++it) {
            int bytes = 0;
            const double* src = B;
            if (vB[it] && kB[it] < krem) {
                src = pB[it] + k0;
                bytes = (kB[it] + 1 < krem) ? 16 : 8;
            }
            cp_async16(Bs + sB[it], src, bytes);
        }
        if (kb + 1 < nkb) fetch_idx(kb + 1);
    };

#pragma unroll
    for (int s = 0; s < DG_STAGES - 1; ++s) {
        if (s < nkb) load_stage(s, s);
        cp_async_commit();
    }
    for (int kb = 0; kb < nkb; ++kb) {
        cp_async_wait<DG_STAGES - 2>();
        __syncthreads();
        {
            const int nxt = kb + DG_STAGES - 1;
            if (nxt < nkb) load_stage(nxt % DG_STAGES, nxt);
            cp_async_commit();
        }
        const double* As = smem + (size_t)(kb % DG_STAGES) * DG_STAGE;
        const double* Bs = As + DG_BK * DG_SA;
#pragma unroll
        for (int kk = 0; kk < DG_BK; kk += 4) {
            double a[MI], b[4];
#pragma unroll
            for (int i = 0; i < MI; ++i) a[i] = As[(kk + t) * DG_SA + wm0 + 8 * i + g];
#pragma unroll
            for (int j = 0; j < 4; ++j) b[j] = Bs[(wn0 + 8 * j + g) * DG_SB + kk + t];
#pragma unroll
            for (int i = 0; i < MI; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) dmma884p(acc[i][j][0], acc[i][j][1], a[i], b[j]);
        }
    }
    cp_async_wait<0>();

#pragma unroll
    for (int i = 0; i < MI; ++i) {
        const int row = m0 + wm0 + 8 * i + g;
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int col = n0 + wn0 + 8 * j + 2 * t + e;
                if (row < d.M && col < d.N) C[row + (int64_t)col * p.ldc] = acc[i][j][e];
            }
    }
}

// batch >= 1 problems; maxM / maxN bound the grid.  Returns cudaError_t as int.
int dgemm_launch_desc(const DgemmArgs& a, int batch, int maxM, int maxN, cudaStream_t stream, int64_t* launches);

}  // namespace eigh
