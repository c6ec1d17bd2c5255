// zgemm.cu -- instantiations and host launcher of the complex-FP64 DMMA GEMM engine (zgemm.cuh).
#include "zgemm.cuh"

namespace eigh {

template <int WM, int WN, bool TA, bool TB, int MODE, int MINB, int NJ = 4, bool M3 = false>
static int launch_inst(const ZgemmArgs& a, cudaStream_t stream, int64_t* launches) {
    using Cfg = ZgemmCfg<WM, WN, TA, TB, MODE, NJ>;
    auto kern = zgemm_kernel<WM, WN, TA, TB, MODE, MINB, NJ, M3>;
    {   // per device / context, cheap: set on every launch
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)Cfg::SMEM_BYTES);
        if (e != cudaSuccess) return (int)e;
    }
    dim3 grid((unsigned)((a.M + Cfg::BM - 1) / Cfg::BM), (unsigned)((a.N + Cfg::BN - 1) / Cfg::BN),
              (unsigned)a.splitk);
    kern<<<grid, Cfg::NT, Cfg::SMEM_BYTES, stream>>>(a);
    if (launches) ++*launches;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return (int)e;
    if (a.splitk > 1) {
        const int64_t total = (int64_t)a.M * a.N;
        int blocks = (int)((total + 255) / 256);
        if (blocks > 148 * 16) blocks = 148 * 16;
        zgemm_splitk_reduce_kernel<<<blocks, 256, 0, stream>>>(a.M, a.N, a.splitk, a.partial, a.alpha, a.beta,
                                                               a.C, a.ldc, a.lower_only, Cfg::BM, Cfg::BN);
        if (launches) ++*launches;
        e = cudaGetLastError();
        if (e != cudaSuccess) return (int)e;
    }
    return 0;
}

bool g_zgemm_big_tiles = false;   // test hook (eigh_k_zgemm lower_only bit 2)
bool g_zgemm_3m = true;

int zgemm_launch(const ZgemmArgs& a, bool ta, bool tb, int mode, bool small_tile, cudaStream_t stream,
                 int64_t* launches) {
    if (a.M <= 0 || a.N <= 0) return 0;
    if (g_zgemm_3m && !g_zgemm_big_tiles) {
        // 3M kernels: CTA tile 64 x 32 (4 warps of 32 x 16), three CTAs per SM
        if (mode == ZMODE_HEMM) return launch_inst<2, 2, false, false, ZMODE_HEMM, 3, 2, true>(a, stream, launches);
        if (!ta && !tb) return launch_inst<2, 2, false, false, ZMODE_GEMM, 3, 2, true>(a, stream, launches);
        if (!ta && tb) return launch_inst<2, 2, false, true, ZMODE_GEMM, 3, 2, true>(a, stream, launches);
        if (ta && !tb) return launch_inst<2, 2, true, false, ZMODE_GEMM, 3, 2, true>(a, stream, launches);
        return (int)cudaErrorInvalidValue;
    }
    if (mode == ZMODE_HEMM) return launch_inst<2, 2, false, false, ZMODE_HEMM, 2>(a, stream, launches);
    // 64x64 tiles with two resident CTAs per SM are the default: measured faster than 128x64 with one
    // CTA per SM in every shape the solver uses (profiles/r01_gemm_shapes.md)
    if (small_tile || !g_zgemm_big_tiles) {
        if (!ta && !tb) return launch_inst<2, 2, false, false, ZMODE_GEMM, 2>(a, stream, launches);
        if (!ta && tb) return launch_inst<2, 2, false, true, ZMODE_GEMM, 2>(a, stream, launches);
        if (ta && !tb) return launch_inst<2, 2, true, false, ZMODE_GEMM, 2>(a, stream, launches);
        return (int)cudaErrorInvalidValue;
    }
    if (!ta && !tb) return launch_inst<4, 2, false, false, ZMODE_GEMM, 1>(a, stream, launches);
    if (!ta && tb) return launch_inst<4, 2, false, true, ZMODE_GEMM, 1>(a, stream, launches);
    if (ta && !tb) return launch_inst<4, 2, true, false, ZMODE_GEMM, 1>(a, stream, launches);
    return (int)cudaErrorInvalidValue;
}

}  // namespace eigh
