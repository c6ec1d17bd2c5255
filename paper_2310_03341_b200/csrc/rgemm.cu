// rgemm.cu -- instantiations and host launcher of the real FP64 DMMA GEMM engine (rgemm.cuh).
#include "rgemm.cuh"

namespace eigh {

template <bool TA, bool TB>
static int rg_launch_inst(const RgemmArgs& a, cudaStream_t stream, int64_t* launches) {
    auto kern = rgemm_kernel<TA, TB>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RG_SMEM_BYTES);
    if (e != cudaSuccess) return (int)e;
    dim3 grid((unsigned)((a.M + RG_BM - 1) / RG_BM), (unsigned)((a.N + RG_BN - 1) / RG_BN), (unsigned)a.splitk);
    kern<<<grid, RG_NT, RG_SMEM_BYTES, stream>>>(a);
    if (launches) ++*launches;
    e = cudaGetLastError();
    if (e != cudaSuccess) return (int)e;
    if (a.splitk > 1) {
        const int64_t total = (int64_t)a.M * a.N;
        int blocks = (int)((total + 255) / 256);
        if (blocks > 148 * 16) blocks = 148 * 16;
        rgemm_splitk_reduce_kernel<<<blocks, 256, 0, stream>>>(a.M, a.N, a.splitk, a.partial, a.alpha, a.beta, a.C, a.ldc,
                                                               a.lower_only);
        if (launches) ++*launches;
        e = cudaGetLastError();
        if (e != cudaSuccess) return (int)e;
    }
    return 0;
}

int rgemm_launch(const RgemmArgs& a, bool ta, bool tb, cudaStream_t stream, int64_t* launches) {
    if (a.M <= 0 || a.N <= 0) return 0;
    if (!ta && !tb) return rg_launch_inst<false, false>(a, stream, launches);
    if (!ta && tb) return rg_launch_inst<false, true>(a, stream, launches);
    if (ta && !tb) return rg_launch_inst<true, false>(a, stream, launches);
    return rg_launch_inst<true, true>(a, stream, launches);
}

}  // namespace eigh
