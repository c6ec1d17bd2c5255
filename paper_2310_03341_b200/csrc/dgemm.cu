// dgemm.cu -- host launcher of the real FP64 DMMA GEMM (dgemm.cuh).
#include "dgemm.cuh"

namespace eigh {

int g_dgemm_mi = 8;      // warp-tile height in 8-row fragments (4 or 8): test hook, see dgemm.cuh

template <int MI>
static int dgemm_launch_t(const DgemmArgs& a, dim3 grid, cudaStream_t stream) {
    cudaError_t e = cudaFuncSetAttribute(dgemm_kernel_t<MI>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)DG_SMEM_BYTES);
    if (e != cudaSuccess) return (int)e;
    dgemm_kernel_t<MI><<<grid, MI == 4 ? 256 : 128, DG_SMEM_BYTES, stream>>>(a);
    return (int)cudaGetLastError();
}

int dgemm_launch_desc(const DgemmArgs& a, int batch, int maxM, int maxN, cudaStream_t stream, int64_t* launches) {
    if (batch <= 0 || maxM <= 0 || maxN <= 0) return 0;
    dim3 grid((unsigned)((maxM + DG_BM - 1) / DG_BM), (unsigned)((maxN + DG_BN - 1) / DG_BN), (unsigned)batch);
    if (launches) ++*launches;
    return g_dgemm_mi == 8 ? dgemm_launch_t<8>(a, grid, stream) : dgemm_launch_t<4>(a, grid, stream);
}

}  // namespace eigh
