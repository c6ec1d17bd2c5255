// dgemm.cu -- host launcher of the real FP64 DMMA GEMM (dgemm.cuh).
#include "dgemm.cuh"

namespace eigh {

int dgemm_launch_desc(const DgemmArgs& a, int batch, int maxM, int maxN, cudaStream_t stream, int64_t* launches) {
    if (batch <= 0 || maxM <= 0 || maxN <= 0) return 0;
    {
        cudaError_t e = cudaFuncSetAttribute(dgemm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)DG_SMEM_BYTES);
        if (e != cudaSuccess) return (int)e;
    }
    dim3 grid((unsigned)((maxM + DG_BM - 1) / DG_BM), (unsigned)((maxN + DG_BN - 1) / DG_BN), (unsigned)batch);
    dgemm_kernel<<<grid, DG_NT, DG_SMEM_BYTES, stream>>>(a);
    if (launches) ++*launches;
    return (int)cudaGetLastError();
}

}  // namespace eigh
