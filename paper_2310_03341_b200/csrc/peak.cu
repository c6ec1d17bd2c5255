// peak.cu -- FP64 roofline microbenchmarks (register-resident loops, no memory traffic) behind eigh_k_fp64_peak /
// eigh_k_fp64_probe.  They give the denominators bench.py reports against and the cost model DESIGN.md uses:
//   kind 0  DFMA loop                       kind 1  mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4) loop
//   kind 2  mma.sync.m16n8k16.f64 loop (ptxas expands it into eight DMMA.8x8x4 on sm_100a)
//   kind 10..13  the inner loop of the 3M GEMM engine (24 DMMAs per k-step on a 32 x 16 warp tile, 128-thread blocks):
//            10 = DMMAs on register operands only, 11 = + LDS.128 fragment loads and the 3M adds,
//            12 = + one __syncthreads per k-block, 13 = + the cp.async traffic of a k-block.
#include "eigh_internal.h"

namespace eigh {

__global__ void peak_dmma_kernel(int64_t iters, double* sink) {
    double c[16][2];
#pragma unroll
    for (int i = 0; i < 16; ++i) { c[i][0] = 0.0; c[i][1] = 0.0; }
    const double a = 1.0 + 1e-9 * threadIdx.x, b = 1.0 - 1e-9 * threadIdx.x;
    for (int64_t it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) dmma884(c[i][0], c[i][1], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += c[i][0] + c[i][1];
    if (s == 123.456) sink[0] = s;
}

__global__ void peak_dmma16816_kernel(int64_t iters, double* sink) {      // 2048 FMAs per instruction
    double c[8][4];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) c[i][j] = 0.0;
    const double a = 1.0 + 1e-9 * threadIdx.x, b = 1.0 - 1e-9 * threadIdx.x;
    for (int64_t it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i)
            asm volatile("mma.sync.aligned.m16n8k16.row.col.f64.f64.f64.f64 {%0,%1,%2,%3}, {%4,%5,%6,%7,%8,%9,%10,%11}, "
                         "{%12,%13,%14,%15}, {%0,%1,%2,%3};"
                         : "+d"(c[i][0]), "+d"(c[i][1]), "+d"(c[i][2]), "+d"(c[i][3])
                         : "d"(a), "d"(b), "d"(a), "d"(b), "d"(a), "d"(b), "d"(a), "d"(b), "d"(b), "d"(a), "d"(b), "d"(a));
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) s += c[i][j];
    if (s == 123.456) sink[0] = s;
}

__global__ void peak_dfma_kernel(int64_t iters, double* sink) {
    double c[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) c[i] = 1e-3 * i;
    const double a = 1.0 + 1e-9 * threadIdx.x, b = 1e-9 * threadIdx.x;
    for (int64_t it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) c[i] = fma(c[i], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += c[i];
    if (s == 123.456) sink[0] = s;
}

// one iteration = one k-block of the 3M engine: 2 k-steps x 24 DMMAs per warp
template <int MODE>
__global__ void __launch_bounds__(128, 3) peak_gemm_loop_kernel(int64_t iters, const c128* __restrict__ g, double* sink) {
    constexpr int TILE = 8 * 66 + 32 * 12;
    __shared__ c128 sm[2][TILE];
    double s1[4][2][2], s2[4][2][2], s3[4][2][2];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 2; ++j)
#pragma unroll
            for (int e = 0; e < 2; ++e) s1[i][j][e] = s2[i][j][e] = s3[i][j][e] = 0.0;
    const int tid = threadIdx.x, lane = tid & 31, gq = lane >> 2, t = lane & 3, warp = tid >> 5;
    for (int i = tid; i < 2 * TILE; i += 128) (&sm[0][0])[i] = g[i % 997];
    __syncthreads();
    double ar[4], ai[4], as[4], br[2], bi[2], bs[2];
#pragma unroll
    for (int i = 0; i < 4; ++i) { ar[i] = 1.0 + 1e-9 * (tid + i); ai[i] = 1.0 - 1e-9 * (tid + i); as[i] = ar[i] + ai[i]; }
#pragma unroll
    for (int j = 0; j < 2; ++j) { br[j] = 1.0 + 2e-9 * (tid + j); bi[j] = 1.0 - 2e-9 * (tid + j); bs[j] = br[j] + bi[j]; }
    for (int64_t it = 0; it < iters; ++it) {
        const c128* As = sm[it & 1];
        const c128* Bs = As + 8 * 66;
#pragma unroll
        for (int kk = 0; kk < 8; kk += 4) {
            if (MODE >= 1) {
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const c128 a = As[(kk + t) * 66 + (warp & 1) * 32 + 8 * i + gq];
                    ar[i] = a.x; ai[i] = a.y; as[i] = a.x + a.y;
                }
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    const c128 b = Bs[((warp >> 1) * 16 + 8 * j + gq) * 12 + kk + t];
                    br[j] = b.x; bi[j] = b.y; bs[j] = b.x + b.y;
                }
            }
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 2; ++j) dmma884(s1[i][j][0], s1[i][j][1], ar[i], br[j]);
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 2; ++j) dmma884(s2[i][j][0], s2[i][j][1], ai[i], bi[j]);
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 2; ++j) dmma884(s3[i][j][0], s3[i][j][1], as[i], bs[j]);
        }
        if (MODE >= 2) __syncthreads();
        if (MODE >= 3) {
#pragma unroll
            for (int q = 0; q < 6; ++q)
                cp_async16(&sm[(it + 1) & 1][(tid + 128 * q) % TILE], g + ((it * 768 + tid + 128 * q) & 0xffff), 16);
            cp_async_commit();
            cp_async_wait<0>();
        }
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 2; ++j)
#pragma unroll
            for (int e = 0; e < 2; ++e) s += s1[i][j][e] + s2[i][j][e] + s3[i][j][e];
    if (s == 123.456) sink[0] = s;
}

}  // namespace eigh

using namespace eigh;

extern "C" int eigh_k_fp64_probe(int kind, int blocks_per_sm, int threads, int64_t iters, double* tflops, double* ms_out,
                                 void* stream) {
    if (!((kind >= 0 && kind <= 2) || (kind >= 10 && kind <= 13))) return -1;
    if (blocks_per_sm < 1 || blocks_per_sm > 16) return -2;
    if (threads < 32 || threads > 1024 || threads % 32) return -3;
    if (iters < 1) return -4;
    if (!tflops) return -5;
    if (kind >= 10) { threads = 128; blocks_per_sm = 3; }
    cudaStream_t s = (cudaStream_t)stream;
    int dev = 0, sms = 0;
    EIGH_CUDA_OK(cudaGetDevice(&dev));
    EIGH_CUDA_OK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    double* sink = nullptr;
    c128* g = nullptr;
    EIGH_CUDA_OK(cudaMalloc(&sink, 8));
    EIGH_CUDA_OK(cudaMalloc(&g, (size_t)(65536 + 1024) * sizeof(c128)));
    EIGH_CUDA_OK(cudaMemsetAsync(g, 0, (size_t)(65536 + 1024) * sizeof(c128), s));
    cudaEvent_t e0, e1;
    EIGH_CUDA_OK(cudaEventCreate(&e0));
    EIGH_CUDA_OK(cudaEventCreate(&e1));
    const int blocks = sms * blocks_per_sm;
    for (int rep = 0; rep < 2; ++rep) {   // first pass = warm-up
        EIGH_CUDA_OK(cudaEventRecord(e0, s));
        switch (kind) {
            case 0: peak_dfma_kernel<<<blocks, threads, 0, s>>>(iters, sink); break;
            case 1: peak_dmma_kernel<<<blocks, threads, 0, s>>>(iters, sink); break;
            case 2: peak_dmma16816_kernel<<<blocks, threads, 0, s>>>(iters, sink); break;
            case 10: peak_gemm_loop_kernel<0><<<blocks, threads, 0, s>>>(iters, g, sink); break;
            case 11: peak_gemm_loop_kernel<1><<<blocks, threads, 0, s>>>(iters, g, sink); break;
            case 12: peak_gemm_loop_kernel<2><<<blocks, threads, 0, s>>>(iters, g, sink); break;
            default: peak_gemm_loop_kernel<3><<<blocks, threads, 0, s>>>(iters, g, sink); break;
        }
        EIGH_CUDA_OK(cudaGetLastError());
        EIGH_CUDA_OK(cudaEventRecord(e1, s));
        EIGH_CUDA_OK(cudaEventSynchronize(e1));
    }
    float ms = 0.f;
    EIGH_CUDA_OK(cudaEventElapsedTime(&ms, e0, e1));
    const double warps = (double)blocks * threads / 32.0;
    double fma_per_warp;
    if (kind == 0) fma_per_warp = 32.0 * (double)iters * 16.0;
    else if (kind == 1) fma_per_warp = (double)iters * 16.0 * 256.0;
    else if (kind == 2) fma_per_warp = (double)iters * 8.0 * 2048.0;
    else fma_per_warp = (double)iters * 48.0 * 256.0;
    *tflops = 2.0 * warps * fma_per_warp / (ms * 1e-3) / 1e12;
    if (ms_out) *ms_out = ms;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    cudaFree(g);
    return 0;
}

// The two historical entry points: DFMA (use_dmma = 0) or DMMA (1) loops with two 256-thread blocks per SM (4 warps per SM
// sub-partition).  With 8 resident warps per sub-partition the same DMMA loop drops to 0.80 of this rate (r01_fp64_peaks.md).
extern "C" int eigh_k_fp64_peak(int use_dmma, int64_t iters, double* tflops, double* ms_out, void* stream) {
    if (iters < 1) return -2;
    if (!tflops) return -3;
    return eigh_k_fp64_probe(use_dmma ? 1 : 0, 2, 256, iters, tflops, ms_out, stream);
}
