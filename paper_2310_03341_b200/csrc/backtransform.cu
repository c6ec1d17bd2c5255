// backtransform.cu -- S4b: the second back-transformation of the eigenvectors
// ("the subsequent back transformation of the eigenvectors also requires two
// stages"), SURVEY.md 8(a) row S4b.  (S4a lives in bt_band.cu.)
//
// S4b  Z <- Q1 Z.  Panels of S1 in reverse order, Z_rows <- (I - V_p T_p V_p^H) Z_rows with the
//      T factors kept from S1:  Y = (V T^H)^H Z_rows ;  Z_rows -= V Y.
#include "eigh_internal.h"
#include "zgemm.cuh"

namespace eigh {

int zgemm_ws(eigh_handle_s* h, bool ta, bool tb, int M, int N, int K, double alpha, const c128* A, int64_t lda,
             const c128* B, int64_t ldb, double beta, c128* C, int64_t ldc, bool small_tile, int splitk,
             cudaStream_t s);

// ------------------------------------------------------------------ S4b
// Vp (m x nb, ldv = m): explicit unit-lower-trapezoidal V of panel p from A
__global__ void bt_extract_v_kernel(const c128* __restrict__ A, int64_t lda, int row0, int col0, int m, int nb, int nr,
                                    c128* __restrict__ Vp, int64_t ldv) {
    const int c = blockIdx.y;
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= m || c >= nb) return;
    c128 v = cmake(0.0, 0.0);
    if (r == c) v = cmake(1.0, 0.0);
    else if (r > c && c < nr) v = A[(row0 + r) + (int64_t)(col0 + c) * lda];
    Vp[r + (int64_t)c * ldv] = v;
}

int phase_backtransform_full(eigh_handle_s* h, const c128* A, int64_t lda, c128* Z, int64_t ldz, cudaStream_t s) {
    const int N = (int)h->N, nev = (int)h->nev, b = h->b;
    const WsPlan& pl = h->plan;
    const c128* T1 = ws_ptr<c128>(h, pl.T1);
    c128* Vp = ws_ptr<c128>(h, pl.Vp);
    c128* VTh = ws_ptr<c128>(h, pl.VT);
    c128* Y = ws_ptr<c128>(h, pl.bt);
    int np = 0;
    while (N - np * b - b >= 2) ++np;                 // panels that S1 factored
    for (int p = np - 1; p >= 0; --p) {
        const int j0 = p * b;
        const int m = N - j0 - b;
        const int nr = std::min(b, m - 1);
        const c128* Tp = T1 + (size_t)p * b * b;
        bt_extract_v_kernel<<<dim3((unsigned)ceil_div(m, 256), (unsigned)b), 256, 0, s>>>(A, lda, j0 + b, j0, m, b, nr, Vp, m);
        ++h->launches;
        int rc = zgemm_ws(h, false, true, m, b, b, 1.0, Vp, m, Tp, b, 0.0, VTh, m, false, 1, s);
        if (rc) return rc;
        rc = zgemm_ws(h, true, false, b, nev, m, 1.0, VTh, m, Z + (j0 + b), ldz, 0.0, Y, b, true, 1, s);
        if (rc) return rc;
        rc = zgemm_ws(h, false, false, m, nev, b, -1.0, Vp, m, Y, b, 1.0, Z + (j0 + b), ldz, m <= 64, 1, s);
        if (rc) return rc;
    }
    const cudaError_t ce = cudaGetLastError();
    return ce != cudaSuccess ? 1000 + (int)ce : 0;
}

}  // namespace eigh
