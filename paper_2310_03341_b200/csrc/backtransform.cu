// backtransform.cu -- S4b: the second back-transformation of the eigenvectors
// ("the subsequent back transformation of the eigenvectors also requires two
// stages"), SURVEY.md 8(a) row S4b.  (S4a lives in bt_band.cu.)
//
// S4b  Z <- Q1 Z,  Q1 = Q_0 Q_1 ... Q_{np-1},  Q_p = I - V_p T_p V_p^H  (panels of S1).
//      Groups of mg adjacent panels are merged into one compact-WY block
//          Q_p0 ... Q_{p0+mg-1} = I - V T V^H,   V = [V_p0 | V_p0+1 | ...]  (m x kb, kb = mg b),
//          T[0:jb, j] = -T[0:jb, 0:jb] (V[:, 0:jb]^H V_j) T_j,  T[j, j] = T_j (kept from S1),
//      so that the rank-kb update  Z_rows -= V (T V^H Z_rows)  runs with inner dimension kb = 256
//      instead of 64 (the C tile of Z is read and written once per 256 inner products).
//      Groups are applied last -> first:  Y = (V T^H)^H Z_rows ;  Z_rows -= V Y.
#include <algorithm>

#include "eigh_internal.h"
#include "zgemm.cuh"

namespace eigh {

int zgemm_ws(eigh_handle_s* h, bool ta, bool tb, int M, int N, int K, double alpha, const c128* A, int64_t lda,
             const c128* B, int64_t ldb, double beta, c128* C, int64_t ldc, bool small_tile, int splitk,
             cudaStream_t s);

// V (m x kb, ldv): explicit unit-lower-trapezoidal reflectors of panels p0 .. p0+cnt-1 taken from A.
// Column c belongs to panel q = c / b; its unit diagonal sits at local row q b + (c % b).
__global__ void bt_extract_vgroup_kernel(const c128* __restrict__ A, int64_t lda, int N, int b, int p0, int cnt,
                                         c128* __restrict__ V, int64_t ldv) {
    const int c = blockIdx.y;
    const int q = c / b, cl = c % b;
    const int row0 = (p0 + 1) * b;            // global row of local row 0
    const int m = N - row0;
    const int mq = m - q * b;                 // rows of panel q
    const int nrq = min(b, mq - 1);           // reflectors of panel q
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= m) return;
    const int rr = r - q * b;                 // row inside panel q
    c128 v = cmake(0.0, 0.0);
    if (rr == cl) v = cmake(1.0, 0.0);
    else if (rr > cl && cl < nrq) v = A[(row0 + r) + (int64_t)((p0 + q) * b + cl) * lda];
    V[r + (int64_t)c * ldv] = v;
}

// T (kb x kb) <- blockdiag(T_p0, ..., T_p0+cnt-1), zero elsewhere
__global__ void bt_tdiag_kernel(const c128* __restrict__ T1, int b, int p0, int cnt, c128* __restrict__ T, int ldt) {
    const int kb = cnt * b;
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < kb * kb; idx += gridDim.x * blockDim.x) {
        const int i = idx % kb, j = idx / kb;
        c128 v = cmake(0.0, 0.0);
        if (i / b == j / b) v = T1[(size_t)(p0 + i / b) * b * b + (i % b) + (size_t)(j % b) * b];
        T[i + (size_t)j * ldt] = v;
    }
}

static int splitk_for(const eigh_handle_s* h, int M, int N, int K) {
    // enough thread blocks for >= 4 waves of 2 x num_sms resident 64x64 tiles
    const int64_t tiles = ceil_div(M, 64) * ceil_div(N, 64);
    const int64_t want = 8 * (int64_t)h->num_sms;
    int sk = (int)ceil_div(want, tiles);
    if (sk < 1) sk = 1;
    while (sk > 1 && K / sk < 256) --sk;
    if (sk > 16) sk = 16;
    return sk;
}

int phase_backtransform_full(eigh_handle_s* h, const c128* A, int64_t lda, c128* Z, int64_t ldz, cudaStream_t s) {
    const int N = (int)h->N, nev = (int)h->nev, b = h->b;
    const WsPlan& pl = h->plan;
    const c128* T1 = ws_ptr<c128>(h, pl.T1);
    c128* V = ws_ptr<c128>(h, pl.b4V);
    c128* VTh = ws_ptr<c128>(h, pl.b4VT);
    c128* Y = ws_ptr<c128>(h, pl.b4Y);
    c128* T = ws_ptr<c128>(h, pl.b4T);
    c128* G = ws_ptr<c128>(h, pl.b4G);
    const int mg = h->p4b_merge < 1 ? 1 : h->p4b_merge;
    c128* tmp = G + (size_t)mg * b * mg * b;
    int np = 0;
    while (N - np * b - b >= 2) ++np;                 // panels that S1 factored
    for (int pend = np; pend > 0;) {
        const int cnt = std::min(mg, pend);
        const int p0 = pend - cnt;
        const int m = N - (p0 + 1) * b;
        const int kb = cnt * b;
        c128* Zr = Z + (p0 + 1) * b;
        bt_extract_vgroup_kernel<<<dim3((unsigned)ceil_div(m, 256), (unsigned)kb), 256, 0, s>>>(A, lda, N, b, p0, cnt, V, m);
        ++h->launches;
        const c128* Tg = T1 + (size_t)p0 * b * b;
        int ldt = b;
        int rc;
        if (cnt > 1) {
            // G = V^H V  (kb x kb)
            rc = zgemm_ws(h, true, false, kb, kb, m, 1.0, V, m, V, m, 0.0, G, kb, true, splitk_for(h, kb, kb, m), s);
            if (rc) return rc;
            bt_tdiag_kernel<<<64, 256, 0, s>>>(T1, b, p0, cnt, T, kb);
            ++h->launches;
            for (int j = 1; j < cnt; ++j) {
                const int jb = j * b;
                // tmp (jb x b) = G[0:jb, jb:jb+b] T_j ;  T[0:jb, jb:jb+b] = -T[0:jb, 0:jb] tmp
                rc = zgemm_ws(h, false, false, jb, b, b, 1.0, G + (size_t)jb * kb, kb, T1 + (size_t)(p0 + j) * b * b, b, 0.0,
                              tmp, jb, true, 1, s);
                if (rc) return rc;
                rc = zgemm_ws(h, false, false, jb, b, jb, -1.0, T, kb, tmp, jb, 0.0, T + (size_t)jb * kb, kb, true, 1, s);
                if (rc) return rc;
            }
            Tg = T;
            ldt = kb;
        }
        // VTh = V T^H
        rc = zgemm_ws(h, false, true, m, kb, kb, 1.0, V, m, Tg, ldt, 0.0, VTh, m, true, 1, s);
        if (rc) return rc;
        // Y = VTh^H Z_rows  (kb x nev, K = m)
        rc = zgemm_ws(h, true, false, kb, nev, m, 1.0, VTh, m, Zr, ldz, 0.0, Y, kb, true, splitk_for(h, kb, nev, m), s);
        if (rc) return rc;
        // Z_rows -= V Y
        rc = zgemm_ws(h, false, false, m, nev, kb, -1.0, V, m, Y, kb, 1.0, Zr, ldz, true, 1, s);
        if (rc) return rc;
        pend = p0;
    }
    const cudaError_t ce = cudaGetLastError();
    return ce != cudaSuccess ? 1000 + (int)ce : 0;
}

}  // namespace eigh
