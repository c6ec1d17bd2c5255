// backtransform.cu -- S4a / S4b: the two back-transformations of the eigenvectors
// ("the subsequent back transformation of the eigenvectors also requires two
// stages"), SURVEY.md 8(a) rows S4a, S4b.
//
// S4a  Z <- Q2 (sgn o Q_T).  Q2 is the product of all bulge-chasing reflectors H_{j,k} (sweep j,
//      step k, rows j+1+k b ..).  Reflectors of g consecutive sweeps at the same step k form a
//      "diamond" WY block  I - V T V^H  with V of size (b+g-1) x g (column t shifted down by t).
//      Valid application order: sweep groups from the last to the first; inside a group k
//      ascending (H_{j',k} and H_{j',k-1} with j' > j must be applied before H_{j,k}).
//      Per diamond:  Y = (V T^H)^H Z_rows ;  Z_rows -= V Y   (two DMMA GEMMs).
// S4b  Z <- Q1 Z.  Panels of S1 in reverse order, Z_rows <- (I - V_p T_p V_p^H) Z_rows with the
//      T factors kept from S1:  Y = (V T^H)^H Z_rows ;  Z_rows -= V Y.
#include "eigh_internal.h"
#include "zgemm.cuh"

namespace eigh {

int zgemm_ws(eigh_handle_s* h, bool ta, bool tb, int M, int N, int K, double alpha, const c128* A, int64_t lda,
             const c128* B, int64_t ldb, double beta, c128* C, int64_t ldc, bool small_tile, int splitk,
             cudaStream_t s);

static inline int64_t bt_ldv(const eigh_handle_s* h) { return round_up(h->b + h->g, 8); }
static inline int64_t bt_kmax(const eigh_handle_s* h) { return ceil_div(h->N, h->b) + 1; }

size_t bt_scratch_bytes(const eigh_handle_s* h) {
    const size_t diamonds = (size_t)bt_kmax(h) * bt_ldv(h) * h->g * sizeof(c128) * 2;   // Vd and VTd
    const size_t y = (size_t)std::max(h->g, h->b) * h->nev * sizeof(c128);
    return diamonds + y + 4096;
}

// ------------------------------------------------------------------ S4a
// Z[r, c] = sgn[r] * Qt[r + c*ldq]
__global__ void bt_expand_kernel(const double* __restrict__ Qt, int64_t ldq, const double* __restrict__ sgn, int N,
                                 int nev, c128* __restrict__ Z, int64_t ldz) {
    const int c = blockIdx.y;
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r < N && c < nev) Z[r + (int64_t)c * ldz] = cmake(sgn[r] * Qt[r + (int64_t)c * ldq], 0.0);
}

// One CTA per diamond (sweep group j0..j0+gs-1, step k = blockIdx.x): gathers the reflectors into
// the dense zero-padded Vd (ldv x gs), forms G = Vd^H Vd, T (tfactor recurrence) and VTd = Vd T^H.
struct DiamondArgs {
    const c128* V2; int N, b, g;
    int j0, gs;
    c128* Vd; c128* VTd; int64_t ldv;     // per diamond: ldv * g elements
};

__global__ void __launch_bounds__(256, 1) bt_diamond_prep_kernel(const DiamondArgs a) {
    extern __shared__ __align__(16) unsigned char dp_raw[];
    const int ldv = (int)a.ldv, g = a.g;
    c128* Vs = reinterpret_cast<c128*>(dp_raw);         // ldv x g
    c128* Gs = Vs + (size_t)ldv * g;                    // g x (g+1): strict upper = G, lower+diag = T^T
    c128* taus = Gs + (size_t)g * (g + 1);              // g
    const int k = blockIdx.x;
    const int N = a.N, b = a.b, gs = a.gs;
    const int R0 = a.j0 + 1 + k * b;
    const int tid = threadIdx.x;
    const int ldg = g + 1;
    // gather: column t = reflector of sweep j = j0+t at rows R0+t .. R0+t+len-1
    for (int idx = tid; idx < ldv * g; idx += 256) {
        const int rl = idx % ldv, t = idx / ldv;
        c128 v = cmake(0.0, 0.0);
        if (t < gs) {
            const int j = a.j0 + t;
            const int row = R0 + rl;
            const int rs = R0 + t;                       // first row of this reflector
            const int len = min(b, N - rs);
            if (len > 0 && row >= rs && row < rs + len) {
                const int64_t voff = (int64_t)j * (N - 1) - (int64_t)j * (j - 1) / 2;
                const c128 e = a.V2[voff + row - j - 1];
                if (row == rs) { taus[t] = e; v = cmake(1.0, 0.0); }
                else v = e;
            } else if (len <= 0 && rl == 0) {
                taus[t] = cmake(0.0, 0.0);
            }
        } else if (rl == 0) {
            taus[t] = cmake(0.0, 0.0);
        }
        Vs[idx] = v;
    }
    __syncthreads();
    // G = Vs^H Vs (upper part is enough)
    for (int idx = tid; idx < g * g; idx += 256) {
        const int i = idx % g, j = idx / g;
        c128 s = cmake(0.0, 0.0);
        if (i < j && j < gs) {
            // reflector i spans rows [i, i+b), reflector j rows [j, j+b): overlap [j, i+b)
            const int lo = j, hi = min(ldv, i + b);
            for (int r = lo; r < hi; ++r) cfmac(s, Vs[r + i * ldv], Vs[r + j * ldv]);
        }
        if (i < j) Gs[i + j * ldg] = s;
    }
    __syncthreads();
    if (tid < g) {
        const int j = tid;
        // T[i,j] (i <= j) lives at Gs[j + i*ldg] (transposed into the lower triangle)
        Gs[j + j * ldg] = taus[j];
        for (int i = j - 1; i >= 0; --i) {
            c128 s = cmake(0.0, 0.0);
            for (int l = i + 1; l <= j; ++l) cfma(s, Gs[i + l * ldg], Gs[j + l * ldg]);
            const c128 ti = taus[i];
            Gs[j + i * ldg] = cmake(-(ti.x * s.x - ti.y * s.y), -(ti.x * s.y + ti.y * s.x));
        }
    }
    __syncthreads();
    // outputs: Vd, VTd = Vd T^H  (VTd[r,j] = sum_{l >= j} Vd[r,l] conj(T[j,l]))
    c128* Vd = a.Vd + (size_t)k * ldv * g;
    c128* VTd = a.VTd + (size_t)k * ldv * g;
    for (int idx = tid; idx < ldv * g; idx += 256) {
        const int rl = idx % ldv, j = idx / ldv;
        Vd[idx] = Vs[idx];
        c128 s = cmake(0.0, 0.0);
        for (int l = j; l < g; ++l) {
            const c128 t = Gs[l + j * ldg];        // T[j,l]
            const c128 v = Vs[rl + l * ldv];
            // v * conj(t)
            s.x += v.x * t.x + v.y * t.y;
            s.y += v.y * t.x - v.x * t.y;
        }
        VTd[idx] = s;
    }
}

int phase_backtransform_band(eigh_handle_s* h, const double* Qt, int64_t ldq, c128* Z, int64_t ldz, cudaStream_t s) {
    const int N = (int)h->N, nev = (int)h->nev, b = h->b, g = h->g;
    const WsPlan& pl = h->plan;
    const double* sgn = ws_ptr<double>(h, pl.sgn);
    const c128* V2 = ws_ptr<c128>(h, pl.V2);
    const int64_t ldv = bt_ldv(h);
    c128* Vd = ws_ptr<c128>(h, pl.bt);
    c128* VTd = Vd + (size_t)bt_kmax(h) * ldv * g;
    c128* Y = VTd + (size_t)bt_kmax(h) * ldv * g;

    bt_expand_kernel<<<dim3((unsigned)ceil_div(N, 256), (unsigned)nev), 256, 0, s>>>(Qt, ldq, sgn, N, nev, Z, ldz);
    ++h->launches;
    if (N < 2) return 0;
    const size_t smem = ((size_t)ldv * g + (size_t)g * (g + 1) + g) * sizeof(c128);
    static size_t attr_smem = 0;
    if (smem > attr_smem) {
        EIGH_CUDA_OK(cudaFuncSetAttribute(bt_diamond_prep_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr_smem = smem;
    }
    const int nsweeps = N - 1;                       // sweeps j = 0..N-2
    const int ngroups = (int)ceil_div(nsweeps, g);
    for (int J = ngroups - 1; J >= 0; --J) {
        const int j0 = J * g;
        const int gs = std::min(g, nsweeps - j0);
        // steps k with a non-empty first reflector: R0 = j0+1+k b <= N-1
        const int nk = (int)ceil_div(N - 1 - j0, b);
        if (nk <= 0) continue;
        DiamondArgs da;
        da.V2 = V2; da.N = N; da.b = b; da.g = g; da.j0 = j0; da.gs = gs; da.Vd = Vd; da.VTd = VTd; da.ldv = ldv;
        bt_diamond_prep_kernel<<<nk, 256, smem, s>>>(da);
        ++h->launches;
        for (int k = 0; k < nk; ++k) {
            const int R0 = j0 + 1 + k * b;
            const int nr = std::min(N - R0, b + gs - 1);
            if (nr <= 0) break;
            const c128* Vk = Vd + (size_t)k * ldv * g;
            const c128* VTk = VTd + (size_t)k * ldv * g;
            int rc = zgemm_ws(h, true, false, gs, nev, nr, 1.0, VTk, ldv, Z + R0, ldz, 0.0, Y, g, true, 1, s);
            if (rc) return rc;
            rc = zgemm_ws(h, false, false, nr, nev, gs, -1.0, Vk, ldv, Y, g, 1.0, Z + R0, ldz, nr <= 64, 1, s);
            if (rc) return rc;
        }
    }
    const cudaError_t ce = cudaGetLastError();
    return ce != cudaSuccess ? 1000 + (int)ce : 0;
}

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
