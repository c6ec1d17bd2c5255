// assemble.cu -- SCF prologue: the dense BdG matrix from its fields.
//
// PAPER.md:103-107 (Eq. 5 / 7): H = [[h, Delta], [Delta^*, -h^*]], h = T + V - mu, T the spectral kinetic term applied
// along each axis (Eq. 8) through dense 1-D matrices, the whole matrix kept dense.
// Grid point r = (ix ny + iy) nz + iz, matrix index s M + r (s = 0: u, 1: v).  Element (i, j) = (s, r; s', r'):
//   s == s':  (+1 for s = 0, -1 for s = 1) * ( Kx[ix,jx] [iy==jy, iz==jz] + Ky[iy,jy] [ix==jx, iz==jz]
//                                             + Kz[iz,jz] [ix==jx, iy==jy] + (V[r] - mu) [r == r'] )
//   s != s':  Delta[r] (s = 0) or conj(Delta[r]) (s = 1) if r == r', else 0.
// The diagonal is summed in the order ((Kx + Ky) + Kz + V) - mu.  Every one of the N^2 elements is written (both
// triangles): the kernel is bound by HBM writes, 16 N^2 bytes; stores are streaming, 512 contiguous bytes per warp.
#include "eigh_internal.h"

namespace eigh {

constexpr int AS_THREADS = 256;
constexpr int AS_COLS = 16;       // columns per thread block: the row decomposition is done once per thread

struct AssembleArgs {
    int nx, ny, nz;
    int64_t M;
    const double *Kx, *Ky, *Kz, *V;
    const c128* Delta;
    double mu, sign;
    c128* A;
    int64_t lda;
};

__global__ void __launch_bounds__(AS_THREADS) assemble_bdg_kernel(const AssembleArgs p) {
    const int64_t N = 2 * p.M;
    const int64_t i = (int64_t)blockIdx.x * AS_THREADS + threadIdx.x;
    const int64_t j0 = (int64_t)blockIdx.y * AS_COLS;
    if (i >= N) return;
    const int M = (int)p.M;
    const int s = i >= M ? 1 : 0;
    const int r = (int)i - s * M;
    const int iz = r % p.nz;
    const int iy = (r / p.nz) % p.ny;
    const int ix = r / (p.nz * p.ny);
    const double hs = (s ? -1.0 : 1.0) * p.sign;
    const double vr = __ldg(p.V + r);
    const c128 dr = __ldg(p.Delta + r);
    // column (s2, jx, jy, jz): decomposed once, then advanced with carries (uniform over the block)
    int s2 = j0 >= M ? 1 : 0;
    int r2 = (int)j0 - s2 * M;
    int jz = r2 % p.nz, jy = (r2 / p.nz) % p.ny, jx = r2 / (p.nz * p.ny);
    c128* out = p.A + i + j0 * p.lda;
#pragma unroll 4
    for (int jj = 0; jj < AS_COLS; ++jj) {
        if (j0 + jj >= N) break;
        c128 val = cmake(0.0, 0.0);
        if (s == s2) {
            double h = 0.0;
            bool any = false;
            if (iy == jy && iz == jz) { h = __ldg(p.Kx + ix + jx * p.nx); any = true; }
            if (ix == jx && iz == jz) { const double k = __ldg(p.Ky + iy + jy * p.ny); h = any ? h + k : k; any = true; }
            if (ix == jx && iy == jy) { const double k = __ldg(p.Kz + iz + jz * p.nz); h = any ? h + k : k; any = true; }
            if (r == r2) h = (h + vr) - p.mu;
            if (any) val.x = hs * h;
        } else if (r == r2) {
            val = cmake(p.sign * dr.x, (s ? -p.sign : p.sign) * dr.y);
        }
        __stcs(out, val);
        out += p.lda;
        ++r2;
        if (++jz == p.nz) { jz = 0; if (++jy == p.ny) { jy = 0; ++jx; } }
        if (r2 == M) { r2 = 0; s2 = 1; jx = jy = jz = 0; }
    }
}

int launch_assemble_bdg(const AssembleArgs& a, cudaStream_t s) {
    const int64_t N = 2 * a.M;
    dim3 grid((unsigned)ceil_div(N, AS_THREADS), (unsigned)ceil_div(N, AS_COLS));
    assemble_bdg_kernel<<<grid, AS_THREADS, 0, s>>>(a);
    EIGH_CUDA_OK(cudaGetLastError());
    return 0;
}

}  // namespace eigh

using namespace eigh;

extern "C" int eigh_assemble_bdg(eigh_handle_t h, int64_t nx, int64_t ny, int64_t nz, const double* Kx_dev,
                                 const double* Ky_dev, const double* Kz_dev, const double* V_dev, const void* Delta_dev,
                                 double mu, double sign, void* A_dev, int64_t lda, void* stream) {
    if (!h) return -1;
    if (nx < 1 || ny < 1 || nz < 1 || nx > 1 << 20 || ny > 1 << 20 || nz > 1 << 20) return -2;
    if (2 * nx * ny * nz != h->N) return set_err(h, -2, "eigh_assemble_bdg: 2 nx ny nz = %lld != N = %lld", (long long)(2 * nx * ny * nz), (long long)h->N);
    if (!Kx_dev) return -5;
    if (!Ky_dev) return -6;
    if (!Kz_dev) return -7;
    if (!V_dev) return -8;
    if (!Delta_dev) return -9;
    if (!(sign == 1.0 || sign == -1.0)) return -11;
    if (!A_dev) return -12;
    if (lda < h->N) return -13;
    AssembleArgs a;
    a.nx = (int)nx; a.ny = (int)ny; a.nz = (int)nz;
    a.M = h->N / 2;
    a.Kx = Kx_dev; a.Ky = Ky_dev; a.Kz = Kz_dev; a.V = V_dev;
    a.Delta = (const c128*)Delta_dev;
    a.mu = mu; a.sign = sign;
    a.A = (c128*)A_dev; a.lda = lda;
    const int rc = launch_assemble_bdg(a, (cudaStream_t)stream);
    if (rc >= 1000) return set_err(h, rc, "assemble_bdg: CUDA error %d (%s)", rc - 1000, cudaGetErrorString((cudaError_t)(rc - 1000)));
    return rc;
}
