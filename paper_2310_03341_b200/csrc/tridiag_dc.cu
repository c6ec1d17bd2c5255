// tridiag_dc.cu -- S3: real symmetric tridiagonal eigensolver by divide & conquer, entirely on the
// GPU ("diagonalizing this tridiagonal form"; method fixed by north_star; SURVEY.md
// 8(a) rows S3.1-S3.5).  Cuppen's rank-one tearing with the Gu-Eisenstat stabilisation:
//
//   T = blockdiag(T1', T2') + rho w w^T,  T1' = Q1 D1 Q1^T, T2' = Q2 D2 Q2^T
//     = blockdiag(Q1,Q2) (D + rho_eff z z^T) blockdiag(Q1,Q2)^T,  z = [last row Q1, first row Q2]/sqrt2
//
//   S3.1 leaves (<= 32) by the implicit symmetric QR iteration with Wilkinson shift, one warp each
//   S3.2 z vector, sort of D (rank by counting), deflation scan (tiny z_i; close d pair -> Givens)
//   S3.3 secular equation 1 + rho sum z_i^2/(d_i - lambda) = 0: one root per thread, stored as
//        (origin, offset) so that d_i - lambda_j keeps full relative accuracy; two-pole rational
//        interpolation with a bisection safeguard
//   S3.4 z_hat from the Loewner product formula, U[:,j] = normalise(z_hat_i / (d_i - lambda_j))
//   S3.5 Q_new[:, :k] = Q_old[:, kept] U on the DMMA path (dgemm.cuh); deflated columns copied
//
// All merges of one tree level run batched (blockIdx.y = merge); the deflation counts k stay on the
// device (worst-case grids, surplus CTAs exit), so the whole phase needs no host round trip except
// the final failure counter.
#include <math.h>

#include <vector>

#include "dgemm.cuh"
#include "eigh_internal.h"

namespace eigh {

struct MergeDesc { int s, mid, e, pad; };

constexpr double DC_EPS = 1.1102230246251565e-16;   // 2^-53 (LAPACK dlamch('E'))
constexpr int DC_LEAF_MAX = 32;

// ------------------------------------------------------------------ arena
struct DcBufs {
    double *QA, *QB, *U;              // ldq x N each
    double *dcur, *dnew, *z, *dk, *zk, *mu, *lam, *zhat, *rot_c, *rot_s, *rho, *zsum, *esgn, *esc, *scale, *stats;
    int *perm, *nd_idx, *df_idx, *org, *rot_a, *rot_b, *kcount, *nrot, *fail, *bnd;
    int *ctype, *ktype, *upos, *acol, *k1c, *k2c;   // block structure of Q_old (column types, U row order)
    MergeDesc* desc;                  // all levels, concatenated
    DgemmDesc* gdesc;
    int64_t ldq;
};

static size_t dc_small_bytes(int64_t N) { return (size_t)(16 * 8 + 18 * 4) * (N + 64) + (size_t)(N + 64) * (sizeof(MergeDesc) + sizeof(DgemmDesc)) * 2 + 16384; }   // (14 double + 15 int arrays, each rounded up to 256 bytes)

size_t dc_arena_bytes(int64_t N) {
    const int64_t ldq = round_up(N, 8);
    return (size_t)3 * ldq * N * sizeof(double) + dc_small_bytes(N) + 4096;
}

// offset of the U buffer inside the arena: dead once the last merge GEMM has run, so the sorted
// N x nev result of the phase is written there (never aliases the final Q, which is QA or QB)
size_t dc_result_offset(int64_t N) {
    const size_t qb = ((size_t)round_up(N, 8) * N * sizeof(double) + 255) / 256 * 256;
    return 2 * qb;
}

static DcBufs dc_carve(void* base, int64_t N) {
    DcBufs b;
    b.ldq = round_up(N, 8);
    char* p = (char*)base;
    auto take = [&](size_t bytes) { char* r = p; p += (bytes + 255) / 256 * 256; return r; };
    const size_t qb = (size_t)b.ldq * N * sizeof(double);
    b.QA = (double*)take(qb);
    b.QB = (double*)take(qb);
    b.U = (double*)take(qb);
    const size_t nd = (size_t)(N + 64) * sizeof(double), ni = (size_t)(N + 64) * sizeof(int);
    b.dcur = (double*)take(nd); b.dnew = (double*)take(nd); b.z = (double*)take(nd);
    b.dk = (double*)take(nd); b.zk = (double*)take(nd); b.mu = (double*)take(nd);
    b.lam = (double*)take(nd); b.zhat = (double*)take(nd); b.rot_c = (double*)take(nd);
    b.rot_s = (double*)take(nd); b.rho = (double*)take(nd); b.zsum = (double*)take(nd);
    b.esgn = (double*)take(nd);
    b.esc = (double*)take(nd);
    b.scale = (double*)take(256);
    b.stats = (double*)take(32 * 3 * sizeof(double));
    b.perm = (int*)take(ni); b.nd_idx = (int*)take(ni); b.df_idx = (int*)take(ni); b.org = (int*)take(ni);
    b.rot_a = (int*)take(ni); b.rot_b = (int*)take(ni); b.kcount = (int*)take(ni); b.nrot = (int*)take(ni);
    b.fail = (int*)take(256); b.bnd = (int*)take(ni);
    b.ctype = (int*)take(ni); b.ktype = (int*)take(ni); b.upos = (int*)take(ni); b.acol = (int*)take(ni);
    b.k1c = (int*)take(ni); b.k2c = (int*)take(ni);
    b.desc = (MergeDesc*)take((size_t)(N + 64) * sizeof(MergeDesc));
    b.gdesc = (DgemmDesc*)take((size_t)(N + 64) * sizeof(DgemmDesc));
    return b;
}

// ------------------------------------------------------------------ S3.0 tearing
// The deflation test of the merge step compares rho |z_i| with 8 eps max(|d|_max, |z|_max), z of unit norm: it assumes a
// matrix of norm ~1 (LAPACK's xSTEDC scales to norm 1 before it calls the merge; without that a matrix of norm 1e-100
// deflates everything and returns its diagonal).  scale[0] = the power of two next to max(|d|, |e|) -- the scaling is then
// exact, and results for matrices of norm >= 1 are bit for bit what they were without it -- scale[1] = 1 / scale[0].
__global__ void __launch_bounds__(1024) dc_norm_kernel(const double* __restrict__ d_in, const double* __restrict__ e_in, int N,
                                                       double* __restrict__ scale) {
    __shared__ double red[32];
    double m = 0.0;
    for (int i = threadIdx.x; i < N; i += 1024) {
        m = fmax(m, fabs(d_in[i]));
        if (i < N - 1) m = fmax(m, fabs(e_in[i]));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 32; ++w) m = fmax(m, red[w]);
        double sg = 1.0;
        if (m > 0.0 && isfinite(m)) {
            int ex;
            frexp(m, &ex);                       // m = f 2^ex, f in [0.5, 1)
            ex -= 1;                             // m / 2^ex in [1, 2)
            if (ex > 1000) ex = 1000;            // (2^-ex must stay a normal number)
            if (ex < -1000) ex = -1000;
            sg = ldexp(1.0, ex);
        }
        scale[0] = sg;
        scale[1] = 1.0 / sg;
    }
}
__global__ void dc_tear_kernel(const double* __restrict__ d_in, const double* __restrict__ e_in, int N,
                               const int* __restrict__ bnd, int L, const double* __restrict__ scale, double* __restrict__ dcur,
                               double* __restrict__ esc) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const double inv = scale[1];
    if (i < N) {
        dcur[i] = d_in[i] * inv;
        esc[i] = (i < N - 1) ? e_in[i] * inv : 0.0;
    }
}
__global__ void dc_tear2_kernel(const double* __restrict__ e_in, const int* __restrict__ bnd, int L,
                                double* __restrict__ dcur) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;   // interior boundary t = 1..L-1
    if (t >= 1 && t < L) {
        const int m = bnd[t];
        const double r = fabs(e_in[m - 1]);
        dcur[m - 1] -= r;
        dcur[m] -= r;
    }
}

// The solver works on |e|: T(d, e) = D T(d, |e|) D with D = diag(sgn), sgn_0 = 1, sgn_{i+1} = sgn_i sign(e_i), so the
// eigenvectors of the signed matrix are the rows of Q scaled by sgn (applied in dc_output_kernel).  One thread block:
// every thread counts the negative entries of its contiguous chunk, a block scan gives the parity at its start.
__global__ void __launch_bounds__(1024) dc_esign_kernel(const double* __restrict__ e_in, int N, double* __restrict__ esgn) {
    __shared__ int cnt[1024];
    const int tid = threadIdx.x;
    const int per = (N + 1023) / 1024;
    const int lo = tid * per, hi = min(N, lo + per);       // sgn[i] for i in [lo, hi) needs e[0 .. i-1]
    int c = 0;
    for (int i = lo; i < hi; ++i) c += (i >= 1 && e_in[i - 1] < 0.0) ? 1 : 0;
    cnt[tid] = c;
    __syncthreads();
    for (int o = 1; o < 1024; o <<= 1) {                     // inclusive scan
        const int v = (tid >= o) ? cnt[tid - o] : 0;
        __syncthreads();
        cnt[tid] += v;
        __syncthreads();
    }
    int par = (cnt[tid] - c) & 1;                            // negatives before this chunk
    for (int i = lo; i < hi; ++i) {
        if (i >= 1 && e_in[i - 1] < 0.0) par ^= 1;
        esgn[i] = par ? -1.0 : 1.0;
    }
}

// ------------------------------------------------------------------ S3.1 leaves
__global__ void __launch_bounds__(128) dc_leaf_kernel(const int* __restrict__ bnd, int L, double* __restrict__ dcur,
                                                      const double* __restrict__ e_in, double* __restrict__ Q,
                                                      int64_t ldq, int* __restrict__ fail) {
    __shared__ double Qs_all[4][DC_LEAF_MAX * (DC_LEAF_MAX + 1)];
    __shared__ double ds_all[4][DC_LEAF_MAX], es_all[4][DC_LEAF_MAX];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int leaf = blockIdx.x * 4 + warp;
    if (leaf >= L) return;
    double* Qs = Qs_all[warp];
    double* ds = ds_all[warp];
    double* es = es_all[warp];
    const int s = bnd[leaf], n = bnd[leaf + 1] - s;
    constexpr int LD = DC_LEAF_MAX + 1;
    if (lane < n) {
        ds[lane] = dcur[s + lane];
        es[lane] = (lane < n - 1) ? fabs(e_in[s + lane]) : 0.0;
        for (int c = 0; c < n; ++c) Qs[lane * LD + c] = (c == lane) ? 1.0 : 0.0;
    }
    __syncwarp();
    int hi = n - 1, iter = 0;
    const int maxit = 40 * n;
    while (hi > 0) {
        if (fabs(es[hi - 1]) <= DC_EPS * (fabs(ds[hi - 1]) + fabs(ds[hi]))) {
            __syncwarp();
            if (lane == 0) es[hi - 1] = 0.0;
            __syncwarp();
            --hi;
            continue;
        }
        int lo = hi - 1;
        while (lo > 0 && fabs(es[lo - 1]) > DC_EPS * (fabs(ds[lo - 1]) + fabs(ds[lo]))) --lo;
        if (++iter > maxit) {
            if (lane == 0) atomicAdd(fail, 1);
            break;
        }
        // implicit symmetric QR step with Wilkinson shift on the unreduced block [lo, hi]
        const double dd = 0.5 * (ds[hi - 1] - ds[hi]);
        const double eh = es[hi - 1];
        const double shift = ds[hi] - eh * eh / (dd + copysign(hypot(dd, eh), dd == 0.0 ? 1.0 : dd));
        double x = ds[lo] - shift, zb = es[lo];
        for (int kk = lo; kk < hi; ++kk) {
            const double r = hypot(x, zb);
            double c = 1.0, sn = 0.0;
            if (r != 0.0) { c = x / r; sn = -zb / r; }
            const double a = ds[kk], bb = es[kk], cc = ds[kk + 1];
            const double en = (kk + 1 < hi) ? es[kk + 1] : 0.0;
            const double dk0 = c * c * a - 2.0 * c * sn * bb + sn * sn * cc;
            const double dk1 = sn * sn * a + 2.0 * c * sn * bb + c * c * cc;
            const double ek = c * sn * (a - cc) + (c * c - sn * sn) * bb;
            __syncwarp();
            if (lane == 0) {
                if (kk > lo) es[kk - 1] = r;
                ds[kk] = dk0;
                ds[kk + 1] = dk1;
                es[kk] = ek;
                if (kk + 1 < hi) es[kk + 1] = c * en;
            }
            if (lane < n) {
                const double q0 = Qs[lane * LD + kk], q1 = Qs[lane * LD + kk + 1];
                Qs[lane * LD + kk] = c * q0 - sn * q1;
                Qs[lane * LD + kk + 1] = sn * q0 + c * q1;
            }
            x = ek;
            zb = -sn * en;
            __syncwarp();
        }
    }
    __syncwarp();
    if (lane < n) {
        dcur[s + lane] = ds[lane];
        for (int c = 0; c < n; ++c) Q[(s + lane) + (int64_t)(s + c) * ldq] = Qs[lane * LD + c];
    }
}

// ------------------------------------------------------------------ S3.2 z, sort, deflation
__global__ void dc_zero_offdiag_kernel(const MergeDesc* __restrict__ desc, double* __restrict__ Q, int64_t ldq) {
    const MergeDesc m = desc[blockIdx.y];
    const int n1 = m.mid - m.s, n2 = m.e - m.mid;
    const int64_t total = (int64_t)2 * n1 * n2;
    for (int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
        if (idx < (int64_t)n1 * n2) {       // rows [mid,e) x cols [s,mid)
            const int r = (int)(idx % n2), c = (int)(idx / n2);
            Q[(m.mid + r) + (int64_t)(m.s + c) * ldq] = 0.0;
        } else {                            // rows [s,mid) x cols [mid,e)
            const int64_t t = idx - (int64_t)n1 * n2;
            const int r = (int)(t % n1), c = (int)(t / n1);
            Q[(m.s + r) + (int64_t)(m.mid + c) * ldq] = 0.0;
        }
    }
}

__global__ void dc_zvec_kernel(const MergeDesc* __restrict__ desc, const double* __restrict__ Q, int64_t ldq,
                               double* __restrict__ z) {
    const MergeDesc m = desc[blockIdx.y];
    const int i = m.s + blockIdx.x * blockDim.x + threadIdx.x;
    if (i < m.e) {
        const int row = (i < m.mid) ? m.mid - 1 : m.mid;
        z[i] = Q[row + (int64_t)i * ldq] * 0.70710678118654752440;
    }
}

// perm[s + rank] = local index i, rank = #{j: d_j < d_i or (d_j == d_i and j < i)}
__global__ void __launch_bounds__(256) dc_rank_kernel(const MergeDesc* __restrict__ desc, const double* __restrict__ dv,
                                                      int* __restrict__ perm) {
    __shared__ double tile[1024];
    const MergeDesc m = desc[blockIdx.y];
    const int n = m.e - m.s;
    if ((int)(blockIdx.x * 256) >= n) return;
    const int i = blockIdx.x * 256 + threadIdx.x;
    const double di = (i < n) ? dv[m.s + i] : 0.0;
    int rank = 0;
    for (int t0 = 0; t0 < n; t0 += 1024) {
        __syncthreads();
        for (int t = threadIdx.x; t < 1024; t += 256) tile[t] = (t0 + t < n) ? dv[m.s + t0 + t] : 0.0;
        __syncthreads();
        const int lim = min(1024, n - t0);
        for (int t = 0; t < lim; ++t) {
            const double dj = tile[t];
            rank += (dj < di) || (dj == di && (t0 + t) < i);
        }
    }
    if (i < n) perm[m.s + rank] = i;
}

constexpr int DF_CH = 2048;
__global__ void __launch_bounds__(256) dc_deflate_kernel(const MergeDesc* __restrict__ desc, const double* __restrict__ e_in,
                                                         double* __restrict__ dcur, double* __restrict__ z,
                                                         const int* __restrict__ perm, int* __restrict__ nd_idx,
                                                         int* __restrict__ df_idx, int* __restrict__ kcount,
                                                         int* __restrict__ nrot, int* __restrict__ rot_a,
                                                         int* __restrict__ rot_b, double* __restrict__ rot_c,
                                                         double* __restrict__ rot_s, double* __restrict__ dk,
                                                         double* __restrict__ zk, double* __restrict__ rho_out,
                                                         double* __restrict__ zsum_out, int* __restrict__ ctype,
                                                         int* __restrict__ ktype, int* __restrict__ upos,
                                                         int* __restrict__ acol, int* __restrict__ k1c,
                                                         int* __restrict__ k2c) {
    __shared__ double ds[DF_CH], zs[DF_CH];
    __shared__ int is[DF_CH];
    __shared__ double red[16];
    const int mi = blockIdx.x;
    const MergeDesc m = desc[mi];
    const int s = m.s, n = m.e - m.s;
    const int tid = threadIdx.x;
    // column types of Q_old = diag(Q_left, Q_right): 1 = non-zero in the top rows only, 3 = bottom rows only,
    // 2 = both (a deflating rotation mixed a left with a right column)
    for (int i = tid; i < n; i += 256) ctype[s + i] = (i < m.mid - m.s) ? 1 : 3;
    // maxima
    double dmax = 0.0, zmax = 0.0;
    for (int i = tid; i < n; i += 256) {
        dmax = fmax(dmax, fabs(dcur[s + i]));
        zmax = fmax(zmax, fabs(z[s + i]));
    }
    for (int o = 16; o > 0; o >>= 1) {
        dmax = fmax(dmax, __shfl_xor_sync(0xffffffffu, dmax, o));
        zmax = fmax(zmax, __shfl_xor_sync(0xffffffffu, zmax, o));
    }
    if ((tid & 31) == 0) { red[tid >> 5] = dmax; red[8 + (tid >> 5)] = zmax; }
    __syncthreads();
    dmax = 0.0; zmax = 0.0;
    for (int w = 0; w < 8; ++w) { dmax = fmax(dmax, red[w]); zmax = fmax(zmax, red[8 + w]); }
    const double rho = 2.0 * fabs(e_in[m.mid - 1]);
    const double tol = 8.0 * DC_EPS * fmax(dmax, zmax);
    if (tid == 0) rho_out[mi] = rho;

    int k = 0, ndf = 0, nr = 0;
    int pj = -1;
    double dpj = 0.0, zpj = 0.0, zs2 = 0.0;
    const bool all_deflate = (rho * zmax <= tol);
    for (int c0 = 0; c0 < n; c0 += DF_CH) {
        __syncthreads();
        for (int t = tid; t < DF_CH && c0 + t < n; t += 256) {
            int i = perm[s + c0 + t];
            if ((unsigned)i >= (unsigned)n) i = 0;
            is[t] = i;
            ds[t] = dcur[s + i];
            zs[t] = z[s + i];
        }
        __syncthreads();
        if (tid == 0) {
            const int lim = min(DF_CH, n - c0);
            for (int t = 0; t < lim; ++t) {
                const int i = is[t];
                double di = ds[t], zi = zs[t];
                if (all_deflate || rho * fabs(zi) <= tol) {
                    df_idx[s + ndf++] = i;
                    continue;
                }
                if (pj < 0) { pj = i; dpj = di; zpj = zi; continue; }
                double sn = zpj, c = zi;
                const double tau = hypot(c, sn);
                const double tt = di - dpj;
                c /= tau;
                sn = -sn / tau;
                if (fabs(tt * c * sn) <= tol) {
                    // deflate pj: rotate columns (pj, i)
                    zi = tau;
                    rot_a[s + nr] = pj; rot_b[s + nr] = i; rot_c[s + nr] = c; rot_s[s + nr] = sn;
                    ++nr;
                    if (ctype[s + pj] != ctype[s + i]) { ctype[s + pj] = 2; ctype[s + i] = 2; }
                    const double tnew = dpj * c * c + di * sn * sn;
                    di = dpj * sn * sn + di * c * c;
                    dcur[s + pj] = tnew;
                    z[s + pj] = 0.0;
                    df_idx[s + ndf++] = pj;
                } else {
                    dcur[s + pj] = dpj; z[s + pj] = zpj;
                    nd_idx[s + k] = pj; dk[s + k] = dpj; zk[s + k] = zpj; zs2 += zpj * zpj;
                    ktype[s + k] = ctype[s + pj];
                    ++k;
                }
                pj = i; dpj = di; zpj = zi;
            }
        }
    }
    if (tid == 0) {
        if (pj >= 0) {
            dcur[s + pj] = dpj; z[s + pj] = zpj;
            nd_idx[s + k] = pj; dk[s + k] = dpj; zk[s + k] = zpj; zs2 += zpj * zpj;
            ktype[s + k] = ctype[s + pj];
            ++k;
        }
        // memory order of the kept columns (= row order of U): [type 1 | type 2 | type 3], so that the merge GEMM
        // runs as  top rows x K-range [0, k1+k2)  and  bottom rows x K-range [k1, k)
        int k1 = 0, k2 = 0;
        for (int i = 0; i < k; ++i) { const int t = ktype[s + i]; k1 += (t == 1); k2 += (t == 2); }
        int p1 = 0, p2 = k1, p3 = k1 + k2;
        for (int i = 0; i < k; ++i) {
            const int t = ktype[s + i];
            const int pos = (t == 1) ? p1++ : (t == 2) ? p2++ : p3++;
            upos[s + i] = pos;
            acol[s + pos] = nd_idx[s + i];
        }
        k1c[mi] = k1;
        k2c[mi] = k2;
        kcount[mi] = k;
        nrot[mi] = nr;
        zsum_out[mi] = zs2;
    }
}

// apply the recorded Givens rotations, in order, to columns of Q (one thread per row)
__global__ void __launch_bounds__(256) dc_apply_rot_kernel(const MergeDesc* __restrict__ desc, double* __restrict__ Q,
                                                           int64_t ldq, const int* __restrict__ nrot,
                                                           const int* __restrict__ rot_a, const int* __restrict__ rot_b,
                                                           const double* __restrict__ rot_c, const double* __restrict__ rot_s) {
    const MergeDesc m = desc[blockIdx.y];
    const int n = m.e - m.s;
    const int r = blockIdx.x * 256 + threadIdx.x;
    const int nr = nrot[blockIdx.y];
    if (r >= n || nr == 0) return;
    double* Qr = Q + (m.s + r) + (int64_t)m.s * ldq;
    for (int t = 0; t < nr; ++t) {
        const int a = rot_a[m.s + t], b = rot_b[m.s + t];
        const double c = rot_c[m.s + t], sn = rot_s[m.s + t];
        const double x = Qr[(int64_t)a * ldq], y = Qr[(int64_t)b * ldq];
        Qr[(int64_t)a * ldq] = c * x + sn * y;
        Qr[(int64_t)b * ldq] = c * y - sn * x;
    }
}

// ------------------------------------------------------------------ S3.3 secular equation
struct SecEval { double psi, dpsi, phi, dphi; };

__device__ __forceinline__ SecEval sec_eval(int k, const double* __restrict__ dk, const double* __restrict__ zk,
                                            double rho, int o, double mu, int isplit) {
    SecEval r = {0.0, 0.0, 0.0, 0.0};
    const double dorg = dk[o];
    for (int i = 0; i <= isplit; ++i) {
        const double inv = 1.0 / ((dk[i] - dorg) - mu);
        const double t = rho * zk[i] * zk[i] * inv;
        r.psi += t;
        r.dpsi += t * inv;
    }
    for (int i = isplit + 1; i < k; ++i) {
        const double inv = 1.0 / ((dk[i] - dorg) - mu);
        const double t = rho * zk[i] * zk[i] * inv;
        r.phi += t;
        r.dphi += t * inv;
    }
    return r;
}

__global__ void __launch_bounds__(128) dc_secular_kernel(const MergeDesc* __restrict__ desc, const int* __restrict__ kcount,
                                                         const double* __restrict__ dk_all, const double* __restrict__ zk_all,
                                                         const double* __restrict__ rho_all, const double* __restrict__ zsum_all,
                                                         int* __restrict__ org_all, double* __restrict__ mu_all,
                                                         double* __restrict__ lam_all, int* __restrict__ fail) {
    const int mi = blockIdx.y;
    const int k = kcount[mi];
    const int j = blockIdx.x * 128 + threadIdx.x;
    if (j >= k) return;
    const int s = desc[mi].s;
    const double* dk = dk_all + s;
    const double* zk = zk_all + s;
    const double rho = rho_all[mi];
    if (k == 1) {
        org_all[s] = 0;
        mu_all[s] = rho * zk[0] * zk[0];
        lam_all[s] = dk[0] + mu_all[s];
        return;
    }
    const bool last = (j == k - 1);
    const int iL = last ? k - 2 : j, iR = last ? k - 1 : j + 1;
    const int isplit = iL;
    int o;
    double mu, lo, hi;
    SecEval ev;
    if (!last) {
        const double gap = dk[j + 1] - dk[j];
        o = j;
        mu = 0.5 * gap;
        ev = sec_eval(k, dk, zk, rho, o, mu, isplit);
        if (1.0 + ev.psi + ev.phi >= 0.0) { lo = 0.0; hi = mu; }
        else { o = j + 1; mu = -0.5 * gap; lo = mu; hi = 0.0; }
        // (ev stays valid: the same point expressed against the other origin)
    } else {
        o = k - 1;
        lo = 0.0;
        hi = rho * zsum_all[mi];
        mu = 0.5 * hi;
        ev = sec_eval(k, dk, zk, rho, o, mu, isplit);
    }
    const double dL = dk[iL] - dk[o], dR = dk[iR] - dk[o];
    bool ok = false;
    for (int it = 0; it < 80; ++it) {
        const double g = 1.0 + ev.psi + ev.phi;
        const double err = DC_EPS * (8.0 * (fabs(ev.psi) + fabs(ev.phi)) + 2.0 + fabs(mu) * (ev.dpsi + ev.dphi));
        if (fabs(g) <= err) { ok = true; break; }
        if (g < 0.0) lo = mu; else hi = mu;
        const double AL = dL - mu, AR = dR - mu;
        const double p = ev.dpsi * AL * AL, sL = ev.psi - ev.dpsi * AL;
        const double q = ev.dphi * AR * AR, sR = ev.phi - ev.dphi * AR;
        const double c = 1.0 + sL + sR;
        const double a2 = c, b2 = -(c * (AL + AR) + p + q), c2 = AL * AR * g;
        double eta;
        bool have = false;
        if (a2 == 0.0) {
            if (b2 != 0.0) { eta = -c2 / b2; have = true; }
        } else {
            double disc = b2 * b2 - 4.0 * a2 * c2;
            if (disc < 0.0) disc = 0.0;
            const double sq = sqrt(disc);
            const double qq = -0.5 * (b2 + copysign(sq, b2));
            const double r1 = qq / a2;
            const double r2 = (qq != 0.0) ? c2 / qq : 0.0;
            const bool in1 = (mu + r1 > lo) && (mu + r1 < hi);
            const bool in2 = (qq != 0.0) && (mu + r2 > lo) && (mu + r2 < hi);
            if (in1 && in2) { eta = (fabs(r1) < fabs(r2)) ? r1 : r2; have = true; }
            else if (in1) { eta = r1; have = true; }
            else if (in2) { eta = r2; have = true; }
        }
        double munew = have ? mu + eta : 0.5 * (lo + hi);
        if (!(munew > lo && munew < hi)) munew = 0.5 * (lo + hi);
        if (munew == mu || (hi - lo) <= 4.0 * DC_EPS * fmax(fabs(lo), fabs(hi))) { ok = true; mu = munew; break; }
        mu = munew;
        ev = sec_eval(k, dk, zk, rho, o, mu, isplit);
    }
    if (!ok) atomicAdd(fail, 1);
    org_all[s + j] = o;
    mu_all[s + j] = mu;
    lam_all[s + j] = dk[o] + mu;
}

// ------------------------------------------------------------------ S3.4 z_hat and U
// z_hat_i = sign(z_i) sqrt( prod_j (lambda_j - d_i) / prod_{j != i} (d_j - d_i) )
__global__ void __launch_bounds__(128) dc_zhat_kernel(const MergeDesc* __restrict__ desc, const int* __restrict__ kcount,
                                                      const double* __restrict__ dk_all, const double* __restrict__ zk_all,
                                                      const int* __restrict__ org_all, const double* __restrict__ mu_all,
                                                      double* __restrict__ zhat_all) {
    const int mi = blockIdx.y;
    const int k = kcount[mi];
    const int i = blockIdx.x * 128 + threadIdx.x;
    if (i >= k) return;
    const int s = desc[mi].s;
    const double* dk = dk_all + s;
    const int* org = org_all + s;
    const double* mu = mu_all + s;
    const double di = dk[i];
    double prod = (dk[org[i]] - di) + mu[i];
    for (int j = 0; j < k; ++j) {
        if (j == i) continue;
        prod *= ((dk[org[j]] - di) + mu[j]) / (dk[j] - di);
    }
    zhat_all[s + i] = copysign(sqrt(fabs(prod)), zk_all[s + i]);
}

// U[i,j] = z_hat_i / ((d_i - d_org(j)) - mu_j), column-normalised; one CTA per column j
__global__ void __launch_bounds__(256) dc_build_u_kernel(const MergeDesc* __restrict__ desc, const int* __restrict__ kcount,
                                                         const double* __restrict__ dk_all, const int* __restrict__ org_all,
                                                         const double* __restrict__ mu_all, const double* __restrict__ zhat_all,
                                                         const int* __restrict__ upos_all, double* __restrict__ U, int64_t ldq) {
    __shared__ double red[8];
    const int mi = blockIdx.y;
    const int k = kcount[mi];
    const int j = blockIdx.x;
    if (j >= k) return;
    const int s = desc[mi].s;
    const double* dk = dk_all + s;
    const double* zh = zhat_all + s;
    const double dorg = dk[org_all[s + j]], muj = mu_all[s + j];
    double* Uc = U + s + (int64_t)(s + j) * ldq;
    double ss = 0.0;
    const int* upos = upos_all + s;
    for (int i = threadIdx.x; i < k; i += 256) {
        const double v = zh[i] / ((dk[i] - dorg) - muj);
        Uc[upos[i]] = v;                   // row order of U = memory order of the gathered columns
        ss += v * v;
    }
    for (int o = 16; o > 0; o >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = ss;
    __syncthreads();
    double tot = 0.0;
    for (int w = 0; w < 8; ++w) tot += red[w];
    const double inv = 1.0 / sqrt(tot);
    for (int i = threadIdx.x; i < k; i += 256) Uc[i] *= inv;
}

// ------------------------------------------------------------------ S3.5 merge GEMM descriptors, deflated columns
// Last merge with nev < N: only the secular roots among the lowest nev values of the merged spectrum need their
// eigenvector.  The roots are ascending in j, so those are a prefix j < kn; root j is wanted when fewer than nev
// values lie below it: j roots plus the deflated values < lam_j (ties counted in favour of keeping the root).
__global__ void __launch_bounds__(256) dc_wanted_kernel(const MergeDesc* __restrict__ desc, const int* __restrict__ kcount,
                                                        const int* __restrict__ df_idx, const double* __restrict__ dcur,
                                                        const double* __restrict__ lam, int nev, int* __restrict__ kn) {
    const MergeDesc m = desc[0];
    const int n = m.e - m.s, k = kcount[0];
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= k) return;
    const double lj = lam[m.s + j];
    int below = j;
    for (int t = 0; t < n - k && below < nev; ++t) below += (dcur[m.s + df_idx[m.s + t]] < lj) ? 1 : 0;
    if (below < nev) atomicMax(kn, j + 1);
}

// (also accumulates the level's statistics for eigh_dc_stats: executed GEMM flops, sum of k, sum of n)
__global__ void dc_gemm_desc_kernel(const MergeDesc* __restrict__ desc, const int* __restrict__ kcount,
                                    const int* __restrict__ k1c, const int* __restrict__ k2c, int nmerge, int64_t ldq,
                                    DgemmDesc* __restrict__ g, const int* __restrict__ kn, double* __restrict__ stats) {
    const int mi = blockIdx.x * blockDim.x + threadIdx.x;
    if (mi >= nmerge) return;
    const MergeDesc m = desc[mi];
    const int k = kcount[mi], k1 = k1c[mi], k2 = k2c[mi];
    const int k1e = k1 & ~1;                 // even start of the bottom K-range (16-byte aligned rows of U); a type-1
                                             // column that falls into it only contributes exact zeros
    DgemmDesc d;
    // top rows: columns of type 1 and 2
    d.offA = d.offB = d.offC = m.s + (int64_t)m.s * ldq;
    d.offIdx = m.s;
    d.M = m.mid - m.s;
    d.N = kn ? min(k, *kn) : k;          // columns of U that are wanted (all of them unless this is the last merge, nev < N)
    d.K = k1 + k2;
    d.pad = 0;
    g[2 * mi] = d;
    // bottom rows: columns of type 2 and 3
    d.offA = d.offC = m.mid + (int64_t)m.s * ldq;
    d.offB = (m.s + k1e) + (int64_t)m.s * ldq;
    d.offIdx = m.s + k1e;
    d.M = m.e - m.mid;
    d.K = k - k1e;
    g[2 * mi + 1] = d;
    const double ncols = (double)d.N;
    atomicAdd(stats + 0, 2.0 * ncols * ((double)(m.mid - m.s) * (k1 + k2) + (double)(m.e - m.mid) * (k - k1e)));
    atomicAdd(stats + 1, (double)k);
    atomicAdd(stats + 2, (double)(m.e - m.s));
}

__global__ void __launch_bounds__(256) dc_finish_kernel(const MergeDesc* __restrict__ desc, const int* __restrict__ kcount,
                                                        const int* __restrict__ df_idx, const double* __restrict__ Qold,
                                                        double* __restrict__ Qnew, int64_t ldq,
                                                        const double* __restrict__ dcur, const double* __restrict__ lam,
                                                        double* __restrict__ dnew) {
    const int mi = blockIdx.y;
    const MergeDesc m = desc[mi];
    const int n = m.e - m.s, k = kcount[mi];
    const int t = blockIdx.x;            // output column index (local)
    if (t >= n) return;
    if (t < k) {
        if (threadIdx.x == 0) dnew[m.s + t] = lam[m.s + t];
        return;
    }
    const int src = df_idx[m.s + t - k];
    if (threadIdx.x == 0) dnew[m.s + t] = dcur[m.s + src];
    const double* a = Qold + m.s + (int64_t)(m.s + src) * ldq;
    double* b = Qnew + m.s + (int64_t)(m.s + t) * ldq;
    for (int r = threadIdx.x; r < n; r += 256) b[r] = a[r];
}

// final: W[rank] = d, Qout[:, rank] = Q[:, j] for rank < nev
__global__ void __launch_bounds__(256) dc_output_kernel(int N, int col0, int nev, const int* __restrict__ perm, const double* __restrict__ dcur,
                                                        const double* __restrict__ Q, int64_t ldq, double* __restrict__ W,
                                                        double* __restrict__ Qout, int64_t ldo,
                                                        const double* __restrict__ esgn, const double* __restrict__ scale) {
    const int rank = blockIdx.x;
    const int j = perm[rank];
    if (threadIdx.x == 0) W[rank] = dcur[j] * scale[0];      // back from the unit-norm matrix (a power of two: exact)
    if (rank < col0 || rank >= col0 + nev) return;           // (col0 > 0: this handle's column shard)
    const double* a = Q + (int64_t)j * ldq;
    double* b = Qout + (int64_t)(rank - col0) * ldo;
    for (int r = threadIdx.x; r < N; r += 256) b[r] = esgn[r] * a[r];
}

// ------------------------------------------------------------------ driver
int phase_tridiag_dc(eigh_handle_s* h, const double* d, const double* e, double* W, double* Qout, int64_t ldo,
                     cudaStream_t st, int* nfail) {
    const int N = (int)h->N, nev = (int)h->nev, col0 = h->col0;
    const int nwant = col0 + nev;                             // eigenvectors 0 .. nwant-1 must exist after the last merge
    DcBufs B = dc_carve(ws_ptr<char>(h, h->plan.dc), N);
    const int64_t ldq = B.ldq;
    // ---- tree (host): L = 2^p leaves, even boundaries
    int leaf_target = h->leaf - 2;
    if (leaf_target < 2) leaf_target = 2;
    int L = 1;
    while ((N + L - 1) / L > leaf_target) L *= 2;
    if (N < 4) L = 1;
    std::vector<int> bnd(L + 1);
    for (int i = 0; i <= L; ++i) bnd[i] = (int)(2 * (((int64_t)i * N + L) / (2 * L)));
    bnd[0] = 0; bnd[L] = N;
    for (int i = 1; i <= L; ++i) if (bnd[i] <= bnd[i - 1] && i < L) bnd[i] = bnd[i - 1] + 2;
    // (N >= 4, leaf_target >= 2 keeps every leaf non-empty and <= 32)
    for (int i = 0; i < L; ++i)
        if (bnd[i + 1] - bnd[i] < 1 || bnd[i + 1] - bnd[i] > DC_LEAF_MAX)
            return set_err(h, -100, "internal: bad D&C leaf partition (N=%d, L=%d)", N, L);
    std::vector<MergeDesc> descs;
    std::vector<int> level_off, level_cnt, level_maxn, level_maxhalf;
    for (int width = 1; width < L; width *= 2) {
        level_off.push_back((int)descs.size());
        int cnt = 0, maxn = 0, maxhalf = 0;
        for (int i = 0; i + 2 * width <= L; i += 2 * width) {
            MergeDesc m = {bnd[i], bnd[i + width], bnd[i + 2 * width], 0};
            descs.push_back(m);
            ++cnt;
            maxn = std::max(maxn, m.e - m.s);
            maxhalf = std::max(maxhalf, std::max(m.mid - m.s, m.e - m.mid));
        }
        level_cnt.push_back(cnt);
        level_maxn.push_back(maxn);
        level_maxhalf.push_back(maxhalf);
    }
    { MergeDesc all = {0, 0, N, 0}; descs.push_back(all); }    // descriptor used by the final sort
    const int final_desc = (int)descs.size() - 1;
    EIGH_CUDA_OK(cudaMemcpyAsync(B.bnd, bnd.data(), (size_t)(L + 1) * sizeof(int), cudaMemcpyHostToDevice, st));
    EIGH_CUDA_OK(cudaMemcpyAsync(B.desc, descs.data(), descs.size() * sizeof(MergeDesc), cudaMemcpyHostToDevice, st));
    EIGH_CUDA_OK(cudaMemsetAsync(B.fail, 0, sizeof(int), st));
    EIGH_CUDA_OK(cudaMemsetAsync(B.stats, 0, 32 * 3 * sizeof(double), st));
    EIGH_CUDA_OK(cudaStreamSynchronize(st));   // host vectors go out of scope; copies are tiny

    // ---- tearing + leaves
    dc_norm_kernel<<<1, 1024, 0, st>>>(d, e, N, B.scale);
    dc_tear_kernel<<<(unsigned)ceil_div(N, 256), 256, 0, st>>>(d, e, N, B.bnd, L, B.scale, B.dcur, B.esc);
    e = B.esc;                                               // from here on: the scaled copy
    dc_tear2_kernel<<<(unsigned)ceil_div(L, 256), 256, 0, st>>>(e, B.bnd, L, B.dcur);
    dc_leaf_kernel<<<(unsigned)ceil_div(L, 4), 128, 0, st>>>(B.bnd, L, B.dcur, e, B.QA, ldq, B.fail);
    dc_esign_kernel<<<1, 1024, 0, st>>>(e, N, B.esgn);
    h->launches += 5;

    double* Qcur = B.QA;
    double* Qnew = B.QB;
    double* dcur = B.dcur;
    double* dnew = B.dnew;
    for (size_t lv = 0; lv < level_cnt.size(); ++lv) {
        const MergeDesc* dd = B.desc + level_off[lv];
        const int cnt = level_cnt[lv], maxn = level_maxn[lv];
        const unsigned gx256 = (unsigned)ceil_div(maxn, 256), gx128 = (unsigned)ceil_div(maxn, 128);
        {
            int64_t work = (int64_t)maxn * maxn / 2;
            unsigned gx = (unsigned)std::min<int64_t>(ceil_div(work, 256), 148 * 8);
            if (gx < 1) gx = 1;
            dc_zero_offdiag_kernel<<<dim3(gx, cnt), 256, 0, st>>>(dd, Qcur, ldq);
        }
        dc_zvec_kernel<<<dim3(gx256, cnt), 256, 0, st>>>(dd, Qcur, ldq, B.z);
        dc_rank_kernel<<<dim3(gx256, cnt), 256, 0, st>>>(dd, dcur, B.perm);
        dc_deflate_kernel<<<cnt, 256, 0, st>>>(dd, e, dcur, B.z, B.perm, B.nd_idx, B.df_idx, B.kcount, B.nrot, B.rot_a,
                                               B.rot_b, B.rot_c, B.rot_s, B.dk, B.zk, B.rho, B.zsum, B.ctype, B.ktype, B.upos, B.acol, B.k1c,
                                               B.k2c);
        dc_apply_rot_kernel<<<dim3(gx256, cnt), 256, 0, st>>>(dd, Qcur, ldq, B.nrot, B.rot_a, B.rot_b, B.rot_c, B.rot_s);
        dc_secular_kernel<<<dim3(gx128, cnt), 128, 0, st>>>(dd, B.kcount, B.dk, B.zk, B.rho, B.zsum, B.org, B.mu, B.lam, B.fail);
        dc_zhat_kernel<<<dim3(gx128, cnt), 128, 0, st>>>(dd, B.kcount, B.dk, B.zk, B.org, B.mu, B.zhat);
        dc_build_u_kernel<<<dim3(maxn, cnt), 256, 0, st>>>(dd, B.kcount, B.dk, B.org, B.mu, B.zhat, B.upos, B.U, ldq);
        const int* kn = nullptr;
        if (nwant < N && lv + 1 == level_cnt.size() && cnt == 1) {
            EIGH_CUDA_OK(cudaMemsetAsync(B.fail + 16, 0, sizeof(int), st));
            dc_wanted_kernel<<<gx256, 256, 0, st>>>(dd, B.kcount, B.df_idx, dcur, B.lam, nwant, B.fail + 16);
            ++h->launches;
            kn = B.fail + 16;          // second counter in the 256-byte block of `fail`
        }
        dc_gemm_desc_kernel<<<(unsigned)ceil_div(cnt, 128), 128, 0, st>>>(dd, B.kcount, B.k1c, B.k2c, cnt, ldq, B.gdesc, kn,
                                                                          B.stats + 3 * std::min<size_t>(lv, 31));
        h->launches += 9;
        DgemmArgs ga;
        memset(&ga, 0, sizeof(ga));
        ga.A = Qcur; ga.lda = ldq; ga.B = B.U; ga.ldb = ldq; ga.C = Qnew; ga.ldc = ldq;
        ga.a_col_idx = B.acol; ga.desc = B.gdesc;
        int rc = dgemm_launch_desc(ga, 2 * cnt, level_maxhalf[lv], maxn, st, &h->launches);
        if (rc) return 1000 + rc;
        dc_finish_kernel<<<dim3(maxn, cnt), 256, 0, st>>>(dd, B.kcount, B.df_idx, Qcur, Qnew, ldq, dcur, B.lam, dnew);
        ++h->launches;
        std::swap(Qcur, Qnew);
        std::swap(dcur, dnew);
    }
    // ---- final ascending order
    dc_rank_kernel<<<dim3((unsigned)ceil_div(N, 256), 1), 256, 0, st>>>(B.desc + final_desc, dcur, B.perm);
    dc_output_kernel<<<N, 256, 0, st>>>(N, col0, nev, B.perm, dcur, Qcur, ldq, W, Qout, ldo, B.esgn, B.scale);
    h->launches += 2;
    int fail = 0;
    double stats[32 * 3];
    EIGH_CUDA_OK(cudaMemcpyAsync(&fail, B.fail, sizeof(int), cudaMemcpyDeviceToHost, st));
    EIGH_CUDA_OK(cudaMemcpyAsync(stats, B.stats, sizeof(stats), cudaMemcpyDeviceToHost, st));
    EIGH_CUDA_OK(cudaStreamSynchronize(st));
    h->dc_levels = (int)std::min<size_t>(level_cnt.size(), 32);
    for (int l = 0; l < h->dc_levels; ++l) {
        h->dc_flops[l] = stats[3 * l]; h->dc_ksum[l] = stats[3 * l + 1]; h->dc_nsum[l] = stats[3 * l + 2];
    }
    EIGH_CUDA_OK(cudaGetLastError());
    if (nfail) *nfail = fail;
    return 0;
}

}  // namespace eigh
