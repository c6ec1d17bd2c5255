// band_reduce.cu -- S1: full -> band reduction ("transforming the dense matrix in a
// banded matrix"), SURVEY.md 8(a) rows S1.1-S1.5.
//
// For each block column p (width b):  panel = A[j0+b:, j0:j0+b]  (m x b)
//   S1.1  panel QR by Householder reflectors h_j = I - tau_j v_j v_j^H (LAPACK zlarfg convention),
//         one cooperative multi-CTA kernel: rows are split over CTAs, one grid barrier per column.
//   S1.2  T from  T^{-1} = striu(V^H V) + diag(1/tau)   (Q_p = I - V T V^H)
//   S1.3  X = Herm(A22) (V T)                 (HEMM-lower on the DMMA path)
//   S1.4  W = X - 1/2 V ((V T)^H X)
//   S1.5  A22 <- A22 - V W^H - W V^H          (HER2K-lower on the DMMA path, one fused K = 2b GEMM)
// A keeps R and the reflectors in place; an explicit copy of V (ones/zeros filled in) is used by
// the GEMMs.  The band is extracted once at the end.
#include "eigh_internal.h"
#include "zgemm.cuh"

namespace eigh {

// ------------------------------------------------------------------ small utility kernels
// Fill the strict upper triangle of every 64-aligned diagonal block from the lower triangle and
// zero the imaginary part of the diagonal (only the lower triangle of A is an input).
__global__ void symmetrize_diag_blocks_kernel(c128* A, int64_t lda, int N) {
    const int d0 = blockIdx.x * 64;
    for (int idx = threadIdx.x; idx < 64 * 64; idx += blockDim.x) {
        const int i = d0 + idx % 64, j = d0 + idx / 64;
        if (i >= N || j >= N) continue;
        if (i == j) A[i + (int64_t)j * lda].y = 0.0;
        else if (i > j) A[j + (int64_t)i * lda] = cconj(A[i + (int64_t)j * lda]);
    }
}

// band[(i-c) + c*ldab] = A[i,c] for 0 <= i-c <= b; rows b+1..ldab-1 zeroed.
__global__ void extract_band_kernel(const c128* __restrict__ A, int64_t lda, int N, int b, c128* __restrict__ band,
                                    int64_t ldab) {
    const int c = blockIdx.x;
    for (int o = threadIdx.x; o < ldab; o += blockDim.x) {
        c128 v = cmake(0.0, 0.0);
        const int i = c + o;
        if (o <= b && i < N) {
            v = A[i + (int64_t)c * lda];
            if (o == 0) v.y = 0.0;
        }
        band[o + (int64_t)c * ldab] = v;
    }
}

// T (b x b upper triangular, zero below) from G = V^H V and tau:
//   T[j,j] = tau_j,  T[i,j] = -tau_i * sum_{l=i+1..j} G[i,l] T[l,j]   (i < j)
__global__ void tfactor_kernel(const c128* __restrict__ G, int ldg, const c128* __restrict__ tau, int nb,
                               c128* __restrict__ T, int ldt) {
    extern __shared__ __align__(16) unsigned char tf_raw[];
    c128* Gs = reinterpret_cast<c128*>(tf_raw);       // nb x (nb+1)
    c128* Ts = Gs + nb * (nb + 1);
    c128* ts = Ts + nb * (nb + 1);
    const int lds = nb + 1;
    for (int idx = threadIdx.x; idx < nb * nb; idx += blockDim.x) {
        const int i = idx % nb, j = idx / nb;
        Gs[i + j * lds] = G[i + (int64_t)j * ldg];
        Ts[i + j * lds] = cmake(0.0, 0.0);
    }
    for (int i = threadIdx.x; i < nb; i += blockDim.x) ts[i] = tau[i];
    __syncthreads();
    const int j = threadIdx.x;
    if (j < nb) {
        Ts[j + j * lds] = ts[j];
        for (int i = j - 1; i >= 0; --i) {
            c128 s = cmake(0.0, 0.0);
            for (int l = i + 1; l <= j; ++l) cfma(s, Gs[i + l * lds], Ts[l + j * lds]);
            const c128 ti = ts[i];
            Ts[i + j * lds] = cmake(-(ti.x * s.x - ti.y * s.y), -(ti.x * s.y + ti.y * s.x));
        }
    }
    __syncthreads();
    for (int idx = threadIdx.x; idx < nb * nb; idx += blockDim.x) {
        const int i = idx % nb, jj = idx / nb;
        T[i + (int64_t)jj * ldt] = Ts[i + jj * lds];
    }
}

// ------------------------------------------------------------------ cooperative panel QR
struct PanelArgs {
    c128* P;  int64_t ld;      // panel, m x nb
    int m, nb, nr;             // rows, columns, reflectors (nr = min(nb, m-1))
    c128* Vp; int64_t ldv;     // explicit V out, m x nb
    c128* tau;                 // nb
    unsigned* counter;         // grid barrier counter, zero on entry
    c128* part;                // [2][gridDim.x][nb]
    c128* pivrow;              // [2][nb]
    int rows_per_cta;
};

__device__ __forceinline__ void grid_barrier(unsigned* ctr, unsigned nblocks, unsigned& epoch) {
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        atomicAdd(ctr, 1u);
        const unsigned target = (epoch + 1) * nblocks;
        while (*(volatile unsigned*)ctr < target) {}
        __threadfence();
    }
    ++epoch;
    __syncthreads();
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

constexpr int PQ_NT = 256, PQ_WARPS = 8, PQ_CG = 8;

__global__ void __launch_bounds__(PQ_NT, 1) panel_qr_kernel(const PanelArgs a) {
    extern __shared__ __align__(16) unsigned char pq_raw[];
    c128* red = reinterpret_cast<c128*>(pq_raw);     // [PQ_WARPS][nb]
    c128* wv = red + PQ_WARPS * a.nb;                // [nb]  w_c
    c128* scal = wv + a.nb;                          // [4]: tau, s, beta, flag
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int G = gridDim.x, cta = blockIdx.x;
    const int r_begin = cta * a.rows_per_cta;
    const int r_end = min(a.m, r_begin + a.rows_per_cta);
    const int nb = a.nb;
    unsigned epoch = 0;

    for (int jj = 0; jj < a.nr; ++jj) {
        const int par = jj & 1;
        const int ncol = nb - jj;
        c128* part = a.part + ((size_t)par * G + cta) * nb;
        c128* piv = a.pivrow + (size_t)par * nb;
        const int lo = max(r_begin, jj + 1);
        // ---- phase A: partial dots over own rows r > jj:  dots[c] = sum conj(P[r,jj]) P[r,c]
        for (int cg0 = jj; cg0 < nb; cg0 += PQ_CG) {
            c128 acc[PQ_CG];
#pragma unroll
            for (int q = 0; q < PQ_CG; ++q) acc[q] = cmake(0.0, 0.0);
            for (int r = lo + warp * 32 + lane; r < r_end; r += PQ_WARPS * 32) {
                const c128 x = a.P[r + (int64_t)jj * a.ld];
#pragma unroll
                for (int q = 0; q < PQ_CG; ++q) {
                    const int c = cg0 + q;
                    if (c < nb) cfmac(acc[q], x, a.P[r + (int64_t)c * a.ld]);
                }
            }
#pragma unroll
            for (int q = 0; q < PQ_CG; ++q) {
                const double sx = warp_sum(acc[q].x), sy = warp_sum(acc[q].y);
                if (lane == 0 && cg0 + q < nb) red[warp * nb + cg0 + q - jj] = cmake(sx, sy);
            }
        }
        __syncthreads();
        if (tid < ncol) {
            c128 s = cmake(0.0, 0.0);
#pragma unroll
            for (int w = 0; w < PQ_WARPS; ++w) s = cadd(s, red[w * nb + tid]);
            part[tid] = s;
        }
        if (jj >= r_begin && jj < r_end && tid < ncol) piv[tid] = a.P[jj + (int64_t)(jj + tid) * a.ld];
        grid_barrier(a.counter, G, epoch);

        // ---- phase B: total dots, reflector scalars, w
        if (tid < ncol) {
            c128 s = cmake(0.0, 0.0);
            const c128* pp = a.part + (size_t)par * G * nb + tid;
            for (int g = 0; g < G; ++g) {
                const c128 v = __ldcg(pp + (size_t)g * nb);
                s.x += v.x; s.y += v.y;
            }
            red[tid] = s;      // red[0..ncol) now holds the total dots (phase-A contents are dead)
        }
        __syncthreads();
        if (tid == 0) {
            const c128 alpha = __ldcg(piv);
            const double xnorm2 = red[0].x;
            c128 tau = cmake(0.0, 0.0), s = cmake(0.0, 0.0);
            double beta = alpha.x;
            double flag = 0.0;
            if (xnorm2 > 0.0 || alpha.y != 0.0) {
                beta = -copysign(sqrt(alpha.x * alpha.x + alpha.y * alpha.y + xnorm2), alpha.x);
                tau = cmake((beta - alpha.x) / beta, -alpha.y / beta);
                const double dr = alpha.x - beta, di = alpha.y;
                const double den = dr * dr + di * di;
                s = cmake(dr / den, -di / den);           // 1 / (alpha - beta)
                flag = 1.0;
            }
            scal[0] = tau; scal[1] = s; scal[2] = cmake(beta, 0.0); scal[3] = cmake(flag, 0.0);
            if (cta == 0) a.tau[jj] = tau;
        }
        __syncthreads();
        const c128 tau = scal[0], s = scal[1];
        const double beta = scal[2].x;
        const bool active = scal[3].x != 0.0;
        if (tid > 0 && tid < ncol) {
            // w_c = P[jj,c] + conj(s) * dots[c]
            const c128 pj = __ldcg(piv + tid);
            const c128 d = red[tid];
            wv[tid] = cadd(pj, cmulc(s, d));
        }
        __syncthreads();
        const c128 ctau = cconj(tau);
        // ---- update own rows r > jj
        if (active) {
            for (int r = lo + tid; r < r_end; r += PQ_NT) {
                const c128 v = cmul(s, a.P[r + (int64_t)jj * a.ld]);
                const c128 f = cmul(ctau, v);
                for (int c = jj + 1; c < nb; ++c) {
                    c128* e = a.P + r + (int64_t)c * a.ld;
                    const c128 t = cmul(f, wv[c - jj]);
                    c128 o = *e;
                    o.x -= t.x; o.y -= t.y;
                    *e = o;
                }
                a.P[r + (int64_t)jj * a.ld] = v;
                a.Vp[r + (int64_t)jj * a.ldv] = v;
            }
        } else {
            for (int r = lo + tid; r < r_end; r += PQ_NT) a.Vp[r + (int64_t)jj * a.ldv] = cmake(0.0, 0.0);
        }
        // rows r <= jj of column jj of Vp (zeros above, one on the diagonal)
        for (int r = r_begin + tid; r < min(r_end, jj + 1); r += PQ_NT)
            a.Vp[r + (int64_t)jj * a.ldv] = (r == jj) ? cmake(1.0, 0.0) : cmake(0.0, 0.0);
        // pivot row (its owner)
        if (jj >= r_begin && jj < r_end && active) {
            if (tid == 0) a.P[jj + (int64_t)jj * a.ld] = cmake(beta, 0.0);
            if (tid > 0 && tid < ncol) {
                c128* e = a.P + jj + (int64_t)(jj + tid) * a.ld;
                const c128 t = cmul(ctau, wv[tid]);
                c128 o = *e;
                o.x -= t.x; o.y -= t.y;
                *e = o;
            }
        }
        __syncthreads();
    }
    // columns without a reflector
    for (int jj = a.nr; jj < nb; ++jj) {
        if (cta == 0 && tid == 0) a.tau[jj] = cmake(0.0, 0.0);
        for (int r = r_begin + tid; r < r_end; r += PQ_NT)
            a.Vp[r + (int64_t)jj * a.ldv] = (r == jj) ? cmake(1.0, 0.0) : cmake(0.0, 0.0);
    }
}

// ------------------------------------------------------------------ shared-memory resident panel QR
// The same Householder QR (zlarfg convention) with the CTA's rows of the panel held in shared memory
// for the whole factorisation, so that a column step costs one lean grid barrier plus two passes over
// shared memory instead of three passes over L2:
//   dots pass   d[c] = sum_{r > jj, own rows} conj(P[r,jj]) P[r,c]  for ALL 64 columns c
//               (c >= jj: norm and v^H P as before; c < jj: conj(d[c]) = V[:,c]^H P[:,jj], the Gram
//               entries from which the compact-WY T factor is built on the fly);
//   barrier     partial dots + the pivot row go through L2; arrival = red.release, wait = ld.acquire;
//   update pass every CTA forms the reflector scalars redundantly and updates its rows.
// One extra CTA (the last) owns no rows: it accumulates T,
//   T[0:jj, jj] = -tau_jj T[0:jj, 0:jj] g,   g_i = v_i^H v_jj = conj(P[jj,i]) + s conj(d[i]),   T[jj,jj] = tau_jj,
// which replaces the V^H V GEMM, its split-K reduction and the serial T recurrence kernel.
constexpr int PS_NT = 256, PS_MAXROWS = 192, PS_LD = 65, PS_B = 64;

struct PanelSmemArgs {
    c128* P;  int64_t ld;      // panel, m x 64, column-major in A
    int m, nr;                 // rows, reflectors (= 64 here)
    c128* Vp; int64_t ldv;     // explicit V out, m x 64
    c128* tau;                 // 64
    c128* T;  int ldt;         // compact-WY T out (64 x 64, upper triangular, zero below)
    unsigned* counter;         // grid barrier counter, zero on entry
    c128* part;                // [2][gridDim.x][64]
    c128* pivrow;              // [2][64]
    int rows_per_cta;
};

__device__ __forceinline__ void ps_grid_barrier(unsigned* ctr, unsigned target) {
    __syncthreads();
    if (threadIdx.x == 0) {
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(ctr) : "memory");
        unsigned v;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(ctr) : "memory");
        } while (v < target);
    }
    __syncthreads();
}

__global__ void __launch_bounds__(PS_NT, 1) panel_qr_smem_kernel(const PanelSmemArgs a) {
    extern __shared__ __align__(16) unsigned char ps_raw[];
    c128* Ps = reinterpret_cast<c128*>(ps_raw);            // [rows][PS_LD] row-major tile (row CTAs) or T (T CTA)
    c128* red = Ps + PS_MAXROWS * PS_LD;                   // [4][64]
    c128* tot = red + 4 * PS_B;                            // [64]
    c128* wv = tot + PS_B;                                 // [64]
    c128* pv = wv + PS_B;                                  // [64] pivot row
    const int tid = threadIdx.x;
    const int c = tid & 63, q = tid >> 6;
    const int G = gridDim.x - 1;                           // row CTAs; CTA G accumulates T
    const int cta = blockIdx.x;
    const bool tcta = cta == G;
    const int r_begin = tcta ? a.m : cta * a.rows_per_cta;
    const int r_end = tcta ? a.m : min(a.m, r_begin + a.rows_per_cta);
    const int nrows = r_end - r_begin;

    // ---- load the tile (coalesced along rows in global, padded rows in shared)
    for (int idx = tid; idx < nrows * PS_B; idx += PS_NT) {
        const int rr = idx % nrows, cc = idx / nrows;
        Ps[rr * PS_LD + cc] = a.P[(r_begin + rr) + (int64_t)cc * a.ld];
    }
    if (tcta)
        for (int idx = tid; idx < PS_B * PS_LD; idx += PS_NT) Ps[idx] = cmake(0.0, 0.0);
    __syncthreads();

    for (int jj = 0; jj < a.nr; ++jj) {
        const int par = jj & 1;
        // ---- dots pass over own rows r > jj
        {
            const int lo = max(0, jj + 1 - r_begin);       // first local row with global index > jj
            c128 acc = cmake(0.0, 0.0);
            for (int rr = lo + q; rr < nrows; rr += 4) cfmac(acc, Ps[rr * PS_LD + jj], Ps[rr * PS_LD + c]);
            red[q * PS_B + c] = acc;
        }
        __syncthreads();
        if (!tcta && tid < PS_B) {
            const c128 s4 = cadd(cadd(red[tid], red[PS_B + tid]), cadd(red[2 * PS_B + tid], red[3 * PS_B + tid]));
            a.part[((size_t)par * G + cta) * PS_B + tid] = s4;
            if (jj >= r_begin && jj < r_end) a.pivrow[(size_t)par * PS_B + tid] = Ps[(jj - r_begin) * PS_LD + tid];
        }
        ps_grid_barrier(a.counter, (unsigned)(jj + 1) * gridDim.x);
        // ---- totals (every CTA, redundantly), reflector scalars, w
        {
            c128 s4 = cmake(0.0, 0.0);
            const c128* pp = a.part + (size_t)par * G * PS_B + c;
            for (int g = q; g < G; g += 4) {
                const c128 v = __ldcg(pp + (size_t)g * PS_B);
                s4.x += v.x; s4.y += v.y;
            }
            red[q * PS_B + c] = s4;
            if (tid < PS_B) pv[tid] = __ldcg(a.pivrow + (size_t)par * PS_B + tid);
        }
        __syncthreads();
        if (tid < PS_B) tot[tid] = cadd(cadd(red[tid], red[PS_B + tid]), cadd(red[2 * PS_B + tid], red[3 * PS_B + tid]));
        __syncthreads();
        c128 tau = cmake(0.0, 0.0), s = cmake(0.0, 0.0);
        double beta;
        bool active = false;
        {
            const c128 alpha = pv[jj];
            const double xnorm2 = tot[jj].x;
            beta = alpha.x;
            if (xnorm2 > 0.0 || alpha.y != 0.0) {
                beta = -copysign(sqrt(alpha.x * alpha.x + alpha.y * alpha.y + xnorm2), alpha.x);
                tau = cmake((beta - alpha.x) / beta, -alpha.y / beta);
                const double dr = alpha.x - beta, di = alpha.y;
                const double den = dr * dr + di * di;
                s = cmake(dr / den, -di / den);            // 1 / (alpha - beta)
                active = true;
            }
        }
        if (tcta) {
            // g_i = v_i^H v_jj (i < jj); T[0:jj, jj] = -tau T[0:jj, 0:jj] g; T[jj, jj] = tau
            if (tid < PS_B) {
                c128 g = cmake(0.0, 0.0);
                if (tid < jj) {
                    g = cconj(pv[tid]);
                    if (active) g = cadd(g, cmul(s, cconj(tot[tid])));
                }
                wv[tid] = g;
            }
            __syncthreads();
            {
                c128 acc = cmake(0.0, 0.0);
                if (c < jj)
                    for (int l = c + q; l < jj; l += 4) cfma(acc, Ps[c * PS_LD + l], wv[l]);
                red[q * PS_B + c] = acc;
            }
            __syncthreads();
            if (tid < PS_B) {
                if (tid < jj) {
                    const c128 t4 = cadd(cadd(red[tid], red[PS_B + tid]), cadd(red[2 * PS_B + tid], red[3 * PS_B + tid]));
                    const c128 v = cmul(tau, t4);
                    Ps[tid * PS_LD + jj] = cmake(-v.x, -v.y);
                } else if (tid == jj) {
                    Ps[tid * PS_LD + jj] = tau;
                }
            }
            if (tid == 0) a.tau[jj] = tau;
            __syncthreads();
            continue;
        }
        // ---- row CTAs: w_c = P[jj,c] + conj(s) d[c] (c > jj); rows r > jj: v_r = s x_r, P[r,c] -= conj(tau) v_r w_c
        if (tid < PS_B) wv[tid] = (tid > jj) ? cadd(pv[tid], cmulc(s, tot[tid])) : cmake(0.0, 0.0);
        __syncthreads();
        const c128 ctau = cconj(tau);
        if (active) {
            const int lo = max(0, jj + 1 - r_begin);
            if (c > jj) {
                const c128 wc = wv[c];
                for (int rr = lo + q; rr < nrows; rr += 4) {
                    const c128 f = cmul(ctau, cmul(s, Ps[rr * PS_LD + jj]));
                    const c128 t4 = cmul(f, wc);
                    c128 o = Ps[rr * PS_LD + c];
                    o.x -= t4.x; o.y -= t4.y;
                    Ps[rr * PS_LD + c] = o;
                }
            }
            // pivot row (its owner)
            if (jj >= r_begin && jj < r_end && q == 0) {
                const int rr = jj - r_begin;
                if (c > jj) {
                    const c128 t4 = cmul(ctau, wv[c]);
                    c128 o = Ps[rr * PS_LD + c];
                    o.x -= t4.x; o.y -= t4.y;
                    Ps[rr * PS_LD + c] = o;
                }
            }
            __syncthreads();
            // column jj becomes v (rows > jj) and beta (pivot)
            for (int rr = lo + tid; rr < nrows; rr += PS_NT) Ps[rr * PS_LD + jj] = cmul(s, Ps[rr * PS_LD + jj]);
            if (jj >= r_begin && jj < r_end && tid == 0) Ps[(jj - r_begin) * PS_LD + jj] = cmake(beta, 0.0);
        } else {
            // H = I: v = e_jj; entries below the pivot are already zero (xnorm2 = 0)
        }
        __syncthreads();
    }
    if (tcta) {
        for (int idx = tid; idx < PS_B * PS_B; idx += PS_NT) {
            const int i = idx & 63, j = idx >> 6;
            a.T[i + (size_t)j * a.ldt] = (i <= j && j < a.nr) ? Ps[i * PS_LD + j] : cmake(0.0, 0.0);
        }
        for (int jj = a.nr + tid; jj < PS_B; jj += PS_NT) a.tau[jj] = cmake(0.0, 0.0);
        return;
    }
    // ---- write back: A keeps R (rows <= column) and v below; Vp gets the explicit unit-lower-trapezoidal V
    for (int idx = tid; idx < nrows * PS_B; idx += PS_NT) {
            const int rr = idx % nrows, cc = idx / nrows;
            const int r = r_begin + rr;
            const c128 v = Ps[rr * PS_LD + cc];
            a.P[r + (int64_t)cc * a.ld] = v;
            c128 e = cmake(0.0, 0.0);
            if (r == cc) e = cmake(1.0, 0.0);
            else if (r > cc && cc < a.nr) e = v;
            a.Vp[r + (int64_t)cc * a.ldv] = e;
        }
}

// ------------------------------------------------------------------ host driver
static int zg(eigh_handle_s* h, bool ta, bool tb, int M, int N, int K, double alpha, const c128* A, int64_t lda,
              const c128* B, int64_t ldb, double beta, c128* C, int64_t ldc, bool small_tile, int splitk,
              cudaStream_t s, int lower_only = 0, int K2 = 0, const c128* A2 = nullptr, int64_t lda2 = 0,
              const c128* B2 = nullptr, int64_t ldb2 = 0, int mode = ZMODE_GEMM) {
    ZgemmArgs a;
    memset(&a, 0, sizeof(a));
    a.M = M; a.N = N; a.K1 = K; a.K2 = K2;
    a.A1 = A; a.B1 = B; a.lda1 = lda; a.ldb1 = ldb;
    a.A2 = A2; a.B2 = B2; a.lda2 = lda2; a.ldb2 = ldb2;
    a.C = C; a.ldc = ldc; a.alpha = alpha; a.beta = beta; a.lower_only = lower_only;
    a.partial = ws_ptr<c128>(h, h->plan.gemm_partial);
    const size_t per = (size_t)M * N * sizeof(c128);
    int sk = splitk < 1 ? 1 : splitk;
    while (sk > 1 && per * sk > h->plan.gemm_partial_bytes) --sk;
    a.splitk = sk;
    const int rc = zgemm_launch(a, ta, tb, mode, small_tile, s, &h->launches);
    return rc ? 1000 + rc : 0;
}

int zgemm_ws(eigh_handle_s* h, bool ta, bool tb, int M, int N, int K, double alpha, const c128* A, int64_t lda,
             const c128* B, int64_t ldb, double beta, c128* C, int64_t ldc, bool small_tile, int splitk,
             cudaStream_t s) {
    return zg(h, ta, tb, M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, small_tile, splitk, s);
}

int zgemm_ws2(eigh_handle_s* h, bool ta, bool tb, int M, int N, int K, double alpha, const c128* A, int64_t lda,
              const c128* B, int64_t ldb, double beta, c128* C, int64_t ldc, bool small_tile, int splitk, cudaStream_t s,
              int lower_only, int K2, const c128* A2, int64_t lda2, const c128* B2, int64_t ldb2) {
    return zg(h, ta, tb, M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, small_tile, splitk, s, lower_only, K2, A2, lda2, B2, ldb2);
}

static int splitk_for_small_output(int K) {
    int sk = K / 256;
    if (sk < 1) sk = 1;
    if (sk > 296) sk = 296;
    return sk;
}

int phase_reduce_to_band(eigh_handle_s* h, c128* A, int64_t lda, c128* band, int64_t ldab, cudaStream_t s) {
    const int N = (int)h->N, b = h->b;
    const WsPlan& pl = h->plan;
    c128* tau1 = ws_ptr<c128>(h, pl.tau1);
    c128* T1 = ws_ptr<c128>(h, pl.T1);
    c128* Vp = ws_ptr<c128>(h, pl.Vp);
    c128* VT = ws_ptr<c128>(h, pl.VT);
    c128* X = ws_ptr<c128>(h, pl.X);
    c128* small = ws_ptr<c128>(h, pl.small);
    unsigned* counter = ws_ptr<unsigned>(h, pl.panel_sync);
    c128* part = reinterpret_cast<c128*>(reinterpret_cast<char*>(counter) + 256);
    const int maxG = 160;
    c128* pivrow = part + (size_t)2 * maxG * b;

    symmetrize_diag_blocks_kernel<<<(unsigned)ceil_div(N, 64), 256, 0, s>>>(A, lda, N);
    ++h->launches;
    EIGH_CUDA_OK(cudaMemsetAsync(tau1, 0, (size_t)N * sizeof(c128), s));

    const size_t ps_smem = (size_t)(PS_MAXROWS * PS_LD + 4 * PS_B + 3 * PS_B) * sizeof(c128);
    const size_t pq_smem = (size_t)(PQ_WARPS * b + b + 4) * sizeof(c128);
    const size_t tf_smem = (size_t)(2 * b * (b + 1) + b) * sizeof(c128);
    // (set on every call: the attribute is per device / context, and the call is cheap)
    EIGH_CUDA_OK(cudaFuncSetAttribute(tfactor_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tf_smem));
    EIGH_CUDA_OK(cudaFuncSetAttribute(panel_qr_smem_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ps_smem));
    int max_coop = 0;
    EIGH_CUDA_OK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&max_coop, panel_qr_kernel, PQ_NT, pq_smem));
    if (max_coop < 1) return set_err(h, EIGH_ERR_CUDA, "panel_qr_kernel cannot be resident");
    const int coop_limit = min(maxG, h->num_sms);   // one CTA per SM

    for (int p = 0;; ++p) {
        const int j0 = p * b;
        const int m = N - j0 - b;
        if (m < 2) break;
        c128* panel = A + (j0 + b) + (int64_t)j0 * lda;
        c128* A22 = A + (j0 + b) + (int64_t)(j0 + b) * lda;
        c128* Tp = T1 + (size_t)p * b * b;
        // S1.1 + S1.2: panel QR and T factor
        int rc;
        const bool smem_panel = b == PS_B && h->panel_smem && m >= 2 * PS_B && m <= (int64_t)(coop_limit - 1) * PS_MAXROWS;
        EIGH_CUDA_OK(cudaMemsetAsync(counter, 0, 256, s));
        if (smem_panel) {
            PanelSmemArgs pa;
            pa.P = panel; pa.ld = lda; pa.m = m; pa.nr = b;
            pa.Vp = Vp; pa.ldv = m; pa.tau = tau1 + j0; pa.T = Tp; pa.ldt = b;
            pa.counter = counter; pa.part = part; pa.pivrow = pivrow;
            int G = coop_limit - 1;
            int rows = (int)ceil_div(m, G);
            if (rows < h->panel_rows_min) rows = h->panel_rows_min;
            if (rows > PS_MAXROWS) rows = PS_MAXROWS;
            pa.rows_per_cta = rows;
            G = (int)ceil_div(m, rows);
            void* kargs[] = {(void*)&pa};
            EIGH_CUDA_OK(cudaLaunchCooperativeKernel((void*)panel_qr_smem_kernel, dim3(G + 1), dim3(PS_NT), kargs, ps_smem, s));
            ++h->launches;
        } else {
            PanelArgs pa;
            pa.P = panel; pa.ld = lda; pa.m = m; pa.nb = b; pa.nr = min(b, m - 1);
            pa.Vp = Vp; pa.ldv = m; pa.tau = tau1 + j0; pa.counter = counter; pa.part = part; pa.pivrow = pivrow;
            int G = (int)ceil_div(m, 64);
            if (G > coop_limit) G = coop_limit;
            pa.rows_per_cta = (int)ceil_div(m, G);
            G = (int)ceil_div(m, pa.rows_per_cta);
            void* kargs[] = {(void*)&pa};
            EIGH_CUDA_OK(cudaLaunchCooperativeKernel((void*)panel_qr_kernel, dim3(G), dim3(PQ_NT), kargs, pq_smem, s));
            ++h->launches;
            rc = zg(h, true, false, b, b, m, 1.0, Vp, m, Vp, m, 0.0, small, b, true, splitk_for_small_output(m), s);
            if (rc) return rc;
            tfactor_kernel<<<1, 128, tf_smem, s>>>(small, b, tau1 + j0, b, Tp, b);
            ++h->launches;
        }
        // VT = V T
        rc = zg(h, false, false, m, b, b, 1.0, Vp, m, Tp, b, 0.0, VT, m, false, 1, s);
        if (rc) return rc;
        // S1.3 X = Herm(A22) VT
        {
            const int tiles = (int)ceil_div(m, 64);
            int sk = (int)ceil_div((int64_t)h->hemm_waves * h->num_sms, tiles);
            if (sk > 16) sk = 16;
            if (m / sk < 512) sk = max(1, m / 512);
            rc = zg(h, false, false, m, b, m, 1.0, A22, lda, VT, m, 0.0, X, m, true, sk, s, 0, 0, nullptr, 0, nullptr,
                    0, ZMODE_HEMM);
            if (rc) return rc;
        }
        // S1.4 S = VT^H X ; W = X - 1/2 V S
        rc = zg(h, true, false, b, b, m, 1.0, VT, m, X, m, 0.0, small + (size_t)b * b, b, true,
                splitk_for_small_output(m), s);
        if (rc) return rc;
        rc = zg(h, false, false, m, b, b, -0.5, Vp, m, small + (size_t)b * b, b, 1.0, X, m, false, 1, s);
        if (rc) return rc;
        // S1.5 A22 -= V W^H + W V^H (lower tiles)
        rc = zg(h, false, true, m, m, b, -1.0, Vp, m, X, m, 1.0, A22, lda, false, 1, s, 1, b, X, m, Vp, m);
        if (rc) return rc;
    }
    extract_band_kernel<<<N, 128, 0, s>>>(A, lda, N, b, band, ldab);
    ++h->launches;
    const cudaError_t ce = cudaGetLastError();
    return ce != cudaSuccess ? 1000 + (int)ce : 0;
}

}  // namespace eigh
