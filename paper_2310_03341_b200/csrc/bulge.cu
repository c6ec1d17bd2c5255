// bulge.cu -- S2: band -> tridiagonal by bulge chasing ("transforming the banded
// matrix into a tridiagonal form"), SURVEY.md 8(a) rows S2 / S2.1.
//
// Sweep j (j = 0..N-2) annihilates column j below the subdiagonal with a Householder reflector of
// length <= b on rows r_0 = j+1.., applies it two-sided to the diagonal block D_0 and from the right
// to the block S_1 below it (creating a bulge), then chases: at iteration k (r_k = j+1+k b) the
// reflector v_k is applied two-sided to D_k = B[r_k:r_k+b, r_k:r_k+b] and from the right to
// S_{k+1} = B[r_k+b:r_k+2b, r_k:r_k+b]; the first column of S_{k+1} defines v_{k+1}, which is applied
// from the left to the other columns of S_{k+1}.  Every block is loaded once and stored once per
// sweep.  The band keeps up to 2b-1 subdiagonals (lower band storage, ldab >= 2b).
//
// Parallelism: one CTA per sweep in flight (persistent grid, sweeps round-robin over CTAs); sweep
// j+1 may run iteration k once sweep j has finished iteration k+1 (progress counters in global
// memory, acquire/release through L2; all band reads bypass L1).  The grid is launched
// cooperatively so that every CTA is resident (the wait chain always ends at a running sweep).
//
// Reflectors (LAPACK zlarfg convention, H = I - tau v v^H, v_0 = 1 stored explicitly) are packed:
// V2[off(j) + row - j - 1], off(j) = j (N-1) - j (j-1)/2; tau of (sweep j, step k) at tau2[j kmax + k].
#include <limits.h>

#include "eigh_internal.h"

namespace eigh {

constexpr int BC_B = 64;          // band width handled by this kernel
constexpr int BC_LD = BC_B + 1;   // padded shared-memory leading dimension
constexpr int BC_NT = 256;

struct BcArgs {
    c128* band; int64_t ldab;
    int N;
    c128* V2;
    c128* tau2;       // [N][kmax]: tau of reflector (sweep j, step k) at tau2[j*kmax + k]
    int kmax;
    int* progress;    // [N], zero on entry
};

__device__ __forceinline__ double bc_block_sum(double v, double* red) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) red[warp] = v;
    __syncthreads();
    double s = 0.0;
#pragma unroll
    for (int w = 0; w < BC_NT / 32; ++w) s += red[w];
    return s;
}

// x[0..len) in xs -> v (v_0 = 1) in vs; returns tau; beta via *beta_out.  All threads call.
__device__ __forceinline__ c128 bc_make_reflector(const c128* xs, c128* vs, int len, double* red, c128* scal,
                                                  double* beta_out) {
    const int tid = threadIdx.x;
    double part = 0.0;
    if (tid >= 1 && tid < len) part = cabs2(xs[tid]);
    const double xnorm2 = bc_block_sum(part, red);
    if (tid == 0) {
        const c128 alpha = xs[0];
        c128 tau = cmake(0.0, 0.0), s = cmake(0.0, 0.0);
        double beta = alpha.x;
        if (xnorm2 > 0.0 || alpha.y != 0.0) {
            beta = -copysign(sqrt(alpha.x * alpha.x + alpha.y * alpha.y + xnorm2), alpha.x);
            tau = cmake((beta - alpha.x) / beta, -alpha.y / beta);
            const double dr = alpha.x - beta, di = alpha.y;
            const double den = dr * dr + di * di;
            s = cmake(dr / den, -di / den);
        }
        scal[0] = tau; scal[1] = s; scal[2] = cmake(beta, 0.0);
    }
    __syncthreads();
    const c128 tau = scal[0], s = scal[1];
    *beta_out = scal[2].x;
    c128 x = cmake(0.0, 0.0);
    if (tid < len) x = xs[tid];
    __syncthreads();       // xs may alias vs
    if (tid < len) vs[tid] = (tid == 0) ? cmake(1.0, 0.0) : cmul(s, x);
    __syncthreads();
    return tau;
}

__device__ __forceinline__ void bc_wait(const int* progress, int sweep, int need) {
    if (sweep >= 0) {
        if (threadIdx.x == 0) {
            while (*(volatile const int*)(progress + sweep) < need) {}
            __threadfence();
        }
    }
    __syncthreads();
}

__global__ void __launch_bounds__(BC_NT, 1) bulge_chase_kernel(const BcArgs a) {
    extern __shared__ __align__(16) unsigned char bc_raw[];
    c128* D = reinterpret_cast<c128*>(bc_raw);      // [BC_B][BC_LD]
    c128* S = D + BC_B * BC_LD;                     // [BC_B][BC_LD]
    c128* v = S + BC_B * BC_LD;                     // [BC_B]
    c128* vn = v + BC_B;                            // [BC_B]
    c128* w = vn + BC_B;                            // [BC_B]
    c128* y = w + BC_B;                             // [BC_B]
    c128* wpart = y + BC_B;                         // [4][BC_B]
    c128* scal = wpart + 4 * BC_B;                  // [4]
    double* red = reinterpret_cast<double*>(scal + 4);   // [8]

    const int tid = threadIdx.x;
    const int r = tid & 63, q = tid >> 6;           // row / quarter
    const int N = a.N;
    const int64_t ldab = a.ldab;

    for (int j = blockIdx.x; j <= N - 2; j += gridDim.x) {
        const int64_t voff = (int64_t)j * (N - 1) - (int64_t)j * (j - 1) / 2;   // packed column j
        c128* Vj = a.V2 + voff - j - 1;              // Vj[row] for row in j+1..N-1
        bc_wait(a.progress, j - 1, 2);
        int len = min(BC_B, N - 1 - j);
        // ---- step 0: reflector from column j
        c128* colj = a.band + (int64_t)j * ldab;
        if (tid < len) v[tid] = __ldcg(colj + 1 + tid);
        __syncthreads();
        double beta;
        c128 tau = bc_make_reflector(v, v, len, red, scal, &beta);
        if (tid < len) {
            colj[1 + tid] = (tid == 0) ? cmake(beta, 0.0) : cmake(0.0, 0.0);
            Vj[j + 1 + tid] = v[tid];
            if (tid == 0) a.tau2[(int64_t)j * a.kmax] = tau;
        }
        for (int k = 0;; ++k) {
            const int r0 = j + 1 + k * BC_B;
            len = min(BC_B, N - r0);
            if (k > 0) bc_wait(a.progress, j - 1, k + 2);
            // ---- load D_k (lower from band, mirrored)
            for (int cc = q; cc < len; cc += 4) {
                if (r < len && r >= cc) {
                    c128 e = __ldcg(a.band + (r - cc) + (int64_t)(r0 + cc) * ldab);
                    if (r == cc) e.y = 0.0;
                    D[r + cc * BC_LD] = e;
                    if (r != cc) D[cc + r * BC_LD] = cconj(e);
                }
            }
            __syncthreads();
            // ---- w = D v
            {
                c128 acc = cmake(0.0, 0.0);
                if (r < len)
                    for (int cc = q * 16; cc < min(len, q * 16 + 16); ++cc) cfma(acc, D[r + cc * BC_LD], v[cc]);
                wpart[q * BC_B + r] = acc;
            }
            __syncthreads();
            if (tid < BC_B) {
                c128 s = cmake(0.0, 0.0);
                if (tid < len) s = cadd(cadd(wpart[tid], wpart[BC_B + tid]), cadd(wpart[2 * BC_B + tid], wpart[3 * BC_B + tid]));
                w[tid] = s;
            }
            __syncthreads();
            // alpha = v^H w (real)
            double pa = 0.0;
            if (tid < len) pa = v[tid].x * w[tid].x + v[tid].y * w[tid].y;
            const double vhw = bc_block_sum(pa, red);
            // y = tau w - 1/2 |tau|^2 alpha v
            if (tid < len) {
                const double f = 0.5 * (tau.x * tau.x + tau.y * tau.y) * vhw;
                const c128 tw = cmul(tau, w[tid]);
                y[tid] = cmake(tw.x - f * v[tid].x, tw.y - f * v[tid].y);
            }
            __syncthreads();
            // D <- D - v y^H - y v^H ; store lower
            if (r < len) {
                const c128 vr = v[r], yr = y[r];
                for (int cc = q; cc < len; cc += 4) {
                    if (r >= cc) {
                        c128 e = D[r + cc * BC_LD];
                        const c128 yc = y[cc], vc = v[cc];
                        // v_r conj(y_c) + y_r conj(v_c)
                        e.x -= vr.x * yc.x + vr.y * yc.y + yr.x * vc.x + yr.y * vc.y;
                        e.y -= vr.y * yc.x - vr.x * yc.y + yr.y * vc.x - yr.x * vc.y;
                        if (r == cc) e.y = 0.0;
                        a.band[(r - cc) + (int64_t)(r0 + cc) * ldab] = e;
                    }
                }
            }
            const int len2 = min(BC_B, N - (r0 + BC_B));
            if (len2 <= 0) break;
            // ---- load S_{k+1}: rows r0+b+ii (ii < len2), cols r0+cc (cc < len)
            for (int cc = q; cc < len; cc += 4)
                if (r < len2) S[r + cc * BC_LD] = __ldcg(a.band + (BC_B + r - cc) + (int64_t)(r0 + cc) * ldab);
            __syncthreads();
            // u = S v  (len2)
            {
                c128 acc = cmake(0.0, 0.0);
                if (r < len2)
                    for (int cc = q * 16; cc < min(len, q * 16 + 16); ++cc) cfma(acc, S[r + cc * BC_LD], v[cc]);
                wpart[q * BC_B + r] = acc;
            }
            __syncthreads();
            if (tid < BC_B) {
                c128 s = cmake(0.0, 0.0);
                if (tid < len2) s = cadd(cadd(wpart[tid], wpart[BC_B + tid]), cadd(wpart[2 * BC_B + tid], wpart[3 * BC_B + tid]));
                w[tid] = cmul(tau, s);      // tau * u
            }
            __syncthreads();
            // S <- S - (tau u) v^H
            if (r < len2) {
                const c128 ur = w[r];
                for (int cc = q; cc < len; cc += 4) {
                    c128 e = S[r + cc * BC_LD];
                    const c128 vc = v[cc];
                    e.x -= ur.x * vc.x + ur.y * vc.y;
                    e.y -= ur.y * vc.x - ur.x * vc.y;
                    S[r + cc * BC_LD] = e;
                }
            }
            __syncthreads();
            // ---- next reflector from S[:,0]
            double betan;
            if (tid < len2) vn[tid] = S[tid];
            __syncthreads();
            const c128 taun = bc_make_reflector(vn, vn, len2, red, scal, &betan);
            if (tid < len2) S[tid] = (tid == 0) ? cmake(betan, 0.0) : cmake(0.0, 0.0);
            // z_c = vn^H S[:,c], c = 1..len-1 : thread (c = r, rows quarter q)
            {
                c128 acc = cmake(0.0, 0.0);
                if (r >= 1 && r < len)
                    for (int ii = q * 16; ii < min(len2, q * 16 + 16); ++ii) cfmac(acc, vn[ii], S[ii + r * BC_LD]);
                wpart[q * BC_B + r] = acc;
            }
            __syncthreads();
            if (tid < BC_B) {
                c128 s = cmake(0.0, 0.0);
                if (tid >= 1 && tid < len) s = cadd(cadd(wpart[tid], wpart[BC_B + tid]), cadd(wpart[2 * BC_B + tid], wpart[3 * BC_B + tid]));
                w[tid] = cmulc(taun, s);    // conj(tau') z_c
            }
            __syncthreads();
            // S[:,c] -= vn (conj(tau') z_c), c >= 1 ; store S
            if (r < len2) {
                const c128 vr = vn[r];
                for (int cc = q; cc < len; cc += 4) {
                    c128 e = S[r + cc * BC_LD];
                    if (cc >= 1) {
                        const c128 t = cmul(vr, w[cc]);
                        e.x -= t.x; e.y -= t.y;
                    }
                    a.band[(BC_B + r - cc) + (int64_t)(r0 + cc) * ldab] = e;
                }
            }
            if (tid < len2) Vj[r0 + BC_B + tid] = vn[tid];
            if (tid == 0) a.tau2[(int64_t)j * a.kmax + k + 1] = taun;
            __syncthreads();
            if (tid == 0) {
                __threadfence();
                *(volatile int*)(a.progress + j) = k + 1;
            }
            // v <- vn
            if (tid < BC_B) v[tid] = (tid < len2) ? vn[tid] : cmake(0.0, 0.0);
            tau = taun;
            __syncthreads();
        }
        __syncthreads();
        if (tid == 0) {
            __threadfence();
            *(volatile int*)(a.progress + j) = INT_MAX;
        }
        __syncthreads();
    }
}

// d_i = Re B[i,i]; e_i = |B[i+1,i]| (real by construction); sgn_0 = 1, sgn_{i+1} = sgn_i sign(B[i+1,i]).
__global__ void extract_tridiag_kernel(const c128* __restrict__ band, int64_t ldab, int N, double* __restrict__ d,
                                       double* __restrict__ e, double* __restrict__ sgn) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) d[i] = band[(int64_t)i * ldab].x;
    if (i < N - 1) e[i] = fabs(band[1 + (int64_t)i * ldab].x);
    if (i == 0) {
        double s = 1.0;
        sgn[0] = 1.0;
        for (int t = 0; t < N - 1; ++t) {
            if (band[1 + (int64_t)t * ldab].x < 0.0) s = -s;
            sgn[t + 1] = s;
        }
    }
}

int phase_band_to_tridiag(eigh_handle_s* h, c128* band, int64_t ldab, double* d, double* e, cudaStream_t s) {
    const int N = (int)h->N;
    if (h->b != BC_B) return set_err(h, -100, "bulge chasing is built for band width %d", BC_B);
    const WsPlan& pl = h->plan;
    int* progress = ws_ptr<int>(h, pl.bc_progress);
    double* sgn = ws_ptr<double>(h, pl.sgn);
    EIGH_CUDA_OK(cudaMemsetAsync(progress, 0, (size_t)(N + 8) * sizeof(int), s));
    if (N >= 2) {
        const size_t smem = (size_t)(2 * BC_B * BC_LD + 4 * BC_B + 4 * BC_B + 4) * sizeof(c128) + 8 * sizeof(double);
        static bool attr = false;
        if (!attr) {
            EIGH_CUDA_OK(cudaFuncSetAttribute(bulge_chase_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            attr = true;
        }
        int occ = 0;
        EIGH_CUDA_OK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, bulge_chase_kernel, BC_NT, smem));
        if (occ < 1) return set_err(h, EIGH_ERR_CUDA, "bulge_chase_kernel cannot be resident");
        int G = h->num_sms * occ;
        if (G > N - 1) G = N - 1;
        BcArgs a;
        a.band = band; a.ldab = ldab; a.N = N; a.V2 = ws_ptr<c128>(h, pl.V2); a.progress = progress;
        a.tau2 = ws_ptr<c128>(h, pl.tau2); a.kmax = (int)bc_kmax(h);
        void* kargs[] = {(void*)&a};
        EIGH_CUDA_OK(cudaLaunchCooperativeKernel((void*)bulge_chase_kernel, dim3(G), dim3(BC_NT), kargs, smem, s));
        ++h->launches;
    }
    extract_tridiag_kernel<<<(unsigned)ceil_div(N, 256), 256, 0, s>>>(band, ldab, N, d, e, sgn);
    ++h->launches;
    const cudaError_t ce = cudaGetLastError();
    return ce != cudaSuccess ? 1000 + (int)ce : 0;
}

}  // namespace eigh
