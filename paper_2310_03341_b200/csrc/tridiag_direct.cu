// tridiag_direct.cu -- the 1-stage variant: "i) transforming the dense matrix into
// a tridiagonal form, ii) diagonalizing this tridiagonal form, iii) back-transformation of the eigenvectors", the solver
// the paper benchmarks (Figs. 3-4), in a complex (c128) and a real-symmetric (double) instance
// (the paper's scaling runs are real FP64).  Step ii) is the D&C of tridiag_dc.cu.
//
// i)  Blocked Householder tridiagonalisation (LAPACK xHETRD / xLATRD formulation, lower triangle), panels of 64 columns.
//     For column c of a panel starting at j0 (V = reflectors of the panel so far, W the accumulated update vectors):
//        a      = A[c:, c] - V W[c,:]^H - W V[c,:]^H          (delayed rank-2k update of the current column)
//        v, tau = larfg(a[c+1:]),  e_c = beta (real)
//        y      = A22 v - V (W^H v) - W (V^H v)               (A22 = trailing matrix as it was at the start of the panel)
//        w      = tau y,   w += -1/2 tau (w^H v) v
//     and after the panel  A22 <- A22 - V W^H - W V^H  (HER2K / SYR2K-lower on the tensor-core GEMM engine).
//     The matrix-vector product A22 v reads the whole lower triangle once per column: 8/3 N^3 bytes (c128) in total, the
//     HBM-bound half of the method -- roofline = bytes of lower-triangle tiles / time against HBM.
//     ONE persistent cooperative kernel per panel: the 64 x 64 tiles of the lower triangle are dealt round-robin to the
//     thread blocks and streamed through a 3-stage cp.async ring filled by four LOADER warps (mbarrier full / empty
//     handshake per stage; the 8 compute warps never issue a copy); a tile is used for both y_I += A_IJ v_J and
//     y_J += A_IJ^H v_I; per-tile partial vectors are summed in a fixed order by the owner of each row block (no FP64
//     atomics: bit-reproducible, independent of the grid size).  Three grid barriers per column (release/acquire
//     counter).  The compact-WY factor T of the panel is accumulated on the fly from V^H v, which the step needs anyway.
// iii) Z <- Q Z with Q = H_0 H_1 ... H_{N-2}: panels merged 4 at a time into compact-WY blocks (K = 256) applied by
//     the GEMM engine, as S4b does for the 2-stage path.
#include <algorithm>

#include "eigh_internal.h"
#include "rgemm.cuh"
#include "scalar.cuh"
#include "zgemm.cuh"

namespace eigh {

int zgemm_ws2(eigh_handle_s* h, bool ta, bool tb, int M, int N, int K, double alpha, const c128* A, int64_t lda,
              const c128* B, int64_t ldb, double beta, c128* C, int64_t ldc, bool small_tile, int splitk, cudaStream_t s,
              int lower_only, int K2, const c128* A2, int64_t lda2, const c128* B2, int64_t ldb2);   // band_reduce.cu

// ------------------------------------------------------------------ GEMM dispatch (complex: zgemm engine, real: rgemm)
static int gemm_t(eigh_handle_s* h, bool ta, bool tb, int M, int N, int K, double alpha, const c128* A, int64_t lda,
                  const c128* B, int64_t ldb, double beta, c128* C, int64_t ldc, int splitk, cudaStream_t s,
                  int lower_only = 0, int K2 = 0, const c128* A2 = nullptr, int64_t lda2 = 0, const c128* B2 = nullptr,
                  int64_t ldb2 = 0) {
    return zgemm_ws2(h, ta, tb, M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, M <= 64, splitk, s, lower_only, K2, A2, lda2,
                     B2, ldb2);
}
static int gemm_t(eigh_handle_s* h, bool ta, bool tb, int M, int N, int K, double alpha, const double* A, int64_t lda,
                  const double* B, int64_t ldb, double beta, double* C, int64_t ldc, int splitk, cudaStream_t s,
                  int lower_only = 0, int K2 = 0, const double* A2 = nullptr, int64_t lda2 = 0, const double* B2 = nullptr,
                  int64_t ldb2 = 0) {
    RgemmArgs a;
    memset(&a, 0, sizeof(a));
    a.M = M; a.N = N; a.K1 = K; a.K2 = K2;
    a.A1 = A; a.B1 = B; a.lda1 = lda; a.ldb1 = ldb;
    a.A2 = A2; a.B2 = B2; a.lda2 = lda2; a.ldb2 = ldb2;
    a.C = C; a.ldc = ldc; a.alpha = alpha; a.beta = beta; a.lower_only = lower_only;
    a.partial = ws_ptr<double>(h, h->plan.gemm_partial);
    int sk = splitk < 1 ? 1 : splitk;
    while (sk > 1 && (size_t)M * N * sizeof(double) * sk > h->plan.gemm_partial_bytes) --sk;
    a.splitk = sk;
    const int rc = rgemm_launch(a, ta, tb, s, &h->launches);
    return rc ? 1000 + rc : 0;
}

// ------------------------------------------------------------------ the panel kernel
constexpr int HT_NT = 256, HT_B = 64, HT_LD = 65, HT_STG = 3;
// The thread block = HT_NT compute threads + HT_NL LOADER threads (threads HT_NT .. HT_NTB-1) that only issue the
// asynchronous copies of the tile phase: a copy instruction blocks its warp while the SM's queue of outstanding copies is
// full, and a blocked compute warp holds up the block's barriers -- the loader warps take that wait off the compute path.
// (Four warps, not one: with one tile per thread block -- small matrices -- the time to issue a tile is exposed.)
constexpr int HT_NL = 128;
constexpr int HT_NTB = HT_NT + HT_NL;

template <typename T>
struct HtArgs {
    T* A; int64_t lda;
    int N, j0, nb;            // panel = columns j0 .. j0+nb-1 (nb <= 64), trailing order m = N - j0
    T* W; int64_t ldw;        // W[global row + k ldw], k < 64
    double* e; T* tau;        // e[c], tau[c], c = global column
    T* Tout;                  // 64 x 64 compact-WY factor of the panel (upper triangular, zero elsewhere), ld 64
    unsigned* counter;        // grid barrier counter, zero on entry
    double* nrm_part;         // [nblk]
    T* dot_part;              // [nblk]
    T* g_part;                // [nblk][2][64]: W_I^H v_I, V_I^H v_I
    T* Pl; T* Pu;             // [ntiles][64] per-tile partial products
};

template <typename T>
struct HtSmem {
    T tile[HT_STG][HT_B * HT_LD];
    T vec[2][2][HT_B];        // [job parity][0: column-block vector v_J, 1: row-block vector v_I]
    T vraw[HT_STG][2][HT_B];  // the entries of column c of A behind them, fetched with the tile
    unsigned long long full[HT_STG], empty[HT_STG];   // mbarriers: the stage's copies have landed / its readers are done
    T red[2][4][HT_B];
    T xs[HT_B], ys[HT_B];
    T sred[HT_NT / 32];
    double dred[HT_NT / 32];
};

// barrier of the HT_NT compute threads (barrier 0 = the whole block incl. the loader warp: grid barriers only)
__device__ __forceinline__ void ht_sync() { asm volatile("bar.sync 1, %0;" ::"n"(HT_NT) : "memory"); }
__device__ __forceinline__ void ht_mbar_init(unsigned long long* b, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count));
}
__device__ __forceinline__ void ht_mbar_arrive(unsigned long long* b) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
// arrives on b once every cp.async this thread has issued so far has landed (counts as one of the expected arrivals)
__device__ __forceinline__ void ht_mbar_arrive_on_copies(unsigned long long* b) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void ht_mbar_wait(unsigned long long* b, unsigned parity) {
    unsigned ok = 0;
    while (!ok) {
        asm volatile(
            "{\n.reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n}"
            : "=r"(ok)
            : "r"(smem_u32(b)), "r"(parity)
            : "memory");
    }
}

__device__ __forceinline__ void ht_grid_barrier(unsigned* ctr, unsigned target) {
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

template <typename T>
__device__ __forceinline__ T ht_ldcg(const T* p);
template <>
__device__ __forceinline__ double ht_ldcg<double>(const double* p) { return __ldcg(p); }
template <>
__device__ __forceinline__ c128 ht_ldcg<c128>(const c128* p) { return __ldcg(p); }

// deterministic block-wide sums of n values read through L2 (every thread block gets the same bits)
template <typename T>
__device__ __forceinline__ double ht_block_sum_d(const double* src, int n, HtSmem<T>& sm) {
    double s = 0.0;
    for (int i = threadIdx.x; i < n; i += HT_NT) s += __ldcg(src + i);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    ht_sync();
    if ((threadIdx.x & 31) == 0) sm.dred[threadIdx.x >> 5] = s;
    ht_sync();
    double t = 0.0;
#pragma unroll
    for (int w = 0; w < HT_NT / 32; ++w) t += sm.dred[w];
    return t;
}
__device__ __forceinline__ double ht_shfl_xor(double v, int m) { return __shfl_xor_sync(0xffffffffu, v, m); }
__device__ __forceinline__ c128 ht_shfl_xor(c128 v, int m) {
    return cmake(__shfl_xor_sync(0xffffffffu, v.x, m), __shfl_xor_sync(0xffffffffu, v.y, m));
}
template <typename T>
__device__ __forceinline__ T ht_block_sum(const T* src, int n, HtSmem<T>& sm) {
    using S = Sc<T>;
    T s = S::zero();
    for (int i = threadIdx.x; i < n; i += HT_NT) s = S::add(s, ht_ldcg(src + i));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s = S::add(s, ht_shfl_xor(s, o));
    ht_sync();
    if ((threadIdx.x & 31) == 0) sm.sred[threadIdx.x >> 5] = s;
    ht_sync();
    T t = S::zero();
#pragma unroll
    for (int w = 0; w < HT_NT / 32; ++w) t = S::add(t, sm.sred[w]);
    return t;
}

// tiles of the lower triangle in column-strip order: strip J holds (I, J), I = J .. nblk-1; first index of strip J
__device__ __forceinline__ long long ht_strip_start(int J, int nblk) { return (long long)J * nblk - (long long)J * (J - 1) / 2; }
__device__ __forceinline__ void ht_tile_decode(long long t, int nblk, int& I, int& J) {
    // largest J with strip_start(J) <= t
    const double nb = (double)nblk + 0.5;
    int j = (int)(nb - sqrt(fmax(nb * nb - 2.0 * (double)t, 0.0)));
    if (j < 0) j = 0;
    if (j > nblk - 1) j = nblk - 1;
    while (j > 0 && ht_strip_start(j, nblk) > t) --j;
    while (j + 1 < nblk && ht_strip_start(j + 1, nblk) <= t) ++j;
    J = j;
    I = J + (int)(t - ht_strip_start(j, nblk));
}

template <typename T>
__global__ void __launch_bounds__(HT_NTB, 1) hetrd_panel_kernel(const HtArgs<T> a) {
    using S = Sc<T>;
    extern __shared__ __align__(16) unsigned char ht_raw[];
    HtSmem<T>& sm = *reinterpret_cast<HtSmem<T>*>(ht_raw);
    const int tid = threadIdx.x;
    const int r = tid & 63, q = tid >> 6;
    const int G = gridDim.x, cta = blockIdx.x;
    const int N = a.N, j0 = a.j0;
    const int m = N - j0;
    const int nblk = (m + HT_B - 1) / HT_B;
    const long long ntiles = (long long)nblk * (nblk + 1) / 2;
    const bool tcta = cta == G - 1;
    unsigned epoch = 0;

    if (tid == 0) {
        for (int st = 0; st < HT_STG; ++st) { ht_mbar_init(&sm.full[st], HT_NL); ht_mbar_init(&sm.empty[st], 1); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    // job list of this thread block in column i: its tiles (round robin over the column-strip order), then (V_I, W_I) of its
    // row blocks.  The loader warp and the compute threads walk the same list.
    const long long my_tiles = (ntiles > cta) ? (ntiles - cta + G - 1) / G : 0;
    const int my_blocks = (nblk > cta) ? (nblk - cta + G - 1) / G : 0;
    struct TileIt { int I, J; };
    auto tile_next = [&](TileIt& t) {
        t.I += G;
        while (t.I >= nblk && t.J < nblk) { t.I -= nblk; ++t.J; t.I += t.J; }     // (past the last tile: stops at J = nblk)
    };
    auto job_src = [&](int i, long long j, const TileIt& t, int& I, int& J, int& kind, const T*& src, int64_t& ld, int& nr, int& nc) {
        if (j < my_tiles) {
            I = t.I; J = t.J;
            kind = (I == J) ? 1 : 0;
            src = a.A + (j0 + I * HT_B) + (int64_t)(j0 + J * HT_B) * a.lda;
            ld = a.lda;
            nr = min(HT_B, m - I * HT_B);
            nc = min(HT_B, m - J * HT_B);
        } else {
            const long long jj = j - my_tiles;
            I = cta + (int)(jj >> 1) * G;
            J = 0;
            kind = 2 + (int)(jj & 1);                      // 2: V_I, 3: W_I
            nr = min(HT_B, m - I * HT_B);
            nc = i;
            if (kind == 2) { src = a.A + (j0 + I * HT_B) + (int64_t)j0 * a.lda; ld = a.lda; }
            else { src = a.W + (j0 + I * HT_B); ld = a.ldw; }
        }
    };
    unsigned jobno = 0;                          // jobs so far (all columns): stage jobno % HT_STG, use jobno / HT_STG of it

    if (tid >= HT_NT) {
        // ================= the loader warps: per column, between the same grid barriers as the tile phase
        const int lt = tid - HT_NT;
        const int lr = lt & 63, lq = lt >> 6;                  // row lr, columns lq, lq + 2, ...
        for (int i = 0; i < a.nb; ++i) {
            const int c = j0 + i;
            ht_grid_barrier(a.counter, (++epoch) * (unsigned)G);
            const long long njobs = my_tiles + (i > 0 ? 2LL * my_blocks : 0);
            TileIt it;
            ht_tile_decode(cta, nblk, it.I, it.J);
            for (long long j = 0; j < njobs; ++j, ++jobno) {
                int I, J, kind, nr, nc;
                const T* src; int64_t ld;
                job_src(i, j, it, I, J, kind, src, ld, nr, nc);
                if (j < my_tiles) tile_next(it);
                const int st = (int)(jobno % HT_STG);
                if (jobno >= HT_STG) ht_mbar_wait(&sm.empty[st], ((jobno / HT_STG) - 1u) & 1u);     // its readers are done
                T* dst = sm.tile[st];
                if (kind == 0 && nr == HT_B && nc == HT_B) {              // interior tile: no predicates
                    const T* p = src + lr + (int64_t)lq * ld;
                    T* dp = dst + lq * HT_LD + lr;
#pragma unroll 8
                    for (int k = 0; k < HT_B * HT_B / HT_NL; ++k)
                        cp_async_elem(dp + k * (HT_NL / HT_B) * HT_LD, p + (int64_t)(k * (HT_NL / HT_B)) * ld, true);
                } else {
                    // diagonal tiles: only the lower triangle is read (the strict upper part is never valid input);
                    // V_I: only the part strictly below the diagonal of A holds reflector entries.  Columns >= nc of a
                    // (V_I, W_I) job are not written at all: their products are never used.
                    const int ncl = kind >= 2 ? nc : HT_B;
#pragma unroll 4
                    for (int cc = lq; cc < ncl; cc += HT_NL / HT_B) {
                        const bool ok = lr < nr && cc < nc && (kind != 1 || lr >= cc) && (kind != 2 || I * HT_B + lr > cc);
                        cp_async_elem(dst + cc * HT_LD + lr, ok ? src + lr + (int64_t)cc * ld : src, ok);
                    }
                }
                {                                                           // entries of column c behind v_J (0) and v_I (1)
                    const int which = lq;
                    const int gl = j0 + (which ? I : J) * HT_B + lr;
                    const bool ok = gl > c + 1 && gl < N && !(kind >= 2 && which == 0);
                    cp_async_elem(&sm.vraw[st][which][lr], ok ? a.A + gl + (int64_t)c * a.lda : a.A, ok);
                }
                ht_mbar_arrive_on_copies(&sm.full[st]);
            }
            ht_grid_barrier(a.counter, (++epoch) * (unsigned)G);
            ht_grid_barrier(a.counter, (++epoch) * (unsigned)G);
        }
        return;
    }

    if (tcta)      // the compact-WY factor is accumulated in place in global memory (read and written by this block only)
        for (int idx = tid; idx < HT_B * HT_B; idx += HT_NT) a.Tout[idx] = S::zero();
    ht_sync();

    T tau_prev = S::zero();
    for (int i = 0; i <= a.nb; ++i) {
        const int c = j0 + i;
        // ================= phase 1: finish W[:, i-1], update column c, partial norms
        T alpha_prev = S::zero();
        if (i > 0) {
            const T dsum = ht_block_sum<T>(a.dot_part, nblk, sm);            // sum over row blocks of w^H v
            alpha_prev = S::scale(-0.5, S::mul(tau_prev, dsum));
        }
        if (i > 0) {
            // fix the rows of W[:, i-1] this thread block owns:  w += alpha v_{i-1}
            for (int I = cta; I < nblk; I += G) {
                const int gl = j0 + I * HT_B + r;
                // (row c itself keeps its unfixed value during step i: every thread block adds alpha where it uses it,
                //  so no block can see a half-updated element; after step i that element is never read again)
                if (q == 0 && gl < N && (gl > c || (gl == c && i == a.nb))) {
                    T* wp = a.W + gl + (int64_t)(i - 1) * a.ldw;
                    const T vv = (gl == c) ? S::one() : a.A[gl + (int64_t)(c - 1) * a.lda];
                    *wp = S::add(*wp, S::mul(alpha_prev, vv));
                }
            }
        }
        if (i == a.nb) break;                                   // the extra round only finishes the last column of W
        if (i > 0 && tid < i) {
            // row c of W and of V:  xs[k] = conj(W[c, k]), ys[k] = conj(V[c, k])
            T wck = ht_ldcg(a.W + c + (int64_t)tid * a.ldw);
            if (tid == i - 1) wck = S::add(wck, alpha_prev);                 // v_{i-1}[c] = 1
            sm.xs[tid] = S::conj(wck);
            sm.ys[tid] = S::conj(ht_ldcg(a.A + c + (int64_t)(j0 + tid) * a.lda));
        }
        ht_sync();                                         // (also orders the W fix before the reads below)
        for (int I = cta; I < nblk; I += G) {
            const int gl = j0 + I * HT_B + r;
            const bool act = gl >= c && gl < N;
            T acc = S::zero();
            if (act) {
                for (int k = q; k < i; k += 4) {
                    S::fma(acc, a.A[gl + (int64_t)(j0 + k) * a.lda], sm.xs[k]);
                    T wv = a.W[gl + (int64_t)k * a.ldw];
                    if (gl == c && k == i - 1) wv = S::add(wv, alpha_prev);
                    S::fma(acc, wv, sm.ys[k]);
                }
            }
            sm.red[0][q][r] = acc;
            ht_sync();
            double pn = 0.0;
            if (q == 0 && act) {
                const T sum = S::add(S::add(sm.red[0][0][r], sm.red[0][1][r]), S::add(sm.red[0][2][r], sm.red[0][3][r]));
                T v = S::sub(a.A[gl + (int64_t)c * a.lda], sum);
                if (gl == c) v = S::real_part_only(v);
                a.A[gl + (int64_t)c * a.lda] = v;
                if (gl >= c + 2) pn = S::abs2(v);
            }
            // block sum of pn (warps 0, 1 hold the 64 rows)
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) pn += __shfl_xor_sync(0xffffffffu, pn, o);
            if ((tid & 31) == 0) sm.dred[tid >> 5] = pn;
            ht_sync();
            if (tid == 0) a.nrm_part[I] = sm.dred[0] + sm.dred[1];
        }
        ht_grid_barrier(a.counter, (++epoch) * (unsigned)G);

        // ================= phase 2: reflector scalars (redundantly), y partials, W^H v and V^H v partials
        const double xnorm2 = ht_block_sum_d<T>(a.nrm_part, nblk, sm);
        T tau, sc;
        double beta;
        {
            const T alpha = (c + 1 < N) ? ht_ldcg(a.A + (c + 1) + (int64_t)c * a.lda) : S::zero();
            larfg_scalars<T>(alpha, xnorm2, tau, sc, beta);
        }
        if (cta == 0 && tid == 0) { a.e[c] = beta; a.tau[c] = tau; }
        // v at global row gl (0 above the subdiagonal, 1 on it, scaled column below), x = A(gl, c)
        auto vmake = [&](int gl, T x) -> T {
            if (gl <= c || gl >= N) return S::zero();
            if (gl == c + 1) return S::one();
            return S::mul(sc, x);
        };
        {
            // the jobs of this column, in the order the loader warp issues them
            const long long njobs = my_tiles + (i > 0 ? 2LL * my_blocks : 0);
            TileIt it_use;
            ht_tile_decode(cta, nblk, it_use.I, it_use.J);
            for (long long j = 0; j < njobs; ++j, ++jobno) {
                int I, J, kind, nr, nc;
                const T* src; int64_t ld;
                job_src(i, j, it_use, I, J, kind, src, ld, nr, nc);
                if (j < my_tiles) tile_next(it_use);
                const int par = (int)(j & 1);
                const int st = (int)(jobno % HT_STG);
                ht_mbar_wait(&sm.full[st], (jobno / HT_STG) & 1u);     // the loader's copies of this stage have landed
                // Every row of v_J and v_I below the subdiagonal entry (all but the tiles of the block row / column that
                // holds column c): v = sc x there, so the products are taken with the fetched column entries x themselves
                // and the sums scaled by sc -- no pass over the vectors, no barrier before the products.
                const bool clean = j0 + (kind <= 1 ? J : I) * HT_B > c + 1;
                if (!clean) {
                    if (tid < 2 * HT_B) {
                        const int which = tid >> 6;                       // 0: v_J, 1: v_I
                        const int blk = which ? I : J;
                        sm.vec[par][which][r] = (kind >= 2 && which == 0) ? S::zero()
                                                                          : vmake(j0 + blk * HT_B + r, sm.vraw[st][which][r]);
                    }
                    ht_sync();
                }
                const T* St = sm.tile[st];
                const T* vJ = clean ? sm.vraw[st][0] : sm.vec[par][0];
                const T* vI = clean ? sm.vraw[st][1] : sm.vec[par][1];
                T accr = S::zero(), accc = S::zero();
                if (kind == 0) {
                    // row r of A_IJ v_J and column r of A_IJ^H v_I, two accumulators each (independent FMA chains)
                    T accr2 = S::zero(), accc2 = S::zero();
#pragma unroll 4
                    for (int cc = q; cc < HT_B; cc += 8) {
                        S::fma(accr, St[cc * HT_LD + r], vJ[cc]);
                        S::fmac(accc, St[r * HT_LD + cc], vI[cc]);
                        S::fma(accr2, St[(cc + 4) * HT_LD + r], vJ[cc + 4]);
                        S::fmac(accc2, St[r * HT_LD + cc + 4], vI[cc + 4]);
                    }
                    accr = S::add(accr, accr2);
                    accc = S::add(accc, accc2);
                } else if (kind == 1) {
#pragma unroll 4
                    for (int cc = q; cc < HT_B; cc += 4) {
                        T e;
                        if (cc < r) e = St[cc * HT_LD + r];
                        else if (cc == r) e = S::real_part_only(St[cc * HT_LD + r]);
                        else e = S::conj(St[r * HT_LD + cc]);
                        S::fma(accr, e, vI[cc]);
                    }
                } else {
#pragma unroll 4
                    for (int rr = q; rr < HT_B; rr += 4) S::fmac(accc, St[r * HT_LD + rr], vI[rr]);        // (V_I or W_I)^H v_I, entry r = k
                }
                sm.red[0][q][r] = accr;
                sm.red[1][q][r] = accc;
                ht_sync();
                if (tid == 0) ht_mbar_arrive(&sm.empty[st]);          // every compute thread is past its reads of the stage
                if (tid < 2 * HT_B) {
                    const int which = tid >> 6;
                    T sum = S::add(S::add(sm.red[which][0][r], sm.red[which][1][r]),
                                   S::add(sm.red[which][2][r], sm.red[which][3][r]));
                    if (clean) sum = S::mul(sc, sum);
                    if (kind <= 1) {
                        const long long t = cta + j * G;
                        if (which == 0) a.Pl[t * HT_B + r] = sum;
                        else if (kind == 0) a.Pu[t * HT_B + r] = sum;
                    } else if (which == 1) {
                        a.g_part[((size_t)I * 2 + (kind == 2 ? 1 : 0)) * HT_B + r] = sum;      // [I][0] = W^H v, [I][1] = V^H v
                    }
                }
            }
        }
        ht_grid_barrier(a.counter, (++epoch) * (unsigned)G);

        // ================= phase 3: y = sum of the partials, corrections, w = tau y, partial w^H v; T factor
        {
            // g1 = W^H v, g2 = V^H v (k < i), summed over the row blocks in a fixed order
            if (tid < 2 * HT_B) {
                const int which = tid >> 6;
                T s = S::zero();
                if (r < i)
                    for (int I = 0; I < nblk; ++I) s = S::add(s, ht_ldcg(a.g_part + ((size_t)I * 2 + which) * HT_B + r));
                if (which == 0) sm.xs[r] = s; else sm.ys[r] = s;
            }
            ht_sync();
            if (tcta) {
                // T[0:i, i] = -tau T[0:i, 0:i] g2,  T[i, i] = tau
                T acc = S::zero();
                if (r < i)
                    for (int l = r + q; l < i; l += 4) S::fma(acc, a.Tout[r + (size_t)l * HT_B], sm.ys[l]);
                sm.red[0][q][r] = acc;
                ht_sync();
                if (tid < HT_B) {
                    if (tid < i) {
                        const T sum = S::add(S::add(sm.red[0][0][tid], sm.red[0][1][tid]), S::add(sm.red[0][2][tid], sm.red[0][3][tid]));
                        a.Tout[tid + (size_t)i * HT_B] = S::neg(S::mul(tau, sum));
                    } else if (tid == i) {
                        a.Tout[tid + (size_t)i * HT_B] = tau;
                    }
                }
                ht_sync();
            }
            for (int I = cta; I < nblk; I += G) {
                const int gl = j0 + I * HT_B + r;
                const bool act = gl >= c + 1 && gl < N;
                T acc = S::zero();
                // partial vectors of row block I: row products of the tiles (I, J), J <= I, and column products of (I', I), I' > I
                for (int J = q; J <= I; J += 4) acc = S::add(acc, ht_ldcg(a.Pl + (ht_strip_start(J, nblk) + (I - J)) * HT_B + r));
                {
                    const long long base = ht_strip_start(I, nblk);
                    for (int Ip = I + 1 + q; Ip < nblk; Ip += 4) acc = S::add(acc, ht_ldcg(a.Pu + (base + (Ip - I)) * HT_B + r));
                }
                T corr = S::zero();
                if (act) {
                    for (int k = q; k < i; k += 4) {
                        S::fma(corr, a.A[gl + (int64_t)(j0 + k) * a.lda], sm.xs[k]);
                        S::fma(corr, a.W[gl + (int64_t)k * a.ldw], sm.ys[k]);
                    }
                }
                sm.red[0][q][r] = S::sub(acc, corr);
                ht_sync();
                T dot = S::zero();
                if (q == 0 && gl < N) {
                    T w = S::zero();
                    if (act) {
                        const T y = S::add(S::add(sm.red[0][0][r], sm.red[0][1][r]), S::add(sm.red[0][2][r], sm.red[0][3][r]));
                        w = S::mul(tau, y);
                        const T v = vmake(gl, (gl > c + 1 && gl < N) ? ht_ldcg(a.A + gl + (int64_t)c * a.lda) : S::zero());
                        S::fmac(dot, w, v);
                        a.A[gl + (int64_t)c * a.lda] = v;            // the reflector replaces the annihilated column
                    }
                    a.W[gl + (int64_t)i * a.ldw] = w;
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) dot = S::add(dot, ht_shfl_xor(dot, o));
                if ((tid & 31) == 0) sm.sred[tid >> 5] = dot;
                ht_sync();
                if (tid == 0) a.dot_part[I] = S::add(sm.sred[0], sm.sred[1]);
            }
        }
        tau_prev = tau;
        ht_grid_barrier(a.counter, (++epoch) * (unsigned)G);
    }
}

// d_i = Re A[i, i]
template <typename T>
__global__ void ht_diag_kernel(const T* __restrict__ A, int64_t lda, int N, double* __restrict__ d) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) d[i] = Sc<T>::re(A[i + (int64_t)i * lda]);
}

size_t ht_partial_bytes(int64_t N) {
    const int64_t nblk = ceil_div(N, HT_B);
    const int64_t ntiles = nblk * (nblk + 1) / 2;
    return (size_t)(2 * ntiles * HT_B + nblk * (2 * HT_B + 2) + 64) * sizeof(c128) + (size_t)(nblk + 64) * sizeof(double) + 1024;
}

template <typename T>
static int tridiagonalise_direct_t(eigh_handle_s* h, T* A, int64_t lda, double* d, double* e, cudaStream_t s) {
    const int N = (int)h->N;
    const WsPlan& pl = h->plan;
    T* W = ws_ptr<T>(h, pl.X);                       // N x 64
    T* tau = ws_ptr<T>(h, pl.tau1);
    T* T1 = ws_ptr<T>(h, pl.T1);
    unsigned* counter = ws_ptr<unsigned>(h, pl.panel_sync);
    // partial-product arena
    char* pp = ws_ptr<char>(h, pl.ht_part);
    const int64_t nblk0 = ceil_div(N, HT_B);
    const int64_t ntiles0 = nblk0 * (nblk0 + 1) / 2;
    T* Pl = reinterpret_cast<T*>(pp);
    T* Pu = Pl + ntiles0 * HT_B;
    T* g_part = Pu + ntiles0 * HT_B;
    T* dot_part = g_part + nblk0 * 2 * HT_B;
    double* nrm_part = reinterpret_cast<double*>(reinterpret_cast<c128*>(pp) + (2 * ntiles0 * HT_B + nblk0 * (2 * HT_B + 2) + 32));
    const size_t smem = sizeof(HtSmem<T>);
    auto kern = hetrd_panel_kernel<T>;
    EIGH_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 0;
    EIGH_CUDA_OK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, HT_NTB, smem));
    if (occ < 1) return set_err(h, EIGH_ERR_CUDA, "hetrd_panel_kernel cannot be resident");
    if (N > 1) EIGH_CUDA_OK(cudaMemsetAsync(e, 0, (size_t)(N - 1) * sizeof(double), s));
    EIGH_CUDA_OK(cudaMemsetAsync(tau, 0, (size_t)N * sizeof(T), s));
    for (int j0 = 0; j0 < N - 1; j0 += HT_B) {
        const int nb = std::min(HT_B, N - 1 - j0);
        const int m = N - j0;
        const int64_t nblk = ceil_div(m, HT_B);
        const int64_t ntiles = nblk * (nblk + 1) / 2;
        int G = h->num_sms * occ;
        if (h->ht_grid > 0 && h->ht_grid < G) G = h->ht_grid;
        if ((int64_t)G > ntiles + 1) G = (int)ntiles + 1;
        if (G < 1) G = 1;
        EIGH_CUDA_OK(cudaMemsetAsync(counter, 0, 256, s));
        HtArgs<T> a;
        a.A = A; a.lda = lda; a.N = N; a.j0 = j0; a.nb = nb;
        a.W = W; a.ldw = N; a.e = e; a.tau = tau; a.Tout = T1 + (size_t)(j0 / HT_B) * HT_B * HT_B;
        a.counter = counter; a.nrm_part = nrm_part; a.dot_part = dot_part; a.g_part = g_part; a.Pl = Pl; a.Pu = Pu;
        void* kargs[] = {(void*)&a};
        EIGH_CUDA_OK(cudaLaunchCooperativeKernel((void*)kern, dim3(G), dim3(HT_NTB), kargs, smem, s));
        ++h->launches;
        const int mt = N - j0 - nb;                  // trailing order after the panel
        if (mt > 0) {
            // A22 -= V W^H + W V^H (lower tiles): V = A[j0+nb:, j0:j0+nb], W rows j0+nb ..
            T* A22 = A + (j0 + nb) + (int64_t)(j0 + nb) * lda;
            const T* V = A + (j0 + nb) + (int64_t)j0 * lda;
            const T* Wt = W + (j0 + nb);
            const int rc = gemm_t(h, false, true, mt, mt, nb, -1.0, V, lda, Wt, N, 1.0, A22, lda, 1, s, 1, nb, Wt, N, V, lda);
            if (rc) return rc;
        }
    }
    ht_diag_kernel<T><<<(unsigned)ceil_div(N, 256), 256, 0, s>>>(A, lda, N, d);
    ++h->launches;
    const cudaError_t ce = cudaGetLastError();
    return ce != cudaSuccess ? 1000 + (int)ce : 0;
}

// ------------------------------------------------------------------ iii) back-transformation  Z <- Q Z
// V (mrows x kb, ldv): explicit unit-lower-trapezoidal reflectors of panels p0 .. p0+cnt-1 (64 columns each) taken from
// A.  Local row 0 = global row p0 64 + 1; column c = 64 q + cl has its unit element at local row c.
template <typename T>
__global__ void ht_extract_vgroup_kernel(const T* __restrict__ A, int64_t lda, int N, int p0, int cnt, T* __restrict__ V,
                                         int64_t ldv) {
    using S = Sc<T>;
    const int c = blockIdx.y;
    const int row0 = p0 * HT_B + 1;
    const int mrows = N - row0;
    const int rr = blockIdx.x * blockDim.x + threadIdx.x;
    if (rr >= mrows) return;
    const int gc = p0 * HT_B + c;                 // global column of this reflector
    T v = S::zero();
    if (gc <= N - 2) {
        if (rr == c) v = S::one();
        else if (rr > c) v = A[(row0 + rr) + (int64_t)gc * lda];
    }
    V[rr + (int64_t)c * ldv] = v;
}

template <typename T>
__global__ void ht_tdiag_kernel(const T* __restrict__ T1, int p0, int cnt, T* __restrict__ Tm, int ldt) {
    const int kb = cnt * HT_B;
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < kb * kb; idx += gridDim.x * blockDim.x) {
        const int i = idx % kb, j = idx / kb;
        T v = Sc<T>::zero();
        if (i / HT_B == j / HT_B) v = T1[(size_t)(p0 + i / HT_B) * HT_B * HT_B + (i % HT_B) + (size_t)(j % HT_B) * HT_B];
        Tm[i + (size_t)j * ldt] = v;
    }
}

static int ht_splitk_for(const eigh_handle_s* h, int M, int N, int K) {
    const int64_t tiles = ceil_div(M, 64) * ceil_div(N, 64);
    const int64_t want = 8 * (int64_t)h->num_sms;
    int sk = (int)ceil_div(want, tiles);
    if (sk < 1) sk = 1;
    while (sk > 1 && K / sk < 256) --sk;
    if (sk > 16) sk = 16;
    return sk;
}

template <typename T>
static int backtransform_direct_t(eigh_handle_s* h, const T* A, int64_t lda, T* Z, int64_t ldz, cudaStream_t s) {
    const int N = (int)h->N, nev = (int)h->nev, b = HT_B;
    const WsPlan& pl = h->plan;
    const T* T1 = ws_ptr<T>(h, pl.T1);
    T* V = ws_ptr<T>(h, pl.b4V);
    T* VTh = ws_ptr<T>(h, pl.b4VT);
    T* Y = ws_ptr<T>(h, pl.b4Y);
    T* Tm = ws_ptr<T>(h, pl.b4T);
    T* Gm = ws_ptr<T>(h, pl.b4G);
    const int mg = h->p4b_merge < 1 ? 1 : h->p4b_merge;
    T* tmp = Gm + (size_t)mg * b * mg * b;
    const int np = (int)ceil_div(N - 1, b);                  // panels of the tridiagonalisation
    for (int pend = np; pend > 0;) {
        const int cnt = std::min(mg, pend);
        const int p0 = pend - cnt;
        const int mrows = N - (p0 * b + 1);
        const int kb = cnt * b;
        T* Zr = Z + (p0 * b + 1);
        ht_extract_vgroup_kernel<T><<<dim3((unsigned)ceil_div(mrows, 256), (unsigned)kb), 256, 0, s>>>(A, lda, N, p0, cnt, V, mrows);
        ++h->launches;
        const T* Tg = T1 + (size_t)p0 * b * b;
        int ldt = b;
        int rc;
        if (cnt > 1) {
            rc = gemm_t(h, true, false, kb, kb, mrows, 1.0, V, mrows, V, mrows, 0.0, Gm, kb, ht_splitk_for(h, kb, kb, mrows), s);
            if (rc) return rc;
            ht_tdiag_kernel<T><<<64, 256, 0, s>>>(T1, p0, cnt, Tm, kb);
            ++h->launches;
            for (int j = 1; j < cnt; ++j) {
                const int jb = j * b;
                rc = gemm_t(h, false, false, jb, b, b, 1.0, Gm + (size_t)jb * kb, kb, T1 + (size_t)(p0 + j) * b * b, b, 0.0, tmp, jb, 1, s);
                if (rc) return rc;
                rc = gemm_t(h, false, false, jb, b, jb, -1.0, Tm, kb, tmp, jb, 0.0, Tm + (size_t)jb * kb, kb, 1, s);
                if (rc) return rc;
            }
            Tg = Tm;
            ldt = kb;
        }
        rc = gemm_t(h, false, true, mrows, kb, kb, 1.0, V, mrows, Tg, ldt, 0.0, VTh, mrows, 1, s);          // V T^H
        if (rc) return rc;
        rc = gemm_t(h, true, false, kb, nev, mrows, 1.0, VTh, mrows, Zr, ldz, 0.0, Y, kb, ht_splitk_for(h, kb, nev, mrows), s);
        if (rc) return rc;
        rc = gemm_t(h, false, false, mrows, nev, kb, -1.0, V, mrows, Y, kb, 1.0, Zr, ldz, 1, s);
        if (rc) return rc;
        pend = p0;
    }
    const cudaError_t ce = cudaGetLastError();
    return ce != cudaSuccess ? 1000 + (int)ce : 0;
}

// Z[r, c] = Q[r + c ldq]  (real D&C vectors -> the working type)
template <typename T>
__global__ void ht_expand_kernel(const double* __restrict__ Q, int64_t ldq, int N, int nev, T* __restrict__ Z, int64_t ldz) {
    const int c = blockIdx.y;
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r < N && c < nev) Z[r + (int64_t)c * ldz] = Sc<T>::from_real(Q[r + (int64_t)c * ldq]);
}

// ------------------------------------------------------------------ phase drivers (api.cu)
int phase_tridiagonalise_direct(eigh_handle_s* h, void* A, int64_t lda, double* d, double* e, cudaStream_t s) {
    if (h->real_dtype) return tridiagonalise_direct_t<double>(h, (double*)A, lda, d, e, s);
    return tridiagonalise_direct_t<c128>(h, (c128*)A, lda, d, e, s);
}

int phase_backtransform_direct(eigh_handle_s* h, const void* A, int64_t lda, const double* Q, int64_t ldq, void* Z,
                               int64_t ldz, cudaStream_t s) {
    const int N = (int)h->N, nev = (int)h->nev;
    const dim3 grid((unsigned)ceil_div(N, 256), (unsigned)nev);
    if (h->real_dtype) {
        if (Q) { ht_expand_kernel<double><<<grid, 256, 0, s>>>(Q, ldq, N, nev, (double*)Z, ldz); ++h->launches; }
        return backtransform_direct_t<double>(h, (const double*)A, lda, (double*)Z, ldz, s);
    }
    if (Q) { ht_expand_kernel<c128><<<grid, 256, 0, s>>>(Q, ldq, N, nev, (c128*)Z, ldz); ++h->launches; }
    return backtransform_direct_t<c128>(h, (const c128*)A, lda, (c128*)Z, ldz, s);
}

}  // namespace eigh
