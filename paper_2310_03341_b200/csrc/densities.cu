// densities.cu -- SCF epilogue: local densities from the quasiparticle states.
//
// PAPER.md:300-311, Eq. (16a), (16d), (17): with phi_n = [u_n, v_n]^T = column n of Z (rows [0, M) = u, rows
// [M, 2M) = v, M = N/2) and f_T(E) = 1 / (1 + exp(E/T)),
//     n(r)  = 2 sum_{0 < E_n < E_c} ( |v_n(r)|^2 f_T(-E_n) + |u_n(r)|^2 f_T(E_n) )
//     nu(r) =   sum_{0 < E_n < E_c} u_n(r) conj(v_n(r)) ( f_T(-E_n) - f_T(E_n) ).
// Both are sums over columns of Z with per-column weights, so the work is one streaming pass over the active
// columns of Z: HBM-bound, 32 bytes (u and v of one grid point and one state) per 10 FMAs.
//
//   dens_weights_kernel  per column: the weights (wu, wv, wnu) and the "active" flag; one thread block compacts the
//                        active columns, in ascending column order, into a list (ballot + block scan, no atomics).
//   dens_partial_kernel  thread = grid point r, block.y = chunk of the active list; sequential sums over the chunk,
//                        coalesced 16-byte streaming loads (512 B per warp and column half), 8 columns in flight.
//   dens_reduce_kernel   sums the chunk partials in chunk order.
// The order of every sum is fixed by (ncols, M, number of chunks): results are reproducible bit for bit.
#include <math.h>

#include <algorithm>

#include "eigh_internal.h"

namespace eigh {

// 1 / (1 + exp(x)) without overflow.  T = 0 is the step function (Eq. 17's limit); E = 0 is never asked for.
__device__ __forceinline__ double fermi_dev(double E, double T) {
    if (T == 0.0) return E < 0.0 ? 1.0 : (E > 0.0 ? 0.0 : 0.5);
    const double x = E / T;
    if (x >= 0.0) {
        const double t = exp(-x);
        return t / (1.0 + t);
    }
    return 1.0 / (1.0 + exp(x));
}

constexpr int DW_THREADS = 1024;

// One entry per ACTIVE column, in ascending column order: the weights of |u|^2, |v|^2 and u conj(v), and the column.
struct __align__(32) DensCol {
    double wu, wv, wnu;
    int64_t col;
};

// branch = +1: Eq. (16) as written on the columns with 0 < E < Ec.
// branch = -1: columns with -Ec < E < 0 stand for their particle-hole partners [-conj(v), conj(u)] of energy -E
//              (SURVEY.md 8(c) reading 3): |u|^2 and |v|^2 trade places and u conj(v) changes sign.
__global__ void __launch_bounds__(DW_THREADS) dens_weights_kernel(const double* __restrict__ E, int64_t ncols, double T,
                                                                   double Ec, int branch, DensCol* __restrict__ act,
                                                                   int* __restrict__ nact) {
    __shared__ int warp_tot[DW_THREADS / 32];
    __shared__ int base;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (tid == 0) base = 0;
    __syncthreads();
    for (int64_t j0 = 0; j0 < ncols; j0 += DW_THREADS) {
        const int64_t j = j0 + tid;
        int on = 0;
        DensCol dc;
        dc.wu = dc.wv = dc.wnu = 0.0;
        dc.col = j;
        if (j < ncols) {
            const double Ep = branch > 0 ? E[j] : -E[j];   // energy of the positive-branch state this column stands for
            on = (Ep > 0.0 && Ep < Ec) ? 1 : 0;
            if (on) {
                const double fm = fermi_dev(-Ep, T), fp = fermi_dev(Ep, T);
                if (branch > 0) { dc.wu = 2.0 * fp; dc.wv = 2.0 * fm; dc.wnu = fm - fp; }
                else            { dc.wu = 2.0 * fm; dc.wv = 2.0 * fp; dc.wnu = fp - fm; }
            }
        }
        // stable compaction of this batch of 1024 columns (ballot + block scan, no atomics)
        const unsigned m = __ballot_sync(0xffffffffu, on);
        if (lane == 0) warp_tot[wid] = __popc(m);
        __syncthreads();
        int before = 0, total = 0;
        for (int i = 0; i < DW_THREADS / 32; ++i) {
            const int t = warp_tot[i];
            if (i < wid) before += t;
            total += t;
        }
        if (on) act[base + before + __popc(m & ((1u << lane) - 1u))] = dc;
        __syncthreads();
        if (tid == 0) base += total;
        __syncthreads();
    }
    if (tid == 0) *nact = base;
}

constexpr int DP_THREADS = 128;
constexpr int DP_UNROLL = 8;

// part[(3*c + k) * M + r], k = 0: n, 1: Re nu, 2: Im nu, for chunk c of the active list.
__global__ void __launch_bounds__(DP_THREADS) dens_partial_kernel(const c128* __restrict__ Z, int64_t ldz, int64_t M,
                                                                   const DensCol* __restrict__ act,
                                                                   const int* __restrict__ nact_p,
                                                                   double* __restrict__ part) {
    const int64_t r = (int64_t)blockIdx.x * DP_THREADS + threadIdx.x;
    const int nchunks = gridDim.y, c = blockIdx.y;
    const int nact = *nact_p;
    const int len = (nact + nchunks - 1) / nchunks;
    const int a0 = min(c * len, nact), a1 = min(a0 + len, nact);
    if (r >= M) return;
    const c128* zu = Z + r;
    const c128* zv = Z + M + r;
    double n = 0.0, nr = 0.0, ni = 0.0;
    int a = a0;
    for (; a + DP_UNROLL <= a1; a += DP_UNROLL) {
        c128 u[DP_UNROLL], v[DP_UNROLL];
        DensCol dc[DP_UNROLL];
#pragma unroll
        for (int i = 0; i < DP_UNROLL; ++i) dc[i] = act[a + i];
#pragma unroll
        for (int i = 0; i < DP_UNROLL; ++i) {
            u[i] = __ldcs(zu + dc[i].col * ldz);
            v[i] = __ldcs(zv + dc[i].col * ldz);
        }
        asm volatile("" ::: "memory");   // keep the 16 streaming loads of the batch in flight together
#pragma unroll
        for (int i = 0; i < DP_UNROLL; ++i) {
            n = fma(dc[i].wu, cabs2(u[i]), n);
            n = fma(dc[i].wv, cabs2(v[i]), n);
            const c128 p = cmulc(v[i], u[i]);   // conj(v) u
            nr = fma(dc[i].wnu, p.x, nr);
            ni = fma(dc[i].wnu, p.y, ni);
        }
    }
    for (; a < a1; ++a) {
        const DensCol dc = act[a];
        const c128 u = __ldcs(zu + dc.col * ldz), v = __ldcs(zv + dc.col * ldz);
        n = fma(dc.wu, cabs2(u), n);
        n = fma(dc.wv, cabs2(v), n);
        const c128 p = cmulc(v, u);
        nr = fma(dc.wnu, p.x, nr);
        ni = fma(dc.wnu, p.y, ni);
    }
    part[((int64_t)3 * c + 0) * M + r] = n;
    part[((int64_t)3 * c + 1) * M + r] = nr;
    part[((int64_t)3 * c + 2) * M + r] = ni;
}

__global__ void dens_reduce_kernel(const double* __restrict__ part, int nchunks, int64_t M, double* __restrict__ n_out,
                                   c128* __restrict__ nu_out) {
    const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= M) return;
    double n = 0.0, nr = 0.0, ni = 0.0;
    for (int c = 0; c < nchunks; ++c) {
        n += part[((int64_t)3 * c + 0) * M + r];
        nr += part[((int64_t)3 * c + 1) * M + r];
        ni += part[((int64_t)3 * c + 2) * M + r];
    }
    n_out[r] = n;
    nu_out[r] = cmake(nr, ni);
}

// Workspace use (the split-K partial region, idle outside the GEMMs): the active list (ncols entries + its length), then
// the chunk partials.
int launch_densities(eigh_handle_s* h, const double* E, const c128* Z, int64_t ldz, int64_t ncols, double T, double Ec,
                     int branch, double* n_out, c128* nu_out, cudaStream_t s) {
    const int64_t M = h->N / 2;
    char* base = ws_ptr<char>(h, h->plan.gemm_partial);
    size_t off = 0;
    DensCol* act = (DensCol*)(base + off);
    off += (size_t)round_up(ncols * (int64_t)sizeof(DensCol) + 8, 256);
    int* nact = (int*)(base + off) - 2;
    if (off + (size_t)3 * M * sizeof(double) > h->plan.gemm_partial_bytes)
        return set_err(h, -5, "eigh_densities: %lld columns do not fit the workspace", (long long)ncols);
    double* part = (double*)(base + off);
    const int64_t max_chunks = (int64_t)((h->plan.gemm_partial_bytes - off) / ((size_t)3 * M * sizeof(double)));
    const int64_t row_blocks = ceil_div(M, DP_THREADS);
    // one wave: as many chunks as keep every thread block co-resident (a partial second wave would double the time)
    int occ = 0;
    EIGH_CUDA_OK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, dens_partial_kernel, DP_THREADS, 0));
    int64_t nchunks = std::max<int64_t>(1, (int64_t)h->num_sms * std::max(occ, 1) / row_blocks);
    nchunks = std::min(nchunks, ceil_div(std::max<int64_t>(ncols, 1), 2 * DP_UNROLL));
    nchunks = std::max<int64_t>(1, std::min(nchunks, std::min<int64_t>(max_chunks, 65535)));
    dens_weights_kernel<<<1, DW_THREADS, 0, s>>>(E, ncols, T, Ec, branch, act, nact);
    dens_partial_kernel<<<dim3((unsigned)row_blocks, (unsigned)nchunks), DP_THREADS, 0, s>>>(Z, ldz, M, act, nact, part);
    dens_reduce_kernel<<<(unsigned)ceil_div(M, 256), 256, 0, s>>>(part, (int)nchunks, M, n_out, nu_out);
    EIGH_CUDA_OK(cudaGetLastError());
    return 0;
}

}  // namespace eigh
