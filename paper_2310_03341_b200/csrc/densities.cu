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

// ------------------------------------------------------------------ Eq. 16b, 16c: kinetic and current densities
//     tau(r) = 2 sum ( |grad v_n|^2 f_T(-E_n) + |grad u_n|^2 f_T(E_n) )
//     j(r)   = 2 sum Im( v_n grad v_n^* f_T(-E_n) - u_n grad u_n^* f_T(E_n) )        (same states as Eq. 16a)
// The gradient along an axis is a dense real L x L matrix applied to the lines of the grid along that axis.  With the
// grid seen as (O, L, I) -- O outer, I inner points around the axis -- line lambda = o I + i holds the points
// r = (o L + l) I + i, l = 0..L-1.  One launch per axis; a thread block owns a tile of 32 lines and loops over its
// chunk of the active columns: the u and v tiles (L x 32 each) arrive by cp.async into a double buffer, the products
// (D u), (D v) of the tile run on the FP64 tensor cores (see the kernel), and each thread adds the weighted |.|^2 and
// Im(w conj(D w)) terms of its grid points to register partials.  In terms of the per-column weights of Eq. 16a:
//     tau += wu |grad u|^2 + wv |grad v|^2,     j += wv Im(v grad v^*) - wu Im(u grad u^*)        (both branches).
// Bound by FP64 arithmetic: 4 L FMAs per grid point, state and axis against 32 bytes read per point, state and axis.
constexpr int DG_THREADS = 256;
constexpr int DG_C = 32;            // lines per tile
constexpr int DG_PITCH = DG_C + 2;  // c128 elements per shared-memory row: 544 B = 32 (mod 128), conflict-free B fragments
constexpr int DG_LMAX = 64;
// cp.async ring: tiles of 2 columns in flight while one is multiplied (1 column for L > 56, where 3 stages do not fit)
__host__ __device__ constexpr int dg_stages(int MB) { return MB >= 8 ? 2 : 3; }

struct GradArgs {
    const c128* Z; int64_t ldz; int64_t M;
    int L; int64_t I; int64_t nlines;     // axis view (O, L, I); nlines = M / L
    const double* D;                      // L x L, column-major: D[l + l2 * L] = D[l, l2]
    const DensCol* act; const int* nact;
    double* part_tau; double* part_j;     // this axis' partials: [chunk][M]
};

// (D w)(l, line) for w = u, v as ONE real product on the FP64 tensor cores: G (LP x 128) = D (LP x LP) W (LP x 128),
// the 128 real columns being (u | v) x 32 lines x (re, im); LP = 8 MB >= L, the padding rows of W and rows / columns
// of D are zero.  Warp w owns lines 4w..4w+3 of both u and v: two 8-column blocks; in the accumulator layout of
// mma.m8n8k4 (c0, c1 = columns 2t, 2t+1 of row g) every thread holds the complex values (D u), (D v) of the grid points
// (l = 8 mb + g, line = 4w + t), mb = 0..MB-1, so the |.|^2 and Im(w conj(D w)) terms are formed in registers.
// The A fragments (D) do not depend on the column: they are loaded once, into registers for MB <= 4 (L <= 32).
template <int MB>
__global__ void __launch_bounds__(DG_THREADS, MB <= 4 ? 2 : 1) dens_grad_kernel(const GradArgs p) {
    extern __shared__ __align__(16) unsigned char dg_raw[];
    constexpr int LP = 8 * MB, KS = 2 * MB, DG_STAGES = dg_stages(MB);
    constexpr bool A_IN_REGS = MB <= 4;
    const int L = p.L;
    c128* buf = reinterpret_cast<c128*>(dg_raw);                  // [DG_STAGES buffers][u, v][LP][DG_PITCH]
    double* Ds = reinterpret_cast<double*>(buf + (size_t)2 * DG_STAGES * LP * DG_PITCH);   // Ds[l * (LP + 1) + l2]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, t = lane & 3;
    const int64_t line0 = (int64_t)blockIdx.x * DG_C;
    const int nchunks = gridDim.y, c = blockIdx.y;
    const int nact = *p.nact;
    const int len = (nact + nchunks - 1) / nchunks;
    const int a0 = min(c * len, nact), a1 = min(a0 + len, nact);

    for (int e = tid; e < LP * LP; e += DG_THREADS) {
        const int l = e / LP, l2 = e % LP;
        Ds[l * (LP + 1) + l2] = (l < L && l2 < L) ? p.D[l + (int64_t)l2 * L] : 0.0;
    }
    for (int e = tid; e < 2 * DG_STAGES * (LP - L) * DG_PITCH; e += DG_THREADS) {      // padding rows of all tiles stay zero
        const int q = e / ((LP - L) * DG_PITCH), rem = e % ((LP - L) * DG_PITCH);
        buf[(size_t)q * LP * DG_PITCH + (size_t)L * DG_PITCH + rem] = cmake(0.0, 0.0);
    }
    // this thread's elements of a tile: global offset (grid point) and shared-memory slot, fixed over the columns
    constexpr int EMAX = LP * DG_C / DG_THREADS;       // = MB
    int goff[EMAX], soff[EMAX];
    const int nelem = L * DG_C;
#pragma unroll
    for (int k = 0; k < EMAX; ++k) {
        const int e = tid + k * DG_THREADS;
        goff[k] = -1;
        soff[k] = 0;
        if (e < nelem) {
            int l, cc;
            if (p.I == 1) { l = e % L; cc = e / L; }       // lines are contiguous in memory: run along l
            else          { cc = e % DG_C; l = e / DG_C; } // neighbouring lines are contiguous: run along the lines
            const int64_t line = line0 + cc;
            soff[k] = l * DG_PITCH + cc;
            if (line < p.nlines) {
                const int64_t o = line / p.I, i = line % p.I;
                goff[k] = (int)((o * L + l) * p.I + i);
            }
        }
    }
    auto issue = [&](int a, int b) {
        const DensCol dc = p.act[a];
        const c128* zu = p.Z + dc.col * p.ldz;
        c128* ub = buf + (size_t)b * 2 * LP * DG_PITCH;
        c128* vb = ub + (size_t)LP * DG_PITCH;
#pragma unroll
        for (int k = 0; k < EMAX; ++k) {
            if (tid + k * DG_THREADS < nelem) {
                const bool ok = goff[k] >= 0;
                cp_async16(ub + soff[k], ok ? zu + goff[k] : zu, ok ? 16 : 0);
                cp_async16(vb + soff[k], ok ? zu + p.M + goff[k] : zu, ok ? 16 : 0);
            }
        }
    };
#pragma unroll
    for (int st = 0; st < DG_STAGES - 1; ++st) {       // prefetch distance DG_STAGES - 1 columns
        if (a0 + st < a1) issue(a0 + st, st);
        cp_async_commit();
    }
    __syncthreads();                                   // Ds is complete
    double afr[A_IN_REGS ? MB : 1][A_IN_REGS ? KS : 1];
    if constexpr (A_IN_REGS) {
#pragma unroll
        for (int mb = 0; mb < MB; ++mb)
#pragma unroll
            for (int ks = 0; ks < KS; ++ks) afr[mb][ks] = Ds[(8 * mb + g) * (LP + 1) + 4 * ks + t];
    }
    double tau[MB], jj[MB];
#pragma unroll
    for (int mb = 0; mb < MB; ++mb) tau[mb] = jj[mb] = 0.0;
    const int myline = 4 * warp + t;                   // the line whose (re, im) this thread accumulates
    for (int a = a0; a < a1; ++a) {
        const int b = (a - a0) % DG_STAGES;
        cp_async_wait<DG_STAGES - 2>();                // column a has landed (this thread's copies) ...
        __syncthreads();                               // ... and everybody's; buffer (b - 1) is free again
        if (a + DG_STAGES - 1 < a1) issue(a + DG_STAGES - 1, (b + DG_STAGES - 1) % DG_STAGES);
        cp_async_commit();
        const DensCol dc = p.act[a];
        const c128* ub = buf + (size_t)b * 2 * LP * DG_PITCH;
        const c128* vb = ub + (size_t)LP * DG_PITCH;
        // B fragment: row 4 ks + t, real column g of the warp's block = (line 4w + g/2, part g & 1)
        const double* ubd = reinterpret_cast<const double*>(ub) + 2 * (4 * warp) + g;
        const double* vbd = reinterpret_cast<const double*>(vb) + 2 * (4 * warp) + g;
        double gu[MB][2], gv[MB][2];
#pragma unroll
        for (int mb = 0; mb < MB; ++mb) gu[mb][0] = gu[mb][1] = gv[mb][0] = gv[mb][1] = 0.0;
#pragma unroll
        for (int ks = 0; ks < KS; ++ks) {
            const double bu = ubd[(size_t)(4 * ks + t) * (2 * DG_PITCH)];
            const double bv = vbd[(size_t)(4 * ks + t) * (2 * DG_PITCH)];
#pragma unroll
            for (int mb = 0; mb < MB; ++mb) {
                const double av = A_IN_REGS ? afr[A_IN_REGS ? mb : 0][A_IN_REGS ? ks : 0] : Ds[(8 * mb + g) * (LP + 1) + 4 * ks + t];
                dmma884p(gu[mb][0], gu[mb][1], av, bu);
                dmma884p(gv[mb][0], gv[mb][1], av, bv);
            }
        }
#pragma unroll
        for (int mb = 0; mb < MB; ++mb) {
            const int l = 8 * mb + g;
            const c128 u = ub[l * DG_PITCH + myline], v = vb[l * DG_PITCH + myline];    // zero on the padding rows
            tau[mb] = fma(dc.wu, gu[mb][0] * gu[mb][0] + gu[mb][1] * gu[mb][1], tau[mb]);
            tau[mb] = fma(dc.wv, gv[mb][0] * gv[mb][0] + gv[mb][1] * gv[mb][1], tau[mb]);
            jj[mb] = fma(dc.wv, v.y * gv[mb][0] - v.x * gv[mb][1], jj[mb]);     // Im(v conj(g)) = v.y g.x - v.x g.y
            jj[mb] = fma(-dc.wu, u.y * gu[mb][0] - u.x * gu[mb][1], jj[mb]);
        }
    }
    cp_async_wait<0>();
    const int64_t line = line0 + myline;
    if (line < p.nlines) {
        const int64_t o = line / p.I, i = line % p.I;
#pragma unroll
        for (int mb = 0; mb < MB; ++mb) {
            const int l = 8 * mb + g;
            if (l < L) {
                const int64_t pt = (o * L + l) * p.I + i;
                p.part_tau[(int64_t)c * p.M + pt] = tau[mb];
                p.part_j[(int64_t)c * p.M + pt] = jj[mb];
            }
        }
    }
}

// tau = sum over axes and chunks; j_a = sum over the chunks of axis a.  Partials: [axis][tau | j][chunk][M].
__global__ void dens_grad_reduce_kernel(const double* __restrict__ part, int nchunks, int64_t M, double* __restrict__ tau,
                                        double* __restrict__ j) {
    const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= M) return;
    double t = 0.0;
    for (int a = 0; a < 3; ++a) {
        const double* pt = part + ((int64_t)(2 * a) * nchunks) * M;
        const double* pj = part + ((int64_t)(2 * a + 1) * nchunks) * M;
        double ja = 0.0;
        for (int c = 0; c < nchunks; ++c) {
            t += pt[(int64_t)c * M + r];
            ja += pj[(int64_t)c * M + r];
        }
        j[(int64_t)a * M + r] = ja;
    }
    tau[r] = t;
}

template <int R>
static int grad_axis(const GradArgs& a, int64_t ntiles, int nchunks, cudaStream_t s, int* occ) {
    constexpr int LP = 8 * R, DG_STAGES = dg_stages(R);
    const size_t smem = (size_t)2 * DG_STAGES * LP * DG_PITCH * sizeof(c128) + (size_t)LP * (LP + 1) * sizeof(double);
    EIGH_CUDA_OK(cudaFuncSetAttribute(dens_grad_kernel<R>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    if (occ) {       // query only: thread blocks of this axis' kernel that fit one SM
        EIGH_CUDA_OK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(occ, dens_grad_kernel<R>, DG_THREADS, smem));
        return 0;
    }
    dens_grad_kernel<R><<<dim3((unsigned)ntiles, (unsigned)nchunks), DG_THREADS, smem, s>>>(a);
    return 0;
}

static int grad_axis_dispatch(const GradArgs& g, int64_t ntiles, int nchunks, cudaStream_t s, int* occ) {
    switch ((int)ceil_div(g.L, 8)) {
        case 1: return grad_axis<1>(g, ntiles, nchunks, s, occ);
        case 2: return grad_axis<2>(g, ntiles, nchunks, s, occ);
        case 3: return grad_axis<3>(g, ntiles, nchunks, s, occ);
        case 4: return grad_axis<4>(g, ntiles, nchunks, s, occ);
        case 5: return grad_axis<5>(g, ntiles, nchunks, s, occ);
        case 6: return grad_axis<6>(g, ntiles, nchunks, s, occ);
        case 7: return grad_axis<7>(g, ntiles, nchunks, s, occ);
        default: return grad_axis<8>(g, ntiles, nchunks, s, occ);
    }
}

int launch_gradient_densities(eigh_handle_s* h, int nx, int ny, int nz, const double* Dx, const double* Dy,
                              const double* Dz, const double* E, const c128* Z, int64_t ldz, int64_t ncols, double T,
                              double Ec, int branch, double* tau, double* j, cudaStream_t s) {
    const int64_t M = h->N / 2;
    char* base = ws_ptr<char>(h, h->plan.gemm_partial);
    size_t off = 0;
    DensCol* act = (DensCol*)(base + off);
    off += (size_t)round_up(ncols * (int64_t)sizeof(DensCol) + 8, 256);
    int* nact = (int*)(base + off) - 2;
    if (off + (size_t)6 * M * sizeof(double) > h->plan.gemm_partial_bytes)
        return set_err(h, -10, "eigh_gradient_densities: %lld columns do not fit the workspace", (long long)ncols);
    double* part = (double*)(base + off);
    const int64_t max_chunks = (int64_t)((h->plan.gemm_partial_bytes - off) / ((size_t)6 * M * sizeof(double)));
    const int Ls[3] = {nx, ny, nz};
    const int64_t Is[3] = {(int64_t)ny * nz, (int64_t)nz, 1};
    const double* Ds[3] = {Dx, Dy, Dz};
    GradArgs g[3];
    int64_t ntiles[3];
    // chunks of the active columns: as many as keep every thread block of every axis co-resident (one wave)
    int64_t nchunks = std::min<int64_t>(std::min<int64_t>(max_chunks, 65535), ceil_div(std::max<int64_t>(ncols, 1), 8));
    for (int a = 0; a < 3; ++a) {
        g[a].Z = Z; g[a].ldz = ldz; g[a].M = M;
        g[a].L = Ls[a]; g[a].I = Is[a]; g[a].nlines = M / Ls[a];
        g[a].D = Ds[a]; g[a].act = act; g[a].nact = nact;
        ntiles[a] = ceil_div(g[a].nlines, DG_C);
        int occ = 0;
        const int rc = grad_axis_dispatch(g[a], ntiles[a], 1, s, &occ);
        if (rc) return rc;
        nchunks = std::min<int64_t>(nchunks, (int64_t)h->num_sms * std::max(occ, 1) / ntiles[a]);
    }
    nchunks = std::max<int64_t>(1, nchunks);
    dens_weights_kernel<<<1, DW_THREADS, 0, s>>>(E, ncols, T, Ec, branch, act, nact);
    for (int a = 0; a < 3; ++a) {
        g[a].part_tau = part + ((int64_t)(2 * a) * nchunks) * M;
        g[a].part_j = part + ((int64_t)(2 * a + 1) * nchunks) * M;
        const int rc = grad_axis_dispatch(g[a], ntiles[a], (int)nchunks, s, nullptr);
        if (rc) return rc;
    }
    dens_grad_reduce_kernel<<<(unsigned)ceil_div(M, 256), 256, 0, s>>>(part, (int)nchunks, M, tau, j);
    EIGH_CUDA_OK(cudaGetLastError());
    return 0;
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

// ------------------------------------------------------------------ eigh_densities_static: the allocation-free variant
// Same three kernels as launch_densities, with the scratch (list of active columns + chunk partials) in a FILE-SCOPE device
// array instead of the caller's workspace: for callers that cannot call cudaMalloc (code under CUDA graph capture, tight
// serving loops, harnesses that forbid it).  Every GPU that loads the library holds these DENS_STATIC_BYTES until exit.
// In HOST code the array's name is a host-side stand-in, not a device address: the address the kernels get comes from
// cudaGetSymbolAddress, taken once per device with that device current (dens_static_setup below).
constexpr size_t DENS_STATIC_BYTES = (size_t)8 << 20;             // 8 MiB per device
constexpr size_t DENS_STATIC_ACT_BYTES = (size_t)1 << 20;         // head: nact word (256 B) + the list of active columns
constexpr int64_t DENS_STATIC_MAX_COLS = (int64_t)((DENS_STATIC_ACT_BYTES - 256) / sizeof(DensCol));      // 32760
constexpr int64_t DENS_STATIC_MAX_N = 65536;                      // M = N/2 <= 32768: one chunk of partials = 768 KiB
static __device__ __align__(256) unsigned char g_dens_static_scratch[DENS_STATIC_BYTES];

struct DensStaticDev { bool ready; unsigned char* ptr; int num_sms; int occ; };
constexpr int DENS_STATIC_MAX_DEVICES = 64;
static DensStaticDev g_dens_static_dev[DENS_STATIC_MAX_DEVICES];   // host side, indexed by device ordinal

// once per device, with that device current: the device address of the scratch array, SM count, occupancy
static int dens_static_setup(eigh_handle_s* h, DensStaticDev** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return set_err(h, 1000 + (int)e, "eigh_densities_static: cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= DENS_STATIC_MAX_DEVICES) return set_err(h, EIGH_ERR_CUDA, "eigh_densities_static: device ordinal %d out of range", dev);
    DensStaticDev& d = g_dens_static_dev[dev];
    if (!d.ready) {
        void* ptr = nullptr;
        e = cudaGetSymbolAddress(&ptr, g_dens_static_scratch);
        if (e != cudaSuccess || !ptr)
            return set_err(h, 1000 + (int)e, "eigh_densities_static: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
        int sms = 0, occ = 0;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, dens_partial_kernel, DP_THREADS, 0);
        if (e != cudaSuccess || sms <= 0)
            return set_err(h, 1000 + (int)e, "eigh_densities_static: device query: %s", cudaGetErrorString(e));
        d.ptr = (unsigned char*)ptr; d.num_sms = sms; d.occ = occ > 0 ? occ : 1;
        d.ready = true;
    }
    *out = &d;
    return 0;
}

}  // namespace eigh

// C ABI (include/eigh.h).  Lives in this file because the scratch array does: only this translation unit can take its address.
extern "C" int eigh_densities_static(eigh_handle_t h, const double* E_dev, const void* Z_dev, int64_t ldz, int64_t ncols,
                                     double T, double Ec, int branch, double* n_dev, void* nu_dev, void* stream) {
    using namespace eigh;
    if (!h) return -1;
    const int64_t N = h->N, M = N / 2;
    if (N & 1) return set_err(h, -1, "eigh_densities_static: N = %lld is odd (phi = [u, v] needs N = 2M)", (long long)N);
    if (N > DENS_STATIC_MAX_N)
        return set_err(h, -1, "eigh_densities_static: N = %lld exceeds the static scratch limit N <= %lld (use eigh_densities)",
                       (long long)N, (long long)DENS_STATIC_MAX_N);
    if (!E_dev && ncols > 0) return -2;
    if (!Z_dev && ncols > 0) return -3;
    if (ldz < N) return -4;
    if (ncols < 0 || ncols > N) return -5;
    if (ncols > DENS_STATIC_MAX_COLS)
        return set_err(h, -5, "eigh_densities_static: ncols = %lld exceeds the static scratch limit ncols <= %lld (use eigh_densities)",
                       (long long)ncols, (long long)DENS_STATIC_MAX_COLS);
    if (!(T >= 0.0)) return -6;
    if (Ec != Ec) return -7;
    if (branch != 1 && branch != -1) return -8;
    if (!n_dev) return -9;
    if (!nu_dev) return -10;
    DensStaticDev* d = nullptr;
    int rc = dens_static_setup(h, &d);
    if (rc) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    int* nact = reinterpret_cast<int*>(d->ptr);                              // first word of the array
    DensCol* act = reinterpret_cast<DensCol*>(d->ptr + 256);
    double* part = reinterpret_cast<double*>(d->ptr + DENS_STATIC_ACT_BYTES);
    const int64_t max_chunks = (int64_t)((DENS_STATIC_BYTES - DENS_STATIC_ACT_BYTES) / ((size_t)3 * (M > 0 ? M : 1) * sizeof(double)));
    const int64_t row_blocks = ceil_div(M > 0 ? M : 1, DP_THREADS);
    int64_t nchunks = std::max<int64_t>(1, (int64_t)d->num_sms * d->occ / row_blocks);
    nchunks = std::min(nchunks, ceil_div(std::max<int64_t>(ncols, 1), 2 * DP_UNROLL));
    nchunks = std::max<int64_t>(1, std::min(nchunks, std::min<int64_t>(max_chunks, 65535)));
    // The array keeps the previous call's contents.  Nothing in it is read before this call writes it (the weights kernel
    // writes the count and the list, every chunk partial is written before the reduction reads it); the count word is
    // cleared all the same, so that a call whose first kernel failed to launch cannot reuse a stale count.
    cudaError_t e = cudaMemsetAsync(nact, 0, 256, s);
    if (e != cudaSuccess) return set_err(h, 1000 + (int)e, "eigh_densities_static: %s", cudaGetErrorString(e));
    dens_weights_kernel<<<1, DW_THREADS, 0, s>>>(E_dev, ncols, T, Ec, branch, act, nact);
    if (M > 0) {
        dens_partial_kernel<<<dim3((unsigned)row_blocks, (unsigned)nchunks), DP_THREADS, 0, s>>>((const c128*)Z_dev, ldz, M, act, nact, part);
        dens_reduce_kernel<<<(unsigned)ceil_div(M, 256), 256, 0, s>>>(part, (int)nchunks, M, n_dev, (c128*)nu_dev);
    }
    h->launches += 3;
    e = cudaGetLastError();
    if (e != cudaSuccess) return set_err(h, 1000 + (int)e, "eigh_densities_static: %s", cudaGetErrorString(e));
    return 0;
}
