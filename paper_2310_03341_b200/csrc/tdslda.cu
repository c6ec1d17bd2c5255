// tdslda.cu -- one TDSLDA time step for the quasiparticle states just computed.
//
// PAPER.md:91 Eq. (5):  i d/dt [u_n, v_n]^T = [[h, Delta], [Delta^*, -h^*]] [u_n, v_n]^T  (hbar = 1), the same Hamiltonian for
// every state; Eq. (8): the kinetic term is applied spectrally; 5th-order
// Adams-Bashforth-Moulton predictor-corrector, h and Delta evaluated twice per step, densities reduced from the states.
//
//   f = -i H phi   with  h = -1/2 lap + V - mu  (real local potential; toy functional Delta = g nu, reading 11)
//
// Kinetic term: Eq. 8's F^-1 (k^2/2) F is, per axis, a dense real symmetric L x L matrix K_L (the caller passes the
// same matrices eigh_assemble_bdg takes), so -1/2 lap = Kx (x) I (x) I + I (x) Ky (x) I + I (x) I (x) Kz is three small
// dense contractions per state: FP64 tensor-core products (mma.sync m8n8k4, DMMA) over tiles of 32 grid lines, exactly the
// scheme of eigh_gradient_densities.  With L = 24..32 that is 4 L FMAs per point and axis against 16-48 bytes of traffic:
// the three passes are HBM-bound (8 x 16 N bytes per state and evaluation: phi read 3 times, f written 3 times, read
// twice).  The last pass fuses everything local: (V - mu) phi, the Delta coupling and the factor -i.
//   kin_axis_kernel<MB, 0>   f  = K_a phi                          (first axis)
//   kin_axis_kernel<MB, 1>   f += K_a phi                          (second axis)
//   kin_axis_kernel<MB, 2>   f  = -i [ (f + K_a phi) + local ]     (third axis; sign -1 and conj(Delta) for the v half)
//   abm_combine_kernel       y_out = y + dt sum_k c_k f_k          (predictor: AB5; corrector: AM4) -- pure streaming
#include <algorithm>

#include "eigh_internal.h"

namespace eigh {

constexpr int TK_THREADS = 256;
constexpr int TK_C = 32;             // lines per tile
constexpr int TK_PITCH = TK_C + 2;   // c128 per shared-memory row (conflict-free B fragments)
__host__ __device__ constexpr int tk_stages(int MB) { return MB >= 8 ? 2 : 3; }

struct KinArgs {
    const c128* Phi; int64_t ldp;    // states, column j at Phi + j ldp: rows [0, M) = u, [M, 2M) = v
    c128* F; int64_t ldf;            // output, same layout
    int64_t M; int ncols;
    int L; int64_t I; int64_t nlines;   // axis view (O, L, I)
    const double* K;                 // L x L real symmetric, K[l + l2 L]
    const double* V; const c128* Delta; double mu;   // used by MODE 2
};

template <int MB, int MODE>
__global__ void __launch_bounds__(TK_THREADS, MB <= 4 ? 2 : 1) kin_axis_kernel(const KinArgs p) {
    extern __shared__ __align__(16) unsigned char tk_raw[];
    constexpr int LP = 8 * MB, KS = 2 * MB, STAGES = tk_stages(MB);
    constexpr bool A_IN_REGS = MB <= 3;      // (MB = 4 with the fragments in registers spills at two blocks per SM)
    const int L = p.L;
    c128* buf = reinterpret_cast<c128*>(tk_raw);                  // [STAGES][u, v][LP][TK_PITCH]
    double* Ks = reinterpret_cast<double*>(buf + (size_t)2 * STAGES * LP * TK_PITCH);   // Ks[l * (LP + 1) + l2]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, t = lane & 3;
    const int64_t line0 = (int64_t)blockIdx.x * TK_C;
    const int nchunks = gridDim.y, c = blockIdx.y;
    const int len = (p.ncols + nchunks - 1) / nchunks;
    const int a0 = min(c * len, p.ncols), a1 = min(a0 + len, p.ncols);

    for (int e = tid; e < LP * LP; e += TK_THREADS) {
        const int l = e / LP, l2 = e % LP;
        Ks[l * (LP + 1) + l2] = (l < L && l2 < L) ? p.K[l + (int64_t)l2 * L] : 0.0;
    }
    for (int e = tid; e < 2 * STAGES * (LP - L) * TK_PITCH; e += TK_THREADS) {        // padding rows stay zero
        const int q = e / ((LP - L) * TK_PITCH), rem = e % ((LP - L) * TK_PITCH);
        buf[(size_t)q * LP * TK_PITCH + (size_t)L * TK_PITCH + rem] = cmake(0.0, 0.0);
    }
    constexpr int EMAX = LP * TK_C / TK_THREADS;       // = MB
    int goff[EMAX], soff[EMAX];
    const int nelem = L * TK_C;
#pragma unroll
    for (int k = 0; k < EMAX; ++k) {
        const int e = tid + k * TK_THREADS;
        goff[k] = -1;
        soff[k] = 0;
        if (e < nelem) {
            int l, cc;
            if (p.I == 1) { l = e % L; cc = e / L; } else { cc = e % TK_C; l = e / TK_C; }
            const int64_t line = line0 + cc;
            soff[k] = l * TK_PITCH + cc;
            if (line < p.nlines) {
                const int64_t o = line / p.I, i = line % p.I;
                goff[k] = (int)((o * L + l) * p.I + i);
            }
        }
    }
    auto issue = [&](int a, int b) {
        const c128* zu = p.Phi + (int64_t)a * p.ldp;
        c128* ub = buf + (size_t)b * 2 * LP * TK_PITCH;
        c128* vb = ub + (size_t)LP * TK_PITCH;
#pragma unroll
        for (int k = 0; k < EMAX; ++k) {
            if (tid + k * TK_THREADS < nelem) {
                const bool ok = goff[k] >= 0;
                cp_async16(ub + soff[k], ok ? zu + goff[k] : zu, ok ? 16 : 0);
                cp_async16(vb + soff[k], ok ? zu + p.M + goff[k] : zu, ok ? 16 : 0);
            }
        }
    };
#pragma unroll
    for (int st = 0; st < STAGES - 1; ++st) {
        if (a0 + st < a1) issue(a0 + st, st);
        cp_async_commit();
    }
    __syncthreads();
    double afr[A_IN_REGS ? MB : 1][A_IN_REGS ? KS : 1];
    if constexpr (A_IN_REGS) {
#pragma unroll
        for (int mb = 0; mb < MB; ++mb)
#pragma unroll
            for (int ks = 0; ks < KS; ++ks) afr[mb][ks] = Ks[(8 * mb + g) * (LP + 1) + 4 * ks + t];
    }
    const int myline = 4 * warp + t;
    const int64_t line = line0 + myline;
    const bool line_ok = line < p.nlines;
    const int64_t lo = line_ok ? line / p.I : 0, li = line_ok ? line % p.I : 0;
    for (int a = a0; a < a1; ++a) {
        const int b = (a - a0) % STAGES;
        cp_async_wait<STAGES - 2>();
        __syncthreads();
        if (a + STAGES - 1 < a1) issue(a + STAGES - 1, (b + STAGES - 1) % STAGES);
        cp_async_commit();
        const c128* ub = buf + (size_t)b * 2 * LP * TK_PITCH;
        const c128* vb = ub + (size_t)LP * TK_PITCH;
        const double* ubd = reinterpret_cast<const double*>(ub) + 2 * (4 * warp) + g;
        const double* vbd = reinterpret_cast<const double*>(vb) + 2 * (4 * warp) + g;
        double gu[MB][2], gv[MB][2];
#pragma unroll
        for (int mb = 0; mb < MB; ++mb) gu[mb][0] = gu[mb][1] = gv[mb][0] = gv[mb][1] = 0.0;
#pragma unroll
        for (int ks = 0; ks < KS; ++ks) {
            const double bu = ubd[(size_t)(4 * ks + t) * (2 * TK_PITCH)];
            const double bv = vbd[(size_t)(4 * ks + t) * (2 * TK_PITCH)];
#pragma unroll
            for (int mb = 0; mb < MB; ++mb) {
                const double av = A_IN_REGS ? afr[A_IN_REGS ? mb : 0][A_IN_REGS ? ks : 0] : Ks[(8 * mb + g) * (LP + 1) + 4 * ks + t];
                dmma884p(gu[mb][0], gu[mb][1], av, bu);
                dmma884p(gv[mb][0], gv[mb][1], av, bv);
            }
        }
        if (line_ok) {
            c128* fu = p.F + (int64_t)a * p.ldf;
            c128* fv = fu + p.M;
#pragma unroll
            for (int mb = 0; mb < MB; ++mb) {
                const int l = 8 * mb + g;
                if (l < L) {
                    const int64_t pt = (lo * L + l) * p.I + li;
                    c128 tu = cmake(gu[mb][0], gu[mb][1]), tv = cmake(gv[mb][0], gv[mb][1]);
                    if (MODE >= 1) { tu = cadd(tu, fu[pt]); tv = cadd(tv, fv[pt]); }
                    if (MODE == 2) {
                        const c128 u = ub[l * TK_PITCH + myline], v = vb[l * TK_PITCH + myline];
                        const double w = p.V[pt] - p.mu;
                        const c128 dl = p.Delta[pt];
                        const c128 hu = cadd(cadd(tu, cscale(w, u)), cmul(dl, v));          // h u + Delta v
                        const c128 hv = csub(cmulc(dl, u), cadd(tv, cscale(w, v)));         // Delta^* u - h v
                        tu = cmake(hu.y, -hu.x);                                            // -i (.)
                        tv = cmake(hv.y, -hv.x);
                    }
                    fu[pt] = tu;
                    fv[pt] = tv;
                }
            }
        }
    }
    cp_async_wait<0>();
}

// y_out = y + dt sum_{k < nk} c_k f_k, element-wise over n c128 values per column (columns at strides ldy / ldf)
struct CombArgs {
    const c128* y; c128* out; int64_t ldy;
    const c128* f[5]; int64_t ldf;
    double c[5]; int nk;
    int64_t n; int ncols;
};
__global__ void __launch_bounds__(256) abm_combine_kernel(const CombArgs p) {
    const int col = blockIdx.y;
    const int64_t off_y = (int64_t)col * p.ldy, off_f = (int64_t)col * p.ldf;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < p.n; i += (int64_t)gridDim.x * blockDim.x) {
        c128 acc = __ldcs(p.y + off_y + i);
#pragma unroll
        for (int k = 0; k < 5; ++k)
            if (k < p.nk) {
                const c128 f = __ldcs(p.f[k] + off_f + i);
                acc.x = fma(p.c[k], f.x, acc.x);
                acc.y = fma(p.c[k], f.y, acc.y);
            }
        p.out[off_y + i] = acc;
    }
}

__global__ void scale_field_kernel(const c128* __restrict__ nu, double g, int64_t M, c128* __restrict__ Delta) {
    const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r < M) Delta[r] = cscale(g, nu[r]);
}

// ------------------------------------------------------------------ host side
template <int MB, int MODE>
static int kin_launch(const KinArgs& a, int num_sms, cudaStream_t s, int64_t* launches) {
    constexpr int LP = 8 * MB;
    const size_t smem = (size_t)2 * tk_stages(MB) * LP * TK_PITCH * sizeof(c128) + (size_t)LP * (LP + 1) * sizeof(double);
    auto kern = kin_axis_kernel<MB, MODE>;
    EIGH_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 0;
    EIGH_CUDA_OK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, TK_THREADS, smem));
    const int64_t ntiles = ceil_div(a.nlines, TK_C);
    // chunks of the columns: about four waves of thread blocks, at least 4 columns per block (the cp.async ring)
    int64_t nchunks = ceil_div((int64_t)4 * num_sms * std::max(occ, 1), ntiles);
    nchunks = std::min<int64_t>(nchunks, ceil_div(std::max(a.ncols, 1), 4));
    nchunks = std::max<int64_t>(1, std::min<int64_t>(nchunks, 65535));
    kern<<<dim3((unsigned)ntiles, (unsigned)nchunks), TK_THREADS, smem, s>>>(a);
    if (launches) ++*launches;
    EIGH_CUDA_OK(cudaGetLastError());
    return 0;
}

template <int MODE>
static int kin_dispatch(const KinArgs& a, int num_sms, cudaStream_t s, int64_t* launches) {
    switch ((int)ceil_div(a.L, 8)) {
        case 1: return kin_launch<1, MODE>(a, num_sms, s, launches);
        case 2: return kin_launch<2, MODE>(a, num_sms, s, launches);
        case 3: return kin_launch<3, MODE>(a, num_sms, s, launches);
        case 4: return kin_launch<4, MODE>(a, num_sms, s, launches);
        case 5: return kin_launch<5, MODE>(a, num_sms, s, launches);
        case 6: return kin_launch<6, MODE>(a, num_sms, s, launches);
        case 7: return kin_launch<7, MODE>(a, num_sms, s, launches);
        default: return kin_launch<8, MODE>(a, num_sms, s, launches);
    }
}

// F = -i H(V, Delta) Phi for ncols states (three launches)
int launch_tdslda_rhs(eigh_handle_s* h, int nx, int ny, int nz, const double* Kx, const double* Ky, const double* Kz,
                      const double* V, const c128* Delta, double mu, const c128* Phi, int64_t ldp, int64_t ncols, c128* F,
                      int64_t ldf, cudaStream_t s) {
    if (ncols <= 0) return 0;
    const int64_t M = h->N / 2;
    const int Ls[3] = {nx, ny, nz};
    const int64_t Is[3] = {(int64_t)ny * nz, (int64_t)nz, 1};
    const double* Ks[3] = {Kx, Ky, Kz};
    for (int ax = 0; ax < 3; ++ax) {
        KinArgs a;
        a.Phi = Phi; a.ldp = ldp; a.F = F; a.ldf = ldf; a.M = M; a.ncols = (int)ncols;
        a.L = Ls[ax]; a.I = Is[ax]; a.nlines = M / Ls[ax]; a.K = Ks[ax];
        a.V = V; a.Delta = Delta; a.mu = mu;
        int rc;
        if (ax == 0) rc = kin_dispatch<0>(a, h->num_sms, s, &h->launches);
        else if (ax == 1) rc = kin_dispatch<1>(a, h->num_sms, s, &h->launches);
        else rc = kin_dispatch<2>(a, h->num_sms, s, &h->launches);
        if (rc) return rc;
    }
    return 0;
}

static int abm_combine(eigh_handle_s* h, const c128* y, c128* out, int64_t ldy, c128* const* f, const int* idx, const double* c,
                       int nk, int64_t ldf, int64_t n, int64_t ncols, cudaStream_t s) {
    CombArgs a;
    a.y = y; a.out = out; a.ldy = ldy; a.ldf = ldf; a.nk = nk; a.n = n; a.ncols = (int)ncols;
    for (int k = 0; k < 5; ++k) { a.f[k] = k < nk ? f[idx[k]] : nullptr; a.c[k] = k < nk ? c[k] : 0.0; }
    const unsigned gx = (unsigned)std::min<int64_t>(ceil_div(n, 256), 64);
    abm_combine_kernel<<<dim3(gx, (unsigned)ncols), 256, 0, s>>>(a);
    ++h->launches;
    EIGH_CUDA_OK(cudaGetLastError());
    return 0;
}

// One PECE step of the 5th-order Adams-Bashforth-Moulton pair.  F[0..4] = f_n, f_{n-1}, ..., f_{n-4} on
// entry; on return Y holds y_{n+1} and the buffer of f_{n-4} holds f_{n+1} (the caller rotates its pointers).
int launch_tdslda_step(eigh_handle_s* h, int nx, int ny, int nz, const double* Kx, const double* Ky, const double* Kz,
                       const double* V, double g, double mu, const double* E0, double T, double Ec, int branch, double dt,
                       c128* Y, int64_t ldy, c128* const F[5], int64_t ldf, c128* Yp, int64_t ncols, double* n_out,
                       c128* Delta, cudaStream_t s) {
    const int64_t N = h->N, M = N / 2;
    static const double AB5[5] = {1901.0 / 720.0, -2774.0 / 720.0, 2616.0 / 720.0, -1274.0 / 720.0, 251.0 / 720.0};
    static const double AM4[5] = {251.0 / 720.0, 646.0 / 720.0, -264.0 / 720.0, 106.0 / 720.0, -19.0 / 720.0};
    double c[5];
    int rc;
    // P: y_p = y_n + dt sum AB5_k f_{n-k}
    { const int idx[5] = {0, 1, 2, 3, 4};
      for (int k = 0; k < 5; ++k) c[k] = dt * AB5[k];
      rc = abm_combine(h, Y, Yp, ldy, F, idx, c, 5, ldf, N, ncols, s); if (rc) return rc; }
    // E: fields of the predicted state, f_p = -i H y_p  (into the buffer of f_{n-4}, which the corrector does not use)
    rc = launch_densities(h, E0, Yp, ldy, ncols, T, Ec, branch, n_out, Delta, s); if (rc) return rc;
    h->launches += 3;
    scale_field_kernel<<<(unsigned)ceil_div(M, 256), 256, 0, s>>>(Delta, g, M, Delta);
    ++h->launches;
    rc = launch_tdslda_rhs(h, nx, ny, nz, Kx, Ky, Kz, V, Delta, mu, Yp, ldy, ncols, F[4], ldf, s); if (rc) return rc;
    // C: y_{n+1} = y_n + dt (AM4_0 f_p + sum_{k >= 1} AM4_k f_{n-k+1})
    { const int idx[5] = {4, 0, 1, 2, 3};
      for (int k = 0; k < 5; ++k) c[k] = dt * AM4[k];
      rc = abm_combine(h, Y, Y, ldy, F, idx, c, 5, ldf, N, ncols, s); if (rc) return rc; }
    // E: fields of the corrected state, f_{n+1} = -i H y_{n+1}
    rc = launch_densities(h, E0, Y, ldy, ncols, T, Ec, branch, n_out, Delta, s); if (rc) return rc;
    h->launches += 3;
    scale_field_kernel<<<(unsigned)ceil_div(M, 256), 256, 0, s>>>(Delta, g, M, Delta);
    ++h->launches;
    rc = launch_tdslda_rhs(h, nx, ny, nz, Kx, Ky, Kz, V, Delta, mu, Y, ldy, ncols, F[4], ldf, s); if (rc) return rc;
    const cudaError_t ce = cudaGetLastError();
    return ce != cudaSuccess ? 1000 + (int)ce : 0;
}

}  // namespace eigh
