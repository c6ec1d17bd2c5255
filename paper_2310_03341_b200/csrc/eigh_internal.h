// eigh_internal.h -- handle, workspace plan and phase drivers (host side) of b200-eigh.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include "../../include/eigh.h"
#include "common.cuh"

namespace eigh {

// Byte offsets of the regions inside the caller-provided workspace (all 256-byte aligned).
struct WsPlan {
    size_t gemm_partial, gemm_partial_bytes;   // split-K partial sums
    size_t band;                               // ldab x N c128 band storage
    size_t tau1;                               // N c128: stage-1 taus
    size_t T1;                                 // npanels x b x b c128: stage-1 compact-WY T factors
    size_t Vp, VT, X;                          // (N x b) c128 panel temporaries (Vp = explicit V)
    size_t small;                              // b x b c128 scratch (Gram, S) x 4
    size_t panel_sync;                         // cooperative panel kernel: counters + partial dots
    size_t V2;                                 // stage-2 reflectors, tile-major: [(pass, k) stage][32 sweeps][64] c128
    size_t pass_off;                           // int64[npass + 1]: first stage of every pass of 32 sweeps
    size_t tau2;                               // stage-2 taus, N x kmax c128 (kmax = bc_kmax)
    size_t bc_progress;                        // bulge chasing progress counters (N int32)
    size_t d, e, sgn;                          // tridiagonal (N doubles each) and row signs
    size_t dc;                                 // D&C arena
    size_t dc_bytes;
    size_t Qt;                                 // D&C result N x nev real (lives inside dc arena)
    size_t btQ;                                // S4a: q = Re v - Im v of the stage-2 reflectors (after btT when the dead D&C buffers hold both)
    size_t btT;                                // S4a: -T factors of all (pass, k) steps (aliases the dead D&C Q buffers)
    size_t bt;                                 // back-transform scratch (S4b's Y, S4a's counters)
    size_t bt_bytes;
    size_t b4V, b4VT, b4Y, b4T, b4G;           // S4b merged-panel WY blocks: V, V T^H (N x kb), Y (kb x nev), T, G (kb x kb)
    size_t ht_part;                            // 1-stage variant: per-tile partial products and per-row-block partials
    size_t total;
};
}  // namespace eigh

struct eigh_handle_s {
    int64_t N, nev;
    int b;          // band width
    int g;          // WY group size for S4a
    int leaf;       // D&C leaf size
    int p4b_merge;  // panels per WY block in S4b
    int gemm_3m;         // complex GEMMs by the 3M method (1) or with four real products (0)
    int panel_smem;      // S1.1: shared-memory resident panel QR (1) or the L2-resident one (0)
    int panel_rows_min;  // S1.1: fewest panel rows per thread block of the resident kernel
    int hemm_waves;      // S1.3: split-K of HEMM-lower chosen for about this many thread blocks per SM
    int bt_chain;   // S4a: consecutive passes of one slab scheduled back to back (0 = auto)
    int bc_grid;    // S2: CTAs of the bulge-chasing kernel (0 = all that are co-resident)
    int bc_variant;     // S2: 0 = publisher-warp kernel (default), 2 = no publisher warp, full register file
    int bc_dual_steps;  // S2: sweeps with at least this many chase steps run two thread blocks per SM (0 = never)
    int col0;       // first eigenvector column this handle returns (column shard of the back-transformations; default 0)
    int method;     // 2 = two-stage (default), 1 = one-stage direct tridiagonalisation
    int real_dtype; // 0 = complex Hermitian (c128), 1 = real symmetric (double); real needs method = 1
    int ht_grid;    // 1-stage: thread blocks of the panel kernel (0 = all that are co-resident)
    int64_t ldab;   // band storage leading dimension
    void* ws;
    size_t ws_bytes;
    eigh::WsPlan plan;
    bool planned;
    char err[512];
    double phase_ms[5];
    int64_t launches;
    cudaEvent_t ev[6];
    cudaEvent_t ev_sweep[2];   // brackets of the bt_sweep_kernel launch (S4a's dominant kernel)
    double sweep_ms;
    bool events_ok;
    int num_sms;
    // statistics of the last S3 run, per merge level (eigh_dc_stats)
    int dc_levels;
    double dc_flops[32], dc_ksum[32], dc_nsum[32];
    // eigh_solve_host: bounded pinned staging ring (2 buffers) + its events and copy stream, allocated on first use
    void* stage[2];
    size_t stage_bytes;
    cudaEvent_t ev_stage[2];
    cudaStream_t copy_stream;
    bool stage_ok;
};

namespace eigh {

void plan_workspace(eigh_handle_s* h);
template <typename T>
static inline T* ws_ptr(eigh_handle_s* h, size_t off) { return reinterpret_cast<T*>((char*)h->ws + off); }

int set_err(eigh_handle_s* h, int code, const char* fmt, ...);

// steps per bulge-chasing sweep (upper bound over sweeps): reflector (j, k) starts at row j+1+k*b
static inline int64_t bc_kmax(const eigh_handle_s* h) {
    const int64_t k = (h->N - 1 + h->b - 1) / h->b;
    return k < 1 ? 1 : k;
}

// Stage-2 reflector storage.  Sweeps are grouped into passes of 32; (pass p, step k) is one stage of 32
// reflectors x 64 elements, zero padded, stored contiguously (so that S4a fetches a stage with ONE bulk copy):
//   v_{j,k}[i]  at  V2[((pass_off[j / 32] + k) * 32 + j % 32) * 64 + i],   pass p has ceil((N-1-32p)/64) stages.
static inline int64_t v2_npass(int64_t N) { return N >= 2 ? (N - 1 + 31) / 32 : 0; }
static inline int64_t v2_pass_stages(int64_t N, int64_t p) { return (N - 1 - 32 * p + 63) / 64; }
static inline int64_t v2_total_stages(int64_t N) {
    int64_t st = 0;
    for (int64_t p = 0; p < v2_npass(N); ++p) st += v2_pass_stages(N, p);
    return st;
}
int launch_pass_off(eigh_handle_s* h, cudaStream_t s);   // fills plan.pass_off (bt_band.cu)

// phase drivers (each enqueues on `s`; returns 0 or an error code)
int phase_reduce_to_band(eigh_handle_s* h, c128* A, int64_t lda, c128* band, int64_t ldab, cudaStream_t s);
int phase_band_to_tridiag(eigh_handle_s* h, c128* band, int64_t ldab, double* d, double* e, cudaStream_t s);
int phase_tridiag_dc(eigh_handle_s* h, const double* d, const double* e, double* W, double* Q, int64_t ldq,
                     cudaStream_t s, int* nfail);
int phase_backtransform_band(eigh_handle_s* h, const double* Q, int64_t ldq, c128* Z, int64_t ldz,
                             cudaStream_t s);
int phase_backtransform_full(eigh_handle_s* h, const c128* A, int64_t lda, c128* Z, int64_t ldz,
                             cudaStream_t s);
// one TDSLDA step (tdslda.cu)
int launch_tdslda_rhs(eigh_handle_s* h, int nx, int ny, int nz, const double* Kx, const double* Ky, const double* Kz,
                      const double* V, const c128* Delta, double mu, const c128* Phi, int64_t ldp, int64_t ncols, c128* F,
                      int64_t ldf, cudaStream_t s);
int launch_tdslda_step(eigh_handle_s* h, int nx, int ny, int nz, const double* Kx, const double* Ky, const double* Kz,
                       const double* V, double g, double mu, const double* E0, double T, double Ec, int branch, double dt,
                       c128* Y, int64_t ldy, c128* const F[5], int64_t ldf, c128* Yp, int64_t ncols, double* n_out,
                       c128* Delta, cudaStream_t s);
// 1-stage variant (tridiag_direct.cu); A / Z are c128 or double according to h->real_dtype
int phase_tridiagonalise_direct(eigh_handle_s* h, void* A, int64_t lda, double* d, double* e, cudaStream_t s);
int phase_backtransform_direct(eigh_handle_s* h, const void* A, int64_t lda, const double* Q, int64_t ldq, void* Z,
                               int64_t ldz, cudaStream_t s);
size_t ht_partial_bytes(int64_t N);
// SCF epilogue (densities.cu): n(r), nu(r) of Eq. 16a / 16d from the columns of Z
int launch_densities(eigh_handle_s* h, const double* E, const c128* Z, int64_t ldz, int64_t ncols, double T, double Ec,
                     int branch, double* n_out, c128* nu_out, cudaStream_t s);
int launch_gradient_densities(eigh_handle_s* h, int nx, int ny, int nz, const double* Dx, const double* Dy,
                              const double* Dz, const double* E, const c128* Z, int64_t ldz, int64_t ncols, double T,
                              double Ec, int branch, double* tau, double* j, cudaStream_t s);

}  // namespace eigh
