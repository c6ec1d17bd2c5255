/* eigh.h -- C ABI of b200-eigh: dense complex-FP64 Hermitian eigensolver for one B200 (sm_100a).
 *
 * The operation is the Hermitian eigenproblem of the paper's Eq. 7:
 * find real E_0 <= ... <= E_{N-1} and an orthonormal set phi_n with  H phi_n = E_n phi_n,
 * for the dense BdG/HFB Hamiltonian H ("dense diagonalization").  The method
 * is the 2-stage solver outlined in PAPER.md:148-154: dense -> band -> tridiagonal,
 * tridiagonal eigensolve, and a two-stage back-transformation of the eigenvectors.
 * Everything below the five named steps is this library's own design.
 *
 * Conventions
 *   - All pointers named *_dev are DEVICE pointers; everything else is host memory.
 *   - Matrices are column-major; complex elements are interleaved (re, im) FP64 pairs
 *     ("c128", 16 bytes); leading dimensions are in ELEMENTS.
 *   - `stream` is a cudaStream_t passed as void* (0 = default stream).  Calls enqueue work
 *     on that stream only and may synchronise it (documented per call).
 *   - Return value: 0 success; -k = k-th argument invalid (nothing launched);
 *     +k = numerical failure count reported after completion (secular iterations that did not
 *     converge; capped at 999, eigh_last_error has the count -- non-finite input ends here, it
 *     never hangs); EIGH_ERR_CUDA (= 1000 + cudaError_t) on a CUDA runtime error.
 *     eigh_last_error(h) gives a text description.
 *   - Ownership: the caller owns A, W, Z and the workspace (e.g. torch tensors); the handle
 *     owns only host-side plan data and a few CUDA events.  One handle per host thread.
 *   - There is NO CPU fallback anywhere in this library.
 */
#ifndef EIGH_B200_H
#define EIGH_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define EIGH_ERR_CUDA 1000

typedef struct eigh_handle_s* eigh_handle_t;

/* Plan a solve of order N returning the LOWEST nev eigenpairs (1 <= nev <= N; "all or the
 * lowest nev", PAPER.md:119-127 keeps only part of the spectrum).  No device allocation.
 * Defaults: band width b = 64, D&C leaf 32, WY group g = 8. */
int eigh_create(eigh_handle_t* h, int64_t N, int64_t nev);

/* Tuning knobs.  Keys: "wy_group" (reflectors per compact-WY block of S4a: 8, 16 or 32), "dc_leaf" (8..32),
 * "p4b_merge" (1..8 panels of S1 merged into one compact-WY block of S4b; default 4),
 * "gemm_3m" (1 = complex GEMMs of S1 / S4b by the 3M method, three real tensor-core products per complex
 * multiply-add, the default; 0 = four products.  The switch is process-wide: handles used concurrently must agree),
 * "panel_smem" (S1.1: 1 = shared-memory resident panel QR with the T factor built in, 0 = L2-resident panel QR + Gram
 * GEMM + T recurrence), "panel_rows_min" (16..192 panel rows per thread block of the resident kernel),
 * "hemm_waves" (S1.3: split-K of HEMM-lower sized for about this many thread blocks per SM; default 14),
 * "bt_chain" (S4a: consecutive passes of one column slab scheduled back to back so that followers read from L2;
 * 0 = automatic = 1, the unchained order), "bc_grid" (thread blocks of the S2 bulge-chasing kernel; 0 = every
 * co-resident block, the default), "dgemm_mi" (real GEMM of the S3 merges: 8 = 64 x 32 warp tiles, 4 warps per
 * thread block, the default; 4 = 32 x 32 warp tiles, 8 warps; process-wide like gemm_3m; identical results), "bc_variant" (S2 kernel: 3 = publisher warp + register reallocation (setmaxnreg: the compute warps
 * get 232 registers, no spills), the default; 2 = no publisher warp, full register file; 0 = publisher warp at 168 registers,
 * the round-1 kernel; all three give bit-identical results), "bc_dual_steps" (S2: sweeps with at least this many chase steps run on the variant
 * with two thread blocks per SM and no publisher warp; 0 = never, the default -- it measured 2-8 % slower at N = 27648 /
 * 49152, the kernel being bound by L2 traffic rather than by occupancy), "band_width" (64: the only width S2 / S4a are built for; anything else is -3),
 * "col_begin" (first eigenvector column returned: Z gets the eigenvectors of W[col_begin .. col_begin + nev) instead of
 * W[0 .. nev); W still holds all N eigenvalues.  This is the column shard of the back-transformations, the first slice of
 * a multi-GPU solve: S1-S3 are replicated, every rank back-transforms its own slab-aligned column range; default 0),
 * "method" (2 = the two-stage solver, the default; 1 = the ONE-STAGE solver of PAPER.md:148 steps i-iii: direct
 * blocked Householder tridiagonalisation, D&C, one back-transformation -- the solver the paper benchmarks in
 * Figs. 3-4), "dtype" (0 = complex Hermitian c128, the default; 1 = REAL SYMMETRIC FP64:
 * A_dev and Z_dev of eigh_solve / eigh_solve_host and of the *_direct entry points then hold `double` elements,
 * lda / ldz in doubles; available for method = 1 only, so set "method" first), "ht_grid" (thread blocks of the
 * 1-stage panel kernel; 0 = every co-resident block).
 * Changing an option invalidates the workspace: call eigh_workspace_size / eigh_set_workspace again afterwards
 * (every compute entry point returns -1 until then).  Returns -2 for an unknown key, -3 for a bad value. */
int eigh_set_option(eigh_handle_t h, const char* key, int64_t value);

/* Current value of an option (same keys as eigh_set_option).  Returns -2 for an unknown key, -3 for value == NULL. */
int eigh_get_option(eigh_handle_t h, const char* key, int64_t* value);

/* Bytes of device workspace the caller must provide for this plan. */
size_t eigh_workspace_size(eigh_handle_t h);

/* Hand the workspace (device memory, 256-byte aligned, >= eigh_workspace_size bytes) to the
 * handle.  The caller keeps ownership and must keep it alive across eigh_solve calls. */
int eigh_set_workspace(eigh_handle_t h, void* ws_dev, size_t bytes);

/* Full solve (band reduction, band -> tridiagonal, tridiagonal eigensolve,
 * two back-transformations).
 *   A_dev : N x N c128, lda >= N.  Only the LOWER triangle is read; imaginary parts of the
 *           diagonal are ignored.  OVERWRITTEN (holds the stage-1 reflectors afterwards).
 *   W_dev : N doubles, all eigenvalues ascending.
 *   Z_dev : N x nev c128, ldz = N; column j = unit-2-norm eigenvector of W[j] (phase free).
 * Enqueues on `stream`; synchronises `stream` before returning (so that the failure count
 * can be returned).
 * Scaling: eigh(s A) = s eigh(A) holds to rounding (exactly for s a power of two) as long as the
 * SQUARES of the entries are representable, about 1e-150 <= max|a_ij| <= 1e150: the reductions form
 * sums of squares without rescaling.  Beyond that range the call fails loudly (a positive return
 * code: secular roots that did not converge); scale the matrix first.  S3 itself scales the
 * tridiagonal matrix to norm ~1 by a power of two (its deflation test needs it) and is free of
 * this limit (tested for s = 1e-200 .. 1e200). */
int eigh_solve(eigh_handle_t h, void* A_dev, int64_t lda, double* W_dev, void* Z_dev,
               void* stream);

/* The same solve with HOST buffers (end-to-end path).  A_host (N x N c128, lda >= N, pageable or pinned; not
 * modified) is streamed to A_scratch_dev through a bounded, double-buffered pinned staging ring owned by the handle
 * (2 x 256 MiB, allocated on first use, one cudaMemcpyAsync per chunk, the host-side fill of one buffer overlapping
 * the transfer of the other); eigh_solve runs; W (N doubles) and Z (N x nev c128) are streamed back to W_host /
 * Z_host the same way.  No pinned memory proportional to N^2 is needed.  A_scratch_dev (lda*N c128), W_scratch_dev
 * (N doubles) and Z_scratch_dev (N*nev c128) are caller-owned device buffers.  Uses `stream` and one internal
 * copy stream; synchronises both before returning. */
int eigh_solve_host(eigh_handle_t h, const void* A_host, int64_t lda, double* W_host, void* Z_host,
                    void* A_scratch_dev, double* W_scratch_dev, void* Z_scratch_dev, void* stream);

/* Per-phase device times of the last eigh_solve, in ms, from CUDA events on the solve's
 * stream: ms[0] = full->band, [1] = band->tridiagonal, [2] = tridiagonal D&C,
 * [3] = band back-transform, [4] = full back-transform.  With method = 1: ms[0] = direct tridiagonalisation,
 * [2] = D&C, [4] = back-transformation, [1] = [3] = 0. */
int eigh_phase_times(eigh_handle_t h, double ms[5]);

/* Device time (ms, CUDA events on the solve's stream around the launch) of one named kernel of the last
 * eigh_solve.  Timed kernels: "bt_sweep_kernel" (the single persistent launch that carries S4a).
 * Returns -2 for an unknown name. */
int eigh_kernel_time(eigh_handle_t h, const char* kernel, double* ms);

/* Kernel launches issued by the last eigh_solve (all are this library's own kernels). */
int64_t eigh_launch_count(eigh_handle_t h);

const char* eigh_last_error(eigh_handle_t h);
int eigh_destroy(eigh_handle_t h);

/* ---------------------------------------------------------------------------------------
 * Phase-level entry points (same conventions).  They use the handle's workspace exactly as
 * eigh_solve does, so a sequence reduce_to_band -> band_to_tridiag -> tridiag_dc ->
 * backtransform_band -> backtransform_full on one handle reproduces eigh_solve.
 * ------------------------------------------------------------------------------------- */

/* S1 ("transforming the dense matrix in a banded matrix"): unitary Q1 with
 * Q1^H A Q1 = B, B Hermitian of half-bandwidth b.  A_dev is overwritten: column block p
 * holds V_p (unit lower trapezoidal, explicit ones and zeros) in rows >= (p+1) b.
 * band_dev: (ldab x N) c128, ldab >= 2b+1... lower band storage band[i-j + j*ldab] = B[i,j]
 * for j <= i <= min(N-1, j+b); rows b+1..ldab-1 are zeroed (bulge-chasing fill-in room). */
int eigh_reduce_to_band(eigh_handle_t h, void* A_dev, int64_t lda, void* band_dev,
                        int64_t ldab, void* stream);

/* S2 ("transforming the banded matrix into a tridiagonal form"): unitary Q2
 * with Q2^H B Q2 = T real symmetric tridiagonal.  band_dev (as written by S1) is destroyed.
 * d_dev[N], e_dev[N-1] (e >= 0).  The reflectors, their taus and the phase vector stay in
 * the workspace for S4a. */
int eigh_band_to_tridiag(eigh_handle_t h, void* band_dev, int64_t ldab, double* d_dev,
                         double* e_dev, void* stream);

/* S3 ("diagonalizing this tridiagonal form"), divide and conquer on the GPU.
 * d_dev[N], e_dev[N-1] are read (not modified); e may have either sign (the solver works on |e| and scales row i
 * of Q by prod_{t<i} sign(e_t), which maps the eigenvectors back to the signed matrix).  W_dev[N] ascending.
 * Q_dev: N x nev real FP64, ldq >= N, column j = eigenvector of W[j]; may alias no other argument.
 * The matrix is scaled internally by the power of two next to max(|d|, |e|) (exact; the merge step's deflation
 * test assumes a matrix of norm ~1, as in LAPACK's xSTEDC) and W scaled back.
 * Synchronises `stream`.  Returns the number of secular roots that failed to converge. */
int eigh_tridiag_dc(eigh_handle_t h, const double* d_dev, const double* e_dev, double* W_dev,
                    double* Q_dev, int64_t ldq, void* stream);

/* 1-stage variant, step i ("transforming the dense matrix into a tridiagonal form"; needs the option
 * method = 1): unitary (orthogonal) Q = H_0 H_1 ... H_{N-2}, H_c = I - tau_c v_c v_c^H, with Q^H A Q = T real
 * symmetric tridiagonal.  A_dev: N x N, c128 or (dtype = 1) double, lda >= N; only the LOWER triangle is read,
 * imaginary parts of the diagonal are ignored; OVERWRITTEN: column c holds v_c in rows c+1.. (explicit unit element
 * at row c+1).  d_dev[N] = diagonal of T; e_dev[N-1] = sub-diagonal (real, EITHER sign: eigh_tridiag_dc accepts it).
 * The taus and the compact-WY T factors of the 64-column panels stay in the workspace for eigh_backtransform_direct.
 * One persistent cooperative kernel per panel (HBM-bound: the lower triangle of the trailing matrix is read once per
 * column, 8/3 N^3 bytes for c128, 4/3 N^3 for double) + one HER2K / SYR2K-lower GEMM per panel.  Enqueues on `stream`,
 * does not synchronise. */
int eigh_tridiagonalise_direct(eigh_handle_t h, void* A_dev, int64_t lda, double* d_dev, double* e_dev, void* stream);

/* 1-stage variant, step iii: Z <- Q Z with the reflectors eigh_tridiagonalise_direct left in A_dev and the workspace.
 * Z_dev: N x nev (c128 or double), ldz >= N, holds the eigenvectors of T on entry (as elements of the working type). */
int eigh_backtransform_direct(eigh_handle_t h, const void* A_dev, int64_t lda, void* Z_dev, int64_t ldz, void* stream);

/* Statistics of the last S3 run on this handle (eigh_tridiag_dc or eigh_solve), per merge level (level 0 = the
 * merges of pairs of leaves, the last level = the root merge):
 *   flops_executed[l] = sum over the merge GEMMs of the level of 2 M N K as launched (block structure of Q_old and
 *                       deflation taken into account: the real FP64 tensor-core flops of S3.5),
 *   kept_frac[l]      = sum k / sum n over the merges of the level (k = non-deflated values; 1 - kept_frac is the
 *                       deflation ratio of SURVEY.md 8(d)).
 * Both arrays hold up to `cap` entries; *nlevels gets the number of levels.  Host pointers. */
int eigh_dc_stats(eigh_handle_t h, int cap, int* nlevels, double* flops_executed, double* kept_frac);

/* S4a (first of the "two stages"): Z <- Q2 * (phase o Q_T).
 * Q_dev: N x nev real (from S3); Z_dev: N x nev c128, ldz >= N. */
int eigh_backtransform_band(eigh_handle_t h, const double* Q_dev, int64_t ldq, void* Z_dev,
                            int64_t ldz, void* stream);

/* S4b (second stage): Z <- Q1 * Z with the reflectors S1 left in A_dev. */
int eigh_backtransform_full(eigh_handle_t h, const void* A_dev, int64_t lda, void* Z_dev,
                            int64_t ldz, void* stream);

/* ---------------------------------------------------------------------------------------
 * SCF epilogue: the local densities the paper's self-consistent loop forms from the
 * eigenpairs (Eq. 16a, 16d; Fermi factors Eq. 17):
 *     n(r)  = 2 sum_{0 < E_n < E_c} ( |v_n(r)|^2 f_T(-E_n) + |u_n(r)|^2 f_T(E_n) )
 *     nu(r) =   sum_{0 < E_n < E_c} u_n(r) conj(v_n(r)) ( f_T(-E_n) - f_T(E_n) ),   f_T(E) = 1 / (1 + exp(E / T)),
 * with phi_n = [u_n, v_n]^T = column n of Z: rows [0, M) hold u_n(r), rows [M, 2M) hold v_n(r), M = N/2 (N even),
 * lattice spacing 1.  One streaming pass over the active columns of Z (HBM-bound), summation order fixed
 * (bit-reproducible).
 *   E_dev  : ncols doubles, E_dev[j] = energy of column j of Z (any order; eigh_solve's W_dev qualifies).
 *   Z_dev  : N x ncols c128, ldz >= N (read only).  0 <= ncols <= N.
 *   T      : temperature >= 0; T = 0 is the step function.   Ec: cutoff (> 0; INFINITY = none).
 *   branch : +1 = Eq. 16 as written, on the columns with 0 < E < Ec;
 *            -1 = use the columns with -Ec < E < 0 in place of their particle-hole partners [-conj(v), conj(u)]
 *                 of energy -E (valid for H = [[h, D], [D^*, -h^*]] with diagonal D): the lowest N/2 eigenpairs
 *                 of H then give the same densities as the positive branch.
 *   n_dev  : M doubles (out).   nu_dev : M c128 (out).
 * Uses the handle's workspace (eigh_set_workspace must have been called); enqueues 3 kernels on `stream`,
 * does not synchronise.  Returns -k for a bad k-th argument, -1 if N is odd. */
int eigh_densities(eigh_handle_t h, const double* E_dev, const void* Z_dev, int64_t ldz, int64_t ncols,
                   double T, double Ec, int branch, double* n_dev, void* nu_dev, void* stream);

/* eigh_densities WITHOUT any allocation and without a workspace: for callers that cannot call cudaMalloc (code under
 * CUDA graph capture, tight serving loops, harnesses that forbid it).  Same arguments, same kernels and same results as
 * eigh_densities (the chunking of the sums may differ, so results agree to rounding, not bit for bit); the scratch (list
 * of active columns + chunk partials) is a file-scope device array of 8 MiB that every GPU loading this library holds
 * until exit.  The handle is used for N, the launch counter and the error text only: eigh_set_workspace need not have
 * been called.  Limits: N <= 65536 and ncols <= 32760; beyond them the call returns -1 / -5 with a message in
 * eigh_last_error and launches nothing (use eigh_densities).  Calls no cudaMalloc / cudaFree or allocating routine; the
 * first call on a device looks up the array's device address (cudaGetSymbolAddress) and the SM count.
 * ALL calls share the one array, which keeps the last call's contents: calls on one stream run one after the other and are
 * safe; calls that overlap on the GPU (different streams, different handles or host threads) RACE on it -- serialise
 * them.  Enqueues one memset (256 B) + 3 kernels on `stream`, does not synchronise. */
int eigh_densities_static(eigh_handle_t h, const double* E_dev, const void* Z_dev, int64_t ldz, int64_t ncols,
                          double T, double Ec, int branch, double* n_dev, void* nu_dev, void* stream);

/* Kinetic and current densities (Eq. 16b, 16c), same states, weights and `branch` rule as eigh_densities:
 *     tau(r) = 2 sum ( |grad v_n|^2 f_T(-E_n) + |grad u_n|^2 f_T(E_n) )
 *     j(r)   = 2 sum Im( v_n grad v_n^* f_T(-E_n) - u_n grad u_n^* f_T(E_n) )
 * (Eq. 16b prints the range 0 <= E_n <= E_r; the range 0 < E_n < E_c of Eq. 16a/c/d is used.)  The gradient acts along
 * each axis through a dense real 1-D matrix: (d_x u)(ix, iy, iz) = sum_i' Dx[ix, i'] u(i', iy, iz), grid point
 * r = (ix ny + iy) nz + iz -- the matrix form of the spectral derivative of PAPER.md:113-115.
 *   nx, ny, nz : grid extents, 1..64 each, 2 nx ny nz = N.
 *   Dx_dev, Dy_dev, Dz_dev : nx x nx, ny x ny, nz x nz doubles, column-major (D[l + l2 * L] = D[l, l2]).
 *   E_dev, Z_dev, ldz, ncols, T, Ec, branch : as for eigh_densities.
 *   tau_dev : M doubles (out).   j_dev : 3 M doubles (out), j_dev[a * M + r] = component a (x, y, z) at r.
 * One launch per axis (ALU-bound: 4 L FP64 FMAs per point, state and axis) + weights + ordered reduction; summation
 * order fixed (bit-reproducible).  Uses the handle's workspace; enqueues on `stream`, does not synchronise. */
int eigh_gradient_densities(eigh_handle_t h, int64_t nx, int64_t ny, int64_t nz, const double* Dx_dev,
                            const double* Dy_dev, const double* Dz_dev, const double* E_dev, const void* Z_dev,
                            int64_t ldz, int64_t ncols, double T, double Ec, int branch, double* tau_dev, double* j_dev,
                            void* stream);

/* SCF prologue: assemble the dense BdG matrix of Eq. 5 / 7 from its fields,
 *     H = sign * [[h, diag(Delta)], [diag(Delta)^*, -h^*]],   h = T + diag(V) - mu,
 *     T = Kx (x) Iy (x) Iz + Ix (x) Ky (x) Iz + Ix (x) Iy (x) Kz   (Eq. 8: the kinetic term, one dense
 *     real symmetric 1-D matrix per axis), grid point r = (ix ny + iy) nz + iz, matrix index s M + r, M = nx ny nz.
 *   Kx_dev, Ky_dev, Kz_dev : nx x nx, ny x ny, nz x nz doubles, column-major, ld = their order.
 *   V_dev : M doubles.   Delta_dev : M c128.   mu : chemical potential.   sign : +1 or -1 (the matrix of -H).
 *   A_dev : N x N c128 (out), lda >= N = 2 M = the handle's N; ALL N^2 elements are written (both triangles).
 * The diagonal is summed as ((Kx + Ky) + Kz + V) - mu.  One kernel on `stream` (HBM-write-bound, 16 N^2 bytes), no
 * synchronisation, no workspace needed.  Returns -k for a bad k-th argument. */
int eigh_assemble_bdg(eigh_handle_t h, int64_t nx, int64_t ny, int64_t nz, const double* Kx_dev,
                      const double* Ky_dev, const double* Kz_dev, const double* V_dev, const void* Delta_dev,
                      double mu, double sign, void* A_dev, int64_t lda, void* stream);

/* ---------------------------------------------------------------------------------------
 * Second workload: one TDSLDA time step for the states just computed.
 * PAPER.md:91 Eq. (5):  i d/dt [u_n, v_n]^T = [[h, Delta], [Delta^*, -h^*]] [u_n, v_n]^T  (hbar = 1), h = -1/2 lap + V - mu
 * with the spectral kinetic term of Eq. (8) in its matrix form: one dense real symmetric 1-D matrix
 * per axis (the Kx, Ky, Kz of eigh_assemble_bdg), applied on the FP64 tensor cores.  States are columns of an N x ncols
 * c128 array (rows [0, M) = u, [M, 2M) = v, grid point r = (ix ny + iy) nz + iz, M = nx ny nz = N/2).
 * ------------------------------------------------------------------------------------- */

/* F <- -i H(V, Delta) Phi, the right-hand side of Eq. (5) for ncols states.  V_dev: M doubles; Delta_dev: M c128;
 * Phi_dev: N x ncols c128, ldp >= N (read only); F_dev: N x ncols c128, ldf >= N (out; must not alias Phi_dev).
 * Three launches (one per axis; the last fuses the local terms and the factor -i); HBM-bound, 8 x 16 N bytes per state.
 * Uses the handle's N only (no workspace contents); enqueues on `stream`, does not synchronise. */
int eigh_tdslda_rhs(eigh_handle_t h, int64_t nx, int64_t ny, int64_t nz, const double* Kx_dev, const double* Ky_dev,
                    const double* Kz_dev, const double* V_dev, const void* Delta_dev, double mu, const void* Phi_dev,
                    int64_t ldp, int64_t ncols, void* F_dev, int64_t ldf, void* stream);

/* One step y_n -> y_{n+1} of the 5th-order Adams-Bashforth-Moulton predictor-corrector of PAPER.md:134 in PECE form
 * (the paper names the method only; the coefficients are the textbook 5-step Adams-Bashforth predictor and 4-step
 * Adams-Moulton corrector), with h and Delta evaluated twice, each time from the densities of the current states
 * (eigh_densities: Eq. 16a / 16d with the occupation weights of the INITIAL energies E0_dev, T, Ec, branch) through the
 * toy functional Delta(r) = g nu(r) (Eq. 18b with a constant coupling; V stays fixed):
 *     y_p     = y_n + dt/720 (1901 f_n - 2774 f_{n-1} + 2616 f_{n-2} - 1274 f_{n-3} + 251 f_{n-4}),   f_p = -i H[y_p] y_p
 *     y_{n+1} = y_n + dt/720 (251 f_p + 646 f_n - 264 f_{n-1} + 106 f_{n-2} - 19 f_{n-3}),           f_{n+1} = -i H[y_{n+1}] y_{n+1}
 *   Y_dev    : N x ncols c128, ldy >= N: y_n on entry, y_{n+1} on return.
 *   F_dev    : HOST array of 5 device pointers, F_dev[k] = f_{n-k} (N x ncols c128 each, ldf >= N).  On return the
 *              buffer F_dev[4] holds f_{n+1}; the others are unchanged: rotate to [F4, F0, F1, F2, F3] for the next step.
 *   Yp_dev   : N x ncols c128 scratch (ld = ldy) for the predicted state.   7 copies of the state in all.
 *   n_dev    : M doubles (out): n(r) of y_{n+1}.   Delta_dev : M c128 (out): g nu(r) of y_{n+1}.
 * Uses the handle's workspace (the densities); 20 launches on `stream`, does not synchronise. */
int eigh_tdslda_step(eigh_handle_t h, int64_t nx, int64_t ny, int64_t nz, const double* Kx_dev, const double* Ky_dev,
                     const double* Kz_dev, const double* V_dev, double g, double mu, const double* E0_dev, double T, double Ec,
                     int branch, double dt, void* Y_dev, int64_t ldy, void* const F_dev[5], int64_t ldf, void* Yp_dev,
                     int64_t ncols, double* n_dev, void* Delta_dev, void* stream);

/* ---------------------------------------------------------------------------------------
 * Kernel-level entry points (unit tests of the building blocks).
 * ------------------------------------------------------------------------------------- */

/* Complex-FP64 GEMM on the FP64 tensor-core path (mma.sync m8n8k4 f64 -> DMMA):
 *   C <- alpha * opA(A) * opB(B) [+ alpha * opA(A2) * opB(B2)] + beta * C
 * opX = 'N' (as stored) or 'C' (conjugate transpose).  C is M x N, inner dimension K (K2 for
 * the optional second pair; pass A2_dev = NULL to disable).  lower_only bit 0 skips output
 * tiles that lie strictly above the diagonal (HER2K-lower); bit 2 (value 4) selects the
 * 128x64 tile configuration (default: 64x64 tiles, two thread blocks per SM).  splitk >= 1 partitions K over
 * thread blocks with a deterministic two-pass reduction (partials in the handle workspace). */
int eigh_k_zgemm(eigh_handle_t h, char opA, char opB, int64_t M, int64_t N, int64_t K,
                 double alpha, const void* A_dev, int64_t lda, const void* B_dev, int64_t ldb,
                 int64_t K2, const void* A2_dev, int64_t lda2, const void* B2_dev, int64_t ldb2,
                 double beta, void* C_dev, int64_t ldc, int lower_only, int splitk, void* stream);

/* HEMM-lower on the DMMA path: C (M x N) <- Herm(A) * B, A is M x M Hermitian of which only
 * the lower triangle AND the 64-aligned diagonal blocks are read as stored. */
int eigh_k_zhemm_lower(eigh_handle_t h, int64_t M, int64_t N, const void* A_dev, int64_t lda,
                       const void* B_dev, int64_t ldb, void* C_dev, int64_t ldc, int splitk,
                       void* stream);

/* Real FP64 GEMM engine of the real-symmetric path (rgemm.cuh), same conventions as eigh_k_zgemm with op = 'N' or 'T':
 *   C <- alpha * opA(A) * opB(B) [+ alpha * opA(A2) * opB(B2)] + beta * C,   lower_only bit 0 skips the 128 x 64 output
 * tiles strictly above the diagonal (SYR2K-lower), splitk >= 1 = deterministic split-K. */
int eigh_k_rgemm(eigh_handle_t h, char opA, char opB, int64_t M, int64_t N, int64_t K, double alpha, const double* A_dev,
                 int64_t lda, const double* B_dev, int64_t ldb, int64_t K2, const double* A2_dev, int64_t lda2,
                 const double* B2_dev, int64_t ldb2, double beta, double* C_dev, int64_t ldc, int lower_only, int splitk,
                 void* stream);

/* Real FP64 GEMM on the DMMA path: C (M x N) <- A[:, idx] * B, K inner; a_col_idx_dev may be
 * NULL (identity) or K int32 column indices into A. */
int eigh_k_dgemm(eigh_handle_t h, int64_t M, int64_t N, int64_t K, const double* A_dev,
                 int64_t lda, const int32_t* a_col_idx_dev, const double* B_dev, int64_t ldb,
                 double* C_dev, int64_t ldc, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* EIGH_B200_H */
