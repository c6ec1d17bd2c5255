// api.cu -- C ABI (include/eigh.h): handle, workspace plan, eigh_solve, kernel-level entry points.
#include <stdarg.h>
#include <stdlib.h>

#include <algorithm>
#include <new>
#include <thread>
#include <vector>

#include <nvtx3/nvToolsExt.h>

#include "dgemm.cuh"
#include "eigh_internal.h"
#include "rgemm.cuh"
#include "zgemm.cuh"

namespace eigh {

int set_err(eigh_handle_s* h, int code, const char* fmt, ...) {
    if (h) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(h->err, sizeof(h->err), fmt, ap);
        va_end(ap);
    }
    return code;
}

static size_t bump(size_t& off, size_t bytes) {
    const size_t at = off;
    off += (bytes + 255) / 256 * 256;
    return at;
}

extern int g_dgemm_mi;              // dgemm.cu
size_t dc_arena_bytes(int64_t N);   // tridiag_dc.cu
size_t dc_result_offset(int64_t N);
size_t bt_scratch_bytes(const eigh_handle_s* h);   // bt_band.cu
size_t bt_tneg_bytes(int64_t N);
size_t bt_vq_bytes(int64_t N);

void plan_workspace(eigh_handle_s* h) {
    WsPlan& p = h->plan;
    const int64_t N = h->N, b = h->b;
    size_t off = 0;
    h->ldab = 2 * b + 2;
    p.gemm_partial_bytes = (size_t)192 << 20;
    p.gemm_partial = bump(off, p.gemm_partial_bytes);
    p.band = bump(off, (size_t)h->ldab * N * sizeof(c128));
    p.tau1 = bump(off, (size_t)N * sizeof(c128));
    const int64_t npanels = ceil_div(N, b);
    p.T1 = bump(off, (size_t)npanels * b * b * sizeof(c128));
    p.Vp = bump(off, (size_t)N * b * sizeof(c128));
    p.VT = bump(off, (size_t)N * b * sizeof(c128));
    p.X = bump(off, (size_t)N * b * sizeof(c128));
    p.small = bump(off, (size_t)4 * b * b * sizeof(c128));
    p.panel_sync = bump(off, (size_t)(256 + 2 * 160 * (2 * b + 8) * sizeof(c128)));
    p.V2 = bump(off, (size_t)(v2_total_stages(N) * 32 * 64 + 64) * sizeof(c128));
    p.pass_off = bump(off, (size_t)(v2_npass(N) + 8) * sizeof(int64_t));
    p.tau2 = bump(off, (size_t)N * bc_kmax(h) * sizeof(c128));
    p.bc_progress = bump(off, (size_t)(N + 8) * sizeof(int));
    p.d = bump(off, (size_t)N * sizeof(double));
    p.e = bump(off, (size_t)N * sizeof(double));
    p.sgn = bump(off, (size_t)N * sizeof(double));
    p.dc_bytes = dc_arena_bytes(N);
    p.dc = bump(off, p.dc_bytes);
    // S4a keeps its T factors in the first two (dead by then) Q buffers of the D&C arena when they fit
    if (bt_tneg_bytes(N) <= dc_result_offset(N)) p.btT = p.dc;
    else p.btT = bump(off, bt_tneg_bytes(N));
    {
        const size_t tb = (bt_tneg_bytes(N) + 255) / 256 * 256, qb = bt_vq_bytes(N);
        if (p.btT == p.dc && tb + qb <= dc_result_offset(N)) p.btQ = p.dc + tb;
        else p.btQ = bump(off, qb ? qb : 256);
    }
    p.Qt = p.dc + dc_result_offset(N);   // eigh_solve lets S3 write its result over the dead U buffer
    // back-transform scratch aliases the tail of the D&C arena (U and the dead Q buffer)
    p.bt_bytes = bt_scratch_bytes(h);
    p.bt = bump(off, p.bt_bytes);
    {
        const int64_t kb = (int64_t)h->p4b_merge * b;
        p.b4V = bump(off, (size_t)N * kb * sizeof(c128));
        p.b4VT = bump(off, (size_t)N * kb * sizeof(c128));
        p.b4Y = bump(off, (size_t)kb * h->nev * sizeof(c128));
        p.b4T = bump(off, (size_t)kb * kb * sizeof(c128));
        p.b4G = bump(off, (size_t)2 * kb * kb * sizeof(c128));
    }
    p.ht_part = 0;
    if (h->method == 1) p.ht_part = bump(off, ht_partial_bytes(N));
    p.total = off;
    h->planned = true;
}

}  // namespace eigh

using namespace eigh;

extern "C" {

int eigh_create(eigh_handle_t* out, int64_t N, int64_t nev) {
    if (!out) return -1;
    *out = nullptr;
    if (N < 1 || N > (int64_t)1 << 20) return -2;
    if (nev < 1 || nev > N) return -3;
    eigh_handle_s* h = new (std::nothrow) eigh_handle_s();
    if (!h) return -1;
    memset(h, 0, sizeof(*h));
    h->N = N;
    h->nev = nev;
    h->b = 64;
    h->g = 8;
    h->leaf = 32;
    h->p4b_merge = 4;
    h->gemm_3m = 1;
    h->panel_smem = 1;
    h->panel_rows_min = 96;
    h->hemm_waves = 14;
    h->bc_variant = 3;
    h->method = 2;
    h->real_dtype = 0;
    h->num_sms = 0;
    snprintf(h->err, sizeof(h->err), "ok");
    *out = h;
    return 0;
}

int eigh_set_option(eigh_handle_t h, const char* key, int64_t value) {
    if (!h) return -1;
    if (!key) return -2;
    if (!strcmp(key, "band_width")) {
        if (value != 64) return set_err(h, -3, "band_width must be 64 (the width S2 and S4a are built for)");
        h->b = (int)value;
    } else if (!strcmp(key, "wy_group")) {
        if (value != 8 && value != 16 && value != 32) return set_err(h, -3, "wy_group must be 8, 16 or 32");
        h->g = (int)value;
    } else if (!strcmp(key, "dc_leaf")) {
        if (value < 8 || value > 32) return set_err(h, -3, "dc_leaf must be in [8, 32]");
        h->leaf = (int)value;
    } else if (!strcmp(key, "p4b_merge")) {
        if (value < 1 || value > 8) return set_err(h, -3, "p4b_merge must be in [1, 8]");
        h->p4b_merge = (int)value;
    } else if (!strcmp(key, "gemm_3m")) {
        if (value != 0 && value != 1) return set_err(h, -3, "gemm_3m must be 0 or 1");
        h->gemm_3m = (int)value;
    } else if (!strcmp(key, "panel_smem")) {
        if (value != 0 && value != 1) return set_err(h, -3, "panel_smem must be 0 or 1");
        h->panel_smem = (int)value;
    } else if (!strcmp(key, "panel_rows_min")) {
        if (value < 16 || value > 192) return set_err(h, -3, "panel_rows_min must be in [16, 192]");
        h->panel_rows_min = (int)value;
    } else if (!strcmp(key, "bt_chain")) {
        if (value < 0 || value > 16) return set_err(h, -3, "bt_chain must be in [0, 16]");
        h->bt_chain = (int)value;
    } else if (!strcmp(key, "hemm_waves")) {
        if (value < 1 || value > 64) return set_err(h, -3, "hemm_waves must be in [1, 64]");
        h->hemm_waves = (int)value;
    } else if (!strcmp(key, "bc_grid")) {
        if (value < 0 || value > 4096) return set_err(h, -3, "bc_grid must be in [0, 4096]");
        h->bc_grid = (int)value;
    } else if (!strcmp(key, "dgemm_mi")) {
        if (value != 4 && value != 8) return set_err(h, -3, "dgemm_mi must be 4 or 8");
        g_dgemm_mi = (int)value;             // process-wide, like gemm_3m
    } else if (!strcmp(key, "bc_variant")) {
        if (value != 0 && value != 2 && value != 3) return set_err(h, -3, "bc_variant must be 0, 2 or 3");
        h->bc_variant = (int)value;
    } else if (!strcmp(key, "bc_dual_steps")) {
        if (value < 0 || value > (1 << 20)) return set_err(h, -3, "bc_dual_steps must be in [0, 2^20]");
        h->bc_dual_steps = (int)value;
    } else if (!strcmp(key, "col_begin")) {
        if (value < 0 || value + h->nev > h->N) return set_err(h, -3, "col_begin must satisfy 0 <= col_begin <= N - nev");
        h->col0 = (int)value;
    } else if (!strcmp(key, "method")) {
        if (value != 1 && value != 2) return set_err(h, -3, "method must be 1 (one-stage) or 2 (two-stage)");
        if (value == 2 && h->real_dtype) return set_err(h, -3, "the real-symmetric path exists for method = 1 only");
        h->method = (int)value;
    } else if (!strcmp(key, "dtype")) {
        if (value != 0 && value != 1) return set_err(h, -3, "dtype must be 0 (complex Hermitian, c128) or 1 (real symmetric, f64)");
        if (value == 1 && h->method != 1) return set_err(h, -3, "dtype = 1 (real symmetric) needs method = 1: set \"method\" first");
        h->real_dtype = (int)value;
    } else if (!strcmp(key, "ht_grid")) {
        if (value < 0 || value > 4096) return set_err(h, -3, "ht_grid must be in [0, 4096]");
        h->ht_grid = (int)value;
    } else {
        return set_err(h, -2, "unknown option '%s'", key);
    }
    // the plan (and with it the size and the layout of the workspace) depends on the options: the workspace handed
    // over earlier is dropped, so that a buffer sized for the old plan can never be used with the new one
    h->planned = false;
    h->ws = nullptr;
    h->ws_bytes = 0;
    return 0;
}

int eigh_get_option(eigh_handle_t h, const char* key, int64_t* value) {
    if (!h) return -1;
    if (!key) return -2;
    if (!value) return -3;
    if (!strcmp(key, "band_width")) *value = h->b;
    else if (!strcmp(key, "wy_group")) *value = h->g;
    else if (!strcmp(key, "dc_leaf")) *value = h->leaf;
    else if (!strcmp(key, "p4b_merge")) *value = h->p4b_merge;
    else if (!strcmp(key, "gemm_3m")) *value = h->gemm_3m;
    else if (!strcmp(key, "panel_smem")) *value = h->panel_smem;
    else if (!strcmp(key, "panel_rows_min")) *value = h->panel_rows_min;
    else if (!strcmp(key, "bt_chain")) *value = h->bt_chain;
    else if (!strcmp(key, "hemm_waves")) *value = h->hemm_waves;
    else if (!strcmp(key, "bc_grid")) *value = h->bc_grid;
    else if (!strcmp(key, "bc_variant")) *value = h->bc_variant;
    else if (!strcmp(key, "bc_dual_steps")) *value = h->bc_dual_steps;
    else if (!strcmp(key, "col_begin")) *value = h->col0;
    else if (!strcmp(key, "method")) *value = h->method;
    else if (!strcmp(key, "dtype")) *value = h->real_dtype;
    else if (!strcmp(key, "ht_grid")) *value = h->ht_grid;
    else return set_err(h, -2, "unknown option '%s'", key);
    return 0;
}

size_t eigh_workspace_size(eigh_handle_t h) {
    if (!h) return 0;
    plan_workspace(h);
    return h->plan.total;
}

int eigh_set_workspace(eigh_handle_t h, void* ws_dev, size_t bytes) {
    if (!h) return -1;
    if (!h->planned) plan_workspace(h);
    if (!ws_dev || ((uintptr_t)ws_dev & 255)) return set_err(h, -2, "workspace must be a 256-byte aligned device pointer");
    if (bytes < h->plan.total) return set_err(h, -3, "workspace too small: %zu < %zu", bytes, h->plan.total);
    h->ws = ws_dev;
    h->ws_bytes = bytes;
    return 0;
}

static int ensure_ready(eigh_handle_t h) {
    if (!h) return -1;
    g_zgemm_3m = h->gemm_3m != 0;            // process-wide switch of the GEMM engine, set from the handle in use
    if (!h->ws) return set_err(h, -1, "no workspace set (call eigh_set_workspace; eigh_set_option drops an earlier one)");
    if (!h->planned) return set_err(h, -1, "options changed after eigh_set_workspace; call eigh_workspace_size / eigh_set_workspace again");
    if (h->ws_bytes < h->plan.total)
        return set_err(h, -1, "workspace too small for the current plan: %zu < %zu", h->ws_bytes, h->plan.total);
    if (!h->events_ok) {
        for (int i = 0; i < 6; ++i) {
            cudaError_t e = cudaEventCreate(&h->ev[i]);
            if (e != cudaSuccess) return set_err(h, 1000 + (int)e, "cudaEventCreate: %s", cudaGetErrorString(e));
        }
        for (int i = 0; i < 2; ++i) {
            cudaError_t e = cudaEventCreate(&h->ev_sweep[i]);
            if (e != cudaSuccess) return set_err(h, 1000 + (int)e, "cudaEventCreate: %s", cudaGetErrorString(e));
        }
        h->events_ok = true;
    }
    if (!h->num_sms) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&h->num_sms, cudaDevAttrMultiProcessorCount, dev);
        if (h->num_sms <= 0) return set_err(h, EIGH_ERR_CUDA, "no CUDA device");
    }
    return 0;
}

namespace {
struct NvtxRange {
    explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
    ~NvtxRange() { nvtxRangePop(); }
};
}  // namespace

static int cuda_fail(eigh_handle_t h, int rc, const char* where) {
    if (rc >= 1000) return set_err(h, rc, "%s: CUDA error %d (%s)", where, rc - 1000, cudaGetErrorString((cudaError_t)(rc - 1000)));
    return rc;
}

int eigh_reduce_to_band(eigh_handle_t h, void* A_dev, int64_t lda, void* band_dev, int64_t ldab, void* stream) {
    int rc = ensure_ready(h);
    if (rc) return rc;
    if (h->method != 2) return set_err(h, -1, "eigh_reduce_to_band belongs to the two-stage method (option method = 2)");
    if (!A_dev) return -2;
    if (lda < h->N) return -3;
    if (!band_dev) return -4;
    if (ldab < h->ldab) return set_err(h, -5, "ldab must be >= %lld", (long long)h->ldab);
    return cuda_fail(h, phase_reduce_to_band(h, (c128*)A_dev, lda, (c128*)band_dev, ldab, (cudaStream_t)stream), "reduce_to_band");
}

int eigh_band_to_tridiag(eigh_handle_t h, void* band_dev, int64_t ldab, double* d_dev, double* e_dev, void* stream) {
    int rc = ensure_ready(h);
    if (rc) return rc;
    if (!band_dev) return -2;
    if (ldab < h->ldab) return set_err(h, -3, "ldab must be >= %lld", (long long)h->ldab);
    if (!d_dev) return -4;
    if (!e_dev && h->N > 1) return -5;
    return cuda_fail(h, phase_band_to_tridiag(h, (c128*)band_dev, ldab, d_dev, e_dev, (cudaStream_t)stream), "band_to_tridiag");
}

int eigh_tridiag_dc(eigh_handle_t h, const double* d_dev, const double* e_dev, double* W_dev, double* Q_dev,
                    int64_t ldq, void* stream) {
    int rc = ensure_ready(h);
    if (rc) return rc;
    if (!d_dev) return -2;
    if (!e_dev && h->N > 1) return -3;
    if (!W_dev) return -4;
    if (!Q_dev) return -5;
    if (ldq < h->N) return -6;
    int nfail = 0;
    rc = phase_tridiag_dc(h, d_dev, e_dev, W_dev, Q_dev, ldq, (cudaStream_t)stream, &nfail);
    if (rc) return cuda_fail(h, rc, "tridiag_dc");
    if (nfail) set_err(h, nfail, "%d secular roots did not converge", nfail);
    return std::min(nfail, 999);          // (1000 and above are CUDA errors; the text has the count)
}

int eigh_backtransform_band(eigh_handle_t h, const double* Q_dev, int64_t ldq, void* Z_dev, int64_t ldz, void* stream) {
    int rc = ensure_ready(h);
    if (rc) return rc;
    if (!Q_dev) return -2;
    if (ldq < h->N) return -3;
    if (!Z_dev) return -4;
    if (ldz < h->N) return -5;
    return cuda_fail(h, phase_backtransform_band(h, Q_dev, ldq, (c128*)Z_dev, ldz, (cudaStream_t)stream), "backtransform_band");
}

int eigh_backtransform_full(eigh_handle_t h, const void* A_dev, int64_t lda, void* Z_dev, int64_t ldz, void* stream) {
    int rc = ensure_ready(h);
    if (rc) return rc;
    if (!A_dev) return -2;
    if (lda < h->N) return -3;
    if (!Z_dev) return -4;
    if (ldz < h->N) return -5;
    return cuda_fail(h, phase_backtransform_full(h, (const c128*)A_dev, lda, (c128*)Z_dev, ldz, (cudaStream_t)stream), "backtransform_full");
}

static int grid_check(eigh_handle_t h, int64_t nx, int64_t ny, int64_t nz, const char* who) {
    if (h->N & 1) return set_err(h, -1, "%s: N = %lld is odd (phi = [u, v] needs N = 2M)", who, (long long)h->N);
    if (nx < 1 || ny < 1 || nz < 1 || nx > 64 || ny > 64 || nz > 64) return set_err(h, -2, "%s: grid extents must be 1..64 per axis", who);
    if (2 * nx * ny * nz != h->N)
        return set_err(h, -2, "%s: 2 nx ny nz = %lld != N = %lld", who, (long long)(2 * nx * ny * nz), (long long)h->N);
    return 0;
}

int eigh_tdslda_rhs(eigh_handle_t h, int64_t nx, int64_t ny, int64_t nz, const double* Kx_dev, const double* Ky_dev,
                    const double* Kz_dev, const double* V_dev, const void* Delta_dev, double mu, const void* Phi_dev,
                    int64_t ldp, int64_t ncols, void* F_dev, int64_t ldf, void* stream) {
    int rc = ensure_ready(h);
    if (rc) return rc;
    rc = grid_check(h, nx, ny, nz, "eigh_tdslda_rhs");
    if (rc) return rc;
    if (!Kx_dev) return -5;
    if (!Ky_dev) return -6;
    if (!Kz_dev) return -7;
    if (!V_dev) return -8;
    if (!Delta_dev) return -9;
    if (!Phi_dev && ncols > 0) return -11;
    if (ldp < h->N) return -12;
    if (ncols < 0) return -13;
    if (!F_dev && ncols > 0) return -14;
    if (ldf < h->N) return -15;
    if (F_dev == Phi_dev && ncols > 0) return set_err(h, -14, "eigh_tdslda_rhs: F must not alias Phi");
    return cuda_fail(h, launch_tdslda_rhs(h, (int)nx, (int)ny, (int)nz, Kx_dev, Ky_dev, Kz_dev, V_dev, (const c128*)Delta_dev, mu,
                                          (const c128*)Phi_dev, ldp, ncols, (c128*)F_dev, ldf, (cudaStream_t)stream), "tdslda_rhs");
}

int eigh_tdslda_step(eigh_handle_t h, int64_t nx, int64_t ny, int64_t nz, const double* Kx_dev, const double* Ky_dev,
                     const double* Kz_dev, const double* V_dev, double g, double mu, const double* E0_dev, double T, double Ec,
                     int branch, double dt, void* Y_dev, int64_t ldy, void* const F_dev[5], int64_t ldf, void* Yp_dev,
                     int64_t ncols, double* n_dev, void* Delta_dev, void* stream) {
    int rc = ensure_ready(h);
    if (rc) return rc;
    rc = grid_check(h, nx, ny, nz, "eigh_tdslda_step");
    if (rc) return rc;
    if (!Kx_dev) return -5;
    if (!Ky_dev) return -6;
    if (!Kz_dev) return -7;
    if (!V_dev) return -8;
    if (!E0_dev) return -11;
    if (!(T >= 0.0)) return -12;
    if (Ec != Ec) return -13;
    if (branch != 1 && branch != -1) return -14;
    if (!(dt == dt)) return -15;
    if (!Y_dev) return -16;
    if (ldy < h->N) return -17;
    if (!F_dev) return -18;
    for (int k = 0; k < 5; ++k) if (!F_dev[k] || F_dev[k] == Y_dev || F_dev[k] == Yp_dev) return -18;
    if (ldf < h->N) return -19;
    if (!Yp_dev || Yp_dev == Y_dev) return -20;
    if (ncols < 1 || ncols > h->N) return -21;
    if (!n_dev) return -22;
    if (!Delta_dev) return -23;
    c128* F[5];
    for (int k = 0; k < 5; ++k) F[k] = (c128*)F_dev[k];
    NvtxRange r("eigh_tdslda_step");
    return cuda_fail(h, launch_tdslda_step(h, (int)nx, (int)ny, (int)nz, Kx_dev, Ky_dev, Kz_dev, V_dev, g, mu, E0_dev, T, Ec, branch, dt,
                                           (c128*)Y_dev, ldy, F, ldf, (c128*)Yp_dev, ncols, n_dev, (c128*)Delta_dev,
                                           (cudaStream_t)stream), "tdslda_step");
}

int eigh_tridiagonalise_direct(eigh_handle_t h, void* A_dev, int64_t lda, double* d_dev, double* e_dev, void* stream) {
    int rc = ensure_ready(h);
    if (rc) return rc;
    if (h->method != 1) return set_err(h, -1, "eigh_tridiagonalise_direct needs the option method = 1");
    if (!A_dev) return -2;
    if (lda < h->N) return -3;
    if (!d_dev) return -4;
    if (!e_dev && h->N > 1) return -5;
    return cuda_fail(h, phase_tridiagonalise_direct(h, A_dev, lda, d_dev, e_dev, (cudaStream_t)stream), "tridiagonalise_direct");
}

int eigh_backtransform_direct(eigh_handle_t h, const void* A_dev, int64_t lda, void* Z_dev, int64_t ldz, void* stream) {
    int rc = ensure_ready(h);
    if (rc) return rc;
    if (h->method != 1) return set_err(h, -1, "eigh_backtransform_direct needs the option method = 1");
    if (!A_dev) return -2;
    if (lda < h->N) return -3;
    if (!Z_dev) return -4;
    if (ldz < h->N) return -5;
    return cuda_fail(h, phase_backtransform_direct(h, A_dev, lda, nullptr, 0, Z_dev, ldz, (cudaStream_t)stream), "backtransform_direct");
}

int eigh_densities(eigh_handle_t h, const double* E_dev, const void* Z_dev, int64_t ldz, int64_t ncols, double T,
                   double Ec, int branch, double* n_dev, void* nu_dev, void* stream) {
    int rc = ensure_ready(h);
    if (rc) return rc;
    if (h->N & 1) return set_err(h, -1, "eigh_densities: N = %lld is odd (phi = [u, v] needs N = 2M)", (long long)h->N);
    if (!E_dev && ncols > 0) return -2;
    if (!Z_dev && ncols > 0) return -3;
    if (ldz < h->N) return -4;
    if (ncols < 0 || ncols > h->N) return -5;
    if (!(T >= 0.0)) return -6;
    if (Ec != Ec) return -7;
    if (branch != 1 && branch != -1) return -8;
    if (!n_dev) return -9;
    if (!nu_dev) return -10;
    return cuda_fail(h, launch_densities(h, E_dev, (const c128*)Z_dev, ldz, ncols, T, Ec, branch, n_dev, (c128*)nu_dev,
                                         (cudaStream_t)stream), "densities");
}

int eigh_gradient_densities(eigh_handle_t h, int64_t nx, int64_t ny, int64_t nz, const double* Dx_dev,
                            const double* Dy_dev, const double* Dz_dev, const double* E_dev, const void* Z_dev,
                            int64_t ldz, int64_t ncols, double T, double Ec, int branch, double* tau_dev, double* j_dev,
                            void* stream) {
    int rc = ensure_ready(h);
    if (rc) return rc;
    if (nx < 1 || ny < 1 || nz < 1 || nx > 64 || ny > 64 || nz > 64)
        return set_err(h, -2, "eigh_gradient_densities: grid extents must be 1..64 per axis");
    if (2 * nx * ny * nz != h->N)
        return set_err(h, -2, "eigh_gradient_densities: 2 nx ny nz = %lld != N = %lld", (long long)(2 * nx * ny * nz), (long long)h->N);
    if (!Dx_dev) return -5;
    if (!Dy_dev) return -6;
    if (!Dz_dev) return -7;
    if (!E_dev && ncols > 0) return -8;
    if (!Z_dev && ncols > 0) return -9;
    if (ldz < h->N) return -10;
    if (ncols < 0 || ncols > h->N) return -11;
    if (!(T >= 0.0)) return -12;
    if (Ec != Ec) return -13;
    if (branch != 1 && branch != -1) return -14;
    if (!tau_dev) return -15;
    if (!j_dev) return -16;
    return cuda_fail(h, launch_gradient_densities(h, (int)nx, (int)ny, (int)nz, Dx_dev, Dy_dev, Dz_dev, E_dev, (const c128*)Z_dev,
                                                  ldz, ncols, T, Ec, branch, tau_dev, j_dev, (cudaStream_t)stream),
                     "gradient_densities");
}

int eigh_solve(eigh_handle_t h, void* A_dev, int64_t lda, double* W_dev, void* Z_dev, void* stream) {
    int rc = ensure_ready(h);
    if (rc) return rc;
    if (!A_dev) return -2;
    if (lda < h->N) return -3;
    if (!W_dev) return -4;
    if (!Z_dev) return -5;
    cudaStream_t s = (cudaStream_t)stream;
    const WsPlan& p = h->plan;
    c128* band = ws_ptr<c128>(h, p.band);
    double* d = ws_ptr<double>(h, p.d);
    double* e = ws_ptr<double>(h, p.e);
    double* Qt = ws_ptr<double>(h, p.Qt);
    const int64_t ldq = round_up(h->N, 8);
    h->launches = 0;
    int nfail = 0;
    if (h->method == 1) {
        // 1-stage variant (PAPER.md:148 steps i-iii): direct tridiagonalisation, D&C, one back-transformation.
        // phase_ms: [0] = tridiagonalisation, [2] = D&C, [4] = back-transformation; [1] = [3] = 0.
        NvtxRange whole1("eigh_solve (1-stage)");
        cudaEventRecord(h->ev[0], s);
        { NvtxRange r("1-stage tridiagonalisation");
          rc = phase_tridiagonalise_direct(h, A_dev, lda, d, e, s); }
        if (rc) return cuda_fail(h, rc, "tridiagonalise_direct");
        cudaEventRecord(h->ev[1], s);
        cudaEventRecord(h->ev[2], s);
        { NvtxRange r("S3 tridiagonal D&C");
          rc = phase_tridiag_dc(h, d, e, W_dev, Qt, ldq, s, &nfail); }
        if (rc) return cuda_fail(h, rc, "tridiag_dc");
        cudaEventRecord(h->ev[3], s);
        cudaEventRecord(h->ev[4], s);
        { NvtxRange r("1-stage back-transform");
          rc = phase_backtransform_direct(h, A_dev, lda, Qt, ldq, Z_dev, h->N, s); }
        if (rc) return cuda_fail(h, rc, "backtransform_direct");
        cudaEventRecord(h->ev[5], s);
        cudaError_t ce1 = cudaStreamSynchronize(s);
        if (ce1 != cudaSuccess) return set_err(h, 1000 + (int)ce1, "eigh_solve: %s", cudaGetErrorString(ce1));
        for (int i = 0; i < 5; ++i) {
            float ms = 0.f;
            cudaEventElapsedTime(&ms, h->ev[i], h->ev[i + 1]);
            h->phase_ms[i] = ms;
        }
        h->phase_ms[1] = h->phase_ms[3] = 0.0;       // phases the 1-stage method does not have
        h->sweep_ms = 0.0;
        if (nfail) set_err(h, nfail, "%d secular roots did not converge", nfail);
        return std::min(nfail, 999);
    }
    // NVTX ranges mark the host-side enqueue of every phase (the device-side spans are the CUDA events below)
    NvtxRange whole("eigh_solve");
    cudaEventRecord(h->ev[0], s);
    { NvtxRange r("S1 full->band");
      rc = phase_reduce_to_band(h, (c128*)A_dev, lda, band, h->ldab, s); }
    if (rc) return cuda_fail(h, rc, "reduce_to_band");
    cudaEventRecord(h->ev[1], s);
    { NvtxRange r("S2 band->tridiagonal");
      rc = phase_band_to_tridiag(h, band, h->ldab, d, e, s); }
    if (rc) return cuda_fail(h, rc, "band_to_tridiag");
    cudaEventRecord(h->ev[2], s);
    { NvtxRange r("S3 tridiagonal D&C");
      rc = phase_tridiag_dc(h, d, e, W_dev, Qt, ldq, s, &nfail); }
    if (rc) return cuda_fail(h, rc, "tridiag_dc");
    cudaEventRecord(h->ev[3], s);
    { NvtxRange r("S4a band back-transform");
      rc = phase_backtransform_band(h, Qt, ldq, (c128*)Z_dev, h->N, s); }
    if (rc) return cuda_fail(h, rc, "backtransform_band");
    cudaEventRecord(h->ev[4], s);
    { NvtxRange r("S4b full back-transform");
      rc = phase_backtransform_full(h, (const c128*)A_dev, lda, (c128*)Z_dev, h->N, s); }
    if (rc) return cuda_fail(h, rc, "backtransform_full");
    cudaEventRecord(h->ev[5], s);
    cudaError_t ce = cudaStreamSynchronize(s);
    if (ce != cudaSuccess) return set_err(h, 1000 + (int)ce, "eigh_solve: %s", cudaGetErrorString(ce));
    for (int i = 0; i < 5; ++i) {
        float ms = 0.f;
        cudaEventElapsedTime(&ms, h->ev[i], h->ev[i + 1]);
        h->phase_ms[i] = ms;
    }
    h->sweep_ms = 0.0;
    if (h->N >= 2) {                          // the sweeper is not launched for N = 1
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, h->ev_sweep[0], h->ev_sweep[1]) == cudaSuccess) h->sweep_ms = ms;
        else (void)cudaGetLastError();
    }
    if (nfail) set_err(h, nfail, "%d secular roots did not converge", nfail);
    return std::min(nfail, 999);          // (1000 and above are CUDA errors; the text has the count)
}

// ---- eigh_solve_host: host <-> device streaming through a bounded pinned ring -----------------------------------
constexpr size_t STAGE_BYTES = (size_t)256 << 20;

static int stage_init(eigh_handle_s* h) {
    if (h->stage_ok) return 0;
    cudaError_t e = cudaSuccess;
    int nbuf = 0, nev = 0;
    bool have_stream = false;
    for (int i = 0; i < 2 && e == cudaSuccess; ++i) {
        e = cudaMallocHost(&h->stage[i], STAGE_BYTES);
        if (e == cudaSuccess) ++nbuf; else h->stage[i] = nullptr;
    }
    for (int i = 0; i < 2 && e == cudaSuccess; ++i) {
        e = cudaEventCreateWithFlags(&h->ev_stage[i], cudaEventDisableTiming);
        if (e == cudaSuccess) ++nev;
    }
    if (e == cudaSuccess) {
        e = cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking);
        have_stream = e == cudaSuccess;
    }
    if (e != cudaSuccess) {           // undo the part that succeeded: a failed init leaves nothing behind
        for (int i = 0; i < nbuf; ++i) { cudaFreeHost(h->stage[i]); h->stage[i] = nullptr; }
        for (int i = 0; i < nev; ++i) cudaEventDestroy(h->ev_stage[i]);
        if (have_stream) cudaStreamDestroy(h->copy_stream);
        return set_err(h, 1000 + (int)e, "eigh_solve_host staging ring: %s", cudaGetErrorString(e));
    }
    h->stage_bytes = STAGE_BYTES;
    h->stage_ok = true;
    return 0;
}

static bool host_is_pinned(const void* p) {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { (void)cudaGetLastError(); return false; }
    return at.type == cudaMemoryTypeHost;
}

// plain host copy split over a few threads (a single thread fills the ring slower than PCIe drains it)
static void host_copy(void* dst, const void* src, size_t bytes) {
    const int nt = bytes >= ((size_t)8 << 20) ? 8 : 1;
    if (nt == 1) { memcpy(dst, src, bytes); return; }
    std::vector<std::thread> th;
    const size_t per = ((bytes + nt - 1) / nt + 63) / 64 * 64;
    for (int t = 0; t < nt; ++t) {
        const size_t off = (size_t)t * per;
        if (off >= bytes) break;
        const size_t n = std::min(per, bytes - off);
        th.emplace_back([=] { memcpy((char*)dst + off, (const char*)src + off, n); });
    }
    for (auto& t : th) t.join();
}

// host -> device, `bytes` contiguous.  Pinned source: chunked direct copies.  Pageable source: the ring, the fill of
// one buffer overlapping the transfer of the other.  All copies on `cs`.
static cudaError_t stream_h2d(eigh_handle_s* h, void* dst_dev, const void* src_host, size_t bytes, cudaStream_t cs) {
    const bool pinned = host_is_pinned(src_host);
    size_t off = 0;
    for (int i = 0; off < bytes; ++i) {
        const size_t n = std::min(h->stage_bytes, bytes - off);
        cudaError_t e;
        if (pinned) {
            e = cudaMemcpyAsync((char*)dst_dev + off, (const char*)src_host + off, n, cudaMemcpyHostToDevice, cs);
        } else {
            const int b = i & 1;
            e = cudaEventSynchronize(h->ev_stage[b]);          // the transfer that last used this buffer is done
            if (e != cudaSuccess) return e;
            host_copy(h->stage[b], (const char*)src_host + off, n);
            e = cudaMemcpyAsync((char*)dst_dev + off, h->stage[b], n, cudaMemcpyHostToDevice, cs);
            if (e == cudaSuccess) e = cudaEventRecord(h->ev_stage[b], cs);
        }
        if (e != cudaSuccess) return e;
        off += n;
    }
    return cudaSuccess;
}

// device -> host, `bytes` contiguous; the host-side drain of chunk i-1 overlaps the transfer of chunk i.
static cudaError_t stream_d2h(eigh_handle_s* h, void* dst_host, const void* src_dev, size_t bytes, cudaStream_t cs) {
    if (host_is_pinned(dst_host)) {
        for (size_t off = 0; off < bytes; off += h->stage_bytes) {
            const size_t n = std::min(h->stage_bytes, bytes - off);
            cudaError_t e = cudaMemcpyAsync((char*)dst_host + off, (const char*)src_dev + off, n, cudaMemcpyDeviceToHost, cs);
            if (e != cudaSuccess) return e;
        }
        return cudaSuccess;
    }
    size_t off = 0, prev_off = 0, prev_n = 0;
    int i = 0;
    for (; off < bytes; ++i) {
        const size_t n = std::min(h->stage_bytes, bytes - off);
        const int b = i & 1;
        cudaError_t e = cudaMemcpyAsync(h->stage[b], (const char*)src_dev + off, n, cudaMemcpyDeviceToHost, cs);
        if (e == cudaSuccess) e = cudaEventRecord(h->ev_stage[b], cs);
        if (e != cudaSuccess) return e;
        if (prev_n) {
            e = cudaEventSynchronize(h->ev_stage[b ^ 1]);
            if (e != cudaSuccess) return e;
            host_copy((char*)dst_host + prev_off, h->stage[b ^ 1], prev_n);
        }
        prev_off = off; prev_n = n;
        off += n;
    }
    if (prev_n) {
        const int b = (i - 1) & 1;
        cudaError_t e = cudaEventSynchronize(h->ev_stage[b]);
        if (e != cudaSuccess) return e;
        host_copy((char*)dst_host + prev_off, h->stage[b], prev_n);
    }
    return cudaSuccess;
}

int eigh_solve_host(eigh_handle_t h, const void* A_host, int64_t lda, double* W_host, void* Z_host,
                    void* A_scratch_dev, double* W_scratch_dev, void* Z_scratch_dev, void* stream) {
    int rc = ensure_ready(h);
    if (rc) return rc;
    if (!A_host) return -2;
    if (lda < h->N) return -3;
    if (!W_host) return -4;
    if (!Z_host) return -5;
    if (!A_scratch_dev) return -6;
    if (!W_scratch_dev) return -7;
    if (!Z_scratch_dev) return -8;
    rc = stage_init(h);
    if (rc) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    const size_t es = h->real_dtype ? sizeof(double) : sizeof(c128);     // element size of A and Z
    NvtxRange whole("eigh_solve_host");
    // the copies run on the handle's copy stream, ordered against the caller's stream by events
    cudaError_t ce = cudaEventRecord(h->ev[0], s);
    if (ce == cudaSuccess) ce = cudaStreamWaitEvent(h->copy_stream, h->ev[0], 0);
    if (ce == cudaSuccess) {
        NvtxRange r("H2D A");
        ce = stream_h2d(h, A_scratch_dev, A_host, (size_t)lda * h->N * es, h->copy_stream);
    }
    if (ce == cudaSuccess) ce = cudaEventRecord(h->ev[1], h->copy_stream);
    if (ce == cudaSuccess) ce = cudaStreamWaitEvent(s, h->ev[1], 0);
    if (ce != cudaSuccess) return set_err(h, 1000 + (int)ce, "eigh_solve_host H2D: %s", cudaGetErrorString(ce));
    rc = eigh_solve(h, A_scratch_dev, lda, W_scratch_dev, Z_scratch_dev, stream);     // synchronises `stream`
    if (rc < 0 || rc >= 1000) return rc;
    {
        NvtxRange r("D2H W, Z");
        ce = stream_d2h(h, W_host, W_scratch_dev, (size_t)h->N * sizeof(double), h->copy_stream);
        if (ce == cudaSuccess)
            ce = stream_d2h(h, Z_host, Z_scratch_dev, (size_t)h->N * h->nev * es, h->copy_stream);
    }
    if (ce == cudaSuccess) ce = cudaStreamSynchronize(h->copy_stream);
    if (ce != cudaSuccess) return set_err(h, 1000 + (int)ce, "eigh_solve_host D2H: %s", cudaGetErrorString(ce));
    return rc;
}

int eigh_dc_stats(eigh_handle_t h, int cap, int* nlevels, double* flops_executed, double* kept_frac) {
    if (!h) return -1;
    if (cap < 0) return -2;
    if (!nlevels) return -3;
    *nlevels = h->dc_levels;
    for (int l = 0; l < h->dc_levels && l < cap; ++l) {
        if (flops_executed) flops_executed[l] = h->dc_flops[l];
        if (kept_frac) kept_frac[l] = h->dc_nsum[l] > 0.0 ? h->dc_ksum[l] / h->dc_nsum[l] : 0.0;
    }
    return 0;
}

int eigh_phase_times(eigh_handle_t h, double ms[5]) {
    if (!h) return -1;
    if (!ms) return -2;
    for (int i = 0; i < 5; ++i) ms[i] = h->phase_ms[i];
    return 0;
}

int eigh_kernel_time(eigh_handle_t h, const char* kernel, double* ms) {
    if (!h) return -1;
    if (!kernel) return -2;
    if (!ms) return -3;
    if (!strcmp(kernel, "bt_sweep_kernel")) { *ms = h->sweep_ms; return 0; }
    return set_err(h, -2, "no timer for kernel '%s'", kernel);
}

int64_t eigh_launch_count(eigh_handle_t h) { return h ? h->launches : -1; }

const char* eigh_last_error(eigh_handle_t h) { return h ? h->err : "null handle"; }

int eigh_destroy(eigh_handle_t h) {
    if (!h) return -1;
    if (h->events_ok)
    {
        for (int i = 0; i < 6; ++i) cudaEventDestroy(h->ev[i]);
        for (int i = 0; i < 2; ++i) cudaEventDestroy(h->ev_sweep[i]);
    }
    if (h->stage_ok) {
        for (int i = 0; i < 2; ++i) { cudaFreeHost(h->stage[i]); cudaEventDestroy(h->ev_stage[i]); }
        cudaStreamDestroy(h->copy_stream);
    }
    delete h;
    return 0;
}

// ------------------------------------------------------------------------- kernel-level entries
int eigh_k_zgemm(eigh_handle_t h, char opA, char opB, int64_t M, int64_t N, int64_t K, double alpha,
                 const void* A_dev, int64_t lda, const void* B_dev, int64_t ldb, int64_t K2, const void* A2_dev,
                 int64_t lda2, const void* B2_dev, int64_t ldb2, double beta, void* C_dev, int64_t ldc,
                 int lower_only, int splitk, void* stream) {
    int rc = ensure_ready(h);
    if (rc) return rc;
    const bool ta = (opA == 'C' || opA == 'c'), tb = (opB == 'C' || opB == 'c');
    if (!ta && opA != 'N' && opA != 'n') return -2;
    if (!tb && opB != 'N' && opB != 'n') return -3;
    if (ta && tb) return set_err(h, -3, "opA = opB = 'C' is not instantiated");
    if (M < 0 || N < 0 || K < 0) return -4;
    if (splitk < 1) return -20;
    ZgemmArgs a;
    memset(&a, 0, sizeof(a));
    a.M = (int)M; a.N = (int)N; a.K1 = (int)K; a.K2 = (int)K2;
    a.A1 = (const c128*)A_dev; a.B1 = (const c128*)B_dev; a.lda1 = lda; a.ldb1 = ldb;
    a.A2 = (const c128*)A2_dev; a.B2 = (const c128*)B2_dev; a.lda2 = lda2; a.ldb2 = ldb2;
    a.C = (c128*)C_dev; a.ldc = ldc; a.alpha = alpha; a.beta = beta;
    a.lower_only = lower_only & 1; a.splitk = splitk;
    a.partial = ws_ptr<c128>(h, h->plan.gemm_partial);
    if (splitk > 1 && (size_t)splitk * M * N * sizeof(c128) > h->plan.gemm_partial_bytes)
        return set_err(h, -20, "splitk partials exceed workspace");
    const bool small_tile = (M <= 64) || (lower_only & 2);
    g_zgemm_big_tiles = (lower_only & 4) != 0;
    rc = zgemm_launch(a, ta, tb, ZMODE_GEMM, small_tile, (cudaStream_t)stream, &h->launches);
    g_zgemm_big_tiles = false;
    return rc ? cuda_fail(h, 1000 + rc, "zgemm") : 0;
}

int eigh_k_zhemm_lower(eigh_handle_t h, int64_t M, int64_t N, const void* A_dev, int64_t lda, const void* B_dev,
                       int64_t ldb, void* C_dev, int64_t ldc, int splitk, void* stream) {
    int rc = ensure_ready(h);
    if (rc) return rc;
    if (M < 0 || N < 0) return -2;
    if (splitk < 1) return -10;
    ZgemmArgs a;
    memset(&a, 0, sizeof(a));
    a.M = (int)M; a.N = (int)N; a.K1 = (int)M;
    a.A1 = (const c128*)A_dev; a.B1 = (const c128*)B_dev; a.lda1 = lda; a.ldb1 = ldb;
    a.C = (c128*)C_dev; a.ldc = ldc; a.alpha = 1.0; a.beta = 0.0; a.splitk = splitk;
    a.partial = ws_ptr<c128>(h, h->plan.gemm_partial);
    if (splitk > 1 && (size_t)splitk * M * N * sizeof(c128) > h->plan.gemm_partial_bytes)
        return set_err(h, -10, "splitk partials exceed workspace");
    rc = zgemm_launch(a, false, false, ZMODE_HEMM, true, (cudaStream_t)stream, &h->launches);
    return rc ? cuda_fail(h, 1000 + rc, "zhemm") : 0;
}

int eigh_k_rgemm(eigh_handle_t h, char opA, char opB, int64_t M, int64_t N, int64_t K, double alpha, const double* A_dev,
                 int64_t lda, const double* B_dev, int64_t ldb, int64_t K2, const double* A2_dev, int64_t lda2,
                 const double* B2_dev, int64_t ldb2, double beta, double* C_dev, int64_t ldc, int lower_only, int splitk,
                 void* stream) {
    int rc = ensure_ready(h);
    if (rc) return rc;
    const bool ta = (opA == 'T' || opA == 't'), tb = (opB == 'T' || opB == 't');
    if (!ta && opA != 'N' && opA != 'n') return -2;
    if (!tb && opB != 'N' && opB != 'n') return -3;
    if (M < 0 || N < 0 || K < 0) return -4;
    if (splitk < 1) return -20;
    if (splitk > 1 && (size_t)splitk * M * N * sizeof(double) > h->plan.gemm_partial_bytes)
        return set_err(h, -20, "splitk partials exceed workspace");
    RgemmArgs a;
    memset(&a, 0, sizeof(a));
    a.M = (int)M; a.N = (int)N; a.K1 = (int)K; a.K2 = (int)K2;
    a.A1 = A_dev; a.B1 = B_dev; a.lda1 = lda; a.ldb1 = ldb;
    a.A2 = A2_dev; a.B2 = B2_dev; a.lda2 = lda2; a.ldb2 = ldb2;
    a.C = C_dev; a.ldc = ldc; a.alpha = alpha; a.beta = beta; a.lower_only = lower_only & 1; a.splitk = splitk;
    a.partial = ws_ptr<double>(h, h->plan.gemm_partial);
    rc = rgemm_launch(a, ta, tb, (cudaStream_t)stream, &h->launches);
    return rc ? cuda_fail(h, 1000 + rc, "rgemm") : 0;
}

int eigh_k_dgemm(eigh_handle_t h, int64_t M, int64_t N, int64_t K, const double* A_dev, int64_t lda,
                 const int32_t* a_col_idx_dev, const double* B_dev, int64_t ldb, double* C_dev, int64_t ldc,
                 void* stream) {
    int rc = ensure_ready(h);
    if (rc) return rc;
    if (M < 0 || N < 0 || K < 0) return -2;
    if ((lda & 1) || (ldb & 1) || ((uintptr_t)A_dev & 15) || ((uintptr_t)B_dev & 15))
        return set_err(h, -6, "dgemm needs 16-byte aligned A, B and even lda, ldb");
    DgemmArgs a;
    memset(&a, 0, sizeof(a));
    a.A = A_dev; a.lda = lda; a.B = B_dev; a.ldb = ldb; a.C = C_dev; a.ldc = ldc;
    a.a_col_idx = a_col_idx_dev; a.desc = nullptr;
    a.one.M = (int)M; a.one.N = (int)N; a.one.K = (int)K;
    rc = dgemm_launch_desc(a, 1, (int)M, (int)N, (cudaStream_t)stream, &h->launches);
    return rc ? cuda_fail(h, 1000 + rc, "dgemm") : 0;
}

}  // extern "C"

