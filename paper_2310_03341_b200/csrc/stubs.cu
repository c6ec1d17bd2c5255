// stubs.cu -- phases not implemented yet fail loudly (removed as the phases land).
#include "eigh_internal.h"
namespace eigh {
size_t dc_arena_bytes(int64_t N) { return 3 * (size_t)round_up(N, 8) * N * sizeof(double) + (size_t)64 * N * 8 + (1 << 20); }
size_t bt_scratch_bytes(const eigh_handle_s* h) { return (size_t)256 << 20; }
int phase_band_to_tridiag(eigh_handle_s* h, c128*, int64_t, double*, double*, cudaStream_t) { return set_err(h, -100, "band_to_tridiag not implemented"); }
int phase_tridiag_dc(eigh_handle_s* h, const double*, const double*, double*, double*, int64_t, cudaStream_t, int*) { return set_err(h, -100, "tridiag_dc not implemented"); }
int phase_backtransform_band(eigh_handle_s* h, const double*, int64_t, c128*, int64_t, cudaStream_t) { return set_err(h, -100, "backtransform_band not implemented"); }
int phase_backtransform_full(eigh_handle_s* h, const c128*, int64_t, c128*, int64_t, cudaStream_t) { return set_err(h, -100, "backtransform_full not implemented"); }
}
