"""Thin ctypes binding of the C ABI in include/eigh.h (argument marshalling only).

Every step of the path runs in the CUDA library; PyTorch is used for device memory and
streams.  There is no fallback: if libeigh_b200.so is missing or fails to load, every
entry point raises.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libeigh_b200.so")
_lib = None

_i64, _int, _dbl, _vp, _sz = ctypes.c_int64, ctypes.c_int, ctypes.c_double, ctypes.c_void_p, ctypes.c_size_t
_dp = ctypes.POINTER(ctypes.c_double)

# name -> (restype, argtypes); must list every function declared in include/eigh.h
SIGNATURES = {
    "eigh_create": (_int, [ctypes.POINTER(_vp), _i64, _i64]),
    "eigh_set_option": (_int, [_vp, ctypes.c_char_p, _i64]),
    "eigh_get_option": (_int, [_vp, ctypes.c_char_p, ctypes.POINTER(_i64)]),
    "eigh_workspace_size": (_sz, [_vp]),
    "eigh_set_workspace": (_int, [_vp, _vp, _sz]),
    "eigh_solve": (_int, [_vp, _vp, _i64, _vp, _vp, _vp]),
    "eigh_solve_host": (_int, [_vp, _vp, _i64, _vp, _vp, _vp, _vp, _vp, _vp]),
    "eigh_phase_times": (_int, [_vp, _dp]),
    "eigh_kernel_time": (_int, [_vp, ctypes.c_char_p, _dp]),
    "eigh_launch_count": (_i64, [_vp]),
    "eigh_dc_stats": (_int, [_vp, _int, ctypes.POINTER(_int), _dp, _dp]),
    "eigh_last_error": (ctypes.c_char_p, [_vp]),
    "eigh_destroy": (_int, [_vp]),
    "eigh_reduce_to_band": (_int, [_vp, _vp, _i64, _vp, _i64, _vp]),
    "eigh_band_to_tridiag": (_int, [_vp, _vp, _i64, _vp, _vp, _vp]),
    "eigh_tridiag_dc": (_int, [_vp, _vp, _vp, _vp, _vp, _i64, _vp]),
    "eigh_backtransform_band": (_int, [_vp, _vp, _i64, _vp, _i64, _vp]),
    "eigh_backtransform_full": (_int, [_vp, _vp, _i64, _vp, _i64, _vp]),
    "eigh_tridiagonalise_direct": (_int, [_vp, _vp, _i64, _vp, _vp, _vp]),
    "eigh_backtransform_direct": (_int, [_vp, _vp, _i64, _vp, _i64, _vp]),
    "eigh_densities": (_int, [_vp, _vp, _vp, _i64, _i64, _dbl, _dbl, _int, _vp, _vp, _vp]),
    "eigh_densities_static": (_int, [_vp, _vp, _vp, _i64, _i64, _dbl, _dbl, _int, _vp, _vp, _vp]),
    "eigh_gradient_densities": (_int, [_vp, _i64, _i64, _i64, _vp, _vp, _vp, _vp, _vp, _i64, _i64, _dbl, _dbl, _int,
                                       _vp, _vp, _vp]),
    "eigh_assemble_bdg": (_int, [_vp, _i64, _i64, _i64, _vp, _vp, _vp, _vp, _vp, _dbl, _dbl, _vp, _i64, _vp]),
    "eigh_tdslda_rhs": (_int, [_vp, _i64, _i64, _i64, _vp, _vp, _vp, _vp, _vp, _dbl, _vp, _i64, _i64, _vp, _i64, _vp]),
    "eigh_tdslda_step": (_int, [_vp, _i64, _i64, _i64, _vp, _vp, _vp, _vp, _dbl, _dbl, _vp, _dbl, _dbl, _int, _dbl, _vp,
                                _i64, ctypes.POINTER(_vp), _i64, _vp, _i64, _vp, _vp, _vp]),
    "eigh_k_zgemm": (_int, [_vp, ctypes.c_char, ctypes.c_char, _i64, _i64, _i64, _dbl, _vp, _i64, _vp, _i64,
                            _i64, _vp, _i64, _vp, _i64, _dbl, _vp, _i64, _int, _int, _vp]),
    "eigh_k_zhemm_lower": (_int, [_vp, _i64, _i64, _vp, _i64, _vp, _i64, _vp, _i64, _int, _vp]),
    "eigh_k_rgemm": (_int, [_vp, ctypes.c_char, ctypes.c_char, _i64, _i64, _i64, _dbl, _vp, _i64, _vp, _i64,
                            _i64, _vp, _i64, _vp, _i64, _dbl, _vp, _i64, _int, _int, _vp]),
    "eigh_k_dgemm": (_int, [_vp, _i64, _i64, _i64, _vp, _i64, _vp, _vp, _i64, _vp, _i64, _vp]),
}


def load():
    """Load the CUDA library; raises (loudly) if it is missing -- there is no fallback."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(
                f"{LIB_PATH} not found: build it with `python -c 'import __graft_entry__ as g; g.build()'` "
                "(b200-eigh has no CPU fallback)")
        lib = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            f = getattr(lib, name)
            f.restype = res
            f.argtypes = args
        _lib = lib
    return _lib


class EighError(RuntimeError):
    pass


def _ptr(t):
    return ctypes.c_void_p(t.data_ptr()) if t is not None else None


def _stream():
    import torch
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


class Eigh:
    """Handle + workspace for one problem size.  A is N x N complex128 with COLUMN-MAJOR
    storage: pass a torch tensor `At` of shape (N, N) holding A^T row-major (i.e. `At[j, i] =
    A[i, j]`), which is the same memory as A column-major."""

    def __init__(self, N: int, nev: Optional[int] = None, device="cuda", **options):
        import torch
        self.lib = load()
        self.N = int(N)
        self.nev = int(nev if nev is not None else N)
        self.device = torch.device(device)
        h = ctypes.c_void_p()
        rc = self.lib.eigh_create(ctypes.byref(h), self.N, self.nev)
        if rc != 0:
            raise EighError(f"eigh_create({N}, {nev}) -> {rc}")
        self.h = h
        for k, v in options.items():
            rc = self.lib.eigh_set_option(self.h, k.encode(), int(v))
            if rc != 0:
                raise EighError(f"eigh_set_option({k}, {v}) -> {rc}: {self.last_error()}")
        self.ws_bytes = int(self.lib.eigh_workspace_size(self.h))
        self.ws = torch.empty(self.ws_bytes + 256, dtype=torch.uint8, device=self.device)
        base = self.ws.data_ptr()
        self._ws_ptr = (base + 255) // 256 * 256
        rc = self.lib.eigh_set_workspace(self.h, ctypes.c_void_p(self._ws_ptr), self.ws_bytes)
        self._check(rc, "eigh_set_workspace")

    # ------------------------------------------------------------------ plumbing
    def last_error(self) -> str:
        return self.lib.eigh_last_error(self.h).decode()

    def _check(self, rc, what, allow_positive=False):
        if rc < 0 or rc >= 1000 or (rc > 0 and not allow_positive):
            raise EighError(f"{what} -> {rc}: {self.last_error()}")
        return rc

    def close(self):
        if getattr(self, "h", None):
            self.lib.eigh_destroy(self.h)
            self.h = None
            self.ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ------------------------------------------------------------------ full solve
    def solve(self, At, W=None, Zt=None):
        """eigh_solve.  At: (N, N) complex128 CUDA tensor = A^T row-major (A column-major); it
        is OVERWRITTEN.  Returns (W [N] float64, Zt [(nev, N)] complex128 with Zt[j] = eigenvector
        j, i.e. Z column-major).  Positive return codes (non-converged secular roots) raise."""
        import torch
        dt = self.dtype
        assert At.is_cuda and At.dtype == dt and At.is_contiguous() and At.shape == (self.N, self.N)
        if W is None:
            W = torch.empty(self.N, dtype=torch.float64, device=At.device)
        if Zt is None:
            Zt = torch.empty((self.nev, self.N), dtype=dt, device=At.device)
        rc = self.lib.eigh_solve(self.h, _ptr(At), self.N, _ptr(W), _ptr(Zt), _stream())
        self._check(rc, "eigh_solve")
        return W, Zt

    def solve_host(self, At_host, W_host, Zt_host, At_dev, W_dev, Zt_dev):
        """eigh_solve_host: host tensors in/out (pinned for speed), device scratch supplied by the
        caller.  At_host is not modified."""
        rc = self.lib.eigh_solve_host(self.h, _ptr(At_host), self.N, _ptr(W_host), _ptr(Zt_host),
                                      _ptr(At_dev), _ptr(W_dev), _ptr(Zt_dev), _stream())
        self._check(rc, "eigh_solve_host")
        return W_host, Zt_host

    # ------------------------------------------------------------------ SCF epilogue
    def densities(self, E, Zt, T: float = 0.0, Ec: float = float("inf"), branch: int = 1, n=None, nu=None):
        """eigh_densities (Eq. 16a, 16d, 17).  E: (ncols,) float64 energies of the rows of Zt; Zt: (ncols, N)
        complex128 = Z column-major (as `solve` returns it; a row stride >= N is allowed).
        Returns (n [N/2] float64, nu [N/2] complex128).  Enqueues only; no synchronisation."""
        import torch
        ncols = int(Zt.shape[0])
        assert Zt.is_cuda and Zt.dtype == torch.complex128 and Zt.shape[1] == self.N
        assert ncols == 0 or (Zt.stride(1) == 1 and (ncols == 1 or Zt.stride(0) >= self.N))
        assert E.is_cuda and E.dtype == torch.float64 and E.is_contiguous() and E.numel() >= ncols
        ldz = int(Zt.stride(0)) if ncols > 1 else self.N
        M = self.N // 2
        if n is None:
            n = torch.empty(M, dtype=torch.float64, device=Zt.device)
        if nu is None:
            nu = torch.empty(M, dtype=torch.complex128, device=Zt.device)
        rc = self.lib.eigh_densities(self.h, _ptr(E), _ptr(Zt), ldz, ncols, float(T), float(Ec), int(branch),
                                     _ptr(n), _ptr(nu), _stream())
        self._check(rc, "eigh_densities")
        return n, nu

    def densities_static(self, E, Zt, n, nu, T: float = 0.0, Ec: float = float("inf"), branch: int = 1):
        """eigh_densities_static: eigh_densities with its scratch in a static device array (no allocation, no workspace;
        N <= 65536, ncols <= 32760).  n [N/2] float64 and nu [N/2] complex128 are caller-provided outputs."""
        ncols = int(Zt.shape[0])
        ldz = int(Zt.stride(0)) if ncols > 1 else self.N
        rc = self.lib.eigh_densities_static(self.h, _ptr(E), _ptr(Zt), ldz, ncols, float(T), float(Ec), int(branch),
                                            _ptr(n), _ptr(nu), _stream())
        self._check(rc, "eigh_densities_static")
        return n, nu

    def gradient_densities(self, shape, Dx, Dy, Dz, E, Zt, T: float = 0.0, Ec: float = float("inf"), branch: int = 1):
        """eigh_gradient_densities (Eq. 16b, 16c).  Dx, Dy, Dz: (L, L) float64 CUDA tensors holding D^T row-major, i.e.
        D column-major (pass `D.t().contiguous()` of the logical matrix).  E, Zt as for `densities`.
        Returns (tau [M] float64, j [3, M] float64)."""
        import torch
        nx, ny, nz = (int(v) for v in shape)
        ncols = int(Zt.shape[0])
        for D, L in ((Dx, nx), (Dy, ny), (Dz, nz)):
            assert D.is_cuda and D.dtype == torch.float64 and D.shape == (L, L) and D.is_contiguous()
        assert Zt.is_cuda and Zt.dtype == torch.complex128 and Zt.shape[1] == self.N
        assert ncols == 0 or (Zt.stride(1) == 1 and (ncols == 1 or Zt.stride(0) >= self.N))
        assert E.is_cuda and E.dtype == torch.float64 and E.is_contiguous() and E.numel() >= ncols
        ldz = int(Zt.stride(0)) if ncols > 1 else self.N
        M = self.N // 2
        tau = torch.empty(M, dtype=torch.float64, device=Zt.device)
        j = torch.empty((3, M), dtype=torch.float64, device=Zt.device)
        rc = self.lib.eigh_gradient_densities(self.h, nx, ny, nz, _ptr(Dx), _ptr(Dy), _ptr(Dz), _ptr(E), _ptr(Zt), ldz,
                                              ncols, float(T), float(Ec), int(branch), _ptr(tau), _ptr(j), _stream())
        self._check(rc, "eigh_gradient_densities")
        return tau, j

    def assemble_bdg(self, shape, Kx, Ky, Kz, V, Delta, mu: float, At=None, sign: float = 1.0):
        """eigh_assemble_bdg (Eq. 5/7/8).  Kx, Ky, Kz: (L, L) float64 symmetric 1-D kinetic matrices; V: (M,) float64;
        Delta: (M,) complex128; all CUDA tensors.  Returns At, (N, N) complex128 = H column-major (ready for solve)."""
        import torch
        nx, ny, nz = (int(v) for v in shape)
        for K, L in ((Kx, nx), (Ky, ny), (Kz, nz)):
            assert K.is_cuda and K.dtype == torch.float64 and K.shape == (L, L) and K.is_contiguous()
        M = nx * ny * nz
        assert V.is_cuda and V.dtype == torch.float64 and V.numel() == M and V.is_contiguous()
        assert Delta.is_cuda and Delta.dtype == torch.complex128 and Delta.numel() == M and Delta.is_contiguous()
        if At is None:
            At = torch.empty((self.N, self.N), dtype=torch.complex128, device=V.device)
        assert At.is_cuda and At.dtype == torch.complex128 and At.shape == (self.N, self.N) and At.is_contiguous()
        # symmetric K: row-major storage equals column-major storage
        rc = self.lib.eigh_assemble_bdg(self.h, nx, ny, nz, _ptr(Kx), _ptr(Ky), _ptr(Kz), _ptr(V), _ptr(Delta),
                                        float(mu), float(sign), _ptr(At), self.N, _stream())
        self._check(rc, "eigh_assemble_bdg")
        return At

    # ------------------------------------------------------------------ second workload: TDSLDA step
    def tdslda_rhs(self, shape, Kx, Ky, Kz, V, Delta, mu, Phit, Ft=None):
        """eigh_tdslda_rhs: Ft <- -i H Phi.  Phit, Ft: (ncols, N) complex128 (states = rows, i.e. column-major N x ncols)."""
        import torch
        nx, ny, nz = (int(v) for v in shape)
        if Ft is None:
            Ft = torch.empty_like(Phit)
        rc = self.lib.eigh_tdslda_rhs(self.h, nx, ny, nz, _ptr(Kx), _ptr(Ky), _ptr(Kz), _ptr(V), _ptr(Delta), float(mu),
                                      _ptr(Phit), int(Phit.stride(0)) if Phit.shape[0] > 1 else self.N, int(Phit.shape[0]),
                                      _ptr(Ft), int(Ft.stride(0)) if Ft.shape[0] > 1 else self.N, _stream())
        self._check(rc, "eigh_tdslda_rhs")
        return Ft

    def tdslda_step(self, shape, Kx, Ky, Kz, V, g, mu, E0, dt, Yt, Flist, Ypt, n, Delta, T=0.0, Ec=float("inf"), branch=1):
        """eigh_tdslda_step.  Yt, Ypt and the five tensors of Flist ([f_n, ..., f_{n-4}]): (ncols, N) complex128 contiguous.
        Returns the rotated list [f_{n+1}, f_n, ..., f_{n-3}] (same tensors, no copy)."""
        nx, ny, nz = (int(v) for v in shape)
        ncols = int(Yt.shape[0])
        for t in [Yt, Ypt] + list(Flist):
            assert t.is_cuda and t.is_contiguous() and t.shape == (ncols, self.N)
        arr = (_vp * 5)(*[t.data_ptr() for t in Flist])
        rc = self.lib.eigh_tdslda_step(self.h, nx, ny, nz, _ptr(Kx), _ptr(Ky), _ptr(Kz), _ptr(V), float(g), float(mu), _ptr(E0),
                                       float(T), float(Ec), int(branch), float(dt), _ptr(Yt), self.N, arr, self.N, _ptr(Ypt),
                                       ncols, _ptr(n), _ptr(Delta), _stream())
        self._check(rc, "eigh_tdslda_step")
        return [Flist[4]] + list(Flist[:4])

    def phase_times_ms(self):
        ms = (ctypes.c_double * 5)()
        self.lib.eigh_phase_times(self.h, ms)
        return list(ms)

    def kernel_time_ms(self, kernel: str) -> float:
        ms = ctypes.c_double()
        rc = self.lib.eigh_kernel_time(self.h, kernel.encode(), ctypes.byref(ms))
        self._check(rc, "eigh_kernel_time")
        return float(ms.value)

    def launch_count(self) -> int:
        return int(self.lib.eigh_launch_count(self.h))

    # ------------------------------------------------------------------ phases
    @property
    def dtype(self):
        """torch dtype of A and Z: complex128, or float64 with the option dtype = 1 (real symmetric, method = 1)."""
        import torch
        return torch.float64 if self.get_option("dtype") == 1 else torch.complex128

    def tridiagonalise_direct(self, At, d, e):
        """eigh_tridiagonalise_direct (1-stage, needs method = 1).  At: (N, N) storage of A column-major, overwritten."""
        rc = self.lib.eigh_tridiagonalise_direct(self.h, _ptr(At), self.N, _ptr(d), _ptr(e), _stream())
        self._check(rc, "eigh_tridiagonalise_direct")

    def backtransform_direct(self, At, Zt):
        rc = self.lib.eigh_backtransform_direct(self.h, _ptr(At), self.N, _ptr(Zt), Zt.shape[1], _stream())
        self._check(rc, "eigh_backtransform_direct")

    def rgemm(self, opA, opB, M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, K2=0, A2=None, lda2=0, B2=None, ldb2=0,
              lower_only=0, splitk=1):
        rc = self.lib.eigh_k_rgemm(self.h, opA.encode(), opB.encode(), M, N, K, alpha, _ptr(A), lda, _ptr(B), ldb, K2,
                                   _ptr(A2), lda2, _ptr(B2), ldb2, beta, _ptr(C), ldc, lower_only, splitk, _stream())
        self._check(rc, "eigh_k_rgemm")

    def get_option(self, key: str) -> int:
        v = _i64()
        rc = self.lib.eigh_get_option(self.h, key.encode(), ctypes.byref(v))
        self._check(rc, f"eigh_get_option({key})")
        return int(v.value)

    def dc_stats(self):
        """Per merge level of the last S3 run: (executed GEMM flops, kept fraction k/n) -- eigh_dc_stats."""
        n = _int()
        fl = (ctypes.c_double * 32)()
        kf = (ctypes.c_double * 32)()
        rc = self.lib.eigh_dc_stats(self.h, 32, ctypes.byref(n), fl, kf)
        self._check(rc, "eigh_dc_stats")
        return [float(fl[i]) for i in range(min(n.value, 32))], [float(kf[i]) for i in range(min(n.value, 32))]

    @property
    def ldab(self) -> int:
        return 2 * self.band_width + 2

    @property
    def band_width(self) -> int:
        return self.get_option("band_width")

    def reduce_to_band(self, At, band):
        rc = self.lib.eigh_reduce_to_band(self.h, _ptr(At), self.N, _ptr(band), band.shape[1], _stream())
        self._check(rc, "eigh_reduce_to_band")

    def band_to_tridiag(self, band, d, e):
        rc = self.lib.eigh_band_to_tridiag(self.h, _ptr(band), band.shape[1], _ptr(d), _ptr(e), _stream())
        self._check(rc, "eigh_band_to_tridiag")

    def tridiag_dc(self, d, e, W, Qt):
        """Qt: (nev, ldq) float64 row-major = Q column-major with ldq = Qt.shape[1]."""
        rc = self.lib.eigh_tridiag_dc(self.h, _ptr(d), _ptr(e), _ptr(W), _ptr(Qt), Qt.shape[1], _stream())
        return self._check(rc, "eigh_tridiag_dc", allow_positive=True)

    def backtransform_band(self, Qt, Zt):
        rc = self.lib.eigh_backtransform_band(self.h, _ptr(Qt), Qt.shape[1], _ptr(Zt), Zt.shape[1], _stream())
        self._check(rc, "eigh_backtransform_band")

    def backtransform_full(self, At, Zt):
        rc = self.lib.eigh_backtransform_full(self.h, _ptr(At), self.N, _ptr(Zt), Zt.shape[1], _stream())
        self._check(rc, "eigh_backtransform_full")

    # ------------------------------------------------------------------ kernels
    def zgemm(self, opA, opB, M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, K2=0, A2=None, lda2=0,
              B2=None, ldb2=0, lower_only=0, splitk=1):
        rc = self.lib.eigh_k_zgemm(self.h, opA.encode(), opB.encode(), M, N, K, alpha, _ptr(A), lda, _ptr(B),
                                   ldb, K2, _ptr(A2), lda2, _ptr(B2), ldb2, beta, _ptr(C), ldc, lower_only,
                                   splitk, _stream())
        self._check(rc, "eigh_k_zgemm")

    def zhemm_lower(self, M, N, A, lda, B, ldb, C, ldc, splitk=1):
        rc = self.lib.eigh_k_zhemm_lower(self.h, M, N, _ptr(A), lda, _ptr(B), ldb, _ptr(C), ldc, splitk, _stream())
        self._check(rc, "eigh_k_zhemm_lower")

    def dgemm(self, M, N, K, A, lda, B, ldb, C, ldc, col_idx=None):
        rc = self.lib.eigh_k_dgemm(self.h, M, N, K, _ptr(A), lda, _ptr(col_idx), _ptr(B), ldb, _ptr(C), ldc,
                                   _stream())
        self._check(rc, "eigh_k_dgemm")
