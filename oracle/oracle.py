"""ctypes front end of the C oracle (oracle_eigh.c).  TEST INFRASTRUCTURE ONLY.

Every function marshals numpy arrays into the C entry points and back; all of the
arithmetic is in oracle_eigh_impl.inc (steps O1..O5, PAPER.md:148 / SURVEY.md 8(c)).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle_eigh.so")
_SRC = [os.path.join(_HERE, "oracle_eigh.c"), os.path.join(_HERE, "oracle_eigh_impl.inc")]
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (building the checker is not using it)."""
    stale = (not os.path.exists(_SO)) or any(
        os.path.getmtime(s) > os.path.getmtime(_SO) for s in _SRC)
    if force or stale:
        cmd = ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-std=gnu11",
               _SRC[0], "-o", _SO, "-lm"]
        subprocess.check_call(cmd, cwd=_HERE)
    return _SO


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_SO)
        dp = ctypes.POINTER(ctypes.c_double)
        for sfx in ("_d", "_ld"):
            f = getattr(lib, "oracle_eigh" + sfx)
            f.argtypes = [ctypes.c_int64, dp, dp, dp]
            f.restype = ctypes.c_int
            f = getattr(lib, "oracle_tridiag_ql" + sfx)
            f.argtypes = [ctypes.c_int64, dp, dp, dp, dp]
            f.restype = ctypes.c_int
            f = getattr(lib, "oracle_tridiagonalise" + sfx)
            f.argtypes = [ctypes.c_int64, dp, dp, dp, dp]
            f.restype = ctypes.c_int
        lib.oracle_num_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double)) if a is not None else None


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def _eigh(H, vectors, sfx):
    H = np.asarray(H)
    n = H.shape[0]
    assert H.shape == (n, n)
    Hf = np.asfortranarray(H, dtype=np.complex128)
    W = np.empty(n, dtype=np.float64)
    Z = np.empty((n, n), dtype=np.complex128, order="F") if vectors else None
    info = getattr(_load(), "oracle_eigh" + sfx)(
        n, _dp(Hf), _dp(W), _dp(Z))
    if info != 0:
        raise RuntimeError(f"oracle_eigh{sfx} failed, info={info}")
    return (W, Z) if vectors else W


def eigh(H, vectors: bool = True):
    """FP64 oracle: (W ascending, Z columns = eigenvectors) of Hermitian H (lower triangle read)."""
    return _eigh(H, vectors, "_d")


def eigh_ld(H, vectors: bool = True):
    """Same steps evaluated in x87 long double; results rounded to FP64 on return."""
    return _eigh(H, vectors, "_ld")


def tridiagonalise(H, sfx: str = "_d"):
    """O1-O3 only: returns (d, e, Q) with H = Q tridiag(d,e) Q^H, e >= 0 real."""
    H = np.asarray(H)
    n = H.shape[0]
    Hf = np.asfortranarray(H, dtype=np.complex128)
    d = np.empty(n)
    e = np.empty(max(n - 1, 0))
    Q = np.empty((n, n), dtype=np.complex128, order="F")
    info = getattr(_load(), "oracle_tridiagonalise" + sfx)(
        n, _dp(Hf), _dp(d), _dp(e), _dp(Q))
    if info != 0:
        raise RuntimeError(f"oracle_tridiagonalise failed, info={info}")
    return d, e, Q


def _tql(d, e, vectors, sfx):
    d = np.ascontiguousarray(d, dtype=np.float64)
    e = np.ascontiguousarray(e, dtype=np.float64)
    n = d.shape[0]
    assert e.shape[0] == max(n - 1, 0)
    W = np.empty(n)
    Q = np.empty((n, n), order="F") if vectors else None
    ep = e if n > 1 else np.zeros(1)
    info = getattr(_load(), "oracle_tridiag_ql" + sfx)(n, _dp(d), _dp(ep), _dp(W), _dp(Q))
    if info != 0:
        raise RuntimeError(f"oracle_tridiag_ql{sfx} failed, info={info}")
    return (W, Q) if vectors else W


def tridiag_ql(d, e, vectors: bool = True):
    """O4+O5 on a real symmetric tridiagonal (FP64)."""
    return _tql(d, e, vectors, "_d")


def tridiag_ql_ld(d, e, vectors: bool = True):
    return _tql(d, e, vectors, "_ld")


def sturm_count(d, e, sigma):
    """Number of eigenvalues of the real symmetric tridiagonal T = tridiag(d, e) that are < sigma
    (Sylvester's law of inertia on the LDL^T pivots of T - sigma I; Golub & Van Loan 8.4.1 /
    SURVEY.md 8(c) "Sturm-count spot checks").  Plain recurrence
        q_0 = d_0 - sigma,   q_i = (d_i - sigma) - e_{i-1}^2 / q_{i-1},
    count = #{i : q_i < 0}; a zero pivot is replaced by a tiny negative number.  `sigma` may be an
    array: the recurrence is vectorised over the shifts only (O(N) steps, each elementwise).
    TEST INFRASTRUCTURE ONLY; shares nothing with the CUDA path."""
    d = np.asarray(d, dtype=np.float64)
    e = np.asarray(e, dtype=np.float64)
    sig = np.atleast_1d(np.asarray(sigma, dtype=np.float64))
    n = d.shape[0]
    scale = max(np.abs(d).max(initial=0.0), np.abs(e).max(initial=0.0), 1e-300)
    tiny = scale * np.finfo(np.float64).tiny ** 0.5
    q = d[0] - sig
    q = np.where(q == 0.0, -tiny, q)
    cnt = (q < 0).astype(np.int64)
    for i in range(1, n):
        q = (d[i] - sig) - (e[i - 1] * e[i - 1]) / q
        q = np.where(q == 0.0, -tiny, q)
        cnt += q < 0
    return cnt if np.ndim(sigma) else int(cnt[0])
